// Register-window kernel: placeholder until the kernel lands (the generic kernel runs instead).
#include "dd_internal.h"

struct dd_window_plan {};

namespace dd {
int build_window_plan(dd_plan* p) { p->window = nullptr; return DD_OK; }
void destroy_window_plan(dd_plan* p) { delete p->window; p->window = nullptr; }
bool window_plan_usable(const dd_plan* p) { return p->window != nullptr; }
bool window_args_ok(const dd_plan*, const void*, int64_t, int64_t, int64_t, int64_t) { return false; }
int launch_window(const dd_plan*, const ExecArgs&) { return fail(DD_ERR_UNSUPPORTED, "window kernel not built"); }
}  // namespace dd
