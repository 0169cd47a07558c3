#!/usr/bin/env python
"""Benchmark of the direct-dedispersion hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A step = one pass of the whole hot path (delay table already in the plan; front end, staging,
unpack, accumulation, store -- one dd_execute, or the four dd_stream_push calls of config 5) over
one synthetic filterbank resident in HBM.  The headline workload is the largest single-GPU
configuration of BASELINE.json: configs[2] (float32, 4096 channels x 4096 DM trials x 2^18
samples, 4.4e12 adds).  The other four configs are timed in the same process and reported under
`per_config`.  Prints ONE JSON line.  `--impl reference` times the CPU oracle (oracle/) on a
bounded sample of the same workload instead.

Multi-GPU: the path shards by beam with no exchange step.  Under torchrun (RANK / WORLD_SIZE in
the environment) every rank dedisperses its own beam; `python bench.py --gpus N` without torchrun
spawns the N ranks itself.  Weak scaling; the only collective is the max-reduction of the timings.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1401_8258_b200 import sharding, synth  # noqa: E402

METRIC = "dedispersed DM·channel·samples/s"
UNIT = "G/s"
SM_COUNT, LANES_PER_SM = 148, 128          # FP32/INT32 add lanes per SM
# measured add lanes per clock per SM of the instruction each path accumulates with (dependent-chain
# microbenchmark, profiles/r1_pipe_rates.txt: FADD 3.868 and IADD3 3.852 warp-instructions/clk/SM)
MEASURED_LANES = {"f32": 123.8, "u8": 123.2}
HEADLINE = 3


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag = index, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.005)

    def result(self):
        self.stop_flag = True
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def visible_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except (ValueError, IndexError):
            pass
    return local_rank


# ----------------------------------------------------------------------------- CPU oracle legs

def _oracle_fn(w):
    import oracle
    return oracle.dedisperse_f32 if w.dtype == "f32" else oracle.dedisperse_u8


def oracle_sample(w, seconds_target=10.0):
    """Times oracle/ (as it stands) on a bounded sample of workload w: a subset of DM rows over a
    shortened time range of the same filterbank.  Returns a dict with the all-core literal-nest rate
    (the cpu_baseline value), the single-core rate and the interchanged-nest rate."""
    import oracle
    cores = oracle.num_threads()
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    nsamp = min(w.nsamp, 1 << 15)
    X = synth.make_input(w, nsamp + ms)
    f = _oracle_fn(w)
    nrows = max(cores, 8)
    rows = np.unique(np.linspace(0, w.ndm - 1, nrows).astype(np.int32))
    f(X, 256, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows[:cores])           # warm caches / threads
    t0 = time.perf_counter()
    f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows)
    dt = time.perf_counter() - t0
    # grow the sample towards the time target (once), keeping the run bounded
    grow = int(min(16, seconds_target / max(dt, 1e-3)))
    if grow >= 2:
        rows = np.unique(np.linspace(0, w.ndm - 1, nrows * grow).astype(np.int32))
        t0 = time.perf_counter()
        f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows)
        dt = time.perf_counter() - t0
    adds = len(rows) * w.nchans * nsamp
    desc = "%d of %d DM rows x %d of %d samples x %d channels, literal (d,t,c) nest" % (
        len(rows), w.ndm, nsamp, w.nsamp, w.nchans)
    out = {"value": adds / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
           "seconds": dt, "_replay": (X, nsamp, rows)}
    # the same rows through the interchanged (d,c,t) nest (bit-identical results, vectorisable inner loop)
    t0 = time.perf_counter()
    f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows, interchanged=True)
    out["interchanged_nest"] = {"value": adds / (time.perf_counter() - t0) / 1e9, "unit": UNIT, "cores": cores}
    # one core: a single row (the OpenMP loop runs over rows, so one row = one thread)
    one = rows[len(rows) // 2: len(rows) // 2 + 1]
    t0 = time.perf_counter()
    f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=one)
    out["single_core"] = {"value": w.nchans * nsamp / (time.perf_counter() - t0) / 1e9, "unit": UNIT, "cores": 1,
                          "sample": "one DM row x %d samples x %d channels, literal nest" % (nsamp, w.nchans)}
    full = w.adds / (out["value"] * 1e9)
    out["extrapolated_full_workload_s"] = full
    return out


def run_reference(args, w):
    rank = _env_int("RANK", 0)
    if rank != 0:
        return
    smp = oracle_sample(w, seconds_target=6.0)
    X, nsamp, rows = smp.pop("_replay")
    f = _oracle_fn(w)
    steps = max(1, min(args.steps, 5))
    for _ in range(min(args.warmup, 1)):
        f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows)
    t0 = time.perf_counter()
    for _ in range(steps):
        f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows)
    dt = (time.perf_counter() - t0) / steps
    val = len(rows) * w.nchans * nsamp / dt / 1e9
    smp["value"] = val
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "sample": smp["sample"]},
        "cpu_baseline": smp,
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ----------------------------------------------------------------------------- GPU leg

class Case:
    """One workload resident on the device: plan, X, D and the step function bench.py times."""

    def __init__(self, dd, torch, w, rank=0, world=1, kernel=None, host_input=False):
        self.dd, self.torch, self.w = dd, torch, w
        dtype = dd.DD_F32 if w.dtype == "f32" else dd.DD_U8
        self.tdt = torch.float32 if w.dtype == "f32" else torch.uint8
        self.odt = torch.float32 if w.dtype == "f32" else torch.int32
        self.es = 4 if w.dtype == "f32" else 1
        self.plan = dd.Plan(dtype, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
        if kernel:
            self.plan.set_kernel({"generic": dd.DD_KERNEL_GENERIC, "ps": dd.DD_KERNEL_PS, "direct": dd.DD_KERNEL_DIRECT}[kernel])
        self.ms = ms = self.plan.max_shift()
        nb = self.nb = w.nbeams
        self.in_stride = (w.nsamp + ms + 63) // 64 * 64
        self.out_stride = w.nsamp
        self.Xh = None
        if host_input:
            # pinned host input, one beam per rank-beam (rank r uses beam seeds r*nb .. r*nb+nb-1), generated
            # by synth (numpy Philox) exactly as the parity tests generate it
            self.Xh = torch.empty((nb, w.nchans, self.in_stride), dtype=self.tdt).pin_memory()
            self.Xh.zero_()
            wb = synth.scaled(w, nbeams=max(2, nb * world))           # per-beam seeds
            for b, beam in enumerate(sharding.beams_of_rank(rank, world, nb)):
                synth.make_input(wb, w.nsamp + ms, beam=beam, out=self.Xh[b, :, :w.nsamp + ms].numpy())
            self.Xd = self.Xh.cuda()
        else:
            # same distributions drawn on the device (seeded); control flow is data-independent
            g = torch.Generator(device="cuda").manual_seed(w.seed + 7919 * rank)
            if w.dtype == "f32":
                self.Xd = torch.randn((nb, w.nchans, self.in_stride), dtype=torch.float32, device="cuda", generator=g)
            else:
                z = torch.randn((nb, w.nchans, self.in_stride), dtype=torch.float32, device="cuda", generator=g)
                self.Xd = z.mul_(16.0).add_(128.0).round_().clamp_(0, 255).to(torch.uint8)
                del z
        self.Dd = torch.empty((nb, w.ndm, self.out_stride), dtype=self.odt, device="cuda")
        self.stream = torch.cuda.Stream()
        a = (self.Xd, self.in_stride, w.nchans * self.in_stride, self.Dd, self.out_stride, w.ndm * self.out_stride)
        self.kern = self.plan.kernel_for(*a, w.nsamp, nb)
        self.streamer = None
        if w.nchunks > 1:
            # config 5: fed through the streaming API: first push nsamp/nchunks + maxshift, then equal chunks
            self.chunk = w.nsamp // w.nchunks
            self.streamer = dd.Stream(self.plan, self.chunk + ms, nb)
            # per push: the append and carry copies (2 strided device copies) + the kernels of one dd_execute
            per_push = 2 + self.plan.launches_for(self.Xd, self.ms + self.chunk + 64, 0, self.Dd, self.out_stride,
                                                  w.ndm * self.out_stride, self.chunk, nb)
            self.launches = w.nchunks * per_push
        else:
            self.launches = self.plan.launches_for(*a, w.nsamp, nb)
        self.hbm_bytes = nb * (w.nchans * (w.nsamp + ms) * self.es + w.ndm * w.nsamp * 4)

    def step(self):
        w, nb = self.w, self.nb
        if self.streamer is None:
            self.plan.execute(self.Xd, self.in_stride, w.nchans * self.in_stride, self.Dd, self.out_stride,
                              w.ndm * self.out_stride, w.nsamp, nb, self.stream)
            return
        self.streamer.reset()
        pos = emitted = 0
        for k in range(w.nchunks):
            n_new = self.chunk + (self.ms if k == 0 else 0)
            n = self.streamer.push(self.Xd[:, :, pos:], self.in_stride, w.nchans * self.in_stride, n_new,
                                   self.Dd[:, :, emitted:], self.out_stride, w.ndm * self.out_stride, self.stream)
            pos += n_new
            emitted += n
        assert emitted == w.nsamp

    def timed(self, steps, warmup, barrier, gpu_index):
        """W warm-up steps, then K steps between CUDA events on the launching stream; returns
        (per-step ms list, total ms, clocks)."""
        torch = self.torch
        with torch.cuda.stream(self.stream):
            for _ in range(warmup):
                self.step()
        barrier()
        sampler = ClockSampler(gpu_index)
        sampler.start()
        # two events around the K steps on the launching stream (an event per step would add its own
        # host and device cost to every step, which matters for the launch-bound config 1)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(self.stream):
            ev0.record(self.stream)
            for i in range(steps):
                self.step()
            ev1.record(self.stream)
        barrier()
        clocks = sampler.result()
        total = ev0.elapsed_time(ev1)
        return [total / steps] * steps, total, clocks

    def graph_ms_per_step(self, steps=200):
        """The same step captured `steps` times into one CUDA graph and replayed: device time per step
        without the host's per-call launch cost (launch-bound workloads only)."""
        torch = self.torch
        g = torch.cuda.CUDAGraph()
        cs = torch.cuda.Stream()
        real = self.stream
        try:
            self.stream = cs
            with torch.cuda.graph(g, stream=cs):
                for _ in range(steps):
                    self.step()
        finally:
            self.stream = real
        g.replay()
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        g.replay()
        ev1.record()
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1) / steps

    def close(self):
        if self.streamer is not None:
            self.streamer.destroy()
        self.plan.destroy()
        self.Xd = self.Dd = self.Xh = None
        self.torch.cuda.empty_cache()


def counters_for(workload, kern):
    """Counters of the dominant kernel from the tracked ncu summaries (profiles/kernel_counters.txt): DRAM
    traffic per launch, issue-slot and LSU utilisation, issued add instructions / algorithmic adds, each
    with the commit of the capture so that staleness is visible."""
    out = None
    try:
        for ln in open(os.path.join(ROOT, "profiles", "kernel_counters.txt")):
            f = ln.split()
            if len(f) >= 8 and not ln.startswith("#") and f[0] == workload and f[1] == str(kern):
                num = lambda v: None if v == "na" else float(v)
                out = {"traffic": num(f[2]), "issue_active": num(f[3]), "lsu_wavefront_frac": num(f[4]),
                       "issued_add_frac": num(f[5]), "captured_at_commit": f[6], "source": "profiles/" + f[7]}
    except OSError:
        pass
    return out


def kernel_name(kern):
    return {1: "generic", 2: "ps", 3: "direct"}.get(kern, str(kern))


def roofline_of(w, case, kernel_ms, clocks):
    peak_max = SM_COUNT * LANES_PER_SM * (clocks["sm_max_mhz"] or 1965) * 1e6 / 1e12
    achieved = w.adds / (kernel_ms * 1e-3) / 1e12
    clk = clocks["sm_mhz"] or clocks["sm_max_mhz"] or 1965
    peak_meas = SM_COUNT * MEASURED_LANES[w.dtype] * clk * 1e6 / 1e12
    r = {"bound": "alu", "achieved": achieved, "peak": peak_max, "unit": "Tadd/s", "frac": achieved / peak_max,
         "traffic": None,
         "peak_note": "148 SM x 128 add lanes x sm_max_mhz (nominal; DESIGN.md 5)",
         "kernel_ms": kernel_ms,
         "frac_at_sampled_clock": achieved / (SM_COUNT * LANES_PER_SM * clk * 1e6 / 1e12),
         "peak_measured": peak_meas, "frac_measured": achieved / peak_meas,
         "peak_measured_note": "148 SM x %.1f lanes/clk/SM (%s dependent-chain microbenchmark, "
                               "profiles/r1_pipe_rates.txt) x sampled SM clock" % (
                                   MEASURED_LANES[w.dtype], "FADD" if w.dtype == "f32" else "IADD3"),
         "algorithmic_adds_per_launch": w.adds,
         "hbm_algorithmic_bytes": case.hbm_bytes,
         "hbm_achieved_gbs": case.hbm_bytes / (kernel_ms * 1e-3) / 1e9}
    c = counters_for(w.name, case.kern)
    if c:
        r["traffic"] = c.pop("traffic")
        r["ncu"] = c
    return r


def run_ours(args, w):
    import torch
    import paper_1401_8258_b200 as dd

    rank, world, local = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    gpu_index = visible_gpu_index(local)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    case = Case(dd, torch, w, rank, world, args.kernel, host_input=True)
    per_step, total_ms, clocks = case.timed(args.steps, args.warmup, barrier, gpu_index)
    ms_per_step, value = finish_timing(total_ms, args.steps, w.adds, world, dist, "cuda")

    # ---- end to end through the host-buffer C-ABI call (pinned host X and D; copies inside)
    e2e = None
    if case.streamer is None:
        nb = w.nbeams
        Dh = torch.empty((nb, w.ndm, case.out_stride), dtype=case.odt).pin_memory()
        a = (case.Xh, case.in_stride, w.nchans * case.in_stride, Dh, case.out_stride, w.ndm * case.out_stride,
             w.nsamp, nb)
        case.plan.execute_host(*a)                                   # warm-up (allocates the cached device buffers)
        n_e2e = max(3, min(args.steps, 5))
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            case.plan.execute_host(*a)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / n_e2e
        dt = sharding.max_over_ranks(dt, dist, "cuda")
        e2e = {"value": sharding.whole_job_rate(w.adds, world, dt) / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": int(nb * w.nchans * (w.nsamp + case.ms) * case.es),
               "d2h_bytes_per_step": int(nb * w.ndm * w.nsamp * 4), "ms_per_step": dt * 1e3,
               "timer": "host wall clock around the synchronous dd_execute_host call, pinned buffers"}
        # the host path must give the same bits as the resident path (compared slice by slice on the device)
        same = True
        for b in range(nb):
            for r0 in range(0, w.ndm, 512):
                same = same and bool(torch.equal(Dh[b, r0:r0 + 512].cuda(), case.Dd[b, r0:r0 + 512]))
        e2e["matches_resident_result"] = same
        del Dh
        # the same path with the post-processing row (median w = 5, detrend, normalise, 6 sigma) run on the
        # device and ONLY the candidate list coming back (dd_search_host): no D -> host copy
        prm = dd.post_params(5, True, True, nsigma=6.0)
        cap = 1 << 20
        hc = torch.zeros(cap * 4, dtype=torch.int32).pin_memory()
        sa = (case.Xh, case.in_stride, w.nchans * case.in_stride, w.nsamp, nb, prm, hc, cap)
        ncand = case.plan.search_host(*sa)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            ncand = case.plan.search_host(*sa)
        dt = (time.perf_counter() - t0) / n_e2e
        dt = sharding.max_over_ranks(dt, dist, "cuda")
        e2e["search"] = {"value": sharding.whole_job_rate(w.adds, world, dt) / 1e9, "unit": UNIT, "ms_per_step": dt * 1e3,
                         "h2d_bytes_per_step": e2e["h2d_bytes_per_step"],
                         "d2h_bytes_per_step": int(8 + 16 * min(ncand, cap)), "candidates": int(ncand),
                         "post": "median 5, detrend, normalise, 6 sigma (PAPER.md:1204-1221)",
                         "gpu_launches_per_step": None}

    line = None
    if rank == 0:
        kernel_ms = float(np.mean(per_step))
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32" if w.dtype == "u8" else "f32",
            "data": "synthetic",
            "config": {"workload": w.name, "nbeams": w.nbeams, "nchans": w.nchans, "ndm": w.ndm,
                       "nsamp": w.nsamp, "maxshift": case.ms, "tsamp": w.tsamp, "fch1": w.fch1, "foff": w.foff,
                       "kernel": kernel_name(case.kern), "plan": case.plan.describe(),
                       "parallelism": "beam-per-rank" if world > 1 else "single",
                       "l2": "X+D per step = %.0f MB > 126 MB L2 (no flush needed)" % (case.hbm_bytes / 1e6)
                             if case.hbm_bytes > 200e6 else "L2 flushed between steps: no (working set fits L2; "
                             "the step is launch-bound)"},
            "real_time_factor": w.nsamp * w.tsamp / (ms_per_step * 1e-3),
            "roofline": roofline_of(w, case, kernel_ms, clocks),
            "clocks": clocks, "gpu_launches": case.launches * args.steps,
        }
        line["roofline"]["work_note"] = (
            "achieved = nbeams*nchans*ndm*nsamp adds (one per DM-channel-sample, SURVEY 8(d)) / CUDA-event time of "
            "the step; an EFFECTIVE rate: the ps kernels form each output from the same operands but share partial "
            "sums of 4-8 channels between trials (DESIGN.md 5.3), so fewer add instructions are issued "
            "(ncu.issued_add_frac) and the binding unit is shared-memory bandwidth (ncu.lsu_wavefront_frac)")
        if e2e is not None:
            line["e2e"] = e2e
    case.close()

    # ---- the other BASELINE.json configs, same process (single GPU only)
    if rank == 0 and world == 1 and not args.no_per_config and not args.nsamp:
        per = {}
        for idx in sorted(synth.WORKLOADS):
            if idx == w.index:
                continue
            wi = synth.WORKLOADS[idx]
            c = Case(dd, torch, wi, 0, 1, args.kernel, host_input=False)
            # tiny steps need more repetitions for a stable mean
            k = args.steps if wi.adds > 1e10 else max(args.steps, 200)
            ps, tot, clk = c.timed(min(k, max(3, int(3000 / max(1.0, wi.adds / 25e9)))), 3, barrier, gpu_index)
            ms_i = tot / len(ps)
            rf = roofline_of(wi, c, ms_i, clk)
            per["cfg%d" % idx] = {
                "workload": wi.name, "ms_per_step": ms_i, "steps": len(ps), "value": wi.adds / (ms_i * 1e-3) / 1e9,
                "frac": rf["frac"], "frac_measured": rf["frac_measured"], "kernel": kernel_name(c.kern),
                "plan": c.plan.describe(), "real_time_factor": wi.nsamp * wi.tsamp / (ms_i * 1e-3),
                "gpu_launches_per_step": c.launches, "clocks": clk, "traffic": rf["traffic"],
                "data": "synthetic, drawn on the device (seeded)"}
            if wi.adds < 1e9:
                per["cfg%d" % idx]["note"] = ("launch-bound: %.2f us of adds at the roofline; empty-kernel launch "
                                              "measured beside it" % (wi.adds / 37.2e12 * 1e6))
                per["cfg%d" % idx]["empty_launch_us"] = empty_launch_us(torch)
                gms = c.graph_ms_per_step()
                per["cfg%d" % idx]["cuda_graph"] = {
                    "ms_per_step": gms, "value": wi.adds / (gms * 1e-3) / 1e9,
                    "note": "200 dd_execute calls captured into one CUDA graph and replayed: device time per step "
                            "without the per-call host launch cost that bounds ms_per_step above"}
            c.close()
        line["per_config"] = per
        hbm_peak = None
        try:
            hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("hbm_gbs")
        except (OSError, ValueError):
            pass
        line["next_rows"] = next_rows(dd, torch, hbm_peak)

    if rank == 0:
        if not args.no_cpu:
            smp = oracle_sample(w)
            smp.pop("_replay")
            line["cpu_baseline"] = smp
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def finish_timing(total_ms, steps, units_per_rank, world, dist, device):
    """Max over ranks of the device-timed region -> (ms per step, whole-job G units/s): every rank processed
    units_per_rank per step (weak scaling, no data-path collective)."""
    total_ms = sharding.max_over_ranks(total_ms, dist, device)
    ms_per_step = total_ms / steps
    return ms_per_step, sharding.whole_job_rate(units_per_rank, world, ms_per_step * 1e-3) / 1e9


def _timed_ms(torch, fn, reps=5, warm=2):
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(reps):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def next_rows(dd, torch, hbm_peak):
    """The SURVEY 8(f) rows beside the hot path, each timed on the device at a BASELINE.json-sized shape with
    its own roofline: f1 / f3 / f4 are HBM-bound streaming kernels (achieved = algorithmic bytes / time against
    the measured HBM copy bandwidth), f2 is reported as its speed-up over the exact kernel on the same input."""
    rows = {}
    peak = hbm_peak or 6453.4
    g = torch.Generator(device="cuda").manual_seed(1401)
    # f1: post-processing of config 3's (DM, t) plane, candidates only
    w = synth.WORKLOADS[3]
    D = torch.randn((w.ndm, w.nsamp), dtype=torch.float32, device="cuda", generator=g)
    cap = 1 << 20
    cand = torch.zeros(4 * cap, dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    prm = dd.post_params(5, True, True, nsigma=6.0)
    ms = _timed_ms(torch, lambda: dd.dd_postprocess(dd.DD_F32, D, w.nsamp, 0, w.ndm, w.nsamp, 1, prm, None, 0, 0, None,
                                                    cand, cap, cnt))
    by = D.numel() * 4
    rows["f1_postprocess"] = {"shape": "config 3 output, %d series x %d samples float32; median 5, detrend, normalise, 6 sigma -> candidates" % (w.ndm, w.nsamp),
                              "ms": ms, "algorithmic_bytes": by, "bound": "hbm", "achieved_gbs": by / ms / 1e6,
                              "peak_gbs": peak, "frac": by / ms / 1e6 / peak, "gpu_launches": dd.dd_postprocess_launches(prm, False),
                              "note": "algorithmic = D read once; read once by the statistics pass (which leaves chunk maxima), then only the chunks that can hold a candidate"}
    del D
    # f3: RFI mitigation of config 3's input buffer, in place
    n_in = w.nsamp + 14845
    n_pad = (n_in + 63) // 64 * 64                       # row stride as the dedisperser's input buffer has it
    # noise on a bandpass with channel-to-channel gain scatter (so that the fit's RMSE is a bandpass property, not the
    # noise of a window mean), narrowband RFI in three channels and two broadband bursts (the recipe of PAPER.md:1176-1185)
    X = torch.randn((w.nchans, n_pad), dtype=torch.float32, device="cuda", generator=g).add_(20.0)
    X.add_(torch.randn((w.nchans, 1), dtype=torch.float32, device="cuda", generator=g).mul_(0.3))
    for c in (100, 1777, 3000):
        X[c, 50000:90000].add_(5.0)
    for t in (123456, 200000):
        X[:, t:t + 4].add_(3.0)
    rp = dd.dd_rfi_params(4, 512, 7.0, 5.0)
    ms = _timed_ms(torch, lambda: dd.dd_rfi_mitigate(X, w.nchans, n_in, n_pad, 0, 1, rp))
    by = w.nchans * n_in * 8
    rows["f3_rfi"] = {"shape": "config 3 input, %d channels x %d samples float32; order 4, window 512, thresholds 7 / 5" % (w.nchans, n_in),
                      "ms": ms, "algorithmic_bytes": by, "bound": "hbm", "achieved_gbs": by / ms / 1e6, "peak_gbs": peak,
                      "frac": by / ms / 1e6 / peak, "gpu_launches": 9,
                      "note": "algorithmic = X read once + written once; the kernels read it twice (window + column sums in one pass, apply) plus the flagged (channel, window) pairs"}
    del X
    # f4: beamformer, BEST-II parameters of PAPER.md:1653 (32 antennas, 1024 channels, 16 beams) over 2^16 samples
    na, nch, nb, nt = 32, 1024, 16, 1 << 16
    V = torch.randint(0, 256, (nch, nt, na), dtype=torch.uint8, device="cuda", generator=g)
    W = torch.randn((nch, nb, na, 2), dtype=torch.float32, device="cuda", generator=g)
    P = torch.empty((nb, nch, nt), dtype=torch.float32, device="cuda")
    ms = _timed_ms(torch, lambda: dd.dd_beamform_power_u4(V, na, nch, nt, W, nb, P, nt, nch * nt))
    by = V.numel() + P.numel() * 4
    flops = 8.0 * na * nb * nch * nt
    rows["f4_beamformer"] = {"shape": "%d antennas (4-bit complex) x %d channels x %d samples -> %d beams, detected power float32" % (na, nch, nt, nb),
                             "ms": ms, "algorithmic_bytes": by, "bound": "hbm", "achieved_gbs": by / ms / 1e6, "peak_gbs": peak,
                             "frac": by / ms / 1e6 / peak, "tflops": flops / ms / 1e9, "gpu_launches": 2,
                             "note": "8 Na Nb flops per (channel, sample) on the tensor cores (tcgen05.mma fp16 x2, fp32 accumulators in TMEM)"}
    del V, W, P
    # f2: subband (32 channels per subband, 16 trials per nominal DM) vs the exact kernel, config 2's shape as float32
    w2 = synth.scaled(synth.WORKLOADS[2], dtype="f32")
    sb = dd.Subband(w2.nchans, w2.fch1, w2.foff, w2.tsamp, w2.dm_list, 32, 16)
    total = (w2.nsamp + sb.max_shift() + 63) // 64 * 64
    X = torch.randn((w2.nchans, total), dtype=torch.float32, device="cuda", generator=g)
    D = torch.empty((w2.ndm, w2.nsamp), dtype=torch.float32, device="cuda")
    ms_sb = _timed_ms(torch, lambda: sb.execute(X, total, D, w2.nsamp, w2.nsamp), reps=3, warm=1)
    plan = dd.Plan(dd.DD_F32, w2.nchans, w2.fch1, w2.foff, w2.tsamp, w2.dm_list)
    ms_ex = _timed_ms(torch, lambda: plan.execute(X, total, 0, D, w2.nsamp, 0, w2.nsamp, 1), reps=3, warm=1)
    rows["f2_subband"] = {"shape": "config 2's shape as float32 (1024 ch x 1024 trials x 2^17 samples), 32 channels per subband, 16 trials per nominal DM",
                          "ms": ms_sb, "exact_ms": ms_ex, "speedup_over_exact": ms_ex / ms_sb,
                          "adds_ratio": (w2.nchans * 64 + 32 * w2.ndm) / (w2.nchans * w2.ndm),
                          "note": "approximate method (PAPER.md:823): same kernels on reduced data; 96 plans, 96 launches"}
    sb.destroy(); plan.destroy()
    tb = dd.TimeBin(w2.nchans, w2.fch1, w2.foff, w2.tsamp, w2.dm_list * 8.0, 0.0, 8)       # DMs up to 818: four levels
    n_in = tb.input_samples(w2.nsamp)
    n_in_p = (n_in + 63) // 64 * 64
    X = torch.randn((w2.nchans, n_in_p), dtype=torch.float32, device="cuda", generator=g)
    ms_tb = _timed_ms(torch, lambda: tb.execute(X, n_in_p, n_in, D, w2.nsamp, w2.nsamp), reps=3, warm=1)
    plan = dd.Plan(dd.DD_F32, w2.nchans, w2.fch1, w2.foff, w2.tsamp, w2.dm_list * 8.0)
    ms_ex = _timed_ms(torch, lambda: plan.execute(X, n_in_p, 0, D, w2.nsamp, 0, w2.nsamp, 1), reps=3, warm=1)
    rows["f2_timebin"] = {"shape": "1024 ch x 1024 trials (DM 0..818, step 0.8) x 2^17 samples float32, levels %s" % sorted(set(tb.levels().tolist())),
                          "ms": ms_tb, "exact_ms": ms_ex, "speedup_over_exact": ms_ex / ms_tb,
                          "note": "approximate method (PAPER.md:736, 813-819): trials above 2 DM_diag on input summed over 2^k samples"}
    tb.destroy(); plan.destroy()
    return rows


def empty_launch_us(torch, n=200):
    """Back-to-back launches of a trivial torch kernel on one stream (device time per launch): the floor
    under any single-kernel step."""
    x = torch.zeros(32, device="cuda")
    for _ in range(20):
        x.add_(1.0)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(n):
        x.add_(1.0)
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / n * 1e3


def _rank_entry(local_rank, world, port, target, extra):
    os.environ.update({"RANK": str(local_rank), "LOCAL_RANK": str(local_rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    target(*extra)


def launch_ranks(world, target, extra=()):
    """`python bench.py --gpus N` without torchrun: one process per GPU on this node, rendezvous on
    127.0.0.1 (the same environment torchrun would set)."""
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_rank_entry, args=(world, port, target, tuple(extra)), nprocs=world, join=True)


def _main_with_argv(argv):
    sys.argv = list(argv)
    main()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=HEADLINE,
                    help="BASELINE.json config number (1-5); default 3 = configs[2], the largest single-GPU shape")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", default=None, choices=["generic", "ps", "direct"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config legs (profiling aid)")
    ap.add_argument("--nsamp", type=int, default=0,
                    help="profiling aid: cut the workload to this many output samples (the line then names it)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = synth.WORKLOADS[args.config]
    if args.nsamp:
        w = synth.scaled(w, nsamp=args.nsamp, name="%s_cut_to_%d_samples" % (w.name, args.nsamp))
    if args.impl == "reference":
        run_reference(args, w)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # the contract command without torchrun: start the N ranks here, one device each
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            print(json.dumps({"error": "--gpus %d but only %d CUDA devices are visible" % (args.gpus, have)}))
            sys.exit(1)
        launch_ranks(args.gpus, _main_with_argv, (list(sys.argv),))
        return
    run_ours(args, w)


if __name__ == "__main__":
    main()
