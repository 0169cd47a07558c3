"""B200-native direct incoherent dedispersion (arxiv/paper_1401_8258, §2.1.1 / §2.4).

``binding`` wraps the C ABI of ``include/dedisp_b200.h`` one to one; ``synth`` holds the seeded
input generators and the BASELINE.json workload shapes (no arithmetic of the method).
"""
from .binding import (  # noqa: F401
    DD_OK, DD_ERR_BAD_ARG, DD_ERR_UNSUPPORTED, DD_ERR_NOMEM, DD_ERR_CUDA, DD_ERR_STATE,
    DD_F32, DD_U8, DD_KERNEL_AUTO, DD_KERNEL_GENERIC, DD_KERNEL_PS, DD_KERNEL_DIRECT,
    DedispError, Plan, Stream, TimeBin, Subband, lib, dd_diagonal_dm, dd_downsample2_f32,
    dd_version, dd_max_shift, dd_shift_table, dd_release_workspaces,
    dd_rfi_params, dd_rfi_mitigate, dd_beamform_power_u4, dd_post_params, post_params, CANDIDATE_DTYPE, dd_postprocess, dd_postprocess_launches,
    dd_postprocess_static, POSTPROCESS_STATIC_MAX_SERIES,
    dd_dedisperse_f32, dd_dedisperse_u8_i32, dd_dedisperse_f32_host, dd_dedisperse_u8_i32_host,
)
