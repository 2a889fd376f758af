"""EPIC (E-field Parallel Imaging Correlator, arXiv 1904.11422) hot path on one NVIDIA B200:
hand-written sm_100a CUDA kernels behind the C ABI of include/epic.h, plus this thin binding.
Build the library with ``python -m paper_1904_11422_b200.build``."""
from .binding import (  # noqa: F401
    EPIC_ERR_ARG, EPIC_ERR_CUDA, EPIC_ERR_NOMEM, EPIC_ERR_RANGE, EPIC_ERR_SCRATCH, EPIC_OK, EPIC_ORDER_TCAP, EPIC_ORDER_TCPA,
    EPIC_PATH_AUTO, EPIC_PATH_FUSED, EPIC_PATH_STREAM, EPIC_PATH_TENSOR, EPIC_PATH_TILED, EPIC_PATH_TWOPASS, LIB_PATH, SYMBOLS,
    EpicError, Plan, epic_autocorr_remove, epic_debug_unpack, epic_fp32_peak_probe, epic_image, epic_image_cf32, epic_image_host, epic_image_noalloc, epic_noalloc_scratch_bytes,
    epic_plan_create, epic_plan_create_per_channel, epic_plan_destroy, lib,
)
