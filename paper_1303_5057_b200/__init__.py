"""gray-b200: photon null geodesics in Kerr spacetime on one B200 (the hot path of GRay, arXiv 1303.5057).

Thin Python binding of the C-ABI library libgray (include/gray.h).  All arithmetic runs in the CUDA
kernels of csrc/; PyTorch is used for device memory and streams only.  There is no CPU path: the
functions raise if libgray.so or a CUDA device is missing.
"""
from .gray import (  # noqa: F401
    GRAY_F32, GRAY_F64, STEP_REL, STEP_EQ2, SYS_FULL, SYS_REDUCED, LIVE, CAPTURED, ESCAPED, BAD, EQUATOR, N_STATUS, SCHED_REFILL, SCHED_STATIC,
    GrayError, PhotonBatch, StepParams, lib, lib_path, gray_init_rays, gray_init_rays_random, gray_init_rays_polar, gray_ring_polar, gray_integrate,
    gray_integrate_counters, gray_classify, gray_shadow_edge, gray_fma_peak, gray_packed_peak, gray_device_info, gray_workspace_bytes,
    gray_version, trace_image, gray_integrate_host, gray_host_scratch_bytes, gray_shadow_edge_noalloc, gray_noalloc_max_angles,
)
