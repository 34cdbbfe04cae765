"""paper_1002_3675_b200 — B200-native (sm_100a) hot path of TV-regularised cone-beam CT
reconstruction by forward-backward splitting (arXiv 1002.3675).

Thin Python binding over the C ABI of `libcbct.so` (include/cbct.h): argument marshalling only —
every step of the path runs in the hand-written CUDA kernels under `csrc/`.  PyTorch supplies
device memory and streams.  There is no CPU fallback: loading fails loudly if the library is
missing, and every compute call fails if there is no CUDA device.
"""
from .binding import (  # noqa: F401
    CbctError, Geometry, load, lib_path, launch_count,
    forward, backproject, backproject_eq2, set_backprojector, BACKPROJECTOR_EXACT, BACKPROJECTOR_EQ2, tv_prox, fbs_reconstruct, fbs_reconstruct_until, data_gradient, prox_step, energy, prolong, restrict, bin2x2,
    profile_enable, profile_read, PROFILE_TAGS, set_guard_mode,
    forward_host, backproject_host, tv_prox_host, fbs_reconstruct_host,
    fbs_vcycle, fdk_reconstruct, tv_value_noalloc, fbs_reconstruct_sharded, CascadeOps, ALLREDUCE_FN,
)
