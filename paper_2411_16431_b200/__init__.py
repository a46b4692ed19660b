"""B200-native boundary-MPS / branch-and-bound hot path of arXiv 2411.16431.

Thin ctypes binding of the C ABI declared in include/tn.h (argument marshalling only; every
step of the path runs in the CUDA kernels of libtn_b200.so).  PyTorch is used for device
memory (its caching allocator, through tn_set_allocator) and the stream.  There is no CPU
fallback: importing works without a GPU, computing does not.
"""
from .binding import (TnError, TensorNetwork, lib, tn_branch_and_bound, tn_contract, tn_create, tn_destroy,
                      tn_energy, tn_fp64_peak, tn_kernel_check, tn_kernel_bench, CHECK_ORTH, CHECK_GEMM_N, CHECK_GEMM_T, tn_get_stats, tn_last_error, tn_log_z, tn_mps_shape, tn_mps_tensor,
                      tn_row_lognorm, tn_set_allocator, tn_set_beta, tn_set_option, tn_set_stream, TnStats,
                      EXPORTED_SYMBOLS, OPT_GAP_GUARD, OPT_SVD_TOL, OPT_SVD_MAXIT, OPT_OVERSAMPLE, OPT_EXACT_CAP, OPT_SELECT_DIRECT_MAX, OPT_SVD_CHEB, OPT_SVD_LOCK, OPT_MERGE, OPT_MERGE_CAP,
                      OPT_SCHEDULE, OPT_SWEEP_RANGE, OPT_SVD_MODE, OPT_RSVD_ITERS, OPT_TWO_STEP,
                      OPT_DROPLETS, OPT_DROPLET_MAX_DE, OPT_DROPLET_MIN_HAMMING, OPT_DROPLET_MAX_COUNT, OPT_MERGE_SEGMENTED, OPT_SVD_DIRECT, OPT_COND_PIPE, OPT_TS_WIDE_ROWS, OPT_RBLOCK_FACT, OPT_SELECT_ROWS, OPT_LAZY_V, tn_droplets, tn_gemm_t_static,
                      tn_lbp, tn_lbp_message, tn_lbp_marginals, tn_lbp_select)

__all__ = [n for n in dir() if not n.startswith("_")]
