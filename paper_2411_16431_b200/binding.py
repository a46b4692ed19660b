"""ctypes binding of libtn_b200.so: same names and argument order as include/tn.h."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtn_b200.so")

EXPORTED_SYMBOLS = ["tn_create", "tn_set_stream", "tn_set_allocator", "tn_set_option", "tn_set_beta", "tn_contract",
                    "tn_log_z", "tn_row_lognorm", "tn_mps_shape", "tn_mps_tensor", "tn_branch_and_bound",
                    "tn_get_stats", "tn_droplets", "tn_energy", "tn_kernel_check", "tn_kernel_bench", "tn_gemm_t_static",
                    "tn_lbp", "tn_lbp_message", "tn_lbp_marginals", "tn_lbp_select", "tn_fp64_peak", "tn_last_error", "tn_destroy"]
OPT_GAP_GUARD, OPT_SVD_TOL, OPT_SVD_MAXIT, OPT_OVERSAMPLE, OPT_EXACT_CAP, OPT_SELECT_DIRECT_MAX, OPT_SVD_CHEB, OPT_SVD_LOCK, OPT_MERGE = 1, 2, 3, 4, 5, 6, 7, 8, 9
OPT_MERGE_CAP = 10
OPT_SCHEDULE, OPT_SWEEP_RANGE, OPT_SVD_MODE, OPT_RSVD_ITERS, OPT_TWO_STEP = 11, 12, 13, 14, 15
OPT_DROPLETS, OPT_DROPLET_MAX_DE, OPT_DROPLET_MIN_HAMMING, OPT_DROPLET_MAX_COUNT = 16, 17, 18, 19
OPT_MERGE_SEGMENTED = 20
OPT_SVD_DIRECT = 21
OPT_COND_PIPE = 22
OPT_TS_WIDE_ROWS = 23
OPT_RBLOCK_FACT = 24
OPT_SELECT_ROWS = 25
OPT_LAZY_V = 26


class TnError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("tn error %d: %s" % (code, msg))
        self.code = code


class TnStats(C.Structure):
    _fields_ = [(n, C.c_double) for n in (
        "ms_tables", "ms_contract", "ms_theta_build", "ms_theta_apply", "ms_orth_svd", "ms_search",
        "ms_search_rblocks", "ms_search_cond", "ms_search_select", "flop_theta_build", "flop_theta_apply",
        "bytes_theta_apply", "flop_search", "bytes_search_cond", "bytes_search_select", "min_sigma_rel")] + [(n, C.c_int64) for n in (
            "svd_iterations", "kernel_launches", "negative_u", "rows_contracted", "bytes_device", "jacobi_calls",
            "jacobi_sweeps", "theta_apply_calls", "cheb_steps", "svd_locked_cols", "merged_away", "svd_unconverged",
            "merge_fallback_cells", "select_tie_overflow", "select_tie_dropped", "svd_direct", "droplet_overflow")] + [(n, C.c_double) for n in ("flop_orth_svd", "flop_search_rblocks", "flop_search_cond")]

    def asdict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


_lib = None
ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


def lib():
    """Loads the shared library (building it is `python -m paper_2411_16431_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError("libtn_b200.so is missing: run `python -m paper_2411_16431_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        p_i32, p_f64, p_i8 = C.POINTER(C.c_int32), C.POINTER(C.c_double), C.POINTER(C.c_int8)
        L.tn_create.argtypes = [C.POINTER(C.c_void_p), C.c_int32, C.c_int64, p_i32, p_i32, p_f64, p_f64, C.c_int32,
                                C.c_int32, C.c_int32, C.c_int32, p_i32, p_i32, p_i32, p_i32]
        L.tn_set_stream.argtypes = [C.c_void_p, C.c_void_p]
        L.tn_set_allocator.argtypes = [C.c_void_p, ALLOC_FN, FREE_FN, C.c_void_p]
        L.tn_set_option.argtypes = [C.c_void_p, C.c_int32, C.c_double]
        L.tn_set_beta.argtypes = [C.c_void_p, C.c_double]
        L.tn_contract.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
        L.tn_log_z.argtypes = [C.c_void_p, p_f64]
        L.tn_row_lognorm.argtypes = [C.c_void_p, C.c_int32, p_f64]
        L.tn_mps_shape.argtypes = [C.c_void_p, C.c_int32, C.c_int32, p_i32, p_i32, p_i32, p_i32]
        L.tn_mps_tensor.argtypes = [C.c_void_p, C.c_int32, C.c_int32, p_f64]
        L.tn_branch_and_bound.argtypes = [C.c_void_p, C.c_int32, p_i32, p_i8, p_f64, p_f64, p_f64]
        L.tn_get_stats.argtypes = [C.c_void_p, C.POINTER(TnStats)]
        L.tn_energy.argtypes = [C.c_void_p, C.c_int32, p_i8, p_f64]
        L.tn_droplets.argtypes = [C.c_void_p, C.c_int32, p_i32, p_f64, p_i8]
        L.tn_fp64_peak.argtypes = [p_f64]
        p_u32 = C.POINTER(C.c_uint32)
        L.tn_lbp.argtypes = [C.c_void_p, C.c_int32]
        L.tn_lbp_message.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, p_i32, p_f64]
        L.tn_lbp_marginals.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, p_u32, p_f64]
        L.tn_lbp_select.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, p_i32, p_u32, p_f64]
        L.tn_gemm_t_static.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_int64, C.c_void_p, C.c_int64, C.c_void_p,
                                       C.c_int64, C.c_void_p, C.c_int64]
        L.tn_kernel_bench.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_int32, C.c_int64, C.c_int32, p_f64]
        L.tn_kernel_check.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_int32, C.c_int32, p_f64, p_f64, p_f64]
        L.tn_last_error.restype = C.c_char_p
        L.tn_destroy.argtypes = [C.c_void_p]
        L.tn_destroy.restype = None
        for n in EXPORTED_SYMBOLS:
            if n not in ("tn_last_error", "tn_destroy"):
                getattr(L, n).restype = C.c_int
        _lib = L
    return _lib


def tn_last_error() -> str:
    return lib().tn_last_error().decode()


def _check(rc):
    if rc != 0:
        raise TnError(rc, tn_last_error())


def _ptr(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def tn_create(n_spins, edge_u, edge_v, J, h, Ly, Lx, subs_per_cell, spins_per_sub, cell_y, cell_x, sub, pos):
    eu = np.ascontiguousarray(edge_u, dtype=np.int32)
    ev = np.ascontiguousarray(edge_v, dtype=np.int32)
    Jv = np.ascontiguousarray(J, dtype=np.float64)
    hv = None if h is None else np.ascontiguousarray(h, dtype=np.float64)
    cy, cx, sb, ps = (np.ascontiguousarray(a, dtype=np.int32) for a in (cell_y, cell_x, sub, pos))
    out = C.c_void_p()
    _check(lib().tn_create(C.byref(out), int(n_spins), int(eu.size), _ptr(eu, C.c_int32), _ptr(ev, C.c_int32),
                           _ptr(Jv, C.c_double), None if hv is None else _ptr(hv, C.c_double), int(Ly), int(Lx),
                           int(subs_per_cell), int(spins_per_sub), _ptr(cy, C.c_int32), _ptr(cx, C.c_int32),
                           _ptr(sb, C.c_int32), _ptr(ps, C.c_int32)))
    return out


def tn_set_stream(handle, cuda_stream):
    _check(lib().tn_set_stream(handle, C.c_void_p(cuda_stream)))


def tn_set_allocator(handle, alloc, free_, ctx=None):
    _check(lib().tn_set_allocator(handle, alloc, free_, ctx))


def tn_set_option(handle, key, value):
    _check(lib().tn_set_option(handle, int(key), float(value)))


def tn_set_beta(handle, beta):
    _check(lib().tn_set_beta(handle, float(beta)))


def tn_contract(handle, D, sweeps):
    _check(lib().tn_contract(handle, int(D), int(sweeps)))


def tn_log_z(handle) -> float:
    v = C.c_double()
    _check(lib().tn_log_z(handle, C.byref(v)))
    return v.value


def tn_row_lognorm(handle, y) -> float:
    v = C.c_double()
    _check(lib().tn_row_lognorm(handle, int(y), C.byref(v)))
    return v.value


def tn_mps_shape(handle, y, j):
    n, dl, p, dr = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32()
    _check(lib().tn_mps_shape(handle, int(y), int(j), C.byref(n), C.byref(dl), C.byref(p), C.byref(dr)))
    return n.value, dl.value, p.value, dr.value


def tn_mps_tensor(handle, y, j):
    _, dl, p, dr = tn_mps_shape(handle, y, j)
    out = np.empty((dl, p, dr), dtype=np.float64)
    _check(lib().tn_mps_tensor(handle, int(y), int(j), _ptr(out, C.c_double)))
    return out


def tn_branch_and_bound(handle, M, n_spins):
    """Returns (states [n, n_spins] int8, energies [n], logp [n], log_p_discarded)."""
    states = np.empty((M, n_spins), dtype=np.int8)
    energies = np.empty(M, dtype=np.float64)
    logp = np.empty(M, dtype=np.float64)
    n = C.c_int32()
    pd = C.c_double()
    _check(lib().tn_branch_and_bound(handle, int(M), C.byref(n), _ptr(states, C.c_int8), _ptr(energies, C.c_double),
                                     _ptr(logp, C.c_double), C.byref(pd)))
    k = n.value
    return states[:k], energies[:k], logp[:k], pd.value


def tn_droplets(handle, rank, n_spins, max_count=32):
    """Returns (dE [n], flips [n, n_spins] int8) of the droplets above returned state `rank` (include/tn.h)."""
    n = C.c_int32()
    dE = np.empty(max_count, dtype=np.float64)
    flips = np.empty((max_count, n_spins), dtype=np.int8)
    _check(lib().tn_droplets(handle, int(rank), C.byref(n), _ptr(dE, C.c_double), _ptr(flips, C.c_int8)))
    return dE[:n.value].copy(), flips[:n.value].copy()


def tn_energy(handle, states, n_spins=None):
    s = np.ascontiguousarray(states, dtype=np.int8)
    if s.ndim == 1:
        s = s[None, :]
    if n_spins is not None and (s.ndim != 2 or s.shape[1] != n_spins):   # the C call reads n * n_spins bytes
        raise TnError(-1, "states must have shape [n, %d], got %s" % (n_spins, s.shape))
    out = np.empty(s.shape[0], dtype=np.float64)
    _check(lib().tn_energy(handle, s.shape[0], _ptr(s, C.c_int8), _ptr(out, C.c_double)))
    return out


CHECK_ORTH, CHECK_GEMM_N, CHECK_GEMM_T = 1, 2, 3


def tn_kernel_check(handle, op, A, B=None):
    """Diagnostic: one device building block on host data (see include/tn.h)."""
    A = np.ascontiguousarray(A, dtype=np.float64)
    m, k = A.shape
    if op == CHECK_ORTH:
        n, out, Bp = 1, np.empty((m, k)), None
    else:
        B = np.ascontiguousarray(B, dtype=np.float64)
        n = B.shape[1]
        out = np.empty((m, n) if op == CHECK_GEMM_N else (k, n))
        Bp = _ptr(B, C.c_double)
    _check(lib().tn_kernel_check(handle, int(op), int(m), int(n), int(k), _ptr(A, C.c_double), Bp,
                                 _ptr(out, C.c_double)))
    return out


def tn_kernel_bench(handle, op, m, n, k, iters=10) -> float:
    """Diagnostic: device ms per call of one building block on device-resident random data."""
    v = C.c_double(0.0)
    _check(lib().tn_kernel_bench(handle, int(op), int(m), int(n), int(k), int(iters), C.byref(v)))
    return v.value


def tn_lbp(handle, iterations):
    _check(lib().tn_lbp(handle, int(iterations)))


def tn_lbp_message(handle, y, x, leg):
    n = C.c_int32()
    out = np.empty(256, dtype=np.float64)
    _check(lib().tn_lbp_message(handle, int(y), int(x), int(leg), C.byref(n), _ptr(out, C.c_double)))
    return out[:n.value].copy()


def tn_lbp_marginals(handle, y, x, cell_states):
    st = np.ascontiguousarray(cell_states, dtype=np.uint32)
    out = np.empty(st.size, dtype=np.float64)
    _check(lib().tn_lbp_marginals(handle, int(y), int(x), int(st.size), _ptr(st, C.c_uint32), _ptr(out, C.c_double)))
    return out


def tn_lbp_select(handle, y, x, K):
    st = np.empty(K, dtype=np.uint32)
    lp = np.empty(K, dtype=np.float64)
    n = C.c_int32()
    _check(lib().tn_lbp_select(handle, int(y), int(x), int(K), C.byref(n), _ptr(st, C.c_uint32), _ptr(lp, C.c_double)))
    return st[:n.value].copy(), lp[:n.value].copy()


def tn_gemm_t_static(cuda_stream, m, n, k, dA, lda, dB, ldb, dC, ldc):
    """C [k x n] = A [m x k]^T . B [m x n] on DEVICE pointers (ints), allocation-free (include/tn.h); asynchronous."""
    _check(lib().tn_gemm_t_static(C.c_void_p(cuda_stream), int(m), int(n), int(k), C.c_void_p(dA), int(lda),
                                  C.c_void_p(dB), int(ldb), C.c_void_p(dC), int(ldc)))


def tn_fp64_peak() -> float:
    v = C.c_double()
    rc = lib().tn_fp64_peak(C.byref(v))
    if rc != 0:
        raise TnError(rc, "tn_fp64_peak failed (no CUDA device?)")
    return v.value


def tn_get_stats(handle) -> dict:
    st = TnStats()
    _check(lib().tn_get_stats(handle, C.byref(st)))
    return st.asdict()


def tn_destroy(handle):
    lib().tn_destroy(handle)


class TensorNetwork:
    """Convenience owner of a tn_handle for an `instances.Instance`-like object (attributes n_spins,
    edge_u, edge_v, J, h, Ly, Lx, S, n_s, cell_y, cell_x, sub, pos).  Uses torch's caching allocator
    and current stream when torch sees a CUDA device."""

    def __init__(self, inst, use_torch: bool = True):
        self.n_spins = int(inst.n_spins)
        self.handle = tn_create(inst.n_spins, inst.edge_u, inst.edge_v, inst.J, inst.h, inst.Ly, inst.Lx, inst.S,
                                inst.n_s, inst.cell_y, inst.cell_x, inst.sub, inst.pos)
        self._cb = None
        if use_torch:
            try:
                import torch
                if torch.cuda.is_available():
                    t_alloc = torch.cuda.caching_allocator_alloc      # bound now: module attributes are
                    t_free = torch.cuda.caching_allocator_delete      # gone at interpreter shutdown
                    alloc = ALLOC_FN(lambda n, ctx: t_alloc(n))
                    free_ = FREE_FN(lambda p, ctx: t_free(p))
                    self._cb = (alloc, free_)
                    tn_set_allocator(self.handle, alloc, free_)
                    tn_set_stream(self.handle, torch.cuda.current_stream().cuda_stream)
            except ImportError:
                pass

    def set_option(self, key, value):
        tn_set_option(self.handle, key, value)

    def set_beta(self, beta):
        tn_set_beta(self.handle, beta)

    def contract(self, D, sweeps):
        tn_contract(self.handle, D, sweeps)

    def log_z(self):
        return tn_log_z(self.handle)

    def row_lognorm(self, y):
        return tn_row_lognorm(self.handle, y)

    def mps(self, y):
        n = tn_mps_shape(self.handle, y, 0)[0]
        return [tn_mps_tensor(self.handle, y, j) for j in range(n)]

    def branch_and_bound(self, M):
        return tn_branch_and_bound(self.handle, M, self.n_spins)

    def lbp(self, iterations):
        tn_lbp(self.handle, iterations)

    def lbp_message(self, y, x, leg):
        return tn_lbp_message(self.handle, y, x, leg)

    def lbp_marginals(self, y, x, cell_states):
        return tn_lbp_marginals(self.handle, y, x, cell_states)

    def lbp_select(self, y, x, K):
        return tn_lbp_select(self.handle, y, x, K)

    def droplets(self, rank):
        return tn_droplets(self.handle, rank, self.n_spins)

    def energy(self, states):
        return tn_energy(self.handle, states, self.n_spins)

    def stats(self):
        return tn_get_stats(self.handle)

    def close(self):
        if self.handle is not None:
            tn_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
