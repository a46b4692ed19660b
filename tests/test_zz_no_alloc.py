"""tn_gemm_t_static: the allocation-free variant of the Theta-core^T x skinny apply (static device scratch instead of a
device allocation; include/tn.h) against the existing handle-based path (tn_kernel_check, TN_CHECK_GEMM_T), on two calls
in a row that share the scratch array.  Collected last on purpose (the file name): the suite runs with `pytest -x`."""
import numpy as np
import pytest

import instances

pytestmark = pytest.mark.gpu


def _run_static(tnb, torch, A, B):
    m, k = A.shape
    n = B.shape[1]
    dA = torch.from_numpy(A).cuda()
    dB = torch.from_numpy(B).cuda()
    dC = torch.full((k, n), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    tnb.tn_gemm_t_static(torch.cuda.current_stream().cuda_stream, m, n, k, dA.data_ptr(), k, dB.data_ptr(), n,
                         dC.data_ptr(), n)
    torch.cuda.synchronize()
    return dC.cpu().numpy()


def test_static_scratch_gemm_matches_the_existing_path_twice_in_a_row():
    import torch
    import paper_2411_16431_b200 as tnb
    rng = np.random.default_rng(17)
    # second call: other shape, other data, fewer partial products -- stale scratch contents of the first call must not
    # leak into it; third call: the first shape again
    # (lda = k and ldb = n must be even: 16-byte rows, as in the path's own Theta-core layouts)
    shapes = [(20000, 48, 300), (4097, 24, 514), (20000, 48, 300), (333, 96, 2050), (65, 6, 10)]
    with tnb.TensorNetwork(instances.lattice(2, 2, 2, 2, seed=1)) as t:
        for (m, n, k) in shapes:
            A = rng.standard_normal((m, k))
            B = rng.standard_normal((m, n))
            ref = tnb.tn_kernel_check(t.handle, tnb.CHECK_GEMM_T, A, B)          # existing path (allocates its workspace)
            got = _run_static(tnb, torch, A, B)
            tol = 1e-13 * m * max(1.0, np.abs(ref).max())                        # the tolerance of tests/test_gpu_kernels.py
            assert np.isfinite(got).all()
            assert np.abs(got - ref).max() <= tol, (m, n, k, np.abs(got - ref).max())
            assert np.abs(got - A.T @ B).max() <= tol


def test_static_scratch_gemm_rejects_sizes_beyond_its_scratch():
    import torch
    import paper_2411_16431_b200 as tnb
    x = torch.zeros(16, dtype=torch.float64, device="cuda")
    with pytest.raises(tnb.TnError) as e:                                         # 2 k n > 2^20 doubles
        tnb.tn_gemm_t_static(0, 1024, 96, 8192, x.data_ptr(), 8192, x.data_ptr(), 96, x.data_ptr(), 96)
    assert e.value.code == -1 and "static scratch" in str(e.value)
    with pytest.raises(tnb.TnError) as e:                                         # more than 96 columns
        tnb.tn_gemm_t_static(0, 1024, 100, 64, x.data_ptr(), 64, x.data_ptr(), 100, x.data_ptr(), 100)
    assert e.value.code == -1
