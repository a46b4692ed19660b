"""Kernel-level GPU parity: single device building blocks (through tn_kernel_check of the C ABI) against
their plain definitions in numpy fp64."""
import numpy as np
import pytest

import instances

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tn():
    import paper_2411_16431_b200 as tnb
    with tnb.TensorNetwork(instances.lattice(2, 2, 2, 2, seed=1)) as t:
        yield t


def _check(tn, op, A, B=None):
    import paper_2411_16431_b200 as tnb
    return tnb.tn_kernel_check(tn.handle, op, A, B)


ORTH = [(1, 1), (7, 3), (64, 16), (65, 17), (1000, 32), (4097, 33), (20000, 48), (5000, 64), (9999, 80), (30011, 96),
        (300, 100)]


@pytest.mark.parametrize("m,k", ORTH)
def test_orth_columns_well_conditioned(tn, m, k):
    import paper_2411_16431_b200 as tnb
    rng = np.random.default_rng(m * 131 + k)
    k = min(k, m)
    A = rng.standard_normal((m, k))
    Q = _check(tn, tnb.CHECK_ORTH, A)
    assert np.abs(Q.T @ Q - np.eye(k)).max() <= 1e-13
    # same column space, and (Cholesky-QR keeps the column order) Q^T A is upper triangular
    R = Q.T @ A
    assert np.abs(Q @ R - A).max() <= 1e-12 * np.abs(A).max()
    if k <= 96:
        assert np.abs(np.tril(R, -1)).max() <= 1e-12 * np.abs(R).max()


@pytest.mark.parametrize("m,k,cond", [(2000, 32, 1e8), (2000, 32, 1e14), (5000, 80, 1e12), (3000, 48, 1e20)])
def test_orth_columns_ill_conditioned(tn, m, k, cond):
    """Singular values decaying over `cond` (beyond 1/eps: numerically rank-deficient, reading S6)."""
    import paper_2411_16431_b200 as tnb
    rng = np.random.default_rng(k)
    U, _ = np.linalg.qr(rng.standard_normal((m, k)))
    V, _ = np.linalg.qr(rng.standard_normal((k, k)))
    s = np.logspace(0, -np.log10(cond), k)
    A = (U * s) @ V.T
    Q = _check(tn, tnb.CHECK_ORTH, A)
    assert np.isfinite(Q).all()
    assert np.abs(Q.T @ Q - np.eye(k)).max() <= 1e-10
    # the well-determined part of the column space is reproduced
    keep = s > 1e-6
    P = (U[:, keep] * s[keep]) @ V[:, keep].T
    assert np.abs(Q @ (Q.T @ P) - P).max() <= 1e-9


def test_orth_columns_zero_columns_stay_zero(tn):
    import paper_2411_16431_b200 as tnb
    rng = np.random.default_rng(5)
    A = rng.standard_normal((777, 24))
    A[:, 17:] = 0.0
    Q = _check(tn, tnb.CHECK_ORTH, A)
    assert np.all(Q[:, 17:] == 0.0)
    assert np.abs(Q[:, :17].T @ Q[:, :17] - np.eye(17)).max() <= 1e-13
    Z = _check(tn, tnb.CHECK_ORTH, np.zeros((100, 8)))
    assert np.all(Z == 0.0)


GEMM = [(1, 1, 1), (5, 3, 7), (128, 16, 128), (129, 17, 65), (1000, 32, 515), (4096, 80, 300), (333, 96, 2049),
        (70000, 24, 64), (50, 130, 40),
        (60001, 48, 130), (310, 40, 60002), (57000, 30, 18)]      # 24-row warp tiles (outputs with >= 192 * 2 * SMs rows)


@pytest.mark.parametrize("m,n,k", GEMM)
def test_skinny_gemm_n_and_t(tn, m, n, k):
    import paper_2411_16431_b200 as tnb
    rng = np.random.default_rng(m + 7 * n + 13 * k)
    A = rng.standard_normal((m, k))
    B = rng.standard_normal((k, n))
    C = _check(tn, tnb.CHECK_GEMM_N, A, B)
    ref = A @ B
    assert np.abs(C - ref).max() <= 1e-13 * k * max(1.0, np.abs(ref).max())
    Bt = rng.standard_normal((m, n))
    Ct = _check(tn, tnb.CHECK_GEMM_T, A, Bt)
    reft = A.T @ Bt
    assert np.abs(Ct - reft).max() <= 1e-13 * m * max(1.0, np.abs(reft).max())


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,D", [(3, 3, 3, 4, 0.9, 4, 6), (3, 3, 2, 8, 0.97, 3, 12), (4, 4, 2, 4, 0.95, 2, 5)])
def test_pipelined_conditional_kernel_against_the_generic_route(Ly, Lx, S, ns, p, seed, D):
    """k_cond (cp.async-pipelined conditional GEMM, TN_OPT_COND_PIPE = 1, the default) against the generic batched kernel
    (TN_OPT_COND_PIPE = 0) on the same boundary MPS: identical states, log-probabilities to rounding (the per-beam
    normaliser is summed in another tile order), identical count of clamped negative conditionals; odd bonds (D = 5)
    and ragged projectors included."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    out = []
    for pipe in (1, 0):
        with tnb.TensorNetwork(inst) as t:
            t.set_option(tnb.OPT_COND_PIPE, pipe)
            t.set_beta(1.2)
            t.contract(D, 1)
            lz = t.log_z()
            states, E, logp, pd = t.branch_and_bound(64)
            out.append((lz, states, logp, pd, t.stats()["negative_u"]))
    assert abs(out[0][0] - out[1][0]) <= 1e-13 * abs(out[0][0])
    assert np.array_equal(out[0][1], out[1][1])
    assert np.allclose(out[0][2], out[1][2], rtol=1e-12, atol=0) and abs(out[0][3] - out[1][3]) <= 1e-12 * abs(out[0][3])
    assert out[0][4] == out[1][4]


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,D", [(3, 3, 3, 4, 0.9, 4, 6), (3, 4, 2, 8, 0.97, 3, 12), (3, 4, 2, 4, 0.95, 2, 5),
                                               (3, 3, 3, 2, 0.85, 7, 4)])
def test_factorised_right_blocks_against_the_joint_gemm(Ly, Lx, S, ns, p, seed, D):
    """k_rblock_mma / k_rblock_h (right blocks summed over c_lo first, then over b: TN_OPT_RBLOCK_FACT = 1, the default, on
    the tensor cores; 2: the plain-FMA kernel) against the joint GEMM over (b, c_lo) x (beam, a_hi) (TN_OPT_RBLOCK_FACT = 0)
    on the same boundary MPS: identical states, log-probabilities and log Z to rounding (another summation order)."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    out = []
    for fact in (1, 2, 0):
        with tnb.TensorNetwork(inst) as t:
            t.set_option(tnb.OPT_RBLOCK_FACT, fact)
            t.set_beta(1.2)
            t.contract(D, 1)
            lz = t.log_z()
            states, E, logp, pd = t.branch_and_bound(64)
            out.append((lz, states, logp, pd))
    for o in out[1:]:
        assert abs(out[0][0] - o[0]) <= 1e-12 * abs(out[0][0])
        assert np.array_equal(out[0][1], o[1])
        assert np.allclose(out[0][2], o[2], rtol=1e-11, atol=0) and abs(out[0][3] - o[3]) <= 1e-11 * abs(out[0][3])


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,D,M", [(3, 3, 3, 4, 0.9, 4, 6, 64), (3, 4, 2, 8, 0.97, 3, 12, 256),
                                                 (3, 4, 2, 4, 0.95, 2, 5, 7)])
def test_row_maxima_selection_bound_gives_the_same_lists(Ly, Lx, S, ns, p, seed, D, M):
    """The top-M bound from the row maxima of V (written by k_cond) + the row-skipping prefilter (TN_OPT_SELECT_ROWS = 1,
    the default) against the hashed 1/64 sample + full pass over V (0): any subset of the candidates gives a valid lower
    bound, so the selected lists must be IDENTICAL (bitwise), not merely close.  The sampled route is forced.
    Lazy V (TN_OPT_LAZY_V = 1, the default: k_cond writes no V, k_cond_rows recomputes the rows that reach the bound) is
    compared the same way: the recomputed entries are the ones the row maxima came from, so again bitwise."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    out = []
    for rows, lazy in ((1, 1), (1, 0), (0, 0)):
        with tnb.TensorNetwork(inst) as t:
            t.set_option(tnb.OPT_SELECT_ROWS, rows)
            t.set_option(tnb.OPT_LAZY_V, lazy)
            t.set_option(tnb.OPT_SELECT_DIRECT_MAX, 0)
            t.set_beta(1.2)
            t.contract(D, 1)
            states, E, logp, pd = t.branch_and_bound(M)
            out.append((states, logp, pd, t.stats()["negative_u"]))
    for o in out[1:]:
        assert np.array_equal(out[0][0], o[0]) and np.array_equal(out[0][1], o[1]) and out[0][2] == o[2]
        assert out[0][3] == o[3]
