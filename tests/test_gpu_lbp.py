"""GPU parity of the loopy-belief-propagation stage (f4; Sec. IV, Eqs. (11)-(13) PAPER.md:181-215): tn_lbp /
tn_lbp_message / tn_lbp_marginals / tn_lbp_select through the C ABI against oracle/lbp.py on the same seeded inputs.
The CUDA path sums Eq. (11) through the chain structure of the cell weight, the oracle over all d states of the cell."""
import numpy as np
import pytest

import instances
from oracle import lbp, model

pytestmark = pytest.mark.gpu

LEGS = ("left", "right", "up", "down", "din", "dout")


def _compare(inst, beta, iterations, K, n_eval=4096, rtol=1e-11):
    import paper_2411_16431_b200 as tnb
    m = model.Model(inst).set_beta(beta)
    nu = lbp.messages(m, iterations)
    rng = np.random.default_rng(5)
    d = 1 << (inst.S * inst.n_s)
    with tnb.TensorNetwork(inst) as t:
        t.set_beta(beta)
        with pytest.raises(tnb.TnError) as e:
            t.lbp_select(0, 0, 4)
        assert e.value.code == -3                                   # TN_ERR_STATE: tn_lbp has not run
        t.lbp(iterations)
        for y in range(inst.Ly):
            for x in range(inst.Lx):
                for leg, name in enumerate(LEGS):
                    got = t.lbp_message(y, x, leg)
                    ref = nu[(y, x)][name]
                    assert got.shape == ref.shape, (y, x, name)
                    assert np.allclose(got, ref, rtol=rtol, atol=1e-300), (y, x, name, np.abs(got - ref).max())
                lp = lbp.log_marginals(m, nu, y, x)
                states = np.arange(d, dtype=np.uint32) if d <= n_eval else rng.integers(0, d, size=n_eval).astype(np.uint32)
                got = t.lbp_marginals(y, x, states)
                ref = lp[states]
                fin = np.isfinite(ref)
                assert np.array_equal(np.isfinite(got), fin)
                assert np.allclose(got[fin], ref[fin], rtol=0, atol=1e-9 * max(1.0, np.abs(ref[fin]).max()))
                # selection: same log-probabilities rank by rank; same states wherever the neighbouring gaps are resolved
                st_ref, lp_ref = lbp.select(m, nu, y, x, K)
                st_got, lp_got = t.lbp_select(y, x, K)
                assert st_got.size == min(K, d)
                assert np.allclose(lp_got, lp_ref, rtol=0, atol=1e-9 * max(1.0, np.abs(lp_ref).max()))
                gap = 1e-8
                for r in range(st_got.size):
                    lo = r == 0 or lp_ref[r - 1] - lp_ref[r] > gap
                    hi = r == st_got.size - 1 or lp_ref[r] - lp_ref[r + 1] > gap
                    if lo and hi and r < st_got.size - 1:
                        assert st_got[r] == st_ref[r], (y, x, r)
                assert np.allclose(t.lbp_marginals(y, x, st_got), lp_got, rtol=0, atol=1e-9 * max(1.0, np.abs(lp_got).max()))
        t.set_beta(beta)                                            # a new beta drops the messages
        with pytest.raises(tnb.TnError):
            t.lbp_message(0, 0, 0)


CASES = [  # (Ly, Lx, S, n_s, p_keep, seed, beta, iterations, K)
    (2, 2, 3, 2, 1.0, 4, 0.9, 2, 5),            # all three kinds of inter-cell couplings
    (3, 3, 3, 4, 0.9, 4, 1.0, 5, 64),           # Pegasus-shaped miniature, ragged projectors, 4096 states per cell
    (3, 4, 2, 4, 0.9, 11, 1.3, 7, 300),         # Zephyr-shaped miniature, K > 256 states of a cell
    (4, 4, 1, 4, 1.0, 6, 2.0, 6, 16),           # one sub-cluster per cell (config-1 shape): K = d
    (5, 5, 1, 1, 1.0, 2, 1.0, 10, 2),           # square lattice, one spin per site
    (1, 4, 2, 2, 1.0, 9, 1.3, 0, 4),            # zero iterations: uniform messages, p ~ w
    (3, 3, 2, 8, 0.97, 3, 2.0, 4, 1000),        # full 8-spin sub-clusters: 65536 states per cell, radix selection
]


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta,iters,K", CASES)
def test_lbp_parity(Ly, Lx, S, ns, p, seed, beta, iters, K):
    _compare(instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed), beta, iters, K)


def test_lbp_on_a_tree_is_exact_on_the_gpu_too():
    """The oracle's pin (LBP is exact on trees) carried over: after parity with the oracle on the star of
    Pegasus-shaped cells the CUDA marginals ARE the brute-force marginals; checked directly on the normalisation."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(1, 4, 2, 2, p_keep=1.0, seed=9)
    with tnb.TensorNetwork(inst) as t:
        t.set_beta(1.3)
        t.lbp(3)
        for x in range(4):
            lp = t.lbp_marginals(0, x, np.arange(16, dtype=np.uint32))
            assert abs(np.exp(lp).sum() - 1.0) <= 1e-12
    _compare(inst, 1.3, 3, 16)


@pytest.mark.slow
def test_lbp_full_pegasus_cell():
    """2 x 2 cells of 24 spins: the sum of Eq. (11) runs over 2^24 states per message in the oracle, over the chain
    A - B - C_lo - C_hi on the device; the top-K selection works on all 2^24 marginals of a cell."""
    _compare(instances.lattice(2, 2, 3, 8, p_keep=0.97, seed=5), 1.0, 3, 4096, n_eval=20000)
