"""GPU parity / property tests at the BASELINE.json sizes, in the launch configuration bench.py times.

configs[1] (Zephyr-shaped 6x6x16) is still within reach of the dense CPU oracle, so it is compared element by element.
The real Pegasus cell shape (2^24 states per cell, 4096-dimensional MPO bonds, mediating tensors with the diagonal
legs) is compared with the oracle on a 2x2 lattice.  configs[2] and configs[4] at full size are beyond the oracle
(a dense Theta SVD per chain position); they are checked through properties that hold at any size."""
import numpy as np
import pytest

import instances
from oracle import energy

from test_gpu_parity import compare, mps_overlap

pytestmark = pytest.mark.gpu


def _tn(inst):
    import paper_2411_16431_b200 as tnb
    return tnb.TensorNetwork(inst)


@pytest.mark.slow
def test_config2_full_size_parity():
    inst, run = instances.config(1)
    st = compare(inst, run["beta"][0], run["D"], run["sweeps"], run["M"], 1e-6)
    assert st["theta_apply_calls"] > 0 and st["kernel_launches"] > 1000


@pytest.mark.slow
def test_pegasus_cell_shape_parity():
    """2 x 2 cells of 24 spins (3 sub-clusters of 8): d = 2^24 per cell, thinned edges, D = 4, one pass."""
    inst = instances.lattice(2, 2, 3, 8, p_keep=0.97, seed=5)
    compare(inst, 1.0, 4, 1, 8, 1e-6)


@pytest.mark.slow
def test_config2_fast_mode_against_converged_mode():
    """configs[1] at full size in the fast mode (TN_OPT_SVD_MODE = 1: seeded randomized SVD with 2 subspace iterations,
    PAPER.md:169-177) against the converged mode: fewer Theta applies, every R_y within the truncation error of the
    converged one, log Z within it, the same best energy."""
    import paper_2411_16431_b200 as tnb
    inst, run = instances.config(1)
    out = {}
    for mode in (0, 1):
        with _tn(inst) as t:
            t.set_option(tnb.OPT_SVD_MODE, mode)
            t.set_beta(run["beta"][0])
            t.contract(run["D"], run["sweeps"])
            rows = {y: t.mps(y) for y in range(1, inst.Ly)}
            lz = t.log_z()
            states, E, logp, pd = t.branch_and_bound(run["M"])
            out[mode] = (rows, lz, E, t.stats())
    trunc = out[0][3]["min_sigma_rel"]
    assert 0 < trunc < 1e-2
    for y in range(1, inst.Ly):
        assert 1 - abs(mps_overlap(out[0][0][y], out[1][0][y])) <= 100 * trunc ** 2
    assert abs(out[0][1] - out[1][1]) <= 10 * trunc * abs(out[0][1])
    assert out[0][2].min() == out[1][2].min()
    assert out[1][3]["theta_apply_calls"] < out[0][3]["theta_apply_calls"]
    assert out[1][3]["flop_theta_apply"] < 0.8 * out[0][3]["flop_theta_apply"]


def _properties(inst, states, E, logp, pd, M):
    assert states.shape == (M, inst.n_spins) and set(np.unique(states)) <= {-1, 1}
    assert np.array_equal(E, energy.energies(inst, states))            # bit-exact, fixed order (O-0)
    assert np.all(np.diff(logp) <= 0) and np.all(np.isfinite(logp)) and logp[0] < 0
    assert len({s.tobytes() for s in states}) == M                     # the beam never holds a state twice
    assert np.isfinite(pd) and pd < 0


def test_config5_full_size_properties():
    """Loop-planted 12x12 Zephyr-shaped instance: planted energy reached, +-s* degenerate, unit-norm boundary MPS."""
    inst, run = instances.config(4)
    with _tn(inst) as t:
        t.set_beta(run["beta"][0])
        t.contract(run["D"], run["sweeps"])
        for y in (1, inst.Ly // 2, inst.Ly - 1):
            R = t.mps(y)
            assert abs(mps_overlap(R, R) - 1.0) <= 1e-10                # <R_y|R_y> = 1 after the log-norm is removed
            assert max(max(a.shape[0], a.shape[2]) for a in R) <= run["D"]
        lz = t.log_z()
        states, E, logp, pd = t.branch_and_bound(run["M"])
        st = t.stats()
    _properties(inst, states, E, logp, pd, run["M"])
    assert E.min() == inst.E0                                           # integer couplings: exact
    assert energy.energies(inst, inst.s_star[None, :])[0] == inst.E0
    # h = 0: p(s) = p(-s); log Z bounds: ground-state term <= Z <= 2^N terms of at most that size
    beta, N = run["beta"][0], inst.n_spins
    assert -beta * inst.E0 + np.log(2) - 1e-6 <= lz <= -beta * inst.E0 + N * np.log(2)
    assert st["min_sigma_rel"] < 1e-6
    # beta = 4 on integer couplings: every bond is rank-deficient below D (nothing above 1e-14 sigma_1 is cut), so the
    # contraction is exact to rounding and the chain rule logp = -beta E - log Z holds at every returned state
    assert np.abs(logp + beta * E + lz).max() <= 1e-6 * abs(lz)


@pytest.mark.slow
def test_config3_full_size_properties():
    inst, run = instances.config(2)
    with _tn(inst) as t:
        t.set_beta(run["beta"][0])
        t.contract(run["D"], run["sweeps"])
        lz = t.log_z()
        states, E, logp, pd = t.branch_and_bound(run["M"])
        st = t.stats()
    _properties(inst, states, E, logp, pd, run["M"])
    beta = run["beta"][0]
    # every returned state is one term of Z:  log Z >= -beta E(s)  (up to the contraction error of a truncated MPS)
    assert lz >= -beta * E.min() - 1e-3 * abs(lz)
    # Chain rule at the returned states: exact marginals give logp = -beta E - log Z.  The product of conditionals
    # telescopes row by row, so the residual is a sum of Ly - 1 log-ratios of boundary-MPS amplitudes, each off by at
    # most the relative weight that row's worst cut discarded (min_sigma_rel = the largest smallest-retained sigma over
    # all bonds, Fig. 12(b); measured at this config: 4.2e-3, residual 7.7e-3 nats).
    resid = logp + beta * E + lz
    assert 0 < st["min_sigma_rel"] < 0.02
    assert np.abs(resid).max() <= 2 * (inst.Ly - 1) * st["min_sigma_rel"], (np.abs(resid).max(), st["min_sigma_rel"])


@pytest.mark.slow
def test_config5_droplets_at_full_size():
    """configs[4] (loop-planted 12x12 Zephyr-shaped, M = 1024) with merge + droplets: the run that exposed a shared-memory
    race in k_droplets at scale.  The merge leaves ONE main branch (the last cell has no boundary), it is a planted
    ground state, and every book-kept droplet is a real excitation: flipping its spins raises the energy by exactly
    dE (integer couplings; the beta = 4 contraction is exact to rounding), dE ascending, pairwise Hamming >= 2."""
    import paper_2411_16431_b200 as tnb
    inst, run = instances.config(4)
    beta = run["beta"][0]
    with _tn(inst) as t:
        for k, v in ((tnb.OPT_MERGE, 1), (tnb.OPT_DROPLETS, 1), (tnb.OPT_DROPLET_MAX_COUNT, 16),
                     (tnb.OPT_DROPLET_MAX_DE, 2.0), (tnb.OPT_DROPLET_MIN_HAMMING, 2)):
            t.set_option(k, v)
        t.set_beta(beta)
        t.contract(run["D"], run["sweeps"])
        states, E, logp, pd = t.branch_and_bound(run["M"])
        st = t.stats()
        dE, flips = t.droplets(0)
        assert states.shape[0] == 1 and E[0] == inst.E0
        assert len(dE) > 0 and np.all(np.diff(dE) >= -1e-9) and dE.max() <= 2.0 + 1e-9
        ex = (states[0][None, :].astype(np.int32) * (1 - 2 * flips.astype(np.int32))).astype(np.int8)
        Eex = t.energy(ex)
    assert np.array_equal(Eex, energy.energies(inst, ex))
    assert np.abs((Eex - E[0]) - dE).max() <= 1e-6
    for i in range(len(dE)):
        assert flips[i].sum() > 0
        for j in range(i):
            assert int((flips[i] != flips[j]).sum()) >= 2
    assert st["merge_fallback_cells"] <= 8               # counted, never silent (cells whose survivors exceed 2^20)
