"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

P-numbers follow SURVEY.md section 8(c) / DESIGN.md section 5.
"""
import os

import numpy as np
import pytest

import instances
from oracle import brute, energy, model, mps, search, transfer

GOLD = os.path.join(os.path.dirname(__file__), "golden", "cfg1_bruteforce.txt")

MINIS = [  # (Ly, Lx, S, n_s, p_keep, seed, beta): all small enough for brute force
    (2, 2, 3, 2, 0.8, 3, 1.3),      # Pegasus-shaped miniature (mediating tensors, thinned edges)
    (3, 2, 2, 2, 0.9, 5, 0.7),      # Zephyr-shaped miniature
    (2, 3, 1, 4, 1.0, 1, 1.5),      # config-1 shape, other seed
    (2, 3, 2, 2, 0.9, 7, 0.9),
]


def read_golden():
    lz, rows = None, []
    for line in open(GOLD):
        t = line.split()
        if t[0] == "log_z":
            lz = float(t[1])
        elif t[0] == "state":
            rows.append((int(t[1]), float(t[3])))
    return lz, rows


# ---------------------------------------------------------------- O-0 energy
def test_energy_fixed_order_matches_python_loop():
    inst = instances.lattice(2, 2, 3, 4, p_keep=0.9, seed=11)
    rng = np.random.default_rng(0)
    s = (1 - 2 * rng.integers(0, 2, size=(5, inst.n_spins))).astype(np.int8)
    Ev = energy.energies(inst, s)
    for k in range(5):
        assert Ev[k] == energy.energy(inst, s[k])          # bit-exact
    # independent closed evaluation: quadratic form (different summation order -> tolerance)
    A = np.zeros((inst.n_spins, inst.n_spins))
    A[inst.edge_u, inst.edge_v] += inst.J
    ref = np.einsum("ki,ij,kj->k", s.astype(float), A, s.astype(float)) + s @ inst.h
    assert np.allclose(Ev, ref, rtol=0, atol=1e-12)


def test_energy_hand_example():
    # two spins, one bond: H = J s0 s1 + h0 s0 + h1 s1
    inst = instances.Instance(n_spins=2, edge_u=np.array([0]), edge_v=np.array([1]), J=np.array([0.5]),
                              h=np.array([0.25, -1.0]))
    assert energy.energy(inst, [1, 1]) == 0.5 + 0.25 - 1.0
    assert energy.energy(inst, [1, -1]) == -0.5 + 0.25 + 1.0
    assert energy.energy(inst, [-1, -1]) == 0.5 - 0.25 + 1.0


# ---------------------------------------------------------------- P1: brute force == exact transfer
def test_cfg1_bruteforce_matches_golden_and_transfer(cfg1):
    inst, run, E = cfg1
    beta = run["beta"][0]
    lz_gold, rows = read_golden()
    assert abs(brute.log_z(E, beta) - lz_gold) <= 1e-13 * abs(lz_gold)
    idx, El = brute.lowest(E, 16)
    assert [k for k, _ in rows] == idx.tolist()
    s = brute.index_to_spins(idx, inst.n_spins)
    assert np.allclose(energy.energies(inst, s), [e for _, e in rows], rtol=0, atol=1e-12)
    m = model.Model(inst).set_beta(beta)
    lz, _ = transfer.log_z(m)
    assert abs(lz - lz_gold) <= 1e-12 * abs(lz_gold)


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta", MINIS)
def test_transfer_matches_bruteforce(Ly, Lx, S, ns, p, seed, beta):
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    E = brute.all_energies(inst)
    m = model.Model(inst).set_beta(beta)
    lz, _ = transfer.log_z(m)
    assert abs(lz - brute.log_z(E, beta)) <= 1e-12 * abs(lz)


# ---------------------------------------------------------------- sparse diagrams == explicit MPO
@pytest.mark.parametrize("S,ns", [(1, 4), (2, 2), (3, 2)])
def test_sparse_diagrams_match_dense_mpo(S, ns):
    inst = instances.lattice(2, 3, S, ns, p_keep=0.85, seed=2)
    m = model.Model(inst).set_beta(0.8)
    rng = np.random.default_rng(1)
    for y in range(2):
        for pos in mps.row_positions(m, y):
            W = pos.dense()
            wl, pu, pd, wr = W.shape
            g, al, ar, g2 = 3, 2, 4, 5
            L = rng.normal(size=(g, wl, al))
            A = rng.normal(size=(al, pd, ar))
            R = rng.normal(size=(g2, wr, ar))
            N = rng.normal(size=(g, pu, g2))
            assert np.allclose(pos.update(L, A, R), np.einsum("gwa,wpdv,adb,hvb->gph", L, W, A, R), atol=1e-11)
            assert np.allclose(pos.env_left(L, A, N), np.einsum("gwa,gph,wpdv,adb->hvb", L, N, W, A), atol=1e-11)
            assert np.allclose(pos.env_right(R, A, N), np.einsum("gph,wpdv,adb,hvb->gwa", N, W, A, R), atol=1e-11)
            th = np.einsum("adb,wpdv,hvb->awph", A, W, R).reshape(al * wl, pu * g2)
            assert np.allclose(pos.theta(A, R), th, atol=1e-11)


# ---------------------------------------------------------------- P2: exact-D MPS == exact transfer
def _dense_of_mps(m, T, shape):
    v = mps.mps_to_dense(T)
    if m.has_med:
        n = m.Lx
        v = np.transpose(v, [2 * x for x in range(n)] + [2 * x + 1 for x in range(n - 1)])
    return v.reshape(shape)


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta", MINIS + [(3, 3, 3, 2, 0.85, 7, 0.9)])
def test_exact_mps_reproduces_transfer_vectors(Ly, Lx, S, ns, p, seed, beta):
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    m = model.Model(inst).set_beta(beta)
    _, R = transfer.log_z(m)
    Rm, ln = mps.contract(m, 0, 0)
    acc = 0.0
    for y in range(Ly - 1, 0, -1):
        acc += ln[y]
        arr, ls = R[y]
        v = _dense_of_mps(m, Rm[y], arr.shape)
        assert abs(1 - abs((arr / np.linalg.norm(arr) * v).sum())) < 1e-12
        assert abs(acc - (ls + np.log(np.linalg.norm(arr)))) < 1e-12 * max(1.0, abs(acc))


# ---------------------------------------------------------------- P3: beam at exact D == exact-marginal beam
@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta", MINIS)
def test_beam_exact_D_matches_exact_marginal_beam(Ly, Lx, S, ns, p, seed, beta):
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    E = brute.all_energies(inst)
    lzb = brute.log_z(E, beta)
    m = model.Model(inst).set_beta(beta)
    Rm, ln = mps.contract(m, 0, 0)
    out = search.branch_and_bound(m, Rm, ln, 8)
    ref = search.exact_marginal_beam(m, E, 8)
    assert abs(out["log_z"] - lzb) <= 1e-12 * abs(lzb)
    assert np.array_equal(out["states"], ref["states"])
    assert np.allclose(out["logp"], ref["logp"], rtol=0, atol=1e-10)
    assert abs(out["log_pd"] - ref["log_pd"]) < 1e-10
    assert np.array_equal(out["energies"], ref["energies"])
    # final log-probabilities are Boltzmann: log p(s) = -beta E(s) - log Z   (Eq. (6))
    assert np.allclose(out["logp"], -beta * out["energies"] - lzb, rtol=0, atol=1e-10)
    # conditionals are normalised: sum over the d candidates of one parent (checked through P6's
    # identity: the kept log-probabilities never exceed 0 and p_d is a probability)
    assert out["logp"].max() <= 1e-12 and out["log_pd"] <= 1e-12


def test_cfg1_beam_against_golden(cfg1):
    """Config 1 at its stated settings (beta = 1, exact D, M = 16).  S12: the beam ranks by marginal
    probability, so equality with the brute-force lowest-16 is not a theorem; the ground state and
    the Boltzmann identity are."""
    inst, run, E = cfg1
    beta = run["beta"][0]
    lz_gold, rows = read_golden()
    m = model.Model(inst).set_beta(beta)
    Rm, ln = mps.contract(m, 0, 0)
    out = search.branch_and_bound(m, Rm, ln, run["M"])
    assert abs(out["log_z"] - lz_gold) <= 1e-12 * abs(lz_gold)
    assert abs(out["energies"].min() - rows[0][1]) < 1e-12
    assert np.array_equal(out["states"][0], brute.index_to_spins(np.array([rows[0][0]]), inst.n_spins)[0])
    assert np.allclose(out["logp"], -beta * out["energies"] - lz_gold, atol=1e-10)
    ref = search.exact_marginal_beam(m, E, run["M"])
    assert np.array_equal(out["states"], ref["states"])


# ---------------------------------------------------------------- P4: closed forms (lattices too big for brute force)
def _logz_mps(inst, beta, D=8, sweeps=1):
    m = model.Model(inst).set_beta(beta)
    Rm, ln = mps.contract(m, D, sweeps)
    return search.branch_and_bound(m, Rm, ln, 4)["log_z"]


@pytest.mark.parametrize("S,ns", [(2, 4), (3, 2)])
def test_closed_form_zero_couplings(S, ns):
    inst = instances.lattice(3, 3, S, ns, p_keep=0.9, seed=4)
    inst["J"] = np.zeros_like(inst.J)
    beta = 0.7
    ref = np.log(2 * np.cosh(beta * inst.h)).sum()
    assert abs(_logz_mps(inst, beta) - ref) <= 1e-12 * abs(ref)


@pytest.mark.parametrize("S,ns", [(2, 4), (3, 2)])
def test_closed_form_tree(S, ns):
    """Spanning forest of the lattice graph, h = 0:  Z = 2^(#components) ... = 2^N prod cosh(beta J_e)."""
    inst = instances.lattice(3, 3, S, ns, p_keep=1.0, seed=6, h="zero")
    parent = list(range(inst.n_spins))

    def find(a):
        while parent[a] != a:
            parent[a] = parent[parent[a]]
            a = parent[a]
        return a
    keep = []
    for e, (u, v) in enumerate(zip(inst.edge_u.tolist(), inst.edge_v.tolist())):
        ru, rv = find(u), find(v)
        if ru != rv:
            parent[ru] = rv
            keep.append(e)
    for k in ("edge_u", "edge_v", "J"):
        inst[k] = inst[k][keep]
    beta = 0.9
    ref = inst.n_spins * np.log(2.0) + np.log(np.cosh(beta * inst.J)).sum()
    assert abs(_logz_mps(inst, beta, D=16) - ref) <= 1e-11 * abs(ref)


def test_small_beta_expansion():
    """log Z = N log 2 + beta^2/2 (sum J^2 + sum h^2) + O(beta^3)."""
    inst = instances.lattice(3, 3, 2, 4, p_keep=0.95, seed=8)
    beta = 1e-3
    ref = inst.n_spins * np.log(2.0) + 0.5 * beta ** 2 * ((inst.J ** 2).sum() + (inst.h ** 2).sum())
    got = _logz_mps(inst, beta)
    assert abs(got - ref) < 50 * beta ** 3 * (np.abs(inst.J).sum() + np.abs(inst.h).sum())
    assert abs(got - inst.n_spins * np.log(2.0)) > 0.4 * (ref - inst.n_spins * np.log(2.0))


# ---------------------------------------------------------------- P5: invariances
def test_gauge_invariance_and_z2():
    inst = instances.lattice(2, 3, 2, 2, p_keep=0.9, seed=9)
    beta, M = 1.1, 12
    m = model.Model(inst).set_beta(beta)
    Rm, ln = mps.contract(m, 0, 0)
    out = search.branch_and_bound(m, Rm, ln, M)
    g = np.where(np.random.default_rng(5).random(inst.n_spins) < 0.5, -1.0, 1.0)
    inst2 = instances.Instance(inst)
    inst2["J"] = inst.J * g[inst.edge_u] * g[inst.edge_v]
    inst2["h"] = inst.h * g
    m2 = model.Model(inst2).set_beta(beta)
    R2, ln2 = mps.contract(m2, 0, 0)
    out2 = search.branch_and_bound(m2, R2, ln2, M)
    assert abs(out["log_z"] - out2["log_z"]) < 1e-11
    assert np.allclose(np.sort(out["energies"]), np.sort(out2["energies"]), atol=1e-11)
    a = {tuple(r) for r in (out["states"] * g.astype(np.int8)).tolist()}
    b = {tuple(r) for r in out2["states"].tolist()}
    assert a == b
    # h = 0  =>  p(s) = p(-s): the returned list is closed under global flip (M even, no pruning ties)
    inst3 = instances.lattice(2, 2, 2, 2, p_keep=1.0, seed=10, h="zero")
    m3 = model.Model(inst3).set_beta(0.8)
    R3, ln3 = mps.contract(m3, 0, 0)
    o3 = search.branch_and_bound(m3, R3, ln3, 1 << 16)
    lp = {tuple(r): l for r, l in zip(o3["states"].tolist(), o3["logp"].tolist())}
    for r, l in list(lp.items())[:200]:
        assert abs(lp[tuple(-np.array(r))] - l) < 1e-10


# ---------------------------------------------------------------- P7: no-prune beam == brute-force ordering
def test_no_prune_beam_equals_bruteforce_order():
    inst = instances.lattice(2, 2, 1, 4, p_keep=1.0, seed=12)           # N = 16, d^n = 65536
    beta = 1.0
    E = brute.all_energies(inst)
    m = model.Model(inst).set_beta(beta)
    Rm, ln = mps.contract(m, 0, 0)
    out = search.branch_and_bound(m, Rm, ln, 1 << 16)
    assert out["states"].shape[0] == 1 << 16
    idx, El = brute.lowest(E, 64)
    assert np.allclose(out["energies"][:64], El, rtol=0, atol=1e-12)
    k = (((1 - out["states"][:64].astype(np.int64)) // 2) << np.arange(16)).sum(axis=1)
    gaps = np.diff(El)
    for r in range(64):
        if (r == 0 or gaps[r - 1] > 1e-9) and (r == 63 or gaps[r] > 1e-9):
            assert k[r] == idx[r]
    assert out["log_pd"] == -np.inf


DEGENERATE = [  # (Ly, Lx, S, n_s, p_keep, seed, beta, h): shapes where pieces of the network disappear
    (1, 3, 2, 2, 1.0, 1, 1.0, "uniform"),      # one row: no boundary MPS
    (1, 1, 3, 2, 1.0, 1, 1.0, "uniform"),      # one cell
    (3, 1, 2, 2, 1.0, 2, 1.0, "uniform"),      # one column: all bonds 1
    (1, 3, 3, 2, 0.9, 3, 0.8, "uniform"),      # one row, mediating positions
    (3, 1, 3, 2, 0.9, 3, 0.8, "uniform"),
    (2, 2, 2, 2, 0.0, 5, 1.0, "uniform"),      # no couplings
    (2, 2, 2, 2, 0.9, 6, 6.0, "uniform"),      # cold
]


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta,h", DEGENERATE)
def test_degenerate_shapes_against_bruteforce(Ly, Lx, S, ns, p, seed, beta, h):
    """log Z, the probabilities of the kept states and the discarded mass against plain enumeration."""
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed, h=h)
    E = brute.all_energies(inst)
    lz = brute.log_z(E, beta)
    m = model.Model(inst).set_beta(beta)
    Rm, ln = mps.contract(m, 0, 0)
    M = 8
    out = search.branch_and_bound(m, Rm, ln, M)
    assert abs(out["log_z"] - lz) <= 1e-12 * abs(lz)
    # every returned state carries its exact Boltzmann probability
    assert np.allclose(out["logp"], -beta * energy.energies(inst, out["states"]) - lz, rtol=0, atol=1e-10)
    assert np.all(np.diff(out["logp"]) <= 1e-12)                       # ranks are sorted
    if inst.n_spins > 12:
        return
    # with no pruning the list is the brute-force order and nothing is discarded
    full = search.branch_and_bound(m, Rm, ln, 1 << inst.n_spins)
    assert full["states"].shape[0] == 1 << inst.n_spins and full["log_pd"] == -np.inf
    idx, El = brute.lowest(E, M)
    assert np.allclose(full["energies"][:M], El, rtol=0, atol=1e-12)


def test_uniform_distribution_closed_form():
    """H = 0: Z = 2^N, every state has log p = -N log 2, the beam discards 1 - M 2^-N exactly."""
    inst = instances.lattice(2, 2, 2, 2, p_keep=0.0, seed=5, h="zero")
    m = model.Model(inst).set_beta(1.0)
    Rm, ln = mps.contract(m, 0, 0)
    out = search.branch_and_bound(m, Rm, ln, 16)
    N = inst.n_spins
    assert abs(out["log_z"] - N * np.log(2.0)) < 1e-12
    assert np.allclose(out["logp"], -N * np.log(2.0), rtol=0, atol=1e-12)
    assert len({tuple(r) for r in out["states"].tolist()}) == 16


# ---------------------------------------------------------------- P8: loop-planted ground state
@pytest.mark.parametrize("seed", [0, 1])
def test_loop_planted_ground_state(seed):
    inst = instances.loop_planted(2, 3, 1, 4, seed=seed)                # N = 24
    E = brute.all_energies(inst)
    assert abs(E.min() - inst.E0) < 1e-12
    assert energy.energy(inst, inst.s_star) == inst.E0
    assert energy.energy(inst, -inst.s_star) == inst.E0
    assert np.all((inst.loop_lengths >= 4) & (inst.loop_lengths <= 8))
    m = model.Model(inst).set_beta(2.0)
    Rm, ln = mps.contract(m, 0, 0)
    out = search.branch_and_bound(m, Rm, ln, 16)
    assert out["energies"].min() == inst.E0


def test_loop_planted_zephyr_shape_energy_of_planted_state():
    inst = instances.loop_planted(3, 3, 2, 8, seed=0)
    assert energy.energy(inst, inst.s_star) == inst.E0


# ---------------------------------------------------------------- lattice transformations
@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed", [(2, 3, 2, 2, 0.85, 4), (3, 2, 1, 4, 0.9, 6)])
def test_lattice_transformations_leave_exact_results_unchanged(Ly, Lx, S, ns, p, seed):
    """The 8 transformations only re-index the cluster map: brute force (which never looks at the map) fixes
    log Z and the low-energy states; the exact contraction on every transformed map must reproduce them, and the
    exact-D beam must return the same states (energies bit-exact, spins in the original ids)."""
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    beta = 1.1
    Eall = brute.all_energies(inst)                          # N = 24: 2^24 states
    lz = brute.log_z(Eall, beta)
    idx, El = brute.lowest(Eall, 8)
    assert np.diff(El).min() > 1e-9                          # unique order
    ref_states = brute.index_to_spins(idx, inst.n_spins)
    maps = set()
    for t in range(8):
        it = instances.transformed(inst, t)
        assert np.array_equal(it.edge_u, inst.edge_u) and np.array_equal(it.J, inst.J)
        maps.add((it.Ly, it.Lx, it.cell_y.tobytes(), it.cell_x.tobytes(), it.sub.tobytes(), it.pos.tobytes()))
        m = model.Model(it).set_beta(beta)
        R, ln = mps.contract(m, 0, 0)
        out = search.branch_and_bound(m, R, ln, 8)
        assert abs(out["log_z"] - lz) <= 1e-12 * abs(lz), t
        # beta = 1.1, M = 8: the beam may prune a low-energy state; the ground state it must keep
        assert np.array_equal(out["states"][0], ref_states[0]), t
        assert np.array_equal(out["energies"], energy.energies(inst, out["states"])), t
        # the beam content depends on the search order (that is why the paper runs all 8), but at exact D
        # every state it returns carries its exact Boltzmann log-probability, which brute force fixes
        assert np.allclose(out["logp"], -beta * out["energies"] - lz, rtol=0, atol=1e-10), t
    assert len(maps) == 8                                    # the eight maps are distinct
    with pytest.raises(ValueError):
        instances.transformed(instances.lattice(2, 2, 3, 2), 1)


# ---------------------------------------------------------------- P10-P12: compress
def _row_problem(seed=3, D=4):
    inst = instances.lattice(3, 4, 2, 2, p_keep=0.9, seed=seed)
    m = model.Model(inst).set_beta(0.9)
    Rex, _ = mps.contract(m, 0, 0)
    return m, Rex


def test_compress_gauge_independent_and_monotone():
    m, Rex = _row_problem()
    y = 1
    pos = mps.row_positions(m, y)
    A = Rex[y + 1]
    rng = np.random.default_rng(2)
    A2 = [a.copy() for a in A]
    for j in range(len(A) - 1):                       # random invertible gauge on every bond
        b = A2[j].shape[2]
        G = rng.normal(size=(b, b)) + 2 * np.eye(b)
        A2[j] = np.einsum("apb,bc->apc", A2[j], G)
        A2[j + 1] = np.einsum("ab,bpc->apc", np.linalg.inv(G), A2[j + 1])
    exact = mpo_dense = mps.mpo_mps_dense(pos, A)
    exact = exact / np.linalg.norm(exact)
    fid = {}
    for sweeps in (0, 1, 2):
        st = {}
        N1, l1 = mps.compress(pos, A, 3, sweeps, stats=st)
        N2, l2 = mps.compress(pos, A2, 3, sweeps)
        v1, v2 = mps.mps_to_dense(N1), mps.mps_to_dense(N2)
        assert abs(1 - abs((v1 * v2).sum())) < 1e-10                 # P10
        assert abs(l1 - l2) < 1e-10
        fid[sweeps] = abs((v1 * exact).sum())
        for k in range(0, len(st["pass_norms"][0]), len(pos)):       # P11: norm non-decreasing in a pass
            nrm = st["pass_norms"][0][k:k + len(pos)]
            assert all(b >= a * (1 - 1e-12) for a, b in zip(nrm, nrm[1:]))
    assert fid[1] >= fid[0] - 1e-12 and fid[2] >= fid[1] - 1e-12     # P11: passes do not lower fidelity
    assert fid[0] < 1 - 1e-9                                         # the cut really truncates


def test_compress_fidelity_obeys_eckart_young():
    """Any MPS with bond <= D across a cut has overlap with the unit-norm exact row vector of at most
    sqrt(sum of the D largest sigma^2 of the exact vector's unfolding at that cut) (Eckart-Young, the bound behind
    'truncating the bond dimension'); the variational passes must come within a
    modest factor of the best single-cut infidelity.  Also: the returned bonds really are <= D, the result has
    unit norm, and exp(log-norm) is the norm of the projection of the exact vector on it up to the cut's error."""
    m, Rex = _row_problem()
    y = 1
    pos = mps.row_positions(m, y)
    exact = mps.mpo_mps_dense(pos, Rex[y + 1])
    nex = np.linalg.norm(exact)
    v = exact / nex
    dims = v.shape
    for D in (2, 3, 4):
        cap = 1.0
        for cut in range(1, len(dims)):                         # unfolding: positions < cut | positions >= cut
            sv = np.linalg.svd(v.reshape(int(np.prod(dims[:cut])), -1), compute_uv=False)
            cap = min(cap, float(np.sqrt((sv[:D] ** 2).sum())))
        for sweeps in (0, 2):
            st = {}
            N, ln = mps.compress(pos, Rex[y + 1], D, sweeps, stats=st)
            assert max(st["bonds"][0][:-1]) <= D and st["bonds"][0][-1] == 1
            w = mps.mps_to_dense(N)
            assert abs(np.linalg.norm(w) - 1) < 1e-12
            fid = abs((w * v).sum())
            assert fid <= cap + 1e-12
            if sweeps == 2:                                      # near-optimal: within 4x of the single-cut bound
                assert 1 - fid <= 4 * len(dims) * (1 - cap) + 1e-12
                # one-site variational optimum: the centre tensor is the projection, so norm = <w|exact>
                assert abs(np.exp(ln) - abs((w * exact).sum())) <= 1e-9 * nex


def test_compress_large_D_equals_exact():
    m, Rex = _row_problem()
    y = 1
    pos = mps.row_positions(m, y)
    N0, l0 = mps.compress(pos, Rex[y + 1], 0, 0)
    N1, l1 = mps.compress(pos, Rex[y + 1], 64, 2)                    # P12
    v0, v1 = mps.mps_to_dense(N0), mps.mps_to_dense(N1)
    assert abs(1 - abs((v0 * v1).sum())) < 1e-12 and abs(l0 - l1) < 1e-12
    ex = mps.mpo_mps_dense(pos, Rex[y + 1])
    assert abs(1 - abs((v0 * ex).sum()) / np.linalg.norm(ex)) < 1e-12
    assert abs(l0 - np.log(np.linalg.norm(ex))) < 1e-12


def test_truncate_rank_rules():
    s = np.array([1.0, 0.5, 0.25, 0.25 * (1 - 1e-9), 1e-3, 1e-15, 0.0])
    assert mps.truncate_rank(s, 0) == 5                 # S6: drops <= 1e-14 sigma_1
    assert mps.truncate_rank(s, 3) == 2                 # S5: does not split the degenerate pair
    assert mps.truncate_rank(s, 3, gap_guard=False) == 3
    assert mps.truncate_rank(s, 4) == 4
    assert mps.truncate_rank(np.zeros(3), 2) == 1


def test_truncated_marginals_close_to_exact():
    """Truncated D: conditionals still sum to 1 (logp <= 0) and log Z stays within the truncation error."""
    inst = instances.lattice(3, 3, 2, 4, p_keep=0.95, seed=13)
    m = model.Model(inst).set_beta(1.0)
    Rex, lex = mps.contract(m, 0, 0)
    ex = search.branch_and_bound(m, Rex, lex, 16)
    st = {}
    Rt, lt = mps.contract(m, 4, 2, stats=st)
    tr = search.branch_and_bound(m, Rt, lt, 16)
    assert abs(tr["log_z"] - ex["log_z"]) < 1e-3 * abs(ex["log_z"])
    assert tr["energies"].min() == ex["energies"].min()
    assert max(st["min_sigma"]) < 1.0


# ---------------------------------------------------------------- merge by boundary (Fig. 3(d))
@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta", MINIS)
def test_merge_by_boundary_never_loses_the_most_probable_state(Ly, Lx, S, ns, p, seed, beta):
    """Two prefixes with the same boundary have identical futures (Eqs. (8)-(9) PAPER.md:100-107), so dropping the
    less probable one cannot lose the most probable full state: with merging on and no pruning by the bound
    (M >= number of boundaries) the first returned state is the brute-force ground state with its exact logp,
    while the number of kept prefixes stays far below the unmerged beam."""
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    E = brute.all_energies(inst)
    m = model.Model(inst).set_beta(beta)
    R, ln = mps.contract(m, 0, 0)
    M = 1 << 14
    st = {}
    out = search.branch_and_bound(m, R, ln, M, stats=st, merge=True)
    idx, El = brute.lowest(E, 1)
    gs = brute.index_to_spins(idx, inst.n_spins)[0]
    assert np.array_equal(out["states"][0], gs)
    lz = brute.log_z(E, beta)
    assert abs(out["logp"][0] - (-beta * El[0] - lz)) <= 1e-10 * abs(lz)
    assert st["merged_away"] > 0
    # every survivor is exact too, and no two survivors share a boundary with a better twin: logp = -beta E - log Z
    assert np.allclose(out["logp"], -beta * out["energies"] - lz, rtol=0, atol=1e-9 * abs(lz))
    # without merging the same M gives the same best state (pruning never triggers on these sizes or keeps it)
    ref = search.branch_and_bound(m, R, ln, M)
    assert np.array_equal(ref["states"][0], gs)
    assert out["logp"].size < ref["logp"].size or ref["logp"].size < M


def test_merge_groups_are_boundaries():
    """Survivors of one merge step have pairwise different boundaries; a merged-away candidate has a survivor
    with the same boundary and a score at least as large."""
    inst = instances.lattice(2, 3, 2, 2, p_keep=0.9, seed=7)
    m = model.Model(inst).set_beta(0.9)
    beam = [[3, 1, 0], [5, 1, 0], [3, 9, 2]]                     # three prefixes covering row 0
    pk, sc = search.boundary_codes(m, 1, 0, beam)
    d = m.cells[1][0].d
    rng = np.random.default_rng(3)
    score = rng.standard_normal(len(beam) * d)
    parent = np.repeat(np.arange(len(beam)), d)
    state = np.tile(np.arange(d), len(beam))
    surv = search.merge_by_boundary(score, parent, state, pk, sc)
    key = pk[parent] * (sc.max() + 1) + sc[state]
    assert np.unique(key[surv]).size == surv.size == np.unique(key).size
    best = {}
    for k, s_ in zip(key.tolist(), score.tolist()):
        best[k] = max(best.get(k, -np.inf), s_)
    assert all(score[i] == best[key[i]] for i in surv)


# ---------------------------------------------------------------- f2: paper-preferred schedule, randomized SVD, 2 chi -> chi
def test_hash_uniform_is_splitmix64():
    """The random block of the randomized SVD comes from SplitMix64's output function (public-domain reference
    implementation by S. Vigna; its first output for state 0 is the published test vector 0xE220A8397B1DCDAF) applied
    to a counter made of (seed, p', gamma, column): reproducible, layout-free, uniform on (-1, 1)."""
    u0 = mps.hash_uniform(0, 1, 1, 1)[0, 0]
    assert u0 == 2.0 * ((0xE220A8397B1DCDAF >> 11) * (1.0 / 9007199254740992.0)) - 1.0
    # counter arithmetic against plain Python integers (instances.SplitMix64 is the same generator, written with ints)
    seed, p, g, c = 7, 3, 5, 4
    U = mps.hash_uniform(seed, p, g, c)
    for (pp, gg, cc) in ((0, 0, 0), (2, 4, 3), (1, 0, 2)):
        ctr = (seed * 0x100000001B3 + ((pp * 4096 + gg) * 1024 + cc)) & ((1 << 64) - 1)
        ref = instances.SplitMix64(ctr)               # state = counter: next_u64 adds the golden gamma and mixes
        assert U[pp * g + gg, cc] == 2.0 * ((ref.next_u64() >> 11) * (1.0 / 9007199254740992.0)) - 1.0
    big = mps.hash_uniform(3, 64, 32, 48)
    assert np.all(np.abs(big) < 1) and abs(big.mean()) < 5e-3 and abs(big.var() - 1 / 3) < 5e-3
    assert np.array_equal(big, mps.hash_uniform(3, 64, 32, 48)) and not np.array_equal(big, mps.hash_uniform(4, 64, 32, 48))


def test_randomized_svd_ritz_values_interlace_and_converge():
    """Randomized range finder + subspace iteration (refs [43, 44]): the returned V is orthonormal, the
    Ritz values never exceed the true singular values (Cauchy interlacing for a compression of Theta), approach them
    from below as the number of iterations grows, and with enough iterations the retained subspace is LAPACK's."""
    rng = np.random.default_rng(5)
    pu, g, m = 12, 6, 90
    U, _ = np.linalg.qr(rng.normal(size=(m, pu * g)))
    W, _ = np.linalg.qr(rng.normal(size=(pu * g, pu * g)))
    sv = 0.7 ** np.arange(pu * g)
    Th = (U * sv) @ W.T
    k, ks = 8, 8 + 6
    prev = None
    for iters in (1, 2, 4, 40):
        V, s = mps.randomized_svd(Th, pu, g, ks, iters, seed=11)
        assert np.abs(V.T @ V - np.eye(ks)).max() < 1e-12
        assert np.all(s <= sv[:ks] * (1 + 1e-12))
        if prev is not None:
            assert np.all(s[:k] >= prev[:k] * (1 - 1e-12))
        prev = s
    assert np.allclose(s[:k], sv[:k], rtol=1e-10)
    P = V[:, :k] @ V[:, :k].T
    assert np.abs(P - W[:, :k] @ W[:, :k].T).max() < 1e-8
    # one iteration already obeys the range-finder error bound in the spectral norm up to a modest factor
    V1, _ = mps.randomized_svd(Th, pu, g, ks, 1, seed=11)
    err = np.linalg.norm(Th - Th @ V1 @ V1.T, 2)
    assert sv[ks] * (1 - 1e-12) <= err <= 10 * sv[ks]


def test_truncate_mps_is_canonical_compression():
    """Second step of 2 chi -> chi: D >= every bond leaves the state unchanged; a real cut keeps unit norm, bonds <= D,
    loses at most sqrt(sum over bonds of the discarded Schmidt weight) (the textbook bound of canonical truncation) and
    never beats the single-cut Eckart-Young optimum."""
    rng = np.random.default_rng(9)
    dims = [(1, 3, 6), (6, 4, 6), (6, 3, 5), (5, 2, 1)]
    T = [rng.normal(size=d) * (0.5 ** np.arange(d[2]))[None, None, :] for d in dims]
    v = mps.mps_to_dense(T)
    nv = np.linalg.norm(v)
    T[0] = T[0] / nv
    v = v / nv
    same, ln0 = mps.truncate_mps(T, 8)
    assert abs(1 - abs((mps.mps_to_dense(same) * v).sum())) < 1e-12 and abs(ln0) < 1e-12
    for D in (2, 3):
        N, ln = mps.truncate_mps(T, D, gap_guard=False)
        w = mps.mps_to_dense(N)
        assert abs(np.linalg.norm(w) - 1) < 1e-12 and max(t.shape[2] for t in N) <= D
        fid = abs((w * v).sum())
        disc, cap = 0.0, 1.0
        for cut in range(1, len(dims)):
            sv = np.linalg.svd(v.reshape(int(np.prod(v.shape[:cut])), -1), compute_uv=False)
            disc += (sv[D:] ** 2).sum()
            cap = min(cap, np.sqrt((sv[:D] ** 2).sum()))
        assert fid <= cap + 1e-12
        assert np.linalg.norm(w * np.exp(ln) - v) <= np.sqrt(disc) * (1 + 1e-9) + 1e-12
        assert ln <= 1e-12


def test_interleaved_schedule_beats_plain_zipper():
    """a variational sweep after every zipper step is the paper's preferred schedule, 'a full zipper
    sweep first ... resulting in worse performance'.  On the P11 / P13 row problem: with no global pass the interleaved
    schedule has a higher fidelity with the exact MPO x MPS product than the plain zipper, a longer sweep range does
    not hurt, every variant respects the Eckart-Young cap, unit norm and bond <= D, and the two-step 2 chi -> chi
    truncation is at least as good as the one-step zipper."""
    m, Rex = _row_problem()
    y = 1
    pos = mps.row_positions(m, y)
    exact = mps.mpo_mps_dense(pos, Rex[y + 1])
    nex = np.linalg.norm(exact)
    v = exact / nex
    dims = v.shape

    def infid(D, sweeps, **kw):
        N, ln = mps.compress(pos, Rex[y + 1], D, sweeps, **kw)
        w = mps.mps_to_dense(N)
        assert abs(np.linalg.norm(w) - 1) < 1e-12 and max(t.shape[2] for t in N) <= D
        return 1 - abs((w * v).sum()), ln

    for D in (2, 3):
        cap = 1.0
        for cut in range(1, len(dims)):
            sv = np.linalg.svd(v.reshape(int(np.prod(dims[:cut])), -1), compute_uv=False)
            cap = min(cap, float(np.sqrt((sv[:D] ** 2).sum())))
        z0, _ = infid(D, 0)
        i1, _ = infid(D, 0, schedule=1, sweep_range=1)
        i3, _ = infid(D, 0, schedule=1, sweep_range=3)
        t0, _ = infid(D, 0, two_step=True)
        assert i1 < 0.2 * z0 and i3 <= i1 * (1 + 1e-9) and t0 < z0
        for f in (z0, i1, i3, t0):
            assert f >= (1 - cap) - 1e-12
        # with global passes on top every schedule lands at the same local optimum to the size of the truncation error
        z2, lz2 = infid(D, 2)
        i2, li2 = infid(D, 2, schedule=1, sweep_range=1)
        assert abs(i2 - z2) <= 0.5 * z2 and abs(li2 - lz2) <= 10 * z2
    # range 0 is the plain zipper; schedule 1 with exact D changes nothing
    assert infid(3, 1, schedule=1, sweep_range=0)[0] == infid(3, 1)[0]
    N0, l0 = mps.compress(pos, Rex[y + 1], 0, 0)
    N1, l1 = mps.compress(pos, Rex[y + 1], 0, 0, schedule=1, svd_mode=1, two_step=True)
    assert abs(1 - abs((mps.mps_to_dense(N0) * mps.mps_to_dense(N1)).sum())) < 1e-12 and abs(l0 - l1) < 1e-12


# ---------------------------------------------------------------- P6: consistency identity of the chain rule
@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta,M", [(3, 3, 2, 2, 0.9, 3, 1.1, 8), (2, 3, 3, 2, 0.85, 4, 0.8, 16),
                                                      (3, 2, 1, 4, 1.0, 5, 1.3, 8)])
def test_p6_consistency_identity(Ly, Lx, S, ns, p, seed, beta, M):
    """P6: at exact D the normaliser of a beam element at step n+1, sum_X u(m'; X), equals
    the kept unnormalised conditional of its parent at step n divided by the Boltzmann weights that step n already
    counted (the new cell's w and its edge factors to fixed neighbours), once every recorded scale factor (row
    log-norms, right-block and left-vector scales) is added back -- across cells of a row AND across row changes.
    A wrong scale bookkeeping, a dropped log-norm or a mis-indexed right block breaks it; 'conditionals sum to 1' does
    not see any of those."""
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    m = model.Model(inst).set_beta(beta)
    R, ln = mps.contract(m, 0, 0)
    trace = []
    out = search.branch_and_bound(m, R, ln, M, trace=trace)
    assert len(trace) == Ly * Lx
    # first step: the normaliser of the empty prefix is Z itself (without the table offsets)
    assert abs(trace[0]["log_z_abs"][0] - (out["log_z"] + m.beta * m.offset)) <= 1e-10 * abs(out["log_z"])
    for a, b in zip(trace[:-1], trace[1:]):
        # beam element i of step n+1 is kept candidate i of step n
        assert b["log_z_abs"].shape == a["kept_rest_abs"].shape
        assert np.allclose(b["log_z_abs"], a["kept_rest_abs"], rtol=0, atol=1e-9 * max(1.0, np.abs(b["log_z_abs"]).max()))
    # last step: nothing is left to sum over -- the rest of a complete configuration is 1
    assert np.abs(trace[-1]["kept_rest_abs"]).max() <= 1e-9


# ---------------------------------------------------------------- f1: droplets (Fig. 4)
@pytest.mark.parametrize("S,ns,seed,beta", [(2, 2, 3, 2.0), (1, 4, 8, 1.5)])
def test_droplets_are_the_connected_low_energy_excitations(S, ns, seed, beta):
    """Fig. 4: with exact marginals and no pruning the merge makes the ground state the main branch and
    the book-kept droplets are EXACTLY the singly connected excitations above it within max_dE -- checked against
    brute force over all 2^24 states: same flip sets, dE (from the ratio of marginals) = the exact energy difference
    (O-0), lowest droplet = first excited state; combinations of droplets give further states of the spectrum."""
    inst = instances.lattice(2, 3, S, ns, p_keep=1.0, seed=seed)
    assert inst.n_spins == 24
    m = model.Model(inst).set_beta(beta)
    R, ln = mps.contract(m, 0, 0)
    max_dE = 1.2
    out = search.branch_and_bound(m, R, ln, 4096, merge=True,
                                  droplets=dict(max_dE=max_dE, min_hamming=1, max_count=256))
    E_all = brute.all_energies(inst)
    gs = int(np.argmin(E_all))
    assert out["states"].shape[0] == 1                       # the last cell has no boundary: everything merges
    s0 = out["states"][0]
    bits = ((1 - s0.astype(np.int64)) // 2)
    assert int((bits << np.arange(24)).sum()) == gs and out["energies"][0] == E_all[gs]
    drops = out["droplets"][0]
    got = {}
    for dE, mask in drops:
        s1 = s0.copy()
        s1[mask] *= -1
        e1 = energy.energies(inst, s1[None])[0]
        assert abs(dE - (e1 - out["energies"][0])) <= 1e-9   # ratio of exact marginals = Boltzmann factor
        got[int((mask.astype(np.int64) << np.arange(24)).sum())] = dE
    # brute force: all states within max_dE whose difference from the ground state is one connected piece
    book = search.DropletBook(m)
    want = set()
    for idx in np.flatnonzero(E_all <= E_all[gs] + max_dE):
        diff = int(idx) ^ gs
        if diff == 0:
            continue
        sp = [i for i in range(24) if (diff >> i) & 1]
        todo, seen, inset = [sp[0]], {sp[0]}, set(sp)
        while todo:
            u = todo.pop()
            for v in book.adj[u]:
                if v in inset and v not in seen:
                    seen.add(v)
                    todo.append(v)
        if len(seen) == len(inset):
            want.add(diff)
    assert want and set(got) == want
    first_excited = np.partition(E_all, 1)[1] - E_all[gs]
    assert abs(min(got.values()) - first_excited) <= 1e-9
    # the filters: a large Hamming threshold keeps fewer, pairwise distant droplets; max_count caps the list
    far = search.branch_and_bound(m, R, ln, 4096, merge=True,
                                  droplets=dict(max_dE=max_dE, min_hamming=3, max_count=256))["droplets"][0]
    assert 0 < len(far) <= len(drops)
    for i in range(len(far)):
        for j in range(i):
            assert int((far[i][1] ^ far[j][1]).sum()) >= 3
    few = search.branch_and_bound(m, R, ln, 4096, merge=True,
                                  droplets=dict(max_dE=max_dE, min_hamming=1, max_count=3))["droplets"][0]
    assert [d for d, _ in few] == sorted(d for d, _ in drops)[:3]


# ---------------------------------------------------------------- f4 (partial): square lattice, one spin per site
def test_square_lattice_against_brute_force():
    """App. B PAPER.md:446-454 workload shape: S = 1, n_s = 1 (cells of a single spin, bond dimension 2 everywhere).
    P1 / P2 / P3 / P7 on a 4 x 5 lattice: log Z of the exact contraction = brute force, the no-prune beam returns the
    brute-force order, logp = -beta E - log Z."""
    inst = instances.lattice(4, 5, 1, 1, p_keep=1.0, seed=2)
    E_all = brute.all_energies(inst)
    m = model.Model(inst).set_beta(1.3)
    R, ln = mps.contract(m, 0, 0)
    out = search.branch_and_bound(m, R, ln, 1 << 12)
    lz = brute.log_z(E_all, 1.3)
    assert abs(out["log_z"] - lz) <= 1e-12 * abs(lz)
    low = np.sort(E_all)[:64]
    assert np.allclose(out["energies"][:64], low, rtol=0, atol=1e-12)
    assert np.allclose(out["logp"], -1.3 * out["energies"] - lz, rtol=0, atol=1e-9)


# ---------------------------------------------------------------- f4: LBP local dimensional reduction (Sec. IV)
def _brute_cell_marginals(inst, E_all, beta):
    nb = inst.S * inst.n_s
    ncell = inst.Ly * inst.Lx
    lw = -beta * (E_all - E_all.min())
    p = np.exp(lw)
    p /= p.sum()
    p = p.reshape((1 << nb,) * ncell)                    # axis 0 = LAST cell (highest bits)
    out = []
    for cidx in range(ncell):
        ax = tuple(a for a in range(ncell) if a != ncell - 1 - cidx)
        out.append(p.sum(axis=ax))
    return out


def _drop_edges(inst, pairs):
    """instance without the inter-cell edges between the given pairs of cells ((y, x), (y, x))"""
    cell = inst.cell_y.astype(int) * inst.Lx + inst.cell_x
    bad = {frozenset((a[0] * inst.Lx + a[1], b[0] * inst.Lx + b[1])) for a, b in pairs}
    keep = np.array([frozenset((cell[u], cell[v])) not in bad for u, v in zip(inst.edge_u, inst.edge_v)])
    d = dict(inst)
    d.update(edge_u=inst.edge_u[keep], edge_v=inst.edge_v[keep], J=inst.J[keep])
    return instances.Instance(d)


def test_lbp_is_exact_on_trees():
    """'Such iterations converge to exact results for problems defined on a tree': Eqs. (11)-(13) on a
    star of Pegasus-shaped cells that carries all three kinds of inter-cell couplings (horizontal, vertical, diagonal)
    and on a chain of Zephyr-shaped cells reproduce the brute-force cell marginals once the iteration count reaches the
    diameter of the tree, and do NOT before (so the iteration really propagates)."""
    from oracle import lbp
    full = instances.lattice(2, 2, 3, 2, p_keep=1.0, seed=4)
    star = _drop_edges(full, [((0, 1), (1, 1)), ((1, 0), (1, 1))])
    assert star.n_spins == 24 and len(star.J) < len(full.J)
    beta = 0.9
    ex = _brute_cell_marginals(star, brute.all_energies(star), beta)
    m = model.Model(star).set_beta(beta)
    nu = lbp.messages(m, 2)                                        # diameter of the star: 2
    for cidx in range(4):
        lp = lbp.log_marginals(m, nu, cidx // 2, cidx % 2)
        assert np.abs(np.exp(lp) - ex[cidx]).max() <= 1e-13
        st, l2 = lbp.select(m, nu, cidx // 2, cidx % 2, 5)
        assert np.array_equal(st, np.lexsort((np.arange(64), -ex[cidx]))[:5]) and np.all(np.diff(l2) <= 0)
    chain = instances.lattice(1, 4, 2, 2, p_keep=1.0, seed=9)
    exc = _brute_cell_marginals(chain, brute.all_energies(chain), 1.3)
    mc = model.Model(chain).set_beta(1.3)
    err = []
    for it in (1, 2, 3, 6):
        nuc = lbp.messages(mc, it)
        err.append(max(np.abs(np.exp(lbp.log_marginals(mc, nuc, 0, x)) - exc[x]).max() for x in range(4)))
    assert err[0] > 1e-4 and err[1] > 1e-6 and err[2] <= 1e-13 and err[3] <= 1e-13


def test_lbp_on_loops_is_normalised_and_close_at_high_temperature():
    """On a lattice with loops LBP is an approximation: the marginals are normalised, the error against
    brute force vanishes with beta (the loop corrections are high order in beta: the shortest loop of cells has four
    edge matrices) and is visible at beta = 1."""
    from oracle import lbp
    inst = instances.lattice(2, 3, 2, 2, p_keep=1.0, seed=6)
    E_all = brute.all_energies(inst)
    errs = {}
    for beta in (0.05, 1.0):
        ex = _brute_cell_marginals(inst, E_all, beta)
        m = model.Model(inst).set_beta(beta)
        nu = lbp.messages(m, 10)
        e = 0.0
        for cidx in range(6):
            lp = lbp.log_marginals(m, nu, cidx // 3, cidx % 3)
            assert abs(np.exp(lp).sum() - 1) <= 1e-12
            e = max(e, np.abs(np.exp(lp) - ex[cidx]).max())
        errs[beta] = e
    assert errs[0.05] <= 1e-9 and 1e-6 < errs[1.0] < 0.2
