"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star): log Z and log-marginals 1e-9 relative at exact D, 1e-6 relative at
truncated D; bitstrings identical wherever the oracle's logp gaps exceed the tolerance; energies bit-exact
with the oracle's fixed-order recomputation (O-0)."""
import numpy as np
import pytest

import instances
from oracle import energy, model, mps, search

pytestmark = pytest.mark.gpu


def _tn(inst):
    import paper_2411_16431_b200 as tnb
    return tnb.TensorNetwork(inst)


def mps_overlap(A, B):
    """<A|B> / (|A| |B|) for two MPS given as lists of [dl, p, dr] arrays."""
    def inner(X, Y):
        E = np.ones((1, 1))
        for x, y in zip(X, Y):
            E = np.einsum("ab,apc,bpd->cd", E, x, y, optimize=True)
        return E[0, 0]
    return inner(A, B) / np.sqrt(inner(A, A) * inner(B, B))


def components(inst):
    """Connected components of the interaction graph (edges with J != 0): label per spin."""
    parent = list(range(inst.n_spins))

    def find(i):
        while parent[i] != i:
            parent[i] = parent[parent[i]]
            i = parent[i]
        return i
    for u, v, J in zip(inst.edge_u.tolist(), inst.edge_v.tolist(), inst.J.tolist()):
        if J != 0.0:
            parent[find(u)] = find(v)
    return np.array([find(i) for i in range(inst.n_spins)])


def differ_by_component_flips(inst, s1, s2, comp=None):
    """True iff s2 is s1 with whole connected components flipped: at h = 0 exactly those states are degenerate by
    symmetry (zero energy gap), so which of them holds a rank is not defined."""
    comp = components(inst) if comp is None else comp
    rel = s1.astype(np.int64) * s2.astype(np.int64)
    return all(np.unique(rel[comp == c]).size == 1 for c in np.unique(comp))


def run_oracle(inst, beta, D, sweeps, M, merge=False, oracle_opts=None):
    m = model.Model(inst).set_beta(beta)
    R, ln = mps.contract(m, D, sweeps, **(oracle_opts or {}))
    st = {}
    out = search.branch_and_bound(m, R, ln, M, merge=merge, stats=st)
    out["tied_cuts"] = st.get("tied_cuts", 0)
    return m, R, ln, out


def compare(inst, beta, D, sweeps, M, tol, check_rows=True, options=(), merge=False, oracle_opts=None):
    m, R, ln, ref = run_oracle(inst, beta, D, sweeps, M, merge=merge, oracle_opts=oracle_opts)
    with _tn(inst) as t:
        for key, val in options:
            t.set_option(key, val)
        t.set_beta(beta)
        t.contract(D, sweeps)
        if check_rows:
            for y in range(inst.Ly - 1, 0, -1):
                ov = mps_overlap(R[y], t.mps(y))
                assert abs(1 - abs(ov)) <= max(tol * 1e-1, 1e-12), (y, ov)
                # (row log-norms are not comparable: the two sides shift their local tables by different
                #  minima, per factor here vs per cell in the oracle; the total enters log Z below)
                assert np.isfinite(t.row_lognorm(y))
        lz = t.log_z()
        assert abs(lz - ref["log_z"]) <= tol * abs(ref["log_z"]), (lz, ref["log_z"])
        states, E, logp, pd = t.branch_and_bound(M)
        st = t.stats()
    check_lists(inst, ref, states, E, logp, pd, tol)
    return st


def check_lists(inst, ref, states, E, logp, pd, tol):
    """Final lists of the CUDA path against the oracle's (`ref`: logp, states, log_pd): element by element."""
    n = ref["logp"].size
    assert states.shape[0] == n
    assert np.allclose(logp, ref["logp"], rtol=tol, atol=0), np.abs(logp - ref["logp"]).max()
    # energies: bit-exact with the oracle's fixed-order recomputation of the SAME states
    assert np.array_equal(E, energy.energies(inst, states))
    # bitstrings identical rank by rank wherever the oracle's adjacent logp gaps exceed the tolerance
    # At h = 0 every state is exactly degenerate with its flips of whole connected components (the global flip on a
    # connected graph): which member survives a cut that falls between them is arbitrary (and decides the sign of its
    # descendants), so states are compared up to such flips there; the last rank may also tie with a discarded
    # candidate, which log p_d (the largest discarded probability) bounds.
    z2 = not np.any(inst.h)
    comp = components(inst) if z2 else None
    lp = ref["logp"]
    gap_tol = 10 * tol * np.abs(lp).max()
    for r in range(n):
        lo = r == 0 or lp[r - 1] - lp[r] > gap_tol
        hi = (lp[r] - ref["log_pd"] > gap_tol) if r == n - 1 else lp[r] - lp[r + 1] > gap_tol
        if lo and hi and not np.array_equal(states[r], ref["states"][r]):
            # h = 0: flipping a whole connected component of the interaction graph (the global flip when the graph
            # is connected) costs exactly nothing, so the state of rank r is one of several exactly degenerate ones
            # (energy gap 0 <= 1e-9, which north_star exempts); ANY other difference is a mismatch
            assert z2 and differ_by_component_flips(inst, states[r], ref["states"][r], comp), r
            assert E[r] == energy.energies(inst, ref["states"][r:r + 1])[0], r
    if ref.get("tied_cuts", 0) > 0:
        # some beam cut fell inside a group of tied candidates (exactly degenerate instances: integer couplings, h = 0
        # pairs, J = 0): WHICH tied prefixes survive is decided by rounding noise, and the discarded probabilities of
        # later cells depend on that choice -- log p_d is not unique there; it must still be a valid log-probability
        assert pd <= 1e-12 and (np.isfinite(pd) or pd == -np.inf)
    elif np.isfinite(ref["log_pd"]):
        assert abs(pd - ref["log_pd"]) <= 10 * tol * abs(ref["log_pd"]), (pd, ref["log_pd"])
    else:
        assert pd == ref["log_pd"]


EXACT = [  # (Ly, Lx, S, n_s, p_keep, seed, beta, M)
    (2, 2, 3, 2, 0.8, 3, 1.3, 8),
    (3, 2, 2, 2, 0.9, 5, 0.7, 8),
    (2, 3, 1, 4, 1.0, 1, 1.5, 16),
    (2, 3, 2, 2, 0.9, 7, 0.9, 8),
    (3, 3, 3, 2, 0.85, 7, 0.9, 32),
    (4, 5, 1, 1, 1.0, 2, 1.0, 16),             # square lattice, one spin per site (App. B; f4 workload)
    (3, 4, 1, 3, 0.9, 5, 0.8, 16),             # S = 1 with an odd number of spins per cell
]


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta,M", EXACT)
def test_exact_contraction_parity(Ly, Lx, S, ns, p, seed, beta, M):
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    compare(inst, beta, 0, 0, M, 1e-9)


def test_config1_parity():
    inst, run = instances.config(0)
    compare(inst, run["beta"][0], run["D"], run["sweeps"], run["M"], 1e-9)


TRUNC = [  # (Ly, Lx, S, n_s, p_keep, seed, beta, D, sweeps, M)
    (3, 4, 2, 2, 0.9, 3, 0.9, 3, 0, 16),
    (3, 4, 2, 2, 0.9, 3, 0.9, 3, 1, 16),
    (3, 4, 2, 2, 0.9, 3, 0.9, 3, 2, 16),
    (4, 4, 2, 4, 0.95, 2, 1.0, 6, 1, 64),      # Zephyr-shaped miniature: 256 states per cell, ragged projectors
    (3, 3, 3, 4, 0.9, 4, 1.0, 6, 2, 64),       # Pegasus-shaped miniature: 4096 states per cell, mediating tensors
    (4, 3, 3, 2, 0.85, 9, 1.5, 4, 3, 32),
    (3, 3, 1, 4, 1.0, 6, 2.0, 5, 1, 16),
    (10, 10, 1, 1, 1.0, 3, 1.0, 4, 1, 64),     # square lattice 10 x 10, chi = 4: truncating, 100 cells of one spin
]


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta,D,sweeps,M", TRUNC)
def test_truncated_contraction_parity(Ly, Lx, S, ns, p, seed, beta, D, sweeps, M):
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    compare(inst, beta, D, sweeps, M, 1e-6)


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta,D,sweeps,M", [TRUNC[3], TRUNC[4], TRUNC[6]])
def test_sampled_prefilter_selection_parity(Ly, Lx, S, ns, p, seed, beta, D, sweeps, M):
    """Top-M through the hashed-sample lower bound + prefilter + compact radix passes (the route taken at the
    BASELINE.json sizes), forced here by TN_OPT_SELECT_DIRECT_MAX = 0."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    compare(inst, beta, D, sweeps, M, 1e-6, check_rows=False, options=[(tnb.OPT_SELECT_DIRECT_MAX, 0)])


@pytest.mark.parametrize("D", [8, 12])
def test_svd_variants_agree_and_match_oracle(D):
    """Locked subspace iteration (default), plain iteration and the Chebyshev-filtered fallback converge the same
    truncated SVD: identical results to 1e-9 among themselves, 1e-6 against the oracle (ks = D + 16 >= 24 locks)."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(4, 4, 2, 4, p_keep=0.95, seed=2)
    beta, sweeps, M = 1.2, 1, 64
    st = compare(inst, beta, D, sweeps, M, 1e-6, check_rows=False)
    outs = []
    for lock, cheb in ((1, 1), (0, 1), (0, 0)):
        with _tn(inst) as t:
            t.set_option(tnb.OPT_SVD_LOCK, lock)
            t.set_option(tnb.OPT_SVD_CHEB, cheb)
            t.set_beta(beta)
            t.contract(D, sweeps)
            lz = t.log_z()
            states, E, logp, pd = t.branch_and_bound(M)
            outs.append((lz, logp, states, t.stats()))
    for lz, logp, states, s in outs[1:]:
        assert abs(lz - outs[0][0]) <= 1e-9 * abs(lz)
        assert np.allclose(logp, outs[0][1], rtol=1e-8, atol=0)
        assert np.array_equal(states[0], outs[0][2][0])
        assert s["svd_unconverged"] == 0
    assert outs[1][3]["svd_locked_cols"] == 0


def test_numeric_failure_is_reported_not_hidden():
    """Non-finite inputs are rejected at the boundary (TN_ERR_ARG), beta out of range too; a result that leaves the
    fp64 range (log Z = -beta * offset + ... overflows at beta = 1e307) is TN_ERR_NUMERIC, not a silent inf, and the
    handle stays usable."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(2, 2, 2, 2, seed=1)
    for key in ("J", "h"):
        bad = instances.Instance(inst)
        v = inst[key].copy()
        v[0] = np.nan
        bad[key] = v
        with pytest.raises(tnb.TnError) as e:
            tnb.TensorNetwork(bad)
        assert e.value.code == -1
    with _tn(inst) as t:
        with pytest.raises(tnb.TnError) as e:
            t.set_beta(float("inf"))
        assert e.value.code == -1
        t.set_beta(0.5)
        with pytest.raises(tnb.TnError) as e:
            t.branch_and_bound(0)
        assert e.value.code in (-1, -3)
        with pytest.raises(tnb.TnError) as e:
            t.energy(np.ones((2, inst.n_spins + 1), dtype=np.int8))
        assert e.value.code == -1
        t.set_beta(1e307)
        with pytest.raises(tnb.TnError) as e:
            t.contract(0, 0)
        assert e.value.code == -6, str(e.value)          # TN_ERR_NUMERIC
        with pytest.raises(tnb.TnError) as e:
            t.log_z()
        assert e.value.code == -3                        # no boundary MPS survives the failed call
        t.set_beta(0.5)
        t.contract(0, 0)
        assert np.isfinite(t.log_z())


def test_error_path_releases_device_memory():
    """A failed tn_contract / tn_branch_and_bound leaves the handle at its pre-call device footprint and usable
    (blocks taken through raw dalloc used to stay pinned until tn_destroy)."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(3, 4, 2, 4, p_keep=0.9, seed=11)
    with _tn(inst) as t:
        t.set_beta(1.0)
        base = t.stats()["bytes_device"]
        t.set_option(tnb.OPT_EXACT_CAP, 4)
        for _ in range(3):
            with pytest.raises(tnb.TnError) as e:
                t.contract(0, 0)                         # exact bond 16 > cap 4, thrown in the middle of row 2
            assert e.value.code == -1 and "EXACT_CAP" in str(e.value)
            assert t.stats()["bytes_device"] == base
        t.set_option(tnb.OPT_EXACT_CAP, 512)
        t.contract(6, 1)
        held = t.stats()["bytes_device"]
        assert held > base                               # the boundary MPS
        with pytest.raises(tnb.TnError):
            t.branch_and_bound(1 << 21)                  # rejected before any allocation
        states, E, logp, pd = t.branch_and_bound(32)
        assert t.stats()["bytes_device"] == held
        assert np.array_equal(E, energy.energies(inst, states))


MERGE = [  # (Ly, Lx, S, n_s, p_keep, seed, beta, D, sweeps, M)
    (2, 3, 1, 4, 1.0, 1, 1.5, 0, 0, 16),
    (3, 2, 2, 2, 0.9, 5, 0.7, 0, 0, 8),
    (3, 3, 3, 2, 0.85, 7, 0.9, 0, 0, 32),       # mediating tensors, diagonal legs in the boundary
    (3, 4, 2, 2, 0.9, 3, 0.9, 3, 1, 16),
    (4, 4, 2, 4, 0.95, 2, 1.0, 6, 1, 64),       # ragged projectors: several cell states share one boundary
    (3, 3, 3, 4, 0.9, 4, 1.0, 6, 2, 64),
]


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta,D,sweeps,M", MERGE)
@pytest.mark.parametrize("sampled", [False, True])
def test_merge_by_boundary_parity(Ly, Lx, S, ns, p, seed, beta, D, sweeps, M, sampled):
    """TN_OPT_MERGE (Fig. 3(d)) against the oracle's merge switch, through both selection routes."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    opts = [(tnb.OPT_MERGE, 1)] + ([(tnb.OPT_SELECT_DIRECT_MAX, 0)] if sampled else [])
    st = compare(inst, beta, D, sweeps, M, 1e-9 if D == 0 else 1e-6, check_rows=False, options=opts, merge=True)
    assert st["merged_away"] > 0 and st["merge_fallback_cells"] == 0


@pytest.mark.parametrize("cap,expect_fallback", [(1 << 20, False), (512, False), (8, True)])
def test_merge_routes_and_counted_fallback(cap, expect_fallback):
    """TN_OPT_MERGE has two routes: a segmented arg-max over all candidates when the possible boundaries of a cell fit
    the merge buffers (TN_OPT_MERGE_CAP), else threshold + sort with a bisected threshold.  cap = 512 sends the middle
    cells of this lattice (up to 16384 possible boundaries) through the threshold route with fewer buffer slots than
    the sampled bound leaves survivors (bisection), the rest through the segmented one; both must reproduce the
    oracle's merge=True.  A cell
    that fits neither route (cap = 8) is selected unmerged and COUNTED in merge_fallback_cells -- never silently."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(4, 4, 2, 4, p_keep=0.95, seed=2)
    opts = [(tnb.OPT_MERGE, 1), (tnb.OPT_MERGE_CAP, cap), (tnb.OPT_SELECT_DIRECT_MAX, 0)]
    if not expect_fallback:
        st = compare(inst, 1.0, 6, 1, 64, 1e-6, check_rows=False, options=opts, merge=True)
        assert st["merge_fallback_cells"] == 0 and st["merged_away"] > 0
        return
    with _tn(inst) as t:
        for k, v in opts:
            t.set_option(k, v)
        t.set_beta(1.0)
        t.contract(6, 1)
        states, E, logp, pd = t.branch_and_bound(64)
        st = t.stats()
    assert st["merge_fallback_cells"] > 0
    assert np.array_equal(E, energy.energies(inst, states)) and np.all(np.diff(logp) <= 0)


F2 = [  # (name, oracle options, CUDA options): the paper's preferred schedule and its ingredients
    ("interleaved_r1", dict(schedule=1, sweep_range=1), [("OPT_SCHEDULE", 1), ("OPT_SWEEP_RANGE", 1)]),
    ("interleaved_r2", dict(schedule=1, sweep_range=2), [("OPT_SCHEDULE", 1)]),
    ("interleaved_all", dict(schedule=1, sweep_range=99), [("OPT_SCHEDULE", 1), ("OPT_SWEEP_RANGE", 99)]),
    ("two_step", dict(two_step=True), [("OPT_TWO_STEP", 1)]),
    ("randomized_2it", dict(svd_mode=1, rsvd_iters=2), [("OPT_SVD_MODE", 1)]),
    ("randomized_1it", dict(svd_mode=1, rsvd_iters=1), [("OPT_SVD_MODE", 1), ("OPT_RSVD_ITERS", 1)]),
    ("paper_preferred", dict(schedule=1, sweep_range=2, svd_mode=1, rsvd_iters=2, two_step=True),
     [("OPT_SCHEDULE", 1), ("OPT_SVD_MODE", 1), ("OPT_TWO_STEP", 1)]),
]
F2_CASES = [  # (Ly, Lx, S, n_s, p_keep, seed, beta, D, M)
    (4, 4, 2, 4, 0.95, 2, 1.0, 6, 64),         # Zephyr-shaped miniature, ragged projectors
    (3, 3, 3, 4, 0.9, 4, 1.0, 6, 64),          # Pegasus-shaped miniature: mediating positions inside the local sweeps
    (3, 4, 1, 4, 1.0, 6, 2.0, 5, 16),
]


@pytest.mark.parametrize("name,oopts,copts", F2, ids=[f[0] for f in F2])
@pytest.mark.parametrize("case", range(len(F2_CASES)))
@pytest.mark.parametrize("sweeps", [0, 1])
def test_f2_schedule_parity(name, oopts, copts, case, sweeps):
    """TN_OPT_SCHEDULE / SVD_MODE / TWO_STEP against the oracle's switches of the same names: element by element at
    1e-6, rows included.  The randomized SVD is deterministic given its counter-based random block, which both sides
    generate from (seed, p', gamma, column) (oracle.mps.hash_uniform, k_fill_random_pgc)."""
    import paper_2411_16431_b200 as tnb
    Ly, Lx, S, ns, p, seed, beta, D, M = F2_CASES[case]
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    st = compare(inst, beta, D, sweeps, M, 1e-6, options=[(getattr(tnb, k), v) for k, v in copts], oracle_opts=oopts)
    assert st["svd_unconverged"] == 0


def test_f2_fast_mode_close_to_converged_mode():
    """The fast mode (randomized SVD) is not the parity definition: it is compared with the converged
    mode by R_y overlap and by the final list -- after one variational pass the two agree to the size of the
    truncation error, with a fraction of the Theta applies."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(4, 4, 2, 4, p_keep=0.95, seed=2)
    out = {}
    for mode in (0, 1):
        with _tn(inst) as t:
            t.set_option(tnb.OPT_SVD_MODE, mode)
            t.set_beta(1.0)
            t.contract(6, 1)
            rows = {y: t.mps(y) for y in range(1, inst.Ly)}
            lz = t.log_z()
            states, E, logp, pd = t.branch_and_bound(64)
            out[mode] = (rows, lz, states, E, logp, t.stats())
    trunc = out[0][5]["min_sigma_rel"]
    assert 0 < trunc < 0.1
    for y in range(1, inst.Ly):
        assert 1 - abs(mps_overlap(out[0][0][y], out[1][0][y])) <= 10 * trunc ** 2 + 1e-12
    assert abs(out[0][1] - out[1][1]) <= 10 * trunc * abs(out[0][1])
    assert out[0][3].min() == out[1][3].min()                     # same best energy
    assert out[1][5]["svd_unconverged"] == 0 and out[1][5]["svd_iterations"] > 0


DROPS = [  # (Ly, Lx, S, n_s, p_keep, seed, beta, D, sweeps, M, max_dE, min_hamming, max_count)
    (2, 3, 2, 2, 1.0, 3, 2.0, 0, 0, 64, 1.2, 1, 16),          # the brute-force pin's lattice (exact D)
    (3, 3, 3, 2, 0.85, 7, 0.9, 0, 0, 32, 1.5, 1, 8),          # mediating tensors: c_hi variants are interior droplets
    (4, 4, 2, 4, 0.95, 2, 1.0, 6, 1, 64, 1.0, 2, 8),          # truncated D, ragged projectors, Hamming filter
    (3, 3, 3, 4, 0.9, 4, 1.0, 6, 2, 64, 0.8, 1, 4),           # 4096 states per cell, list capped at 4
    (3, 4, 1, 4, 1.0, 6, 2.0, 5, 1, 16, 2.0, 3, 8),
]


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta,D,sweeps,M,max_dE,min_h,max_count", DROPS)
@pytest.mark.parametrize("route", ["segmented", "threshold"])
def test_droplets_parity(Ly, Lx, S, ns, p, seed, beta, D, sweeps, M, max_dE, min_h, max_count, route):
    """TN_OPT_DROPLETS (Fig. 4) against the oracle's DropletBook: for every returned state the same
    droplets -- identical flip masks, dE within the tolerance that the log-probabilities carry -- through both merge
    routes (segmented arg-max with per-group bounds; threshold + sort, forced by TN_OPT_MERGE_SEGMENTED = 0)."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed)
    tol = 1e-9 if D == 0 else 1e-6
    m = model.Model(inst).set_beta(beta)
    R, ln = mps.contract(m, D, sweeps)
    ref = search.branch_and_bound(m, R, ln, M, merge=True,
                                  droplets=dict(max_dE=max_dE, min_hamming=min_h, max_count=max_count))
    with _tn(inst) as t:
        for k, v in ((tnb.OPT_MERGE, 1), (tnb.OPT_DROPLETS, 1), (tnb.OPT_DROPLET_MAX_DE, max_dE),
                     (tnb.OPT_DROPLET_MIN_HAMMING, min_h), (tnb.OPT_DROPLET_MAX_COUNT, max_count),
                     (tnb.OPT_SELECT_DIRECT_MAX, 0)):
            t.set_option(k, v)
        if route == "threshold":
            t.set_option(tnb.OPT_MERGE_SEGMENTED, 0)
        t.set_beta(beta)
        t.contract(D, sweeps)
        states, E, logp, pd = t.branch_and_bound(M)
        st = t.stats()
        got = [t.droplets(r) for r in range(states.shape[0])]
    assert st["merge_fallback_cells"] == 0 and st["droplet_overflow"] == 0
    check_lists(inst, ref, states, E, logp, pd, tol)
    dtol = 4 * tol * np.abs(ref["logp"]).max() / beta
    total = 0
    for r in range(states.shape[0]):
        if not np.array_equal(states[r], ref["states"][r]):
            continue                                           # a tie inside the tolerance (check_lists accepted it)
        dE, flips = got[r]
        want = ref["droplets"][r]
        assert len(dE) == len(want), (r, len(dE), len(want))
        for k, (wE, wmask) in enumerate(want):
            assert abs(dE[k] - wE) <= dtol, (r, k, dE[k], wE)
            assert np.array_equal(flips[k].astype(bool), wmask), (r, k)
            s1 = states[r].copy()
            s1[wmask] *= -1
            if D == 0:                                         # exact marginals: dE IS the energy of the excitation
                assert abs(energy.energies(inst, s1[None])[0] - E[r] - dE[k]) <= 1e-8
        total += len(want)
    assert total > 0


EDGE = [  # (Ly, Lx, S, n_s, p_keep, seed, beta, D, sweeps, M, h): the degenerate shapes the method has
    (1, 3, 2, 2, 1.0, 1, 1.0, 0, 0, 8, "uniform"),       # one row: no boundary MPS at all
    (1, 1, 3, 2, 1.0, 1, 1.0, 0, 0, 8, "uniform"),       # one cell
    (3, 1, 2, 2, 1.0, 2, 1.0, 0, 0, 8, "uniform"),       # one column: every bond of every MPS is 1
    (1, 4, 3, 2, 0.9, 3, 0.8, 0, 0, 16, "uniform"),      # one row with mediating positions
    (4, 1, 3, 2, 0.9, 3, 0.8, 0, 0, 16, "uniform"),
    (2, 2, 1, 2, 1.0, 4, 1.0, 0, 0, 300, "uniform"),     # M > 2^8 states: everything kept, log p_d = -inf
    (1, 2, 2, 4, 1.0, 9, 1.0, 0, 0, 70000, "uniform"),   # M > 2^16 states through the selection kernels
    (2, 2, 2, 2, 0.0, 5, 1.0, 0, 0, 16, "uniform"),      # no couplings: product distribution
    (2, 2, 2, 2, 0.0, 5, 1.0, 0, 0, 16, "zero"),         # H = 0: uniform distribution, every rank is a tie
    (3, 3, 3, 2, 0.0, 5, 1.0, 2, 1, 16, "uniform"),      # truncated D on rank-1 boundaries
    (2, 3, 2, 2, 0.9, 6, 6.0, 0, 0, 16, "uniform"),      # cold: weights span e^-100
    (2, 3, 2, 2, 0.9, 6, 1e-3, 0, 0, 16, "uniform"),     # hot: nearly uniform
    (2, 2, 2, 2, 1.0, 7, 1.0, 0, 0, 1, "uniform"),       # M = 1: greedy descent
    (3, 3, 2, 2, 0.9, 8, 1.0, 1, 1, 8, "uniform"),       # D = 1
]


@pytest.mark.parametrize("Ly,Lx,S,ns,p,seed,beta,D,sweeps,M,h", EDGE)
def test_degenerate_shapes_parity(Ly, Lx, S, ns, p, seed, beta, D, sweeps, M, h):
    inst = instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=seed, h=h)
    compare(inst, beta, D, sweeps, M, 1e-9 if D == 0 else 1e-6)


@pytest.mark.parametrize("t", range(8))
def test_lattice_transformations_parity(t):
    """The 8 lattice transformations of PAPER.md:270 are re-indexings of the cluster map handed to tn_create
    (instances.transformed): on every map the CUDA path must match the oracle run on the same map, at exact D
    (1e-9, both cell kinds that admit them) and at truncated D with ragged projectors (1e-6)."""
    compare(instances.transformed(instances.lattice(2, 3, 2, 2, p_keep=0.85, seed=4), t), 1.1, 0, 0, 8, 1e-9)
    compare(instances.transformed(instances.lattice(3, 2, 1, 4, p_keep=0.9, seed=6), t), 1.1, 0, 0, 8, 1e-9)
    compare(instances.transformed(instances.lattice(3, 4, 2, 4, p_keep=0.9, seed=11), t), 1.0, 6, 1, 32, 1e-6)


def test_exact_contraction_with_svd_blocks_above_128_columns():
    """Regression: the exact (D <= 0) contraction of this map runs SVD blocks of 256 columns (retained rank 58); the
    residual-flag kernel used a 128-entry shared array for one slot per column (illegal address for k > 128)."""
    inst = instances.transformed(instances.lattice(3, 4, 2, 4, p_keep=0.9, seed=11), 1)
    compare(inst, 1.0, 0, 0, 32, 1e-9)


def test_lattice_transformations_spread_of_log_z():
    """Z-spread diagnostic: log Z is the same number on all 8 maps at exact D, and the truncated
    contractions scatter around it by no more than their truncation error."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(3, 4, 2, 4, p_keep=0.9, seed=11)
    exact, trunc = [], []
    for t in range(8):
        with tnb.TensorNetwork(instances.transformed(inst, t)) as tn:
            tn.set_beta(1.0)
            tn.contract(0, 0)
            exact.append(tn.log_z())
            tn.contract(6, 1)
            trunc.append(tn.log_z())
    exact, trunc = np.array(exact), np.array(trunc)
    assert np.ptp(exact) <= 1e-9 * abs(exact[0])
    assert np.ptp(trunc) > 0 and np.abs(trunc - exact[0]).max() <= 1e-2 * abs(exact[0])


def _random_case(i):
    """Seeded random small case: every cell kind, thinned edges, zero / random fields, exact and truncated D with
    0-2 passes, beam sizes from 1 to 64, lattice transformations, merge by boundary, both selection routes."""
    r = np.random.default_rng(9000 + i)
    S = int(r.integers(1, 4))
    ns = int(r.choice([2, 4])) if S < 3 else 2
    if S == 2 and ns == 4 and r.random() < 0.5:
        ns = 2
    Ly, Lx = int(r.integers(1, 4)), int(r.integers(1, 5))
    if S * ns >= 8:
        Lx = min(Lx, 3)
    p = float(r.choice([0.7, 0.85, 0.95, 1.0]))
    beta = float(r.uniform(0.3, 3.0))
    exact = r.random() < 0.4
    D = 0 if exact else int(r.integers(2, 9))
    sweeps = 0 if exact else int(r.integers(0, 3))
    M = int(r.choice([1, 3, 8, 17, 32, 64]))
    t = int(r.integers(0, 8)) if S < 3 else 0
    merge = bool(r.random() < 0.25)
    h = "zero" if r.random() < 0.2 else "uniform"
    sampled = bool(r.random() < 0.3)
    inst = instances.transformed(instances.lattice(Ly, Lx, S, ns, p_keep=p, seed=9000 + 7 * i, h=h), t)
    return inst, beta, D, sweeps, M, merge, sampled


@pytest.mark.parametrize("block", range(8))
def test_random_small_cases_parity(block):
    """160 seeded random small cases (20 per block) through the full parity comparison.  A case whose truncated
    contraction breaks down in the oracle itself (a non-positive normaliser at tiny D) has no reference and is skipped;
    at most a few may do so."""
    import paper_2411_16431_b200 as tnb
    skipped = 0
    for i in range(20 * block, 20 * block + 20):
        inst, beta, D, sweeps, M, merge, sampled = _random_case(i)
        opts = ([(tnb.OPT_MERGE, 1)] if merge else []) + ([(tnb.OPT_SELECT_DIRECT_MAX, 0)] if sampled else [])
        try:
            with np.errstate(divide="raise", invalid="raise"):
                run_oracle(inst, beta, D, sweeps, M, merge=merge)
        except (FloatingPointError, ValueError):
            skipped += 1
            continue
        try:
            compare(inst, beta, D, sweeps, M, 1e-9 if D == 0 else 1e-6, options=opts, merge=merge)
        except AssertionError as e:
            raise AssertionError(f"random case {i}: {e}") from e
    assert skipped <= 2


def test_zero_field_z2_instance():
    inst = instances.lattice(3, 3, 2, 4, p_keep=1.0, seed=21, h="zero")
    compare(inst, 2.0, 8, 1, 32, 1e-6)


def test_energy_kernel_bit_exact():
    inst = instances.lattice(3, 3, 3, 4, p_keep=0.9, seed=11)
    rng = np.random.default_rng(0)
    s = (1 - 2 * rng.integers(0, 2, size=(37, inst.n_spins))).astype(np.int8)
    with _tn(inst) as t:
        assert np.array_equal(t.energy(s), energy.energies(inst, s))


def test_error_codes():
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(2, 2, 2, 2, seed=1)
    with _tn(inst) as t:
        with pytest.raises(tnb.TnError) as e:
            t.contract(4, 1)
        assert e.value.code == -3          # TN_ERR_STATE: contract before set_beta
        t.set_beta(1.0)
        with pytest.raises(tnb.TnError) as e:
            t.branch_and_bound(4)
        assert e.value.code == -3
    bad = instances.Instance(inst)
    bad["edge_u"] = np.append(inst.edge_u, 0).astype(np.int32)
    bad["edge_v"] = np.append(inst.edge_v, inst.n_spins - 1).astype(np.int32)   # cell (0,0) -- (1,1) on S = 2
    bad["J"] = np.append(inst.J, 1.0)
    with pytest.raises(tnb.TnError) as e:
        tnb.TensorNetwork(bad)
    assert e.value.code == -2              # TN_ERR_GEOMETRY


@pytest.mark.slow
def test_square_lattice_workload_of_appendix_b():
    """App. B: nearest-neighbour square lattice, one spin per site, J ~ U[-1,1] (class I), chi = 16, M = 256,
    beta = 4 -- here 16 x 16 sites (the oracle needs a minute for it), element by element against the oracle.  The
    king's lattice of the same appendix (both diagonals) is outside the accepted geometry."""
    inst = instances.lattice(16, 16, 1, 1, p_keep=1.0, seed=1, h="zero")
    compare(inst, 4.0, 16, 1, 256, 1e-6)


@pytest.mark.parametrize("sampled", [False, True])
def test_exact_ties_beyond_the_candidate_list_follow_the_s8_order(sampled):
    """J = 0, h = 0 on cells of 2^16 states: every candidate of every cell ties exactly, far more of them than the
    candidate list holds.  The whole tie group is then collected and sorted, so the kept prefixes are the
    FIRST ones in the S8 order (parent rank, then cell state) -- bit for bit the oracle's list -- and the run is
    reproducible; select_tie_overflow counts the cells that took this route."""
    import paper_2411_16431_b200 as tnb
    inst = instances.lattice(2, 2, 2, 8, p_keep=0.0, seed=1, h="zero")
    m, R, ln, ref = run_oracle(inst, 1.0, 0, 0, 8)
    outs = []
    for rep in range(2):
        with _tn(inst) as t:
            if sampled:                                   # the sampled-prefilter route (taken at the BASELINE sizes)
                t.set_option(tnb.OPT_SELECT_DIRECT_MAX, 0)
            t.set_beta(1.0)
            t.contract(0, 0)
            lz = t.log_z()
            states, E, logp, pd = t.branch_and_bound(8)
            st = t.stats()
        outs.append((states.copy(), logp.copy(), pd))
        assert abs(lz - inst.n_spins * np.log(2.0)) <= 1e-9 * lz
        assert st["select_tie_overflow"] > 0 and st["select_tie_dropped"] == 0
        assert np.array_equal(states, ref["states"])
        assert np.allclose(logp, ref["logp"], rtol=1e-12, atol=0) and np.allclose(logp, -inst.n_spins * np.log(2.0))
        assert abs(pd - ref["log_pd"]) <= 1e-9 * abs(pd)
    assert np.array_equal(outs[0][0], outs[1][0]) and outs[0][2] == outs[1][2]
