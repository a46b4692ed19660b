"""Seeded synthetic Ising instances shaped like the paper's workloads.

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It holds
no arithmetic of the method (no energies, tables, tensors): it only draws couplings
and lays out the graph + cluster map that `tn_create` / the oracle consume.

The paper's workloads are random-coupling instances on D-Wave Pegasus / Zephyr working
graphs (PAPER.md:225-226 classes I/II); those graphs are not available
offline, so BASELINE.json's "Pegasus-/Zephyr-shaped" lattices stand in for them
(24-/16-spin unit cells made of 8-spin groups, NN + one diagonal coupling, ~3 % missing
couplers).  Recipe (restated in DESIGN.md §4):

* lattice of Ly x Lx cells, cell = chain of S sub-clusters of n_s spins,
  spin id = ((y*Lx + x)*S + sub)*n_s + k, lo = spins [0, n_s/2), hi = [n_s/2, n_s);
* candidate edges, in this order, `for y: for x:`
    for s in 0..S-1:  K(lo x hi) of sub-cluster s (i major, j minor);
                      then hi(s) x lo(s+1) if s+1 < S (i major);
    horizontal k=0..n_s-1:  sub 0 spin k of (x,y) -- sub 0 spin k of (x+1,y);
    vertical   k=0..n_s-1:  sub min(1,S-1) spin k of (x,y) -- same of (x,y+1);
    diagonal (S==3): lo(C) i of (x,y) x hi(C) j of (x+1,y+1) (i major);
* PRNG SplitMix64; u = (z >> 11) * 2^-53; for every candidate edge draw u_keep then
  u_J (both always drawn), keep iff u_keep < p_keep, J = 2 u_J - 1; then h_i = 2u-1
  for i = 0..N-1 (nothing drawn when h is "zero").
"""
from __future__ import annotations

import numpy as np

_MASK = (1 << 64) - 1


class SplitMix64:
    """Counter-based 64-bit generator (public-domain algorithm by S. Vigna)."""

    def __init__(self, seed: int):
        self.state = seed & _MASK

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _MASK
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        return z ^ (z >> 31)

    def u01(self) -> float:
        return (self.next_u64() >> 11) * (1.0 / 9007199254740992.0)

    def below(self, n: int) -> int:
        return min(int(self.u01() * n), n - 1)


class Instance(dict):
    """dict with attribute access; keys: n_spins, edge_u, edge_v, J, h, Ly, Lx, S, n_s,
    cell_y, cell_x, sub, pos (cluster map, one entry per spin), plus free-form metadata."""

    __getattr__ = dict.__getitem__


def spin_id(Lx, S, n_s, y, x, sub, k):
    return ((y * Lx + x) * S + sub) * n_s + k


def candidate_edges(Ly, Lx, S, n_s):
    """Candidate edge list of the synthetic lattice in the documented order."""
    half = n_s // 2
    vsub = min(1, S - 1)
    E = []
    for y in range(Ly):
        for x in range(Lx):
            sid = lambda sub, k, yy=y, xx=x: spin_id(Lx, S, n_s, yy, xx, sub, k)
            for s in range(S):
                for i in range(half):
                    for j in range(half, n_s):
                        E.append((sid(s, i), sid(s, j)))
                if s + 1 < S:
                    for i in range(half, n_s):
                        for j in range(half):
                            E.append((sid(s, i), sid(s + 1, j)))
            if x + 1 < Lx:
                for k in range(n_s):
                    E.append((sid(0, k), sid(0, k, y, x + 1)))
            if y + 1 < Ly:
                for k in range(n_s):
                    E.append((sid(vsub, k), sid(vsub, k, y + 1, x)))
            if S == 3 and x + 1 < Lx and y + 1 < Ly:
                for i in range(half):
                    for j in range(half, n_s):
                        E.append((sid(2, i), sid(2, j, y + 1, x + 1)))
    return E


def cluster_map(Ly, Lx, S, n_s):
    N = Ly * Lx * S * n_s
    ids = np.arange(N, dtype=np.int64)
    pos = (ids % n_s).astype(np.int32)
    sub = ((ids // n_s) % S).astype(np.int32)
    cell = ids // (n_s * S)
    return (cell // Lx).astype(np.int32), (cell % Lx).astype(np.int32), sub, pos


def lattice(Ly, Lx, S, n_s, p_keep=1.0, seed=0, h="uniform", h_scale=1.0, name=""):
    """Random-coupling instance (classes I/II of PAPER.md:225-226 on the synthetic shape).

    h: "uniform" -> h_i ~ U[-h_scale, h_scale]; "zero" -> h = 0 (class I)."""
    assert 1 <= S <= 3 and (n_s % 2 == 0 or S == 1)      # S = 1 has no lo / hi halves: any n_s (square lattice: n_s = 1)
    rng = SplitMix64(seed)
    eu, ev, J = [], [], []
    for (u, v) in candidate_edges(Ly, Lx, S, n_s):
        u_keep = rng.u01()
        u_J = rng.u01()
        if u_keep < p_keep:
            eu.append(u)
            ev.append(v)
            J.append(2.0 * u_J - 1.0)
    N = Ly * Lx * S * n_s
    hv = np.zeros(N, dtype=np.float64)
    if h == "uniform":
        for i in range(N):
            hv[i] = h_scale * (2.0 * rng.u01() - 1.0)
    cy, cx, sub, pos = cluster_map(Ly, Lx, S, n_s)
    return Instance(name=name or f"lattice{Ly}x{Lx}S{S}n{n_s}p{p_keep}s{seed}",
                    n_spins=N, edge_u=np.asarray(eu, dtype=np.int32),
                    edge_v=np.asarray(ev, dtype=np.int32), J=np.asarray(J, dtype=np.float64),
                    h=hv, Ly=Ly, Lx=Lx, S=S, n_s=n_s, cell_y=cy, cell_x=cx, sub=sub, pos=pos,
                    seed=seed, p_keep=p_keep)


def transformed(inst, t: int):
    """One of the 8 lattice transformations of PAPER.md:270 ("8 distinct transformations of the 2D lattice ...
    rotations and reflections") as a pure re-indexing of the cluster map: spin ids, the edge list, J and h are
    untouched, so states and energies of a transformed run compare directly with the original.
    t bit 0: mirror x, bit 1: mirror y, bit 2: transpose (applied last).  The synthetic geometry admits them as
    follows: S = 1 (config 1) and S = 2 (Zephyr-shaped): all 8; under transposition the horizontal sub-cluster A
    and the vertical sub-cluster B swap roles and, for the A_hi x B_lo rule to hold again, lo and hi swap inside
    both.  S = 3 (Pegasus-shaped): only t = 0, the single (x+1, y+1) diagonal of the shape has no mirror image."""
    t = int(t)
    if not 0 <= t < 8:
        raise ValueError("t must be 0..7")
    if inst.S == 3 and t != 0:
        raise ValueError("the Pegasus-shaped lattice (one diagonal direction) admits only the identity")
    cy, cx = inst.cell_y.copy(), inst.cell_x.copy()
    sub, pos = inst.sub.copy(), inst.pos.copy()
    Ly, Lx = inst.Ly, inst.Lx
    if t & 1:
        cx = (Lx - 1 - cx).astype(np.int32)
    if t & 2:
        cy = (Ly - 1 - cy).astype(np.int32)
    if t & 4:
        cy, cx = cx, cy
        Ly, Lx = Lx, Ly
        if inst.S == 2:
            sub = (1 - sub).astype(np.int32)
            pos = ((pos + inst.n_s // 2) % inst.n_s).astype(np.int32)
    out = Instance(inst)
    out.update(name=f"{inst.name}_t{t}", Ly=Ly, Lx=Lx, cell_y=cy, cell_x=cx, sub=sub, pos=pos, transform=t)
    return out


def loop_planted(Ly, Lx, S, n_s, seed=0, n_loops=None, min_len=4, max_len=8, name=""):
    """Loop-planted instance with known ground-state energy (BASELINE.json config 5).

    n_loops (default 3N/4) loops are drawn on the full (p_keep = 1) lattice graph: a seeded
    non-backtracking random walk from a uniform start vertex, closed at its first
    self-intersection, accepted iff the closed loop has min_len..max_len edges.  One uniformly
    chosen edge of the loop gets +1, the others -1 (all-up satisfies all but one edge, so it
    is a ground state of the loop with energy -(len-2)); J is the sum over loops, then gauged
    by a seeded hidden s*: J_ij <- J_ij s*_i s*_j.  E0 = -sum(len-2) is attained by +-s*.
    Every lattice edge stays in the edge list (J may be 0)."""
    rng = SplitMix64(seed)
    E = candidate_edges(Ly, Lx, S, n_s)
    N = Ly * Lx * S * n_s
    if n_loops is None:
        n_loops = (3 * N) // 4
    adj = [[] for _ in range(N)]
    for e, (u, v) in enumerate(E):
        adj[u].append((v, e))
        adj[v].append((u, e))
    Jsum = np.zeros(len(E), dtype=np.float64)
    E0 = 0.0
    accepted = 0
    lens = []
    while accepted < n_loops:
        v = rng.below(N)
        path_v, path_e, seen = [v], [], {v: 0}
        prev = -1
        loop = None
        for _ in range(4 * max_len):
            nb = [(w, e) for (w, e) in adj[v] if w != prev]
            if not nb:
                break
            w, e = nb[rng.below(len(nb))]
            path_e.append(e)
            if w in seen:
                loop = path_e[seen[w]:]
                break
            seen[w] = len(path_v)
            path_v.append(w)
            prev, v = v, w
        if loop is None or not (min_len <= len(loop) <= max_len):
            continue
        frustrated = rng.below(len(loop))
        for i, e in enumerate(loop):
            Jsum[e] += 1.0 if i == frustrated else -1.0
        E0 -= (len(loop) - 2)
        lens.append(len(loop))
        accepted += 1
    s_star = np.array([1 if rng.u01() < 0.5 else -1 for _ in range(N)], dtype=np.int8)
    eu = np.asarray([u for u, _ in E], dtype=np.int32)
    ev = np.asarray([v for _, v in E], dtype=np.int32)
    J = Jsum * s_star[eu].astype(np.float64) * s_star[ev].astype(np.float64)
    cy, cx, sub, pos = cluster_map(Ly, Lx, S, n_s)
    return Instance(name=name or f"loops{Ly}x{Lx}S{S}n{n_s}s{seed}", n_spins=N, edge_u=eu, edge_v=ev,
                    J=J, h=np.zeros(N, dtype=np.float64), Ly=Ly, Lx=Lx, S=S, n_s=n_s,
                    cell_y=cy, cell_x=cx, sub=sub, pos=pos, seed=seed, p_keep=1.0,
                    E0=E0, s_star=s_star, loop_lengths=np.asarray(lens))


# BASELINE.json configs (index = position in BASELINE.json "configs"); run parameters beside them.
CONFIGS = [
    dict(name="cfg1_tiny_2x3x4", kind="lattice", Ly=2, Lx=3, S=1, n_s=4, p_keep=1.0, h="uniform",
         beta=[1.0], D=0, M=16, sweeps=0),
    dict(name="cfg2_zephyr_6x6x16", kind="lattice", Ly=6, Lx=6, S=2, n_s=8, p_keep=0.97, h="uniform",
         beta=[2.0], D=16, M=256, sweeps=1),
    dict(name="cfg3_pegasus_8x8x24", kind="lattice", Ly=8, Lx=8, S=3, n_s=8, p_keep=0.97, h="uniform",
         beta=[2.0], D=32, M=1024, sweeps=1),
    dict(name="cfg4_pegasus_15x15x24", kind="lattice", Ly=15, Lx=15, S=3, n_s=8, p_keep=0.97, h="zero",
         beta=[1.0, 2.0, 4.0], D=64, M=1024, sweeps=3),
    dict(name="cfg5_zephyr_12x12x16_planted", kind="loops", Ly=12, Lx=12, S=2, n_s=8,
         beta=[4.0], D=32, M=1024, sweeps=1),
    # not a BASELINE.json config: the square-lattice workload of App. B (nearest neighbours, one spin per
    # site, class I couplings, chi = 16, M = 256, beta = 4, 50 x 50 sites) -- SURVEY.md section 8(f) f4, first half
    dict(name="appB_square_50x50", kind="lattice", Ly=50, Lx=50, S=1, n_s=1, p_keep=1.0, h="zero",
         beta=[4.0], D=16, M=256, sweeps=1),
]


def config(i: int, seed: int = 0, **override):
    """Instance + run parameters of BASELINE.json config i (0-based)."""
    c = dict(CONFIGS[i])
    c.update(override)
    if c["kind"] == "lattice":
        inst = lattice(c["Ly"], c["Lx"], c["S"], c["n_s"], p_keep=c["p_keep"], seed=seed, h=c["h"],
                       name=c["name"])
    else:
        inst = loop_planted(c["Ly"], c["Lx"], c["S"], c["n_s"], seed=seed, name=c["name"])
    run = dict(beta=c["beta"], D=c["D"], M=c["M"], sweeps=c["sweeps"])
    return inst, run
