"""T-2: branch and bound over cells driven by boundary-MPS conditionals; O-3 exact-marginal beam.
Test infrastructure (see oracle/__init__.py).

PAPER.md:94-98 Eq. (7) chain rule p(x_{n+1}) = p(x_{n+1} | x_n) p(x_n); Fig. 3
(branch to d*M candidates, keep the M most probable); Eqs. (8)-(9) PAPER.md:100-107 (conditionals
depend only on the boundary of the prefix); Fig. 6(b) PAPER.md:143 (fixed legs above, one open site,
boundary MPS R_{y+1} below, contracted numerically exactly, 'up to normalization'); p_d
PAPER.md:113 (largest discarded probability).  Search order: row-major.

For beam element m at cell (x, y) (rows < y and cells < x of row y fixed; S, Q = tensors of R_{y+1}):
  u(m; X) = hvec[Pl X] dvec[Pi X] uvec[Pu X] w(X) * (Lv . S[:,Pd X,:] . Q[:,Po X,:] . RM_x[:, Pr X])
  hvec = Bh_x[Pr(left neighbour state), :], uvec = Bv_x[Pd(upper state), :], dvec = Bd_x[Po(upper-left), :]
  Lv    = product of S.Q of the already fixed cells of row y (row vector)
  RM_x  = right block: contraction of columns > x of rows y (summed) with the fixed row y-1 above,
          RM_{Lx-1} = 1;  RS_x[b', l] = sum_{X: Pl X = l} dvec uvec w(X) (S[b',Pd X,:] Q[:,Po X,:] RM_x[:, Pr X]);
          RM_{x-1}[b', r] = sum_l Bh_x[r, l] RS_x[b', l]
  p = max(u, 0) / sum max(u, 0)   (S7: a truncated MPS can give small negative u; they are clamped)
Ties (S8): candidates are ordered by (logp desc, parent rank asc, cell state asc).
Positive rescalings of Lv and RM cancel in p; their logs are tracked only where log Z needs them.
"""
import numpy as np
from . import energy as _energy


def select_top(scores, parent, state, M):
    """Indices of the M best candidates in the S8 total order, best first, and the best
    discarded score (or -inf)."""
    n = scores.size
    if n > M + 1:                      # prefilter: everything >= the (M+1)-th largest score
        kth = n - (M + 1)
        thr = np.partition(scores, kth)[kth]
        sub = np.flatnonzero(scores >= thr)
    else:
        sub = np.arange(n)
    order = sub[np.lexsort((state[sub], parent[sub], -scores[sub]))]
    keep = order[:M]
    disc = scores[order[M]] if order.size > M else -np.inf
    return keep, disc


class _RowCtx:
    """Per-row tables of the search: cells of row y and the tensors of R_{y+1}."""

    def __init__(self, model, y, Rnext):
        self.cells = model.cells[y]
        Lx = model.Lx
        if model.has_med:
            self.S = [Rnext[2 * x] for x in range(Lx)]
            self.Q = [Rnext[2 * x + 1] if x + 1 < Lx else None for x in range(Lx)]
        else:
            self.S = list(Rnext)
            self.Q = [None] * Lx
        self.G = []          # G[x][pd, po] = S[:,pd,:] @ Q[:,po,:]  -> [n_down, n_dout, Dl, Dr']
        for x in range(Lx):
            S = self.S[x]
            if self.Q[x] is None:
                assert self.cells[x].n["dout"] == 1
                self.G.append(S.transpose(1, 0, 2)[:, None, :, :])
            else:
                self.G.append(np.einsum("apb,bqc->pqac", S, self.Q[x]))


def _right_blocks(model, y, ctx, above):
    """RM_x for x = 0..Lx-1 given the states `above` of row y-1 (None for y = 0).
    Returns list of (RM [D', n_r], log-scale)."""
    Lx = model.Lx
    RM = [None] * Lx
    RM[Lx - 1] = (np.ones((1, 1)), 0.0)
    for x in range(Lx - 1, 0, -1):
        c = ctx.cells[x]
        uvec, dvec = _above_vectors(model, y, x, above)
        rm, ls = RM[x]
        Gx = ctx.G[x][c.P["down"], c.P["dout"]]                     # [d, Dl, Dr']
        v = np.einsum("xab,bx->xa", Gx, rm[:, c.P["right"]])         # [d, Dl]
        v = v * (dvec[c.P["din"]] * uvec[c.P["up"]] * c.w)[:, None]
        RS = np.zeros((c.n["left"], v.shape[1]))
        np.add.at(RS, c.P["left"], v)
        new = (model.Bh[(y, x)] @ RS).T                             # [Dl, n_r(x-1)]
        s = np.abs(new).max()
        RM[x - 1] = (new / s, ls + np.log(s))
    return RM


def _above_vectors(model, y, x, above):
    if y == 0 or above is None:
        return np.ones(1), np.ones(1)
    up = model.cells[y - 1][x]
    uvec = model.Bv[(y, x)][up.P["down"][above[x]], :]
    if x > 0:
        ul = model.cells[y - 1][x - 1]
        dvec = model.Bd[(y, x)][ul.P["dout"][above[x - 1]], :]
    else:
        dvec = np.ones(1)
    return uvec, dvec


def _forward_legs(model, y, x, n_last):
    """Directions of cell (x, y) that lead to a cell visited AFTER cell index n_last (row-major order)."""
    out = []
    for d, (dy, dx) in (("right", (0, 1)), ("down", (1, 0)), ("dout", (1, 1))):
        yy, xx = y + dy, x + dx
        if yy < model.Ly and xx < model.Lx and yy * model.Lx + xx > n_last:
            out.append(d)
    return out


def boundary_codes(model, y, x, beam_states):
    """Boundary of every candidate (parent m, new state X of cell (x, y)), Eq. (8): the
    sub-configuration of the visited spins that couple to not yet visited cells, as
    (id of the parent's part, integer code of the new cell's part [d]).  Only rows y-1 and y can contribute."""
    Lx = model.Lx
    n = y * Lx + x
    ids, keys = {}, []
    for st in beam_states:
        key = []
        for yy in (y - 1, y):
            if yy < 0:
                continue
            for xx in range(Lx):
                idx = yy * Lx + xx
                if idx >= n:
                    break
                c = model.cells[yy][xx]
                for d in _forward_legs(model, yy, xx, n):
                    key.append(int(c.P[d][st[idx]]))
        keys.append(ids.setdefault(tuple(key), len(ids)))
    c = model.cells[y][x]
    code = np.zeros(c.d, dtype=np.int64)
    for d in _forward_legs(model, y, x, n):
        code = code * c.n[d] + c.P[d]
    return np.asarray(keys, dtype=np.int64), code


def merge_by_boundary(score, parent, state, parent_key, state_code):
    """Fig. 3(d): among candidates with the same boundary keep the most probable one
    (ties by the S8 order).  Returns the indices of the survivors."""
    key = parent_key[parent] * (int(state_code.max()) + 1) + state_code[state]
    order = np.lexsort((state, parent, -score, key))
    first = np.r_[True, key[order][1:] != key[order][:-1]]
    return np.sort(order[first])


class DropletBook:
    """Excitation bookkeeping on top of the merge (Fig. 4): every beam element (main branch)
    carries a list of droplets = low-energy excitations above it that do not modify its boundary.

    A droplet is (dE, flips) with flips = {cell index: xor mask on that cell's state bits}.  When candidates merge
    (same boundary), the most probable one is the main branch; every loser L gives the candidate droplet
    diff(L, main) with dE = (logp_main - logp_L) / beta (same boundary => the ratio of the marginals is
    exp(-beta dE) exactly for exact marginals), and every droplet d' already carried by L's parent gives the candidate
    diff(L, main) xor d' with dE_L + dE(d') ('together with excitations above (b) and (b') accumulated in the previous
    steps', Fig. 4 caption).  'To keep their number under control, we keep only those that are singly connected and
    with a hamming distance between any pair of them above a specified threshold': candidates are walked in increasing
    dE (ties: generation order = inherited ones first, then losers in the S8 order, each followed by its compositions)
    and kept iff dE <= max_dE, the flipped spins form ONE connected piece of the interaction graph (edges with
    J != 0), and the Hamming distance to every droplet already kept is >= min_hamming; at most max_count are kept
    (reading S24)."""

    def __init__(self, model, max_dE=1.0, min_hamming=1, max_count=8):
        self.max_dE, self.min_hamming, self.max_count = float(max_dE), int(min_hamming), int(max_count)
        inst = model.inst
        ncell = model.Ly * model.Lx
        self.nbits = model.nbits
        self.spin_of = -np.ones((ncell, model.nbits), dtype=np.int64)       # (cell, bit) -> spin id
        cell = inst.cell_y.astype(np.int64) * model.Lx + inst.cell_x
        bit = inst.sub.astype(np.int64) * inst.n_s + inst.pos
        self.spin_of[cell, bit] = np.arange(inst.n_spins)
        self.adj = [[] for _ in range(inst.n_spins)]
        for u, v, J in zip(inst.edge_u.tolist(), inst.edge_v.tolist(), inst.J.tolist()):
            if J != 0.0:
                self.adj[u].append(v)
                self.adj[v].append(u)

    def spins(self, flips):
        out = []
        for cidx, mask in flips.items():
            for b in range(self.nbits):
                if (mask >> b) & 1:
                    out.append(int(self.spin_of[cidx, b]))
        return out

    def connected(self, flips):
        sp = self.spins(flips)
        if not sp:
            return False
        todo, seen, inset = [sp[0]], {sp[0]}, set(sp)
        while todo:
            u = todo.pop()
            for v in self.adj[u]:
                if v in inset and v not in seen:
                    seen.add(v)
                    todo.append(v)
        return len(seen) == len(inset)

    @staticmethod
    def xor(f1, f2):
        out = dict(f1)
        for k, v in f2.items():
            w = out.get(k, 0) ^ v
            if w:
                out[k] = w
            else:
                out.pop(k, None)
        return out

    @staticmethod
    def hamming(f1, f2):
        return sum(bin(v).count("1") for v in DropletBook.xor(f1, f2).values())

    def select(self, cands):
        """cands: list of (dE, flips) in generation order -> kept list (greedy in increasing dE)."""
        order = sorted(range(len(cands)), key=lambda i: (cands[i][0], i))
        kept = []
        for i in order:
            dE, fl = cands[i]
            if len(kept) >= self.max_count:
                break
            if not (dE <= self.max_dE) or not fl or not self.connected(fl):
                continue
            if all(self.hamming(fl, k[1]) >= self.min_hamming for k in kept):
                kept.append((dE, fl))
        return kept


def branch_and_bound(model, R, lognorm, M, stats=None, merge=False, trace=None, droplets=None):
    """Returns dict(states [n, N] int8 +-1, energies [n], logp [n] (descending), log_pd, log_z,
    cell_states [n, Ly*Lx]).  `trace` (a list) receives, per cell, the absolute log-normaliser log Z_m of every beam
    element and, for every kept candidate, the absolute log of its 'rest' = u / (weights of the new cell) -- the two
    sides of the consistency identity P6, with every recorded scale factor added back.
    merge=True adds the paper's merge-by-boundary step (Fig. 3(d)) before the bound
    (reading S11: off by default; the CUDA path's counterpart is TN_OPT_MERGE).
    droplets=dict(max_dE, min_hamming, max_count) (needs merge=True) adds the excitation bookkeeping of Fig. 4
    (class DropletBook); the result then carries `droplets`: per returned state a list of (dE, flip mask [N] bool)."""
    Ly, Lx = model.Ly, model.Lx
    book = DropletBook(model, **droplets) if droplets is not None else None
    assert book is None or merge, "droplets need merge=True"
    drops = [[]]                        # per beam element: list of (dE, flips)
    beam_states = [[]]                  # per element: list of chosen cell states (row-major)
    beam_logp = np.zeros(1)
    log_pd = -np.inf
    log_z = None
    n_neg = 0
    for y in range(Ly):
        ctx = _RowCtx(model, y, R[y + 1])
        # B-1: right blocks at the row start, memoised by the boundary they depend on (Eq. (9))
        cache = {}
        slots = []
        for st in beam_states:
            above = tuple(st[(y - 1) * Lx:(y - 1) * Lx + Lx]) if y > 0 else None
            if above not in cache:
                cache[above] = _right_blocks(model, y, ctx, above)
            slots.append(cache[above])
        Lv = [np.ones(1) for _ in beam_states]
        Lv_ls = [0.0 for _ in beam_states]               # log of the scale removed from Lv (max-abs normalisation below)
        ls_rows = sum(lognorm[yy] for yy in range(y + 1, Ly))   # R_{y+1} is a unit vector: scale of the rows below
        for x in range(Lx):
            c = ctx.cells[x]
            cand_score, cand_parent, cand_state = [], [], []
            tables = []
            tr_logz, tr_rest = [], []
            for m, st in enumerate(beam_states):
                above = st[(y - 1) * Lx:(y - 1) * Lx + Lx] if y > 0 else None
                uvec, dvec = _above_vectors(model, y, x, above)
                hvec = model.Bh[(y, x)][ctx.cells[x - 1].P["right"][st[-1]], :] if x > 0 else np.ones(1)
                rm, rm_ls = slots[m][x]
                tab = np.einsum("a,pqac->pqc", Lv[m], ctx.G[x])          # Lv.S.Q for every (pd, po)
                val = np.einsum("xc,cx->x", tab[c.P["down"], c.P["dout"]], rm[:, c.P["right"]])
                u = hvec[c.P["left"]] * dvec[c.P["din"]] * uvec[c.P["up"]] * c.w * val
                if trace is not None:
                    with np.errstate(divide="ignore", invalid="ignore"):
                        tr_logz.append(np.log(np.maximum(u, 0.0).sum()) + Lv_ls[m] + rm_ls + ls_rows)
                        tr_rest.append(np.log(val) + Lv_ls[m] + rm_ls + ls_rows)
                n_neg += int(np.count_nonzero(u < 0))
                u = np.maximum(u, 0.0)                                     # S7
                Z = u.sum()
                if y == 0 and x == 0:                                      # C-6
                    log_z = (-model.beta * model.offset + sum(lognorm[yy] for yy in range(1, Ly))
                             + np.log(Z) + rm_ls)
                with np.errstate(divide="ignore"):
                    cand_score.append(beam_logp[m] + np.log(u / Z))
                cand_parent.append(np.full(c.d, m))
                cand_state.append(np.arange(c.d))
                tables.append(tab)
            score = np.concatenate(cand_score)
            parent = np.concatenate(cand_parent)
            state = np.concatenate(cand_state)
            if merge:
                pk, sc = boundary_codes(model, y, x, beam_states)
                if book is not None:
                    all_score, all_parent, all_state = score, parent, state
                    gkey = pk[parent] * (int(sc.max()) + 1) + sc[state]
                    gorder = np.lexsort((state, parent, -score, gkey))     # groups contiguous, winner first, S8 inside
                    gpos = np.empty(gorder.size, dtype=np.int64)
                    gpos[gorder] = np.arange(gorder.size)
                surv = merge_by_boundary(score, parent, state, pk, sc)
                score, parent, state = score[surv], parent[surv], state[surv]
                if stats is not None:
                    stats["merged_away"] = stats.get("merged_away", 0) + int(pk.size * sc.size - surv.size)
            keep, disc = select_top(score, parent, state, M)
            if stats is not None and keep.size == M and np.isfinite(disc):
                # bookkeeping for the parity tests: a cut that falls INSIDE a group of (numerically) tied candidates --
                # which members survive is then decided by rounding noise, and everything downstream that depends on
                # the identity of the survivors (later discarded probabilities, states of tied ranks) is not unique
                last = score[keep[-1]]
                if last - disc <= 1e-9 * max(1.0, abs(last)):
                    stats["tied_cuts"] = stats.get("tied_cuts", 0) + 1
            keep = keep[np.isfinite(score[keep])]                          # never keep p = 0
            new_drops = []
            if book is not None:
                n_cell = y * Lx + x
                for kk in keep:                                            # Fig. 4: losers of the winner's group
                    w = int(surv[kk])
                    mw, Xw, sw = int(all_parent[w]), int(all_state[w]), all_score[w]
                    cands = list(drops[mw])                                # excitations the main branch already carries
                    t = gpos[w] + 1
                    while t < gorder.size and gkey[gorder[t]] == gkey[w]:
                        l = int(gorder[t])
                        dE = (sw - all_score[l]) / model.beta
                        if not (dE <= book.max_dE):
                            break                                          # sorted by score: the rest is further away
                        ml, Xl = int(all_parent[l]), int(all_state[l])
                        base = {k: a ^ b for k, (a, b) in enumerate(zip(beam_states[ml], beam_states[mw])) if a != b}
                        if Xl != Xw:
                            base[n_cell] = Xl ^ Xw
                        cands.append((dE, base))
                        for (d2, f2) in drops[ml]:
                            if dE + d2 <= book.max_dE:
                                cands.append((dE + d2, DropletBook.xor(base, f2)))
                        t += 1
                    new_drops.append(book.select(cands))
            log_pd = max(log_pd, disc)
            new_states, new_Lv, new_slots, new_ls = [], [], [], []
            for k in keep:
                m, X = int(parent[k]), int(state[k])
                new_states.append(beam_states[m] + [X])
                lv = tables[m][c.P["down"][X], c.P["dout"][X]]
                new_Lv.append(lv / np.abs(lv).max())
                new_ls.append(Lv_ls[m] + np.log(np.abs(lv).max()))
                new_slots.append(slots[m])
            if trace is not None:
                trace.append(dict(cell=(y, x), log_z_abs=np.asarray(tr_logz),
                                  kept_rest_abs=np.asarray([tr_rest[int(parent[k])][int(state[k])] for k in keep])))
            beam_states, Lv, slots, Lv_ls = new_states, new_Lv, new_slots, new_ls
            if book is not None:
                drops = new_drops
            beam_logp = score[keep]
    cs = np.asarray(beam_states, dtype=np.int64)
    spins = model.spins_of_cells(cs)
    if stats is not None:
        stats["negative_u"] = n_neg
    out = dict(states=spins, energies=_energy.energies(model.inst, spins), logp=beam_logp,
               log_pd=log_pd, log_z=log_z, cell_states=cs)
    if book is not None:
        out["droplets"] = []
        for lst in drops:
            row = []
            for dE, fl in lst:
                mask = np.zeros(model.inst.n_spins, dtype=bool)
                mask[book.spins(fl)] = True
                row.append((dE, mask))
            out["droplets"].append(row)
    return out


def exact_marginal_beam(model, E_all, M):
    """O-3: the same beam, with conditionals from brute-force prefix marginals (Eq. (7))."""
    from . import brute
    inst = model.inst
    N, nb = inst.n_spins, model.nbits
    ncell = model.Ly * model.Lx
    d = 1 << nb
    prefix = np.zeros(1, dtype=np.int64)      # prefix value = low bits of the global state index
    logp = np.zeros(1)
    log_pd = -np.inf
    for n in range(ncell):
        lm = brute.prefix_log_marginals(E_all, model.beta, N, (n + 1) * nb)
        X = np.arange(d, dtype=np.int64)
        cand_prefix = (prefix[:, None] | (X[None, :] << (n * nb))).reshape(-1)
        score = lm[cand_prefix]
        parent = np.repeat(np.arange(prefix.size), d)
        state = np.tile(X, prefix.size)
        keep, disc = select_top(score, parent, state, M)
        log_pd = max(log_pd, disc)
        prefix, logp = cand_prefix[keep], score[keep]
    cs = (prefix[:, None] >> (np.arange(ncell) * nb)[None, :]) & (d - 1)
    spins = model.spins_of_cells(cs)
    return dict(states=spins, energies=_energy.energies(inst, spins), logp=logp, log_pd=log_pd, cell_states=cs)
