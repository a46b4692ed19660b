"""T-1: boundary MPS by zipper + truncated SVD + one-site variational passes.
Test infrastructure (see oracle/__init__.py).

PAPER.md:137 (boundary MPS, row after row), Sec. III B 1 PAPER.md:149-163 + Fig. 7 (sparse
diagrams: project the legs to the physical space of size d, batched matmul over the chi legs,
apply the local Boltzmann factor, project out), Sec. III B 2 PAPER.md:165-179 + Fig. 8 (zipper
right->left from a left-canonical MPS with the trivial 1x1x1 connector, SVD keeping chi values,
then variational overlap maximisation).  Readings of silent points: DESIGN.md section 3
(S1 converged truncated SVD = LAPACK dense SVD here; S2 schedule = whole zipper, then `sweeps`
passes; S4 one sweep = one pass, alternating, first left->right; S5 gap guard; S6 rank cut).

Conventions.  Row y is a chain of positions: Site_0 [, Med_0.5], Site_1, ...  (Med positions only
for 3-sub-cluster cells; otherwise Bh is folded into the left leg of the next site).
  MPS tensors      A[al, p, ar]          (p = lower physical leg of the row = R_{y+1}'s leg)
  new MPS tensors  N[g, p', g2]          (p' = upper leg = R_y's leg)
  environments     L[g, w, al], R[g2, w, ar]   (g: new bond, w: MPO bond, al/ar: old bond)
  connector        C = right environment (the zipper's U*Sigma IS the overlap environment)
Site MPO tensor (never built, except by `dense()` for the pins):
  W[(l,i), p', p, (r,o)] = sum_x w(x) d(l,Pl x) d(i,Pi x) d(r,Pr x) d(o,Po x) Bv[p',Pu x] d(p,Pd x)
Mediating tensor:  W[(r,o), q', q, (l',i')] = Bh[r,l'] d(q,o) Bd[q',i'].
"""
import numpy as np

RANK_TOL = 1e-14      # S6: singular values <= RANK_TOL * sigma_1 count as zero
GAP_GUARD = 1e-6      # S5: never cut between sigma_k, sigma_{k+1} closer than this (relative)


def _seg(idx, n):
    """stable grouping helper: order, segment starts and segment ids for scatter-add by idx."""
    order = np.argsort(idx, kind="stable")
    sidx = idx[order]
    starts = np.flatnonzero(np.r_[True, sidx[1:] != sidx[:-1]])
    return order, starts, sidx[starts]


def _scatter_add(out, idx, vals, seg=None):
    """out[idx[k]] += vals[k] (first axis)."""
    order, starts, ids = seg if seg is not None else _seg(idx, out.shape[0])
    out[ids] += np.add.reduceat(vals[order], starts, axis=0)
    return out


class SitePos:
    def __init__(self, model, y, x):
        c = model.cells[y][x]
        self.kind = "site"
        self.fold = not model.has_med
        self.w = c.w
        self.n_i, self.n_o = c.n["din"], c.n["dout"]
        self.iL = c.P["left"] * self.n_i + c.P["din"]
        self.iR = c.P["right"] * self.n_o + c.P["dout"]
        self.Pu, self.Pd = c.P["up"], c.P["down"]
        self.n_u = c.n["up"]
        self.nL = c.n["left"] * self.n_i
        self.Bv = model.Bv[(y, x)]                       # [p', u]
        self.Bh = model.Bh[(y, x)] if self.fold else None  # [r_prev, l]
        self.wl = self.Bh.shape[0] if self.fold else self.nL
        self.wr = c.n["right"] * self.n_o
        self.pu, self.pd = self.Bv.shape[0], c.n["down"]
        self.d = c.d
        self.chunk = 1 << 16

    # -- helpers -----------------------------------------------------------------------------
    def _left_in(self, L):
        return np.einsum("gra,rl->gla", L, self.Bh) if self.fold else L

    def _left_out(self, Ll):
        return np.einsum("gla,rl->gra", Ll, self.Bh) if self.fold else Ll

    def _chunks(self):
        for s in range(0, self.d, self.chunk):
            yield slice(s, min(self.d, s + self.chunk))

    # -- Fig. 7(a,b) diagrams ---------------------------------------------------------------
    def update(self, L, A, R):
        """N[g,p',g2] = sum L[g,wl,al] W[wl,p',p,wr] A[al,p,ar] R[g2,wr,ar]."""
        Ll = self._left_in(L)
        N0 = np.zeros((self.n_u, L.shape[0], R.shape[0]))
        for sl in self._chunks():
            Lx = Ll[:, self.iL[sl], :].transpose(1, 0, 2)          # [x, g, al]
            Ax = A[:, self.Pd[sl], :].transpose(1, 0, 2)           # [x, al, ar]
            Rx = R[:, self.iR[sl], :].transpose(1, 2, 0)           # [x, ar, g2]
            T = (Lx @ Ax @ Rx) * self.w[sl, None, None]
            _scatter_add(N0, self.Pu[sl], T)
        return np.einsum("pu,ugd->gpd", self.Bv, N0)

    def env_left(self, L, A, N):
        """L'[g2,wr,ar] = sum L[g,wl,al] N[g,p',g2] W[wl,p',p,wr] A[al,p,ar]."""
        Ll = self._left_in(L)
        Nb = np.einsum("pu,gpd->udg", self.Bv, N)                  # [u, g2, g]
        out = np.zeros((self.wr, N.shape[2], A.shape[2]))
        for sl in self._chunks():
            T = Nb[self.Pu[sl]] @ Ll[:, self.iL[sl], :].transpose(1, 0, 2) @ A[:, self.Pd[sl], :].transpose(1, 0, 2)
            _scatter_add(out, self.iR[sl], T * self.w[sl, None, None])
        return out.transpose(1, 0, 2)

    def env_right(self, R, A, N):
        """R'[g,wl,al] = sum N[g,p',g2] W[wl,p',p,wr] A[al,p,ar] R[g2,wr,ar]."""
        Nb = np.einsum("pu,gpd->ugd", self.Bv, N)                  # [u, g, g2]
        out = np.zeros((self.nL, N.shape[0], A.shape[0]))
        for sl in self._chunks():
            T = Nb[self.Pu[sl]] @ R[:, self.iR[sl], :].transpose(1, 0, 2) @ A[:, self.Pd[sl], :].transpose(1, 2, 0)
            _scatter_add(out, self.iL[sl], T * self.w[sl, None, None])
        return self._left_out(out.transpose(1, 0, 2))

    def theta(self, A, C):
        """Theta[(al,wl),(p',g)] = sum A[al,p,ar] W[wl,p',p,wr] C[g,wr,ar]  (Fig. 8(c) dashed box)."""
        out = np.zeros((self.nL * self.n_u, A.shape[0], C.shape[0]))
        for sl in self._chunks():
            T = A[:, self.Pd[sl], :].transpose(1, 0, 2) @ C[:, self.iR[sl], :].transpose(1, 2, 0)
            _scatter_add(out, self.iL[sl] * self.n_u + self.Pu[sl], T * self.w[sl, None, None])
        T0 = out.reshape(self.nL, self.n_u, A.shape[0], C.shape[0])
        T1 = np.tensordot(self.Bv, T0, axes=([1], [1]))                   # [p', l, al, g] = sum_u Bv[p',u] T0[l,u,al,g]
        if self.fold:
            T1 = np.tensordot(self.Bh, T1, axes=([1], [1]))               # [r, p', al, g] = sum_l Bh[r,l] T1[p',l,al,g]
            T1 = T1.transpose(2, 0, 1, 3)                                 # [al, r, p', g]
        else:
            T1 = T1.transpose(2, 1, 0, 3)                                 # [al, l, p', g]
        return T1.reshape(A.shape[0] * self.wl, self.pu * C.shape[0])

    def dense(self):
        """Explicit W[wl, p', p, wr] (tiny cells only; used by the pins)."""
        W0 = np.zeros((self.nL, self.n_u, self.pd, self.wr))
        np.add.at(W0, (self.iL, self.Pu, self.Pd, self.iR), self.w)
        W = np.einsum("pu,ludr->lpdr", self.Bv, W0)
        return np.einsum("rl,lpdw->rpdw", self.Bh, W) if self.fold else W


class MedPos:
    def __init__(self, model, y, x):
        """Mediating tensor between Site_x and Site_{x+1} of row y (Fig. 5)."""
        cl, cr = model.cells[y][x], model.cells[y][x + 1]
        self.kind = "med"
        self.Bh = model.Bh[(y, x + 1)]        # [r, l']
        self.Bd = model.Bd[(y, x + 1)]        # [q', i']
        self.n_r, self.n_o = cl.n["right"], cl.n["dout"]
        self.n_l, self.n_i = cr.n["left"], cr.n["din"]
        self.wl, self.wr = self.n_r * self.n_o, self.n_l * self.n_i
        self.pu, self.pd = self.Bd.shape[0], self.n_o

    def _L4(self, L):
        return L.reshape(L.shape[0], self.n_r, self.n_o, L.shape[2])

    def _R4(self, R):
        return R.reshape(R.shape[0], self.n_l, self.n_i, R.shape[2])

    def update(self, L, A, R):
        return np.einsum("groa,aob,rl,qi,dlib->gqd", self._L4(L), A, self.Bh, self.Bd, self._R4(R), optimize=True)

    def env_left(self, L, A, N):
        out = np.einsum("groa,gqd,aob,rl,qi->dlib", self._L4(L), N, A, self.Bh, self.Bd, optimize=True)
        return out.reshape(out.shape[0], self.wr, out.shape[3])

    def env_right(self, R, A, N):
        out = np.einsum("gqd,aob,rl,qi,dlib->groa", N, A, self.Bh, self.Bd, self._R4(R), optimize=True)
        return out.reshape(out.shape[0], self.wl, out.shape[3])

    def theta(self, A, C):
        T = np.einsum("aob,rl,qi,glib->aroqg", A, self.Bh, self.Bd, self._R4(C), optimize=True)
        return T.reshape(A.shape[0] * self.wl, self.pu * C.shape[0])

    def dense(self):
        # W[(r,o), q', q, (l',i')] = Bh[r,l'] d(q,o) Bd[q',i']
        W = np.einsum("rl,qi,ko->roqkli", self.Bh, self.Bd, np.eye(self.n_o))
        return W.reshape(self.wl, self.pu, self.pd, self.wr)


def row_positions(model, y):
    pos = []
    for x in range(model.Lx):
        pos.append(SitePos(model, y, x))
        if model.has_med and x + 1 < model.Lx:
            pos.append(MedPos(model, y, x))
    return pos


def trivial_mps(model):
    """R_{Ly} = 1: all legs of size 1."""
    n = 2 * model.Lx - 1 if model.has_med else model.Lx
    return [np.ones((1, 1, 1)) for _ in range(n)]


def left_canonicalize(A):
    """C-1: QR chain left->right (Fig. 8(c) 'initial MPS in the left canonical form').
    Returns the isometries and the final 1x1 factor (the signed norm)."""
    A = [a.copy() for a in A]
    for j in range(len(A)):
        al, p, ar = A[j].shape
        Q, Rf = np.linalg.qr(A[j].reshape(al * p, ar))
        A[j] = Q.reshape(al, p, Q.shape[1])
        if j + 1 < len(A):
            A[j + 1] = np.einsum("ab,bpc->apc", Rf, A[j + 1])
    assert Rf.shape == (1, 1)
    return A, Rf[0, 0]


def truncate_rank(s, D, gap_guard=True):
    """C-3 / S5 / S6: number of singular values kept."""
    if s.size == 0 or s[0] == 0.0:
        return 1
    k = int(np.count_nonzero(s > RANK_TOL * s[0]))
    if D > 0 and k > D:
        k = D
        if gap_guard:
            while k > 1 and s[k] >= (1.0 - GAP_GUARD) * s[k - 1]:
                k -= 1
    return max(k, 1)


_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def hash_uniform(seed, p, g, c):
    """Counter-based uniform(-1, 1) numbers Omega[(p', gamma), col] for the randomized SVD: SplitMix64's finaliser
    (public-domain, S. Vigna) of the counter seed * 0x100000001B3 + ((p' * 4096 + gamma) * 1024 + col).  The numbers the
    method draws are an INPUT of the algorithm (PAPER.md:169-177 'randomized SVD'); the CUDA path implements the same
    generator, indexed by (p', gamma, col) and not by any memory layout."""
    pp, gg, cc = np.meshgrid(np.arange(p, dtype=np.uint64), np.arange(g, dtype=np.uint64),
                             np.arange(c, dtype=np.uint64), indexing="ij")
    with np.errstate(over="ignore"):
        z = np.uint64(seed) * np.uint64(0x100000001B3) + ((pp * np.uint64(4096) + gg) * np.uint64(1024) + cc)
        z = z + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    u = (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    return (2.0 * u - 1.0).reshape(p * g, c)


def randomized_svd(Th, pu, g, ks, iters, seed):
    """Truncated randomized SVD of Theta (refs [43, 44] = randomized range finder with `iters`
    subspace iterations, matrix-free: only Theta x block and Theta^T x block are used):
        Om <- orth(Omega);  repeat iters times:  Y <- orth(Theta Om);  Z <- Theta^T Y;  Om <- orth(Z);
        B = Om^T Z = W diag(s) X^T  (small SVD);   right vectors V = Om W, Ritz values s.
    Returns (V [n, ks], s [ks]).  The connector is Theta V (exact for the chosen V), computed by the caller."""
    Om, _ = np.linalg.qr(hash_uniform(seed, pu, g, ks))
    Z = None
    for _ in range(max(1, iters)):
        Y, _ = np.linalg.qr(Th @ Om)
        Z = Th.T @ Y
        Om, _ = np.linalg.qr(Z)
    W, sv, _ = np.linalg.svd(Om.T @ Z)
    return Om @ W, sv


def truncate_mps(N, D, gap_guard=True, min_sigma=None):
    """Second step of the two-step truncation 2 chi -> chi ('targeting 2 chi singular values with
    randomized SVD, which, after variational refinement, are further truncated to the target chi singular values'):
    canonical MPS compression -- left-canonicalise, then SVD every bond right -> left keeping <= D values.
    Returns (tensors with unit norm, log of the norm removed by the truncation)."""
    N, r_last = left_canonicalize(N)
    n = len(N)
    N[n - 1] = N[n - 1] * r_last
    for j in range(n - 1, 0, -1):
        dl, p, dr = N[j].shape
        U, sv, Vt = np.linalg.svd(N[j].reshape(dl, p * dr), full_matrices=False)
        k = truncate_rank(sv, D, gap_guard)
        if min_sigma is not None and k < np.count_nonzero(sv > RANK_TOL * sv[0]):
            min_sigma.append(sv[k - 1] / sv[0])
        N[j] = Vt[:k].reshape(k, p, dr)
        N[j - 1] = np.einsum("apb,bc->apc", N[j - 1], U[:, :k] * sv[:k])
    nrm = np.linalg.norm(N[0])
    N[0] = N[0] / nrm
    return N, float(np.log(nrm))


def compress(positions, A, D, sweeps, gap_guard=True, stats=None, schedule=0, sweep_range=2, svd_mode=0,
             rsvd_iters=2, oversample=16, two_step=False, seed=None):
    """R_y = compress(T_y R_{y+1}; D, sweeps).  A: tensors of R_{y+1} (any gauge).
    Returns (tensors of R_y with unit norm, log of the norm removed).

    Options (readings S21-S23; the defaults are the parity definition S1-S4):
      schedule   0: whole zipper, then `sweeps` passes (the paper's variant (ii));
                 1: the paper's preferred schedule: every zipper step is followed by a variational sweep
                    of the instantaneous stage of the zipper over the `sweep_range` positions to the right of the
                    centre and back ('limit the range ... to a few tensors in the vicinity of the instantaneous
                    centre'), then `sweeps` global passes as before.
      svd_mode   0: converged truncated SVD (S1; LAPACK here); 1: randomized SVD with `rsvd_iters` subspace iterations
                 and `oversample` extra columns, random block from hash_uniform(seed[0]++).
      two_step   zipper and passes at bond 2 D, then truncate_mps to D.
      seed       one-element list: running count of truncated SVDs of this contraction (the random block's seed).

    Range (reading S19): the norm of a row is exp(-O(beta N_row)) and under/overflows fp64 on
    the large lattices, so every environment is kept at O(1) and the positive scale removed from it is
    carried as a logarithm: the zipper connector is divided by sigma_1 of each step, the variational
    environments by their Frobenius norm; lsR[j] / lsL[j] are the logs of what was removed from
    Renv[j] / Lenv[j].  Positive rescalings change nothing but the bookkeeping."""
    n = len(positions)
    A, r_last = left_canonicalize(A)
    Dz = 2 * D if (two_step and D > 0) else D       # bond kept by the zipper and the passes
    if seed is None:
        seed = [1]
    Renv = [None] * n
    lsR = [0.0] * n
    Renv[n - 1] = np.full((1, 1, 1), r_last)       # trivial unity connector x the folded norm
    N = [None] * n
    Lenv = [None] * n
    min_sigma = []
    ls0 = 0.0
    for j in range(n - 1, -1, -1):                  # C-2 zipper, right -> left
        pos = positions[j]
        Th = pos.theta(A[j], Renv[j])
        g = Renv[j].shape[0]
        if svd_mode == 1 and D > 0 and min(Th.shape) > Dz:
            ks = min(min(Dz, min(Th.shape)) + oversample, min(Th.shape))
            V, s = randomized_svd(Th, pos.pu, g, ks, rsvd_iters, seed[0])
            k = truncate_rank(s, Dz, gap_guard)
            Vk = V[:, :k]
            N[j] = Vk.T.reshape(k, pos.pu, g)
            scale = s[0] if s[0] > 0 else 1.0
            Cn = ((Th @ Vk) / scale).reshape(A[j].shape[0], pos.wl, k)
        else:
            U, s, Vt = np.linalg.svd(Th, full_matrices=False)
            k = truncate_rank(s, Dz, gap_guard)
            N[j] = Vt[:k].reshape(k, pos.pu, g)
            scale = s[0] if s[0] > 0 else 1.0
            Cn = (U[:, :k] * (s[:k] / scale)).reshape(A[j].shape[0], pos.wl, k)
        seed[0] += 1
        min_sigma.append(s[k - 1] / s[0] if s[0] > 0 else 0.0)
        if j > 0:
            Renv[j - 1] = Cn.transpose(2, 1, 0)
            lsR[j - 1] = lsR[j] + np.log(scale)
        else:
            ls0 = lsR[0] + np.log(scale)
        if schedule == 1 and D > 0 and sweep_range > 0 and j < n - 1:
            # ---- variational sweep of the instantaneous stage of the zipper, positions j .. kmax.
            # The block [connector . N_j ... N_kmax ...] approximates (A_j W_j) ... (A_{n-1} W_{n-1}) with its left
            # legs (old bond, MPO bond) open; an orthonormal basis Q of the connector's range on those legs plays the
            # left environment of position j (reading S21).
            kmax = min(n - 1, j + sweep_range)
            al, wl = A[j].shape[0], pos.wl
            Q, _ = np.linalg.qr(Cn.reshape(al * wl, k))
            Lenv[j] = Q.reshape(al, wl, Q.shape[1]).transpose(2, 1, 0)
            for q in range(j, kmax):                                   # left -> right
                N[q] = positions[q].update(Lenv[q], A[q], Renv[q])
                g1, p1, g2 = N[q].shape
                Qq, _ = np.linalg.qr(N[q].reshape(g1 * p1, g2))
                N[q] = Qq.reshape(g1, p1, Qq.shape[1])
                E = positions[q].env_left(Lenv[q], A[q], N[q])
                Lenv[q + 1] = E / np.linalg.norm(E)
            for q in range(kmax, j - 1, -1):                           # right -> left, back to the zipper's centre
                N[q] = positions[q].update(Lenv[q], A[q], Renv[q])
                g1, p1, g2 = N[q].shape
                Qq, _ = np.linalg.qr(N[q].reshape(g1, p1 * g2).T)
                N[q] = Qq.T.reshape(Qq.shape[1], p1, g2)
                E = positions[q].env_right(Renv[q], A[q], N[q])
                nE = np.linalg.norm(E)
                if q > 0:
                    Renv[q - 1] = E / nE
                    lsR[q - 1] = lsR[q] + np.log(nE)
                else:
                    Cn = (E / nE).transpose(2, 1, 0)
                    ls0 = lsR[0] + np.log(nE)
    assert Cn.shape == (1, 1, 1)
    centre = 0
    N[0] = N[0] * Cn[0, 0, 0]
    lsL = [0.0] * n
    log_centre = ls0                                # log of the scale carried beside N[centre]
    norms = []
    if D > 0 and sweeps > 0:                        # C-5: exact mode skips the passes
        Lenv = [None] * n
        Lenv[0] = np.ones((1, 1, 1))
        for sweep in range(sweeps):                 # C-4
            if sweep % 2 == 0:
                for j in range(n):
                    N[j] = positions[j].update(Lenv[j], A[j], Renv[j])
                    log_centre = lsL[j] + lsR[j]
                    norms.append(np.linalg.norm(N[j]) * np.exp(log_centre))
                    if j + 1 < n:
                        g, p, g2 = N[j].shape
                        Q, _ = np.linalg.qr(N[j].reshape(g * p, g2))
                        N[j] = Q.reshape(g, p, Q.shape[1])
                        E = positions[j].env_left(Lenv[j], A[j], N[j])
                        nE = np.linalg.norm(E)
                        Lenv[j + 1] = E / nE
                        lsL[j + 1] = lsL[j] + np.log(nE)
                centre = n - 1
            else:
                for j in range(n - 1, -1, -1):
                    N[j] = positions[j].update(Lenv[j], A[j], Renv[j])
                    log_centre = lsL[j] + lsR[j]
                    norms.append(np.linalg.norm(N[j]) * np.exp(log_centre))
                    if j > 0:
                        g, p, g2 = N[j].shape
                        Q, _ = np.linalg.qr(N[j].reshape(g, p * g2).T)
                        N[j] = Q.T.reshape(Q.shape[1], p, g2)
                        E = positions[j].env_right(Renv[j], A[j], N[j])
                        nE = np.linalg.norm(E)
                        Renv[j - 1] = E / nE
                        lsR[j - 1] = lsR[j] + np.log(nE)
                centre = 0
    nrm = np.linalg.norm(N[centre])
    N[centre] = N[centre] / nrm
    ln_trunc = 0.0
    if two_step and D > 0:
        N, ln_trunc = truncate_mps(N, D, gap_guard, min_sigma)
    log_centre += ln_trunc
    if stats is not None:
        stats.setdefault("min_sigma", []).append(min(min_sigma))
        stats.setdefault("pass_norms", []).append(norms)
        stats.setdefault("bonds", []).append([t.shape[2] for t in N])
    return N, float(np.log(nrm) + log_centre)


def contract(model, D, sweeps, gap_guard=True, stats=None, **options):
    """Boundary MPS R_y for y = Ly .. 1 (R_0 is never needed: log Z comes from the first cell's
    normaliser in the search, C-6).  Returns {y: tensors}, {y: log-norm}.  `options`: see compress."""
    R = {model.Ly: trivial_mps(model)}
    lognorm = {model.Ly: 0.0}
    seed = [1]                                      # running count of truncated SVDs (seed of the random blocks)
    for y in range(model.Ly - 1, 0, -1):
        R[y], lognorm[y] = compress(row_positions(model, y), R[y + 1], D, sweeps, gap_guard, stats, seed=seed,
                                    **options)
    return R, lognorm


def mps_to_dense(T):
    """Boundary MPS -> dense array with one axis per position (tiny only)."""
    v = T[0]
    for t in T[1:]:
        v = np.tensordot(v, t, axes=([v.ndim - 1], [0]))
    return v.reshape(v.shape[1:-1])


def mpo_mps_dense(positions, A):
    """Exact (untruncated) T_y R_{y+1} as a dense array, via the explicit W tensors (tiny only)."""
    v = None
    for pos, a in zip(positions, A):
        t = np.einsum("wpdv,adb->awpvb", pos.dense(), a)         # [al, wl, p', wr, ar]
        if v is None:
            v = t[0, 0]                                            # [p', wr, ar]
        else:
            v = np.tensordot(v, t, axes=([v.ndim - 2, v.ndim - 1], [1, 0]))
    return v.reshape(v.shape[:-2])
