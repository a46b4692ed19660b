"""Local dimensional reduction by loopy belief propagation (Sec. IV, Eqs. (11)-(13), Fig. 9).
Test infrastructure (see oracle/__init__.py).

Dense formulation on the clustered model of oracle/model.py: every cell carries its length-d weight vector
w(x) = exp(-beta (E_x - min)) and the projector index tables P^{mn}; edge matrices are exp(-beta (Ebar - min)).
Messages live on the directed neighbour pairs of the cell grid (left/right, up/down, din/dout):

  nu_{m->n}(xbar_n)   message from the edge <m,n> to cluster n, a vector over P^{nm}(x_n)   [black half-circles of Fig. 9]
  mu_{m->n}(xbar_m)   message from cluster m towards the edge <m,n>, a vector over P^{mn}(x_m) [green half-circles]

  Eq. (11)  mu_{mn}(xbar_m) = sum_{x_m : P^{mn}(x_m) = xbar_m} exp(-beta E_{x_m}) prod_{m' in N(m) \\ n} nu_{m'm}(P^{mm'}(x_m))
  Eq. (12)  nu_{mn}(xbar_n) = sum_{xbar_m} exp(-beta Ebar_{xbar_n xbar_m}) mu_{mn}(xbar_m)
  Eq. (13)  p(x_n) ~ exp(-beta E_{x_n}) prod_{m in N(n)} nu_{mn}(P^{nm}(x_n))

Readings (S26): messages start uniform; one iteration = ALL cluster -> edge messages from the
current nu (Fig. 9(c)), then ALL edge -> cluster messages (Fig. 9(d)) ("a fixed number of such updates");
every nu is normalised to sum 1 after Eq. (12) (a positive rescaling: it cancels in Eq. (13) after normalisation);
neighbours that do not exist, or carry no coupling (a 1 x 1 edge matrix), send the constant message 1; the K most
probable states are taken in the order (p descending, state index ascending).
"""
import numpy as np

# direction of the neighbour as seen from a cell, its grid offset (dy, dx), and the direction back
DIRS = {"left": ((0, -1), "right"), "right": ((0, 1), "left"), "up": ((-1, 0), "down"), "down": ((1, 0), "up"),
        "din": ((-1, -1), "dout"), "dout": ((1, 1), "din")}


def _edge_matrix(model, y, x, d):
    """exp(-beta Ebar) between cell (y, x) and its neighbour in direction d, as [index of the neighbour's leg,
    index of this cell's leg d]."""
    if d == "left":
        return model.Bh[(y, x)]                    # [r of the left cell, l]
    if d == "up":
        return model.Bv[(y, x)]                    # [down of the upper cell, u]
    if d == "din":
        return model.Bd[(y, x)]                    # [dout of the upper-left cell, i]
    (dy, dx), _ = DIRS[d]
    B = {"right": model.Bh, "down": model.Bv, "dout": model.Bd}[d][(y + dy, x + dx)]
    return B.T                                     # stored as [this cell's leg, neighbour's leg]


def messages(model, iterations):
    """nu[(y, x)][d]: message arriving at cell (y, x) from its neighbour in direction d, over the cell's leg d."""
    Ly, Lx = model.Ly, model.Lx

    def exists(y, x, d):
        (dy, dx), _ = DIRS[d]
        if d in ("din", "dout") and not model.has_med:
            return False
        return 0 <= y + dy < Ly and 0 <= x + dx < Lx

    nu = {(y, x): {d: np.ones(model.cells[y][x].n[d]) for d in DIRS} for y in range(Ly) for x in range(Lx)}
    for _ in range(iterations):
        mu = {}
        for y in range(Ly):                                        # Eq. (11), Fig. 9(c)
            for x in range(Lx):
                c = model.cells[y][x]
                for d in DIRS:
                    if not exists(y, x, d):
                        continue
                    f = c.w.copy()
                    for d2 in DIRS:
                        if d2 != d:
                            f = f * nu[(y, x)][d2][c.P[d2]]
                    out = np.zeros(c.n[d])
                    np.add.at(out, c.P[d], f)
                    mu[(y, x, d)] = out
        new = {}
        for y in range(Ly):                                        # Eq. (12), Fig. 9(d)
            for x in range(Lx):
                new[(y, x)] = {}
                for d, ((dy, dx), back) in DIRS.items():
                    n = model.cells[y][x].n[d]
                    if not exists(y, x, d):
                        new[(y, x)][d] = np.ones(n)
                        continue
                    B = _edge_matrix(model, y, x, d)               # [neighbour's leg, this cell's leg]
                    v = mu[(y + dy, x + dx, back)] @ B
                    new[(y, x)][d] = v / v.sum()
        nu = new
    return nu


def log_marginals(model, nu, y, x):
    """Eq. (13): log of the normalised LBP marginal of every state of cell (y, x)."""
    c = model.cells[y][x]
    f = c.w.copy()
    for d in DIRS:
        f = f * nu[(y, x)][d][c.P[d]]
    with np.errstate(divide="ignore"):
        return np.log(f / f.sum())


def select(model, nu, y, x, K):
    """The K most probable states of cell (y, x) according to LBP: (states, log p), p descending,
    ties by ascending state index."""
    lp = log_marginals(model, nu, y, x)
    order = np.lexsort((np.arange(lp.size), -lp))[:K]
    return order, lp[order]
