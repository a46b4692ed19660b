"""O-2: exact row-transfer contraction with dense boundary vectors (tiny lattices only).
Test infrastructure (see oracle/__init__.py).

The PEPS is an exact representation of Z (Eq. (10), Fig. 5).  With R_{Ly} = 1,

  R_y(p', q') = sum_{row-y states X} prod_x [ w_x(X_x) Bv_x[p'_x, P_up X_x] Bd_x[q'_{x-1}, P_din X_x]
                                              Bh_x[P_right X_{x-1}, P_left X_x] ] R_{y+1}(P_down X, P_dout X)

where p'_x = P_down of cell (x, y-1) and q'_x = P_dout of cell (x, y-1) are the legs left open
towards the row above (SURVEY.md section 8.0 recursion).  R_y is stored as
an array with axes (p'_0, ..., p'_{Lx-1}, q'_0, ..., q'_{Lx-2}) and NO truncation or normalisation
beyond a tracked log-scale.  Z = exp(-beta offset) * R_0.
"""
import numpy as np


def _row_apply(model, y, Rn):
    """One application of the recursion; Rn has axes (p_0..p_{Lx-1}, q_0..q_{Lx-2}) of row y."""
    Lx = model.Lx
    cells = model.cells[y]
    d = cells[0].d
    # val[X_0,...,X_{Lx-1}] = prod_x w_x * prod_x Bh_x * R_{y+1}(P_down X, P_dout X)
    grids = np.meshgrid(*[np.arange(d)] * Lx, indexing="ij")
    val = np.ones([d] * Lx)
    for x in range(Lx):
        c = cells[x]
        val = val * c.w[grids[x]]
        if x > 0:
            val = val * model.Bh[(y, x)][cells[x - 1].P["right"][grids[x - 1]], c.P["left"][grids[x]]]
    idx = tuple(cells[x].P["down"][grids[x]] for x in range(Lx)) + \
        tuple(cells[x].P["dout"][grids[x]] for x in range(Lx - 1))
    val = val * Rn[idx]
    # contract each X_x with F_x[(p'_x, q'_{x-1}), X_x] = Bv_x[p'_x, P_up X_x] * Bd_x[q'_{x-1}, P_din X_x]
    # after the loop the axes are (p'_0, q'_-1(=1), p'_1, q'_0, ..., p'_{Lx-1}, q'_{Lx-2})
    for x in range(Lx):
        c = cells[x]
        F = model.Bv[(y, x)][:, c.P["up"]][:, None, :] * model.Bd[(y, x)][:, c.P["din"]][None, :, :]
        val = np.tensordot(val, F, axes=([0], [2]))      # consumed axis first, new axes appended last
    # axis 1 (q'_{-1}) always has size 1: cell x=0 has no din neighbour
    assert val.shape[1] == 1
    val = np.squeeze(val, axis=1)
    p_axes = [0] + [2 * x - 1 for x in range(1, Lx)]
    q_axes = [2 * x for x in range(1, Lx)]
    return np.transpose(val, p_axes + q_axes)


def boundary_vectors(model):
    """Exact R_y for y = Ly .. 0 as (array, log-scale) pairs: R_y_true = array * exp(log-scale)."""
    Ly, Lx = model.Ly, model.Lx
    R = {Ly: (np.ones([1] * (2 * Lx - 1)), 0.0)}
    for y in range(Ly - 1, -1, -1):
        arr, ls = R[y + 1]
        new = _row_apply(model, y, arr)
        s = np.abs(new).max()
        R[y] = (new / s, ls + np.log(s))
    return R


def log_z(model):
    R = boundary_vectors(model)
    arr, ls = R[0]
    return -model.beta * model.offset + ls + np.log(arr.reshape(-1)[0]), R
