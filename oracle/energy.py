"""O-0: Ising energy in a fixed summation order.  Test infrastructure (see oracle/__init__.py).

Eq. (1):  H(s) = sum_<ij> J_ij s_i s_j + sum_i h_i s_i.

Fixed order: ONE running fp64 sum, first over the edges in input order, then over the spins in
index order:  E = (((0 + J_0 s_u0 s_v0) + J_1 s_u1 s_v1) + ...) + h_0 s_0 + ... .  Each term
J*(+-1) is exact, so the result is fully determined by the order; this is what makes energies
bit-comparable between implementations.
"""
import numpy as np


def energy(inst, s):
    """Sequential-order energy of one state s (array of +-1, spin-id order). Pure Python loop."""
    E = 0.0
    for u, v, J in zip(inst.edge_u.tolist(), inst.edge_v.tolist(), inst.J.tolist()):
        E = E + J * float(int(s[u]) * int(s[v]))
    for i, hi in enumerate(inst.h.tolist()):
        E = E + hi * float(int(s[i]))
    return E


def energies(inst, states):
    """Same sum for many states [n, N]; np.cumsum adds strictly left to right."""
    s = np.asarray(states, dtype=np.float64)
    if s.ndim == 1:
        s = s[None, :]
    terms = np.concatenate([inst.J[None, :] * (s[:, inst.edge_u] * s[:, inst.edge_v]),
                            inst.h[None, :] * s], axis=1)
    if terms.shape[1] == 0:
        return np.zeros(s.shape[0])
    return np.cumsum(terms, axis=1)[:, -1]
