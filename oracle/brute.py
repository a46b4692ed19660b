"""O-1: brute-force enumeration of all 2^N states.  Test infrastructure (see oracle/__init__.py).

State index k in [0, 2^N): bit i of k is spin i, s_i = 1 - 2*bit_i (bit 0 -> +1).
Boltzmann distribution Eq. (6), partition function Eq. (10) PAPER.md:119,
prefix marginals / chain rule Eq. (7) PAPER.md:96.  Cells are consecutive in spin-id order, so
the first n cells are the low n*(S*n_s) bits of k.
"""
import numpy as np


def all_energies(inst, chunk_bits=20):
    """Energy of every state, shape [2^N] (N <= 28).  Summation order here is edge-by-edge
    vectorised over states (not bit-comparable with O-0; use energy.energies for that)."""
    N = inst.n_spins
    assert N <= 28
    total = 1 << N
    out = np.empty(total, dtype=np.float64)
    cb = min(chunk_bits, N)
    eu, ev, J, h = inst.edge_u, inst.edge_v, inst.J, inst.h
    for start in range(0, total, 1 << cb):
        k = np.arange(start, start + (1 << cb), dtype=np.int64)
        E = np.zeros(1 << cb)
        for u, v, j in zip(eu.tolist(), ev.tolist(), J.tolist()):
            E += j * (1.0 - 2.0 * (((k >> u) ^ (k >> v)) & 1))
        for i, hi in enumerate(h.tolist()):
            if hi != 0.0:
                E += hi * (1.0 - 2.0 * ((k >> i) & 1))
        out[start:start + (1 << cb)] = E
    return out


def log_z(E, beta):
    m = (-beta * E).max()
    return m + np.log(np.exp(-beta * E - m).sum())


def lowest(E, M):
    """(state indices, energies) of the M lowest energies, ascending (ties by index)."""
    M = min(M, E.size)
    idx = np.argpartition(E, M - 1)[:M] if M < E.size else np.arange(E.size)
    idx = idx[np.lexsort((idx, E[idx]))]
    return idx, E[idx]


def index_to_spins(k, N):
    k = np.asarray(k, dtype=np.int64)
    return (1 - 2 * ((k[..., None] >> np.arange(N)) & 1)).astype(np.int8)


def prefix_log_marginals(E, beta, N, n_bits):
    """log p(low n_bits of the state) for every prefix value, shape [2^n_bits]."""
    lz = log_z(E, beta)
    m = (-beta * E).max()
    w = np.exp(-beta * E - m).reshape(1 << (N - n_bits), 1 << n_bits)
    with np.errstate(divide="ignore"):
        return np.log(w.sum(axis=0)) + m - lz
