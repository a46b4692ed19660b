"""Clustered (Potts) form of the Ising instance, projectors and edge matrices.
Test infrastructure (see oracle/__init__.py).

Eq. (3):  H = sum_<m,n> E_{x_m x_n} + sum_n E_{x_n}   (cells on a square grid with
nearest-neighbour and one diagonal coupling, Fig. 1(b,d) PAPER.md:31).
Eqs. (4)-(5) PAPER.md:78-84:  E_{x_m x_n} = Ebar[P^{mn}(x_m), P^{nm}(x_n)] with P^{mn} projecting the
d cell states onto the distinct sub-configurations of the spins actually coupled to cell n.
Fig. 5(c): bond tensors are exp(-beta Ebar).

Dense formulation: every cell carries explicit length-d tables (d = 2^(spins per cell)); no use
is made of any structure inside the cell.  Cell state x: bit (sub*n_s + pos) of x is that spin,
s = 1 - 2*bit.  Projected index = bits of the coupled spins packed in increasing bit order
(reading S10 in DESIGN.md).  Directions: left/right (x-1 / x+1), up/down (y-1 / y+1),
din/dout (from (x-1,y-1) / to (x+1,y+1)).  "Coupled" = has an edge in the list, even if J = 0 (S9).
"""
import numpy as np

DIRS = ("left", "right", "up", "down", "din", "dout")


class Cell:
    def __init__(self, nbits):
        self.nbits = nbits
        self.d = 1 << nbits
        self.E = np.zeros(self.d)                 # intra-cell energy E_{x_n}, Eq. (3)
        self.coupled = {k: [] for k in DIRS}      # cell-bit indices coupled in each direction
        self.P = {}                               # projector index tables, Eq. (5)
        self.n = {}                               # their ranges d^{mn}

    def finish(self):
        x = np.arange(self.d, dtype=np.int64)
        for k in DIRS:
            bits = sorted(set(self.coupled[k]))
            self.coupled[k] = bits
            idx = np.zeros(self.d, dtype=np.int64)
            for t, b in enumerate(bits):
                idx |= ((x >> b) & 1) << t
            self.P[k] = idx
            self.n[k] = 1 << len(bits)


def _spin_of_proj(bits, b, n):
    """+-1 value of cell-bit b as a function of the projected index (length n)."""
    t = bits.index(b)
    return 1.0 - 2.0 * ((np.arange(n) >> t) & 1)


class Model:
    def __init__(self, inst):
        self.inst = inst
        Ly, Lx = inst.Ly, inst.Lx
        self.Ly, self.Lx = Ly, Lx
        self.nbits = inst.S * inst.n_s
        self.has_med = inst.S == 3
        cy, cx = inst.cell_y, inst.cell_x
        bit = (inst.sub.astype(np.int64) * inst.n_s + inst.pos).tolist()
        self.cells = [[Cell(self.nbits) for _ in range(Lx)] for _ in range(Ly)]
        inter = {"h": {}, "v": {}, "d": {}}       # (y,x) of the right/lower cell -> [(bit_m, bit_n, J)]
        xs = np.arange(1 << self.nbits, dtype=np.int64)
        for u, v, J in zip(inst.edge_u.tolist(), inst.edge_v.tolist(), inst.J.tolist()):
            a, b = (cy[u], cx[u]), (cy[v], cx[v])
            if a == b:
                c = self.cells[a[0]][a[1]]
                c.E += J * (1.0 - 2.0 * (((xs >> bit[u]) ^ (xs >> bit[v])) & 1))
                continue
            if (b[0], b[1]) < (a[0], a[1]):
                u, v, a, b = v, u, b, a
            dy, dx = b[0] - a[0], b[1] - a[1]
            if (dy, dx) == (0, 1):
                kind, da, db = "h", "right", "left"
            elif (dy, dx) == (1, 0):
                kind, da, db = "v", "down", "up"
            elif (dy, dx) == (1, 1):
                kind, da, db = "d", "dout", "din"
            else:
                raise ValueError(f"edge ({u},{v}) joins cells {a} and {b}: not NN or (x+1,y+1) diagonal")
            self.cells[a[0]][a[1]].coupled[da].append(bit[u])
            self.cells[b[0]][b[1]].coupled[db].append(bit[v])
            inter[kind].setdefault((b[0], b[1]), []).append((bit[u], bit[v], J))
        for i, hi in enumerate(inst.h.tolist()):
            if hi != 0.0:
                self.cells[cy[i]][cx[i]].E += hi * (1.0 - 2.0 * ((xs >> bit[i]) & 1))
        for row in self.cells:
            for c in row:
                c.finish()
        # compressed interaction energies Ebar, Eq. (4); key (y,x) = the right / lower / lower-right cell
        self.Eh, self.Ev, self.Ed = {}, {}, {}
        for y in range(Ly):
            for x in range(Lx):
                for kind, tab, (py, px), da, db in (("h", self.Eh, (y, x - 1), "right", "left"),
                                                    ("v", self.Ev, (y - 1, x), "down", "up"),
                                                    ("d", self.Ed, (y - 1, x - 1), "dout", "din")):
                    if py < 0 or px < 0:
                        tab[(y, x)] = np.zeros((1, 1))
                        continue
                    ca, cb = self.cells[py][px], self.cells[y][x]
                    M = np.zeros((ca.n[da], cb.n[db]))
                    for (bu, bv, J) in inter[kind].get((y, x), []):
                        M += J * np.outer(_spin_of_proj(ca.coupled[da], bu, ca.n[da]),
                                          _spin_of_proj(cb.coupled[db], bv, cb.n[db]))
                    tab[(y, x)] = M
        self.beta = None

    def set_beta(self, beta):
        """Boltzmann factors, each table shifted by its minimum; `offset` = sum of the minima, so
        exp(-beta H) = exp(-beta offset) * prod(factors)   (Eq. (6))."""
        self.beta = float(beta)
        self.offset = 0.0
        self.Bh, self.Bv, self.Bd = {}, {}, {}
        for y in range(self.Ly):
            for x in range(self.Lx):
                c = self.cells[y][x]
                m = c.E.min()
                self.offset += m
                c.w = np.exp(-self.beta * (c.E - m))
                for src, dst in ((self.Eh, self.Bh), (self.Ev, self.Bv), (self.Ed, self.Bd)):
                    m = src[(y, x)].min()
                    self.offset += m
                    dst[(y, x)] = np.exp(-self.beta * (src[(y, x)] - m))
        return self

    def spins_of_cells(self, cell_states):
        """cell states [n, Ly*Lx] (row-major) -> +-1 spins [n, N] in spin-id order."""
        cs = np.asarray(cell_states, dtype=np.int64)
        inst = self.inst
        cell = inst.cell_y.astype(np.int64) * self.Lx + inst.cell_x
        bit = inst.sub.astype(np.int64) * inst.n_s + inst.pos
        return (1 - 2 * ((cs[:, cell] >> bit[None, :]) & 1)).astype(np.int8)
