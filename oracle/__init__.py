"""CPU oracle for the boundary-MPS / branch-and-bound hot path of arXiv 2411.16431.

TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 numpy code written from the paper
(/root/reference/PAPER.md; citations are `PAPER.md:<line>` + section/equation).  It shares
no code with the CUDA path (`paper_2411_16431_b200/`), never imports it, and may only be
imported by `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / reference
legs.  Inputs come from `instances/` (seeded generators, no method arithmetic).

Modules
  energy    O-0  fixed-order Ising energy, Eq. (1)
  brute     O-1  enumeration of all 2^N states: log Z, lowest energies, prefix marginals
  model          clustered Potts form, projectors, edge matrices: Eqs. (3)-(5) PAPER.md:69-84
  transfer  O-2  exact (untruncated, dense-vector) row transfer contraction
  mps       T-1  boundary MPS: zipper + truncated SVD + 1-site variational passes,
                 Sec. III B 2 PAPER.md:165-179, Fig. 8
  search    T-2  branch and bound, Eqs. (7)-(9) PAPER.md:94-113, Fig. 3, Fig. 6;  O-3 exact-marginal beam

Pins (tests/test_oracle_*.py, `-m "not gpu"`): brute force == exact transfer matrix == exact-D
MPS (log Z, every boundary vector); closed forms (J = 0, trees, small beta); gauge and Z2
invariances; no-prune beam == brute-force lowest-M; beam at exact D == exact-marginal beam;
final logp == -beta E - log Z; loop-planted E0 by brute force; sparse diagrams == explicit
dense MPO einsum; gauge independence and variational monotonicity of `compress`.
Parity unpinned (no external ground truth exists): truncated-D results on lattices too large
for brute force -- there the oracle is pinned only through the properties above.
"""
