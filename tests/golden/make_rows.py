"""Writes tests/golden/rows_<case>.npz: results of the CPU oracle on cases that are too slow to run inside the test
suite (minutes to an hour each), so that the GPU parity tests can compare against them without re-running them.

    python tests/golden/make_rows.py <case> [<case> ...]        # or: all

Calls only oracle/ (and the shared seeded generators in instances/).  Nothing here comes from the CUDA path: the
stored values are the oracle's, as SURVEY.md section 8(d) "Oracle timing" planned ("the oracle writes R_y and its final
lists to disk keyed by a hash of (instance, beta, D, sweeps, options)").  The full R_y tensors would be tens of MB per
case, so each row is stored as
  * its Schmidt spectrum at every bond (gauge independent, fixes the state up to local unitaries),
  * K = 192 of its amplitudes <p'_0 q'_0 p'_1 ... | R_y> at boundary configurations drawn (seeded) from |R_y|^2 --
    sampled ELEMENTS of the output vector, which the test evaluates on the CUDA path's tensors one by one,
together with the final lists (cell states, log-probabilities, log p_d, log Z, energies).
tests/test_gpu_golden.py rebuilds the instance from the recipe below, checks its hash and compares.
"""
import hashlib
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import instances  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
K_SAMPLES = 192

# name -> (generator, args, run parameters).  Sizes follow VERDICT r1 "Next round" item 1: the code paths that
# produce the headline numbers (D = 32 / 64 bonds, full 8-spin sub-clusters, Pegasus-shaped cells with Ly >= 3 so that
# the Theta-core build and the mediating positions see non-trivial old bonds, rank-deficient loop-planted blocks).
CASES = {
    # (i) Zephyr-shaped full cells, the configs[1]/[4] cell: d = 2^16, Theta 8192 x 8192 per middle position
    "zephyr4x4_D32": ("lattice", dict(Ly=4, Lx=4, S=2, n_s=8, p_keep=0.97, seed=3), dict(beta=2.0, D=32, sweeps=1, M=1024)),
    # (ii) the same shape loop-planted at beta = 4: rank-deficient blocks (reading S6), the configs[4] regime
    "zephyr4x4_planted_D32": ("loops", dict(Ly=4, Lx=4, S=2, n_s=8, seed=3), dict(beta=4.0, D=32, sweeps=1, M=1024)),
    # (iii) Pegasus-shaped full 24-spin cells with three rows: d = 2^24, w_h = 4096
    "pegasus3x2_D8": ("lattice", dict(Ly=3, Lx=2, S=3, n_s=8, p_keep=0.97, seed=5), dict(beta=1.0, D=8, sweeps=2, M=16)),
    # the configs[2] code path itself: D = 32 on full Pegasus cells, Theta 131072 x 8192 at the middle site
    # (M = 0: rows only -- the oracle's right blocks at d = 2^24 and D = 32 need a 128 GiB gather, beyond this host)
    "pegasus3x3_D32": ("lattice", dict(Ly=3, Lx=3, S=3, n_s=8, p_keep=0.97, seed=0), dict(beta=2.0, D=32, sweeps=1, M=0)),
    # (iv) bonds 49..64 at truncated D: the K = 64 instantiations (configs[3] path)
    "zephyr3x3_D56": ("lattice", dict(Ly=3, Lx=3, S=2, n_s=8, p_keep=0.97, seed=7), dict(beta=1.0, D=56, sweeps=1, M=256)),
    "zephyr3x3_D64_h0": ("lattice", dict(Ly=3, Lx=3, S=2, n_s=8, p_keep=0.97, seed=8, h="zero"),
                         dict(beta=2.0, D=64, sweeps=3, M=256)),
}


def build_instance(kind, args):
    if kind == "lattice":
        return instances.lattice(**args)
    if kind == "loops":
        return instances.loop_planted(**args)
    raise ValueError(kind)


def instance_hash(inst):
    h = hashlib.sha256()
    for k in ("edge_u", "edge_v", "J", "h", "cell_y", "cell_x", "sub", "pos"):
        h.update(np.ascontiguousarray(inst[k]).tobytes())
    h.update(repr((inst.n_spins, inst.Ly, inst.Lx, inst.S, inst.n_s)).encode())
    return h.hexdigest()


def schmidt_spectra(T):
    """Singular values at every bond of the MPS T (list of [dl, p, dr]); the state is taken as given (unit norm)."""
    A = [t.copy() for t in T]
    n = len(A)
    for j in range(n - 1):                          # left-canonical up to the last site
        dl, p, dr = A[j].shape
        Q, R = np.linalg.qr(A[j].reshape(dl * p, dr))
        A[j] = Q.reshape(dl, p, Q.shape[1])
        A[j + 1] = np.einsum("ab,bpc->apc", R, A[j + 1])
    out = [None] * (n - 1)
    for j in range(n - 1, 0, -1):                   # sweep the centre back, SVD at every bond
        dl, p, dr = A[j].shape
        U, s, Vt = np.linalg.svd(A[j].reshape(dl, p * dr), full_matrices=False)
        out[j - 1] = s
        A[j - 1] = np.einsum("apb,bc->apc", A[j - 1], U * s)
    return out


def sample_configs(T, K, rng):
    """K boundary configurations drawn from |R|^2 (exact sequential sampling with right environments)."""
    n = len(T)
    E = [None] * (n + 1)
    E[n] = np.ones((1, 1))
    for j in range(n - 1, -1, -1):
        E[j] = np.einsum("apb,bc,dpc->ad", T[j], E[j + 1], T[j], optimize=True)
    cfg = np.zeros((K, n), dtype=np.int32)
    for k in range(K):
        v = np.ones(1)
        for j in range(n):
            w = np.einsum("a,apb->pb", v, T[j])                       # [p, dr]
            pr = np.einsum("pb,bc,pc->p", w, E[j + 1], w)
            pr = np.maximum(pr, 0.0)
            pr /= pr.sum()
            c = int(rng.choice(pr.size, p=pr))
            cfg[k, j] = c
            v = w[c]
            v = v / np.abs(v).max()
    return cfg


def amplitudes(T, cfg):
    out = np.zeros(cfg.shape[0])
    for k in range(cfg.shape[0]):
        v = np.ones(1)
        for j, t in enumerate(T):
            v = v @ t[:, cfg[k, j], :]
        out[k] = v[0]
    return out


def run_case(name):
    from oracle import model, mps, search
    kind, args, run = CASES[name]
    inst = build_instance(kind, args)
    t0 = time.perf_counter()
    m = model.Model(inst).set_beta(run["beta"])
    t1 = time.perf_counter()
    st = {}
    R, ln = mps.contract(m, run["D"], run["sweeps"], stats=st)
    t2 = time.perf_counter()
    data = dict(min_sigma=np.asarray(st["min_sigma"]))
    if run["M"] > 0:
        out = search.branch_and_bound(m, R, ln, run["M"], stats=st)
        data.update(log_z=np.float64(out["log_z"]), logp=out["logp"], log_pd=np.float64(out["log_pd"]),
                    cell_states=out["cell_states"].astype(np.int32), energies=out["energies"],
                    states=out["states"].astype(np.int8), negative_u=np.int64(st.get("negative_u", 0)),
                    tied_cuts=np.int64(st.get("tied_cuts", 0)))
    t3 = time.perf_counter()
    rng = np.random.default_rng(20241116)
    for y in range(1, inst.Ly):
        T = R[y]
        sp = schmidt_spectra(T)
        D = max([s.size for s in sp] + [1])
        S = np.zeros((len(sp), D))
        for j, s in enumerate(sp):
            S[j, :s.size] = s
        cfg = sample_configs(T, K_SAMPLES, rng)
        data["schmidt_%d" % y] = S
        data["cfg_%d" % y] = cfg
        data["amp_%d" % y] = amplitudes(T, cfg)
        data["bonds_%d" % y] = np.asarray([t.shape[2] for t in T], dtype=np.int32)
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1
    meta = dict(case=name, kind=kind, args=args, run=run, instance_sha256=instance_hash(inst),
                oracle_seconds=dict(tables=t1 - t0, contract=t2 - t1, search=t3 - t2), cores=int(cores),
                numpy=np.__version__, written_by="tests/golden/make_rows.py (calls only oracle/)")
    data["meta"] = np.asarray(json.dumps(meta))
    path = os.path.join(HERE, "rows_%s.npz" % name)
    np.savez_compressed(path, **data)
    print("%s: tables %.1fs contract %.1fs search %.1fs -> %s (%.0f KB)"
          % (name, t1 - t0, t2 - t1, t3 - t2, path, os.path.getsize(path) / 1024), flush=True)


if __name__ == "__main__":
    names = sys.argv[1:]
    if names == ["all"]:
        names = list(CASES)
    if not names:
        raise SystemExit(__doc__)
    for n in names:
        run_case(n)
