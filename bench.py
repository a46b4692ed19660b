"""bench.py -- times the whole hot path (a1 tables -> a2-a4 boundary-MPS contraction -> a5 branch and bound)
of one synthetic instance per step, through the C ABI of libtn_b200.so.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl reference]

Workload: BASELINE.json configs[I] (default I = 1, the Zephyr-shaped 6x6x16 instance; configs[0] is the
brute-force parity case).  A step = tn_set_beta + tn_contract(D, sweeps) + tn_branch_and_bound(M) on an
instance that is already resident in HBM (tn_create done before the timed region).  The `e2e` arm repeats
the measurement with tn_create (host -> device copy of the instance) and tn_destroy inside the timed
region; results always come back to caller-allocated host buffers.  Multi-GPU: replicas only (DESIGN.md
section 9) -- every rank solves its own seeded instance, no data-path collective; NCCL is used for the
barrier and the max-over-ranks of the device time.

--impl reference times the CPU oracle (oracle/, numpy fp64) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "bnb_wall_time_per_instance"
UNIT = "s/instance"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs (0-based)")
    ap.add_argument("--beta-index", type=int, default=0, help="which beta of the config's sweep")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--merge", action="store_true", help="TN_OPT_MERGE: merge candidates by boundary (paper Fig. 3(d))")
    ap.add_argument("--transform", type=int, default=0,
                    help="lattice transformation 0..7 (PAPER.md:270; instances.transformed; Zephyr-shaped configs only)")
    return ap.parse_args()


def workload_name(ci, inst, run, beta):
    return "configs[%d] %s N=%d beta=%g D=%d M=%d sweeps=%d" % (ci, inst.name, inst.n_spins, beta, run["D"], run["M"],
                                                              run["sweeps"])


# ----------------------------------------------------------------------------------------------------
# CPU oracle on a bounded sample: the top `rows` rows of the instance, whole path
# ----------------------------------------------------------------------------------------------------
def slice_rows(inst, rows):
    """Sub-instance made of the first `rows` cell rows (spins are row-major, so it is a prefix)."""
    import instances
    keep = inst.cell_y < rows
    n = int(keep.sum())
    ke = keep[inst.edge_u] & keep[inst.edge_v]
    d = dict(inst)
    d.update(n_spins=n, edge_u=inst.edge_u[ke], edge_v=inst.edge_v[ke], J=inst.J[ke], h=inst.h[:n], Ly=rows,
             cell_y=inst.cell_y[:n], cell_x=inst.cell_x[:n], sub=inst.sub[:n], pos=inst.pos[:n])
    return instances.Instance(d)


def oracle_sample(inst, run, beta, rows=2):
    """Runs oracle/ as it stands on the top `rows` rows (tables, rows-1 boundary-MPS rows, B&B over all
    cells of the slice).  Returns (measured seconds, extrapolated seconds per full instance, description)."""
    from oracle import model, mps, search
    s = slice_rows(inst, min(rows, inst.Ly))
    t0 = time.perf_counter()
    m = model.Model(s).set_beta(beta)
    t1 = time.perf_counter()
    R, ln = mps.contract(m, run["D"], run["sweeps"])
    t2 = time.perf_counter()
    search.branch_and_bound(m, R, ln, run["M"])
    t3 = time.perf_counter()
    cells_s, cells = s.Ly * s.Lx, inst.Ly * inst.Lx
    est = (t1 - t0) * cells / cells_s + (t2 - t1) * (inst.Ly - 1) / max(1, s.Ly - 1) + (t3 - t2) * cells / cells_s
    desc = ("oracle/ (numpy fp64) on the top %d of %d cell rows (%d of %d spins): tables %.1fs, %d boundary-MPS "
            "row(s) %.1fs, B&B over %d cells %.1fs; value = extrapolation to the full instance by cell / row "
            "counts" % (s.Ly, inst.Ly, s.n_spins, inst.n_spins, t1 - t0, s.Ly - 1, t2 - t1, cells_s, t3 - t2))
    return t3 - t0, est, desc


# ----------------------------------------------------------------------------------------------------
# multi-rank plumbing (replicas only); backend-agnostic so that the gloo tests cover it
# ----------------------------------------------------------------------------------------------------
def replica_instance(config_index, rank):
    """Rank r solves its own instance of the config: same shape, generator seed r."""
    import instances
    return instances.config(config_index, seed=rank)


def max_over_ranks(v, world, device="cuda"):
    if world == 1:
        return float(v)
    import torch
    import torch.distributed as dist
    x = torch.tensor([v], dtype=torch.float64, device=device)
    dist.all_reduce(x, op=dist.ReduceOp.MAX)
    return float(x.item())


def whole_job_value(ms_total, steps, world):
    """Seconds per instance over the whole job: every rank solves `steps` instances in ms_total (max over ranks)."""
    return ms_total / steps * 1e-3 / world


def diversity_report(inst, states, E, frac=0.01, R=0.25, restarts=100, seed=0):
    """Config-5 harness metrics: gap to the planted E0, states within `frac` of E0 by both
    (E - E0)/|E0| and Eq. (14) d_E = (E - E0)/(2|E0|), and the size of the largest set of those states
    that are pairwise >= R*N Hamming apart (Eq. (15)), found by a randomised greedy clique heuristic
    (footnote [58] PAPER.md:418) after flipping every state to s_0 = +1 (h = 0)."""
    import numpy as np
    E0 = float(inst.E0)
    rel = (E - E0) / abs(E0)
    near = np.flatnonzero(rel <= frac)
    out = {"E0": E0, "gap_to_E0": float(E.min() - E0), "n_within_1pct": int(near.size),
           "n_within_dE_1pct": int(np.count_nonzero(rel / 2.0 <= frac))}
    s = states[near].astype(np.int8)
    s = s * s[:, :1]                                           # Z2 gauge: s_0 = +1
    s = np.unique(s, axis=0)
    n, N = s.shape[0], inst.n_spins
    if n == 0:
        out["diversity"] = 0
        return out
    ham = (N - s.astype(np.int32) @ s.astype(np.int32).T) // 2
    ok = ham >= R * N
    rng = np.random.default_rng(seed)
    best = 1
    for _ in range(restarts):
        order = rng.permutation(n)
        chosen = []
        for i in order:
            if all(ok[i, j] for j in chosen):
                chosen.append(i)
        best = max(best, len(chosen))
    out["diversity"] = int(best)
    out["distinct_up_to_Z2"] = int(n)
    return out


def host_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info()]
        if n:
            return int(max(n))
    except Exception:
        pass
    return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import instances
    inst, run = instances.config(args.config)
    beta = run["beta"][args.beta_index]
    import numpy  # noqa: F401  (loads the BLAS whose thread count is reported)
    for _ in range(args.warmup):
        oracle_sample(inst, run, beta)
    ests, meas, desc = [], [], ""
    for _ in range(args.steps):
        tm, est, desc = oracle_sample(inst, run, beta)
        ests.append(est)
        meas.append(tm)
    v = sum(ests) / len(ests)
    cores = host_threads()
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sum(meas) / len(meas), "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, inst, run, beta)},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------
# clocks during the timed region (profiling recipe's clocks line)
# ----------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
                pw.append(float(f[3]))
            except ValueError:
                continue
            for n, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "power_w_max": max(pw) if pw else None}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0}, "fallback (B200_PROFILING.md)"


STAGES = [  # (stats ms key, label, kernel, flop key, bytes key, bound)
    ("ms_theta_apply", "theta_apply", "k_tsgemm<NT,8,N|T> (Theta-core x skinny: zipper SVD / variational / env applies)",
     "flop_theta_apply", "bytes_theta_apply", "tensor"),
    ("ms_theta_build", "theta_build", "k_bgemm_pipe<.., ArTh, BrTh, EpTh> (Theta-core build) + projector maps", "flop_theta_build",
     None, "tensor"),
    ("ms_orth_svd", "orth_svd", "k_orth_coop (Cholesky-QR rounds, one cooperative launch) + k_jacobi_rows (Rayleigh-Ritz)", None, None, "alu"),
    ("ms_search_rblocks", "search_rblocks", "k_gather_G, k_coef + k_tsgemm + k_rs (right blocks)", None, None, "tensor"),
    ("ms_search_cond", "search_cond", "k_bgemm<.., ArPV, LdPB, EpPV> (conditionals, Z fused in the epilogue)", None,
     "bytes_search_cond", "hbm"),
    ("ms_search_select", "search_select", "k_sel_hist (sample) + k_sel_prefilter + k_csel_* + bitonic (top-M)", None,
     "bytes_search_select", "hbm"),
    ("ms_tables", "tables", "k_tables", None, None, "hbm"),
]


def stored_traffic(workload_key):
    """dram bytes per launch of the dominant kernel from the committed `ncu --set full` capture (profiles/), or None."""
    p = os.path.join(ROOT, "profiles", "r01_traffic.json")
    try:
        with open(p) as f:
            return json.load(f).get(workload_key)
    except (OSError, ValueError):
        return None


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import instances
    import paper_2411_16431_b200 as tnb

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    tnb.lib()   # fails loudly when libtn_b200.so is missing
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    inst, run = replica_instance(args.config, rank)           # one independent replica per rank
    if args.transform:
        import instances
        inst = instances.transformed(inst, args.transform)
    beta = run["beta"][args.beta_index]
    D, sweeps, M = run["D"], run["sweeps"], run["M"]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step(t):
        t.set_beta(beta)
        t.contract(D, sweeps)
        return t.branch_and_bound(M)

    def timed(fn, n):
        """n calls of fn, each bracketed by CUDA events on the launching stream; L2 flushed in between."""
        tot, outs = 0.0, None
        for _ in range(n):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            outs = fn()
            e1.record()
            e1.synchronize()
            tot += e0.elapsed_time(e1)
        return tot, outs

    fp64_peak = tnb.tn_fp64_peak()
    t = tnb.TensorNetwork(inst)
    if args.merge:
        t.set_option(tnb.OPT_MERGE, 1)
    for _ in range(args.warmup):
        step(t)
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    ms_total, outs = timed(lambda: step(t), args.steps)
    barrier()
    st = t.stats()                                               # stage timers of the last timed step
    # the dominant kernel timed alone at this workload's largest apply shape (burst figure, warm L2 for small shapes)
    alone = None
    if rank == 0:
        c0 = 1 << inst.n_s
        nK = c0 * ((1 << (inst.n_s // 2)) if inst.S == 3 else 1)
        mk, nk, sk = D * nK, c0 * D, min(D + 16, 96)
        alone = {"shape": "Tc[%d x %d] x [%d x %d]" % (mk, nk, nk, sk)}
        for op, nm in ((tnb.CHECK_GEMM_N, "N"), (tnb.CHECK_GEMM_T, "T")):
            ms1 = tnb.tn_kernel_bench(t.handle, op, mk, sk, nk, 5)
            alone[nm] = {"ms": round(ms1, 4), "tflops": round(2.0 * mk * nk * sk / ms1 * 1e-9, 2),
                         "frac_fp64_tensor": round(2.0 * mk * nk * sk / ms1 * 1e-9 / fp64_peak, 4),
                         "gbs": round(8.0 * mk * nk / ms1 * 1e-6, 1)}
    t.close()

    # ---- e2e: host buffers in, host buffers out, tn_create / tn_destroy inside the timed region
    def e2e_step():
        with tnb.TensorNetwork(inst) as tt:
            if args.merge:
                tt.set_option(tnb.OPT_MERGE, 1)
            return step(tt)
    e2e_ms = None
    if not args.no_e2e:
        for _ in range(min(args.warmup, 2)):
            e2e_step()
        barrier()
        e2e_ms, _ = timed(e2e_step, args.steps)
        barrier()
    clocks = sampler.stop() if rank == 0 else None

    def maxr(v):
        return max_over_ranks(v, world, device="cuda")

    ms_total = maxr(ms_total)
    if e2e_ms is not None:
        e2e_ms = maxr(e2e_ms)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    states, E, logp, pd = outs
    K = args.steps
    ms_step = ms_total / K
    value = whole_job_value(ms_total, K, world)                  # seconds per instance over the whole job
    h2d = int(inst.edge_u.nbytes + inst.edge_v.nbytes + inst.J.nbytes + inst.h.nbytes + inst.cell_y.nbytes
              + inst.cell_x.nbytes + inst.sub.nbytes + inst.pos.nbytes)
    d2h = int(M * inst.n_spins + 2 * 8 * M + 8 + 4)
    peaks, peak_src = measured_peaks()

    # ---- per-stage table and the roofline of the dominant kernel
    stages = {}
    for key, label, kern, fk, bk, bound in STAGES:
        ms = st[key]
        d = {"ms": round(ms, 3), "share": round(ms / max(st["ms_contract"] + st["ms_search"] + st["ms_tables"], 1e-9), 4),
             "kernel": kern, "bound": bound}
        if fk and ms > 0:
            d["tflops"] = round(st[fk] / ms * 1e-9, 3)
            d["frac_fp64_tensor"] = round(st[fk] / ms * 1e-9 / fp64_peak, 4)
        if bk and ms > 0:
            d["gbs"] = round(st[bk] / ms * 1e-6, 1)
            d["frac_hbm"] = round(st[bk] / ms * 1e-6 / peaks["hbm_gbs"], 4)
        stages[label] = d
    sflop = st["flop_search"]
    if st["ms_search"] > 0:
        stages["search_total"] = {"ms": round(st["ms_search"], 3), "tflops": round(sflop / st["ms_search"] * 1e-9, 3)}
    dom = STAGES[0]                                              # the FLOP carrier: Theta-core x skinny GEMMs (k_tsgemm)
    ms_dom = st[dom[0]]
    achieved = st[dom[3]] / ms_dom * 1e-9 if ms_dom > 0 else 0.0
    tr = stored_traffic("configs[%d]" % args.config)
    roofline = {"bound": "tensor", "achieved": round(achieved, 3), "peak": round(fp64_peak, 2), "unit": "TFLOP/s",
                "frac": round(achieved / fp64_peak, 4), "traffic": tr["dram_bytes_per_launch"] if tr else None,
                "kernel": dom[2], "stage": dom[1], "share_of_step": stages[dom[1]]["share"],
                "launches_per_step": int(st["theta_apply_calls"]),
                "peak_source": "tn_fp64_peak(): mma.sync m8n8k4 f64 (SASS DMMA) chain measured in this run "
                               "(MEASURED_PEAKS.json has no FP64 entry; profiles/r01_fp64_peak.md); HBM peak %s = %.1f GB/s"
                               % (peak_src, peaks["hbm_gbs"]),
                "algorithmic_flop_per_step": st[dom[3]], "algorithmic_bytes_per_step": st["bytes_theta_apply"],
                "achieved_gbs": round(st["bytes_theta_apply"] / ms_dom * 1e-6, 1) if ms_dom > 0 else None,
                "kernel_alone": alone}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "l2": "flushed (256 MiB fill) between timed steps",
            "config": {"workload": workload_name(args.config, inst, run, beta), "D": D, "M": M, "sweeps": sweeps,
                       "beta": beta, "merge": bool(args.merge), "transform": int(args.transform), "parallelism": "replicas x%d" % world, "l2": "flush between steps"},
            "contract_rows_per_s": round(st["rows_contracted"] / max(st["ms_contract"], 1e-9) * 1e3, 3),
            "contract_ms": round(st["ms_contract"], 3), "search_ms": round(st["ms_search"], 3),
            "best_energy": float(E.min()), "n_states": int(len(E)), "log_p_discarded": float(pd),
            "gpu_launches": int(st["kernel_launches"]) * K, "stages": stages, "roofline": roofline, "clocks": clocks,
            "fp64_tensor_peak_tflops": round(fp64_peak, 2)}
    if "E0" in inst:
        line["planted"] = diversity_report(inst, states, E)
    if e2e_ms is not None:
        line["e2e"] = {"value": whole_job_value(e2e_ms, K, world), "unit": UNIT, "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": d2h}
    if world == 1 and not args.no_cpu_baseline:
        tm, est, desc = oracle_sample(inst, run, beta)
        line["cpu_baseline"] = {"value": est, "unit": UNIT, "cores": host_threads(), "kind": "oracle", "sample": desc,
                                "sample_seconds": round(tm, 2)}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
