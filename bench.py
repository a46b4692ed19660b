"""bench.py -- times the whole hot path (a1 tables -> a2-a4 boundary-MPS contraction -> a5 branch and bound)
of one synthetic instance per step, through the C ABI of libtn_b200.so.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl reference] [--no-headline]

Workload: BASELINE.json configs[I].  Default I = 2, the Pegasus-shaped 8x8x24 instance (N = 1536, D = 32, M = 1024):
the largest config whose `--steps 20 --warmup 5` run fits the driver's per-arm time limit (about 3 s per step; every
kernel is in its streaming regime, the Theta-core is 8.6 GB >> L2).  The north_star target workload, configs[3]
(Pegasus-shaped 15x15x24, N = 5400, D = 64, M = 1024, three variational passes, beta = 2), takes about two minutes per
step, so the same JSON line carries a `headline` record of ONE timed step of it (own stage table, roofline and clocks;
`--no-headline` skips it, N = 1 only), and a second one, `headline_fast`, of the same workload with the paper's own
truncated randomized SVD (seeded, reproducible, parity-tested against the oracle's switch on small
lattices; `--no-headline-fast` skips it).  The line's `value` is always the converged (parity-defining) mode.
A step = tn_set_beta + tn_contract(D, sweeps) + tn_branch_and_bound(M) on an instance that is already resident in HBM
(tn_create done before the timed region).  The `e2e` arm repeats the measurement with tn_create (host -> device copy
of the instance) and tn_destroy inside the timed region; results always come back to caller-allocated host buffers.
Multi-GPU: replicas only -- every rank solves its own seeded instance (or, with
`--replicas transforms`, its own lattice transformation of ONE instance), no data-path collective; NCCL
is used for the barrier and the max-over-ranks of the device time.

--impl reference times the CPU oracle (oracle/, numpy fp64) as it stands: the whole instance where it finishes in
bounded time (configs[0], [1]), else the largest whole sub-problem that does, with any scaled figure labelled
"extrapolated".
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
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (0-based); 5 = the 50 x 50 square lattice of the paper's App. B")
    ap.add_argument("--beta-index", type=int, default=0, help="which beta of the config's sweep")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-headline", action="store_true",
                    help="skip the one-step record of configs[3] (the north_star target workload)")
    ap.add_argument("--replicas", default="seeds", choices=["seeds", "transforms"],
                    help="what the N ranks differ by: generator seeds (default) or the 8 lattice transformations "
                         "of one instance (PAPER.md:270; best-of-N energy and log Z spread are reported)")
    ap.add_argument("--streams", type=int, default=1,
                    help="N = 1 with --replicas transforms: run the 8 maps as concurrent replicas on this many "
                         "CUDA streams (one host thread per stream)")
    ap.add_argument("--merge", action="store_true", help="TN_OPT_MERGE: merge candidates by boundary (paper Fig. 3(d))")
    ap.add_argument("--svd-mode", default="converged", choices=["converged", "randomized"],
                    help="TN_OPT_SVD_MODE: converged truncated SVD (parity definition, default) or the paper's seeded "
                         "randomized SVD with 2 subspace iterations (PAPER.md:169-177)")
    ap.add_argument("--schedule", default="zipper-then-sweeps", choices=["zipper-then-sweeps", "interleaved"],
                    help="TN_OPT_SCHEDULE: variant (ii) of PAPER.md:179 (default) or a sweep after every zipper step")
    ap.add_argument("--oversample", type=int, default=None, help="TN_OPT_OVERSAMPLE (extra block columns of the SVD)")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="tn_set_option by numeric key (tuning switches of include/tn.h), e.g. --opt 26=0")
    ap.add_argument("--two-step", action="store_true", help="TN_OPT_TWO_STEP: zipper and passes at 2 D, then cut to D")
    ap.add_argument("--no-headline-fast", action="store_true",
                    help="skip the second one-step record of configs[3], taken in the paper's own mode (seeded randomized "
                         "SVD, --svd-mode randomized)")
    ap.add_argument("--droplets", action="store_true",
                    help="TN_OPT_DROPLETS on top of --merge: book-keep the excitations above every main branch (Fig. 4)")
    ap.add_argument("--droplet-max-de", type=float, default=2.0, help="TN_OPT_DROPLET_MAX_DE (energy units of J)")
    ap.add_argument("--droplet-min-hamming", type=int, default=2, help="TN_OPT_DROPLET_MIN_HAMMING")
    ap.add_argument("--transform", type=int, default=0,
                    help="lattice transformation 0..7 (PAPER.md:270; instances.transformed; Zephyr-shaped configs only)")
    return ap.parse_args()


def config_record(ci, inst, run, beta, merge, transform, world):
    """The `config` object of the JSON line (same keys in both arms, so that the driver sees the same config)."""
    return {"workload": workload_name(ci, inst, run, beta), "D": run["D"], "M": run["M"], "sweeps": run["sweeps"],
            "beta": beta, "merge": bool(merge), "transform": int(transform), "parallelism": "replicas x%d" % world,
            "l2": "flush between steps"}


def workload_name(ci, inst, run, beta):
    return "configs[%d] %s N=%d beta=%g D=%d M=%d sweeps=%d" % (ci, inst.name, inst.n_spins, beta, run["D"], run["M"],
                                                              run["sweeps"])


# ----------------------------------------------------------------------------------------------------
# CPU oracle, as it stands, on the whole instance or on the largest whole sub-problem that finishes in bounded time
# ----------------------------------------------------------------------------------------------------
def sub_lattice(inst, rows, cols):
    """Sub-instance made of the top-left `rows` x `cols` block of cells (spin ids re-numbered, edges inside kept)."""
    import numpy as np
    import instances
    keep = (inst.cell_y < rows) & (inst.cell_x < cols)
    idx = np.flatnonzero(keep)
    remap = -np.ones(inst.n_spins, dtype=np.int64)
    remap[idx] = np.arange(idx.size)
    ke = keep[inst.edge_u] & keep[inst.edge_v]
    d = dict(inst)
    d.update(n_spins=int(idx.size), edge_u=remap[inst.edge_u[ke]].astype(np.int32),
             edge_v=remap[inst.edge_v[ke]].astype(np.int32), J=inst.J[ke], h=inst.h[idx], Ly=rows, Lx=cols,
             cell_y=inst.cell_y[idx], cell_x=inst.cell_x[idx], sub=inst.sub[idx], pos=inst.pos[idx])
    return instances.Instance(d)


# (rows, cols, beam) of the oracle sample per config: None = the whole instance.  Pegasus-shaped cells have 2^24
# states: every oracle operation on one cell costs seconds, so the sample there is a 2 x 2 block with one beam element.
ORACLE_SAMPLE = {0: None, 1: None, 2: (2, 2, 1), 3: (2, 2, 1), 4: (2, 4, 64), 5: None}
ORACLE_SAMPLE_SMALL = {0: None, 1: (2, 6, 256), 2: (2, 1, 1), 3: (2, 1, 1), 4: (2, 4, 64), 5: (10, 50, 256)}   # reference arm, many steps


class OracleSample:
    """Times oracle/ (numpy fp64, never tuned for this) on `spec` of the workload.  The instance preprocessing
    (cluster energies, projectors: oracle.model.Model.__init__, the counterpart of tn_create) is done once and timed
    separately; a step = set_beta + contract(D, sweeps) + branch_and_bound, like the GPU arm's step."""

    def __init__(self, inst, run, beta, spec):
        from oracle import model
        self.full, self.run, self.beta = inst, run, beta
        self.whole = spec is None or (spec[0] >= inst.Ly and spec[1] >= inst.Lx and spec[2] >= run["M"])
        self.rows, self.cols, self.M = (inst.Ly, inst.Lx, run["M"]) if self.whole else spec
        self.inst = inst if self.whole else sub_lattice(inst, self.rows, self.cols)
        t0 = time.perf_counter()
        self.model = model.Model(self.inst)
        self.t_setup = time.perf_counter() - t0

    def step(self):
        from oracle import mps, search
        t0 = time.perf_counter()
        m = self.model.set_beta(self.beta)
        t1 = time.perf_counter()
        R, ln = mps.contract(m, self.run["D"], self.run["sweeps"])
        t2 = time.perf_counter()
        search.branch_and_bound(m, R, ln, self.M)
        t3 = time.perf_counter()
        self.parts = (t1 - t0, t2 - t1, t3 - t2)
        return t3 - t0

    def positions(self, cols):
        return 2 * cols - 1 if self.inst.S == 3 else cols

    def estimate(self):
        """Seconds per FULL instance from the last step: the measurement itself when the sample is the whole instance,
        else scaled by cell / (row x position) / (cell x beam) counts -- a LOWER bound, the old bonds inside a two-row
        sample are 1 where a full-height lattice has up to D."""
        tb, tc, ts = self.parts
        if self.whole:
            return tb + tc + ts
        f, s = self.full, self.inst
        cells = (f.Ly * f.Lx) / (s.Ly * s.Lx)
        rows = (f.Ly - 1) * self.positions(f.Lx) / max(1, (s.Ly - 1) * self.positions(s.Lx))
        return tb * cells + tc * rows + ts * cells * self.run["M"] / self.M

    def describe(self):
        tb, tc, ts = self.parts
        what = ("the WHOLE instance" if self.whole else
                "the top-left %d x %d cells (%d of %d spins) with beam %d of %d"
                % (self.rows, self.cols, self.inst.n_spins, self.full.n_spins, self.M, self.run["M"]))
        tail = "" if self.whole else ("; value = measured parts scaled by cell, row x position and cell x beam counts "
                                      "(extrapolated, a lower bound: old bonds in a 2-row sample are 1, not D)")
        return ("oracle/ (numpy fp64, as it stands) on %s: instance preprocessing %.1fs (once, outside the step), "
                "step = tables %.1fs + %d boundary-MPS row(s) %.1fs + B&B over %d cells %.1fs%s"
                % (what, self.t_setup, tb, self.inst.Ly - 1, tc, self.inst.Ly * self.inst.Lx, ts, tail))


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
    table = ORACLE_SAMPLE if args.steps + args.warmup <= 3 else ORACLE_SAMPLE_SMALL
    smp = OracleSample(inst, run, beta, table[args.config])
    for _ in range(args.warmup):
        smp.step()
    ests, meas = [], []
    for _ in range(args.steps):
        meas.append(smp.step())
        ests.append(smp.estimate())
    v = sum(ests) / len(ests)
    cores = host_threads()
    # value and ms_per_step are the SAME quantity (seconds per full instance); the measured sample time sits beside them
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * v, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "extrapolated": not smp.whole, "sample_seconds_per_step": sum(meas) / len(meas),
            "config": config_record(args.config, inst, run, beta, False, 0, 1),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": smp.describe(),
                             "extrapolated": not smp.whole, "sample_seconds": round(sum(meas) / len(meas), 2)},
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
    ("ms_orth_svd", "orth_svd", "k_orth_coop (Cholesky-QR rounds, one cooperative launch) + k_jacobi_rows (Rayleigh-Ritz)",
     "flop_orth_svd", None, "alu"),
    ("ms_search_rblocks", "search_rblocks", "k_gather_Gy + k_rblock_mma (right blocks, factorised: c_lo first, then b; two DMMA products per stage) + k_rs + k_tsgemm (Bh)",
     "flop_search_rblocks", None, "tensor"),
    ("ms_search_cond", "search_cond", "k_cond<KP> (conditionals: A tile resident, dense operand through a cp.async double buffer; Z fused in the epilogue)",
     "flop_search_cond", "bytes_search_cond", "tensor"),
    ("ms_search_select", "search_select", "k_sel_hist_rows (bound from the row maxima of V) + k_sel_prefilter (reads only rows that reach it) + k_csel_* + bitonic (top-M)", None,
     "bytes_search_select", "hbm"),
    ("ms_tables", "tables", "k_tables", None, None, "hbm"),
]
DFMA_PEAK_TFLOPS = 35.8   # plain FP64 FMA peak measured on this pool's B200 (profiles/r01_fp64_peak.md)


def stored_traffic(config_index, stage):
    """DRAM bytes per launch of the dominant kernel from the committed `ncu --set full` capture OF THAT CONFIG
    (profiles/r02_traffic.json, which names the capture command), or (None, reason)."""
    p = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        with open(p) as f:
            rec = json.load(f).get("configs[%d]:%s" % (config_index, stage))
    except (OSError, ValueError):
        rec = None
    if rec is None:
        return None, "no committed ncu --set full capture of this kernel at configs[%d]" % config_index
    return rec["dram_bytes_per_launch"], rec.get("source", "profiles/r02_traffic.json")


def stage_report(st, ci, fp64_peak, peaks, peak_src):
    """Per-stage table (CUDA-event times and analytic FLOP / byte counters of tn_get_stats) and the roofline record of
    the TIME-DOMINANT stage of this run."""
    total = max(st["ms_contract"] + st["ms_search"] + st["ms_tables"], 1e-9)
    stages = {}
    for key, label, kern, fk, bk, bound in STAGES:
        ms = st[key]
        d = {"ms": round(ms, 3), "share": round(ms / total, 4), "kernel": kern, "bound": bound}
        if fk and ms > 0 and st.get(fk, 0) > 0:
            d["tflops"] = round(st[fk] / ms * 1e-9, 3)
            d["frac_fp64_tensor" if bound != "alu" else "frac_fp64_alu"] = round(
                st[fk] / ms * 1e-9 / (fp64_peak if bound != "alu" else DFMA_PEAK_TFLOPS), 4)
        if bk and ms > 0:
            d["gbs"] = round(st[bk] / ms * 1e-6, 1)
            d["frac_hbm"] = round(st[bk] / ms * 1e-6 / peaks["hbm_gbs"], 4)
        stages[label] = d
    named = sum(st[k[0]] for k in STAGES)
    stages["other"] = {"ms": round(total - named, 3), "share": round((total - named) / total, 4),
                       "kernel": "maps on skinny operands outside the stage timers, copies, host round trips"}
    dom = max(STAGES, key=lambda k: st[k[0]])
    key, label, kern, fk, bk, bound = dom
    ms_dom = st[key]
    tr, tr_src = stored_traffic(ci, label)
    launches = int(st["theta_apply_calls"]) if label == "theta_apply" else None
    roof = {"bound": bound, "kernel": kern, "stage": label, "share_of_step": stages[label]["share"],
            "traffic": tr, "traffic_source": tr_src, "launches_per_step": launches}
    if bound in ("tensor", "alu") and fk:
        ach = st[fk] / ms_dom * 1e-9 if ms_dom > 0 else 0.0
        pk = fp64_peak if bound == "tensor" else DFMA_PEAK_TFLOPS
        roof.update({"achieved": round(ach, 3), "peak": round(pk, 2), "unit": "TFLOP/s", "frac": round(ach / pk, 4),
                     "algorithmic_flop_per_step": st[fk],
                     "peak_source": ("tn_fp64_peak(): mma.sync m8n8k4 f64 (SASS DMMA) chain measured in this run "
                                     "(MEASURED_PEAKS.json has no FP64 entry)" if bound == "tensor" else
                                     "plain DFMA chain measured on this pool (profiles/r01_fp64_peak.md); the stage is "
                                     "latency-bound, see DESIGN.md section 6")})
        if bk:
            roof["algorithmic_bytes_per_step"] = st[bk]
            roof["achieved_gbs"] = round(st[bk] / ms_dom * 1e-6, 1) if ms_dom > 0 else None
            roof["hbm_peak_gbs"] = peaks["hbm_gbs"]
            roof["hbm_peak_source"] = peak_src
        if launches:
            roof["algorithmic_flop_per_launch"] = st[fk] / launches
            roof["algorithmic_bytes_per_launch"] = st[bk] / launches if bk else None
            roof["avg_launch_ms"] = round(ms_dom / launches, 4)
    else:
        ach = st[bk] / ms_dom * 1e-6 if (bk and ms_dom > 0) else 0.0
        roof.update({"achieved": round(ach, 1), "peak": peaks["hbm_gbs"], "unit": "GB/s",
                     "frac": round(ach / peaks["hbm_gbs"], 4), "peak_source": peak_src,
                     "algorithmic_bytes_per_step": st[bk] if bk else None})
    return stages, roof


def zspread(logzs):
    """Z-spread diagnostic of PAPER.md:284, App. C: spread of log Z over the lattice transformations."""
    import numpy as np
    z = np.asarray(logzs, dtype=np.float64)
    return {"log_z": [float(v) for v in z], "ptp": float(np.ptp(z)), "std": float(z.std()),
            "rel_ptp": float(np.ptp(z) / abs(z.mean())) if z.size and z.mean() != 0 else None}


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

    transform = int(args.transform)
    if args.replicas == "transforms":
        inst, run = instances.config(args.config)                 # ONE instance, rank r contracts map r
        if inst.S == 3:
            raise SystemExit("--replicas transforms: the Pegasus-shaped lattice admits only the identity map "
                             "(DESIGN.md section 0, f3); use --config 1 or 4")
        if world > 1:
            transform = rank % 8
    else:
        inst, run = replica_instance(args.config, rank)           # one independent seeded replica per rank
    base_inst = inst
    if transform:
        inst = instances.transformed(inst, transform)
    beta = run["beta"][args.beta_index]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    fp64_peak = tnb.tn_fp64_peak()
    peaks, peak_src = measured_peaks()

    def make_tn(ins):
        t = tnb.TensorNetwork(ins)
        set_contract_options(tnb, t, args)
        if args.merge or args.droplets:
            t.set_option(tnb.OPT_MERGE, 1)
        if args.droplets:
            t.set_option(tnb.OPT_DROPLETS, 1)
            t.set_option(tnb.OPT_DROPLET_MAX_COUNT, 16)
            t.set_option(tnb.OPT_DROPLET_MAX_DE, args.droplet_max_de)
            t.set_option(tnb.OPT_DROPLET_MIN_HAMMING, args.droplet_min_hamming)
        return t

    def step(t, b, r):
        t.set_beta(b)
        t.contract(r["D"], r["sweeps"])
        return t.branch_and_bound(r["M"])

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

    def kernel_alone(t, ins, r):
        """the dominant kernel timed alone at this workload's largest apply shape (burst figure)"""
        c0 = 1 << ins.n_s
        nK = c0 * ((1 << (ins.n_s // 2)) if ins.S == 3 else 1)
        D = r["D"]
        mk, nk, sk = D * nK, c0 * D, min(D + 16, 96)
        alone = {"shape": "Tc[%d x %d] x [%d x %d]" % (mk, nk, nk, sk)}
        for op, nm in ((tnb.CHECK_GEMM_N, "N"), (tnb.CHECK_GEMM_T, "T")):
            ms1 = tnb.tn_kernel_bench(t.handle, op, mk, sk, nk, 5)
            alone[nm] = {"ms": round(ms1, 4), "tflops": round(2.0 * mk * nk * sk / ms1 * 1e-9, 2),
                         "frac_fp64_tensor": round(2.0 * mk * nk * sk / ms1 * 1e-9 / fp64_peak, 4),
                         "gbs": round(8.0 * mk * nk / ms1 * 1e-6, 1)}
        return alone

    # ---- main arm: W warm-up steps, then K timed steps on the resident instance
    t = make_tn(inst)
    for _ in range(args.warmup):
        step(t, beta, run)
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    ms_total, outs = timed(lambda: step(t, beta, run), args.steps)
    barrier()
    st = t.stats()                                               # stage timers of the last timed step
    log_z = t.log_z()
    drop_states = None
    if args.droplets:                                            # main branches and their single-droplet excitations
        states0 = outs[0]
        ex = [states0]
        for r in range(states0.shape[0]):
            dE, flips = t.droplets(r)
            if len(dE):
                ex.append((states0[r][None, :].astype(np.int32) * (1 - 2 * flips.astype(np.int32))).astype(np.int8))
        drop_states = np.concatenate(ex, axis=0)
        drop_E = t.energy(drop_states)                           # O-0 energies on the device (tn_energy)
    alone = kernel_alone(t, inst, run) if (rank == 0 and run["D"] > 0) else None
    t.close()

    # ---- e2e: host buffers in, host buffers out, tn_create / tn_destroy inside the timed region
    def e2e_step():
        with make_tn(inst) as tt:
            return step(tt, beta, run)
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
    states, E, logp, pd = outs
    replicas = None
    if args.replicas == "transforms":
        # best-of-maps energy and the spread of log Z over the maps
        if world > 1:
            got = [None] * world
            dist.all_gather_object(got, (transform, float(E.min()), float(log_z)))
            replicas = {"mode": "one map per rank", "maps": [g[0] for g in got], "best_energy_per_map": [g[1] for g in got],
                        "best_energy": min(g[1] for g in got), "z_spread": zspread([g[2] for g in got])}
        elif rank == 0:
            replicas = transforms_on_streams(tnb, instances, base_inst, run, beta, args, torch)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    K = args.steps
    ms_step = ms_total / K
    value = whole_job_value(ms_total, K, world)                  # seconds per instance over the whole job
    h2d = int(inst.edge_u.nbytes + inst.edge_v.nbytes + inst.J.nbytes + inst.h.nbytes + inst.cell_y.nbytes
              + inst.cell_x.nbytes + inst.sub.nbytes + inst.pos.nbytes)
    d2h = int(run["M"] * inst.n_spins + 2 * 8 * run["M"] + 8 + 4)
    stages, roofline = stage_report(st, args.config, fp64_peak, peaks, peak_src)
    roofline["kernel_alone"] = alone
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "l2": "flushed (256 MiB fill) between timed steps",
            "config": config_record(args.config, inst, run, beta, args.merge, transform, world),
            "contract_rows_per_s": round(st["rows_contracted"] / max(st["ms_contract"], 1e-9) * 1e3, 3),
            "contract_ms": round(st["ms_contract"], 3), "search_ms": round(st["ms_search"], 3),
            "best_energy": float(E.min()), "log_z": float(log_z), "n_states": int(len(E)), "log_p_discarded": float(pd),
            "min_sigma_rel": st["min_sigma_rel"], "negative_u": int(st["negative_u"]),
            "svd_unconverged": int(st["svd_unconverged"]), "merge_fallback_cells": int(st["merge_fallback_cells"]),
            "gpu_launches": int(st["kernel_launches"]) * K, "launches_per_step": int(st["kernel_launches"]),
            "stages": stages, "roofline": roofline, "clocks": clocks,
            "fp64_tensor_peak_tflops": round(fp64_peak, 2)}
    if replicas is not None:
        line["replicas"] = replicas
    if "E0" in inst:
        line["planted"] = diversity_report(inst, states, E)
    if drop_states is not None:
        Ed = drop_E
        line["droplets"] = {"main_branches": int(states.shape[0]), "states_with_single_droplets": int(drop_states.shape[0]),
                            "droplet_overflow": int(st["droplet_overflow"])}
        if "E0" in inst:
            line["droplets"]["planted"] = diversity_report(inst, drop_states, Ed)
    if e2e_ms is not None:
        line["e2e"] = {"value": whole_job_value(e2e_ms, K, world), "unit": UNIT, "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": d2h}
    # ---- the north_star target workload: ONE timed step of configs[3] (N = 5400, D = 64, M = 1024, 3 passes, beta = 2)
    if world == 1 and not args.no_headline and args.config != 3:
        line["headline"] = headline_record(tnb, instances, args, step, timed, fp64_peak, peaks, peak_src, local)
        if not args.no_headline_fast and args.svd_mode == "converged":
            line["headline_fast"] = headline_record(tnb, instances, args, step, timed, fp64_peak, peaks, peak_src, local,
                                                    svd_mode="randomized")
    if world == 1 and not args.no_cpu_baseline:
        smp = OracleSample(base_inst if not transform else inst, run, beta, ORACLE_SAMPLE[args.config])
        tm = smp.step()
        line["cpu_baseline"] = {"value": smp.estimate(), "unit": UNIT, "cores": host_threads(), "kind": "oracle",
                                "sample": smp.describe(), "extrapolated": not smp.whole, "sample_seconds": round(tm, 2)}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def set_contract_options(tnb, t, args, svd_mode=None):
    mode = svd_mode or args.svd_mode
    if mode == "randomized":
        t.set_option(tnb.OPT_SVD_MODE, 1)
    if args.schedule == "interleaved":
        t.set_option(tnb.OPT_SCHEDULE, 1)
    if args.two_step:
        t.set_option(tnb.OPT_TWO_STEP, 1)
    if args.oversample is not None:
        t.set_option(tnb.OPT_OVERSAMPLE, args.oversample)
    for kv in args.opt:
        k, v = kv.split("=")
        t.set_option(int(k), float(v))


def headline_record(tnb, instances, args, step, timed, fp64_peak, peaks, peak_src, local, svd_mode=None):
    """One timed step (after a tables-only warm-up of the handle) of BASELINE.json configs[3] at beta = 2: the
    ~5400-spin D = 64, M = 1024 instance of north_star, with its own stage table, roofline and clocks.  A single step:
    `steps` = 1, `warmup` = 0 -- a record inside the driver-observed run, not the line's `value`."""
    ci, bi = 3, 1
    inst, run = instances.config(ci)
    beta = run["beta"][bi]
    sampler = ClockSampler(local)
    t = tnb.TensorNetwork(inst)
    set_contract_options(tnb, t, args, svd_mode)
    if args.merge:
        t.set_option(tnb.OPT_MERGE, 1)
    sampler.start()
    ms, outs = timed(lambda: step(t, beta, run), 1)
    st = t.stats()
    lz = t.log_z()
    t.close()
    clocks = sampler.stop()
    states, E, logp, pd = outs
    stages, roofline = stage_report(st, ci, fp64_peak, peaks, peak_src)
    return {"config": dict(config_record(ci, inst, run, beta, args.merge, 0, 1), svd_mode=svd_mode or args.svd_mode,
                           schedule=args.schedule, two_step=bool(args.two_step)), "steps": 1, "warmup": 0,
            "svd_iterations": int(st["svd_iterations"]), "theta_apply_calls": int(st["theta_apply_calls"]),
            "value": ms * 1e-3, "unit": UNIT, "ms_per_step": ms, "contract_ms": round(st["ms_contract"], 3),
            "search_ms": round(st["ms_search"], 3), "best_energy": float(E.min()), "log_z": float(lz),
            "log_p_discarded": float(pd), "min_sigma_rel": st["min_sigma_rel"], "negative_u": int(st["negative_u"]),
            "svd_unconverged": int(st["svd_unconverged"]), "launches_per_step": int(st["kernel_launches"]),
            "peak_device_bytes": int(st["bytes_device"]), "stages": stages, "roofline": roofline, "clocks": clocks}


def transforms_on_streams(tnb, instances, inst, run, beta, args, torch):
    """N = 1: the 8 lattice transformations of ONE instance as concurrent replicas ("all 8 ...
    transformations"), one handle per map, `--streams` CUDA streams with one host thread each (a handle is
    single-threaded, distinct handles are independent).  Reports best-of-8, the log Z spread and the wall time of the
    whole batch next to the sum of the per-map device times."""
    import numpy as np
    ns = max(1, min(8, int(args.streams)))
    streams = [torch.cuda.Stream() for _ in range(ns)]
    res = [None] * 8

    def work(k):
        with torch.cuda.stream(streams[k]):
            for tmap in range(k, 8, ns):
                with tnb.TensorNetwork(instances.transformed(inst, tmap)) as t:   # binds the thread's current stream
                    if args.merge:
                        t.set_option(tnb.OPT_MERGE, 1)
                    t.set_beta(beta)
                    t.contract(run["D"], run["sweeps"])
                    lz = t.log_z()
                    states, E, logp, pd = t.branch_and_bound(run["M"])
                    st = t.stats()
                res[tmap] = (float(E.min()), float(lz), st["ms_contract"] + st["ms_search"] + st["ms_tables"])
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    th = [threading.Thread(target=work, args=(k,)) for k in range(ns)]
    for x in th:
        x.start()
    for x in th:
        x.join()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    return {"mode": "8 maps on %d stream(s), one GPU" % ns, "maps": list(range(8)),
            "best_energy_per_map": [r[0] for r in res], "best_energy": min(r[0] for r in res),
            "z_spread": zspread([r[1] for r in res]), "batch_wall_s": round(wall, 4),
            "sum_of_device_ms": round(sum(r[2] for r in res), 3)}


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
