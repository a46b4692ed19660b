"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol include/tn.h declares,
argument validation that precedes any device work, the no-CPU-fallback rule, and the multi-rank (replicas)
plumbing of bench.py under gloo with world_size 2."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

import instances

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    import paper_2411_16431_b200 as tnb
    from paper_2411_16431_b200 import build
    if not os.path.exists(os.path.join(ROOT, "paper_2411_16431_b200", "libtn_b200.so")):
        build.build()
    return tnb, tnb.lib()


def test_library_exports_every_declared_symbol():
    tnb, L = _lib()
    hdr = open(os.path.join(ROOT, "include", "tn.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(tn_[a-z0-9_]+)\s*\(", hdr))
    assert {"tn_create", "tn_set_beta", "tn_contract", "tn_branch_and_bound", "tn_destroy"} <= declared
    assert declared == set(tnb.EXPORTED_SYMBOLS), declared ^ set(tnb.EXPORTED_SYMBOLS)
    for name in sorted(declared):
        assert getattr(L, name) is not None          # ctypes raises AttributeError if the symbol is missing
    # and nothing under oracle/ is linked into, or imported by, the product
    out = subprocess.run(["nm", "-D", "--defined-only", os.path.join(ROOT, "paper_2411_16431_b200", "libtn_b200.so")],
                         capture_output=True, text=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln}
    assert declared <= exported


def test_product_never_imports_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2411_16431_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src.replace(
                    "under oracle/", ""), f


def test_argument_validation_before_device_work():
    tnb, _ = _lib()
    inst = instances.lattice(2, 2, 2, 2, seed=1)
    bad = instances.Instance(inst)
    bad["n_spins"] = inst.n_spins + 1                    # cluster map does not cover Ly*Lx*S*n_s slots
    with pytest.raises(tnb.TnError) as e:
        tnb.tn_create(bad.n_spins, inst.edge_u, inst.edge_v, inst.J, np.zeros(bad.n_spins), inst.Ly, inst.Lx, inst.S,
                      inst.n_s, np.zeros(bad.n_spins), np.zeros(bad.n_spins), np.zeros(bad.n_spins),
                      np.zeros(bad.n_spins))
    assert e.value.code == -2 and "slots" in str(e.value)
    with pytest.raises(tnb.TnError) as e:                # 3 spins per sub-cluster: odd
        tnb.tn_create(12, inst.edge_u[:0], inst.edge_v[:0], inst.J[:0], None, 1, 2, 2, 3, np.zeros(12), np.zeros(12),
                      np.zeros(12), np.zeros(12))
    assert e.value.code == -2


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    tnb, L = _lib()
    inst = instances.lattice(2, 2, 2, 2, seed=1)
    with pytest.raises(tnb.TnError) as e:
        tnb.tn_create(inst.n_spins, inst.edge_u, inst.edge_v, inst.J, inst.h, inst.Ly, inst.Lx, inst.S, inst.n_s,
                      inst.cell_y, inst.cell_x, inst.sub, inst.pos)
    assert e.value.code == -4                            # TN_ERR_CUDA: no silent CPU path
    v = ctypes.c_double(0.0)
    assert L.tn_fp64_peak(ctypes.byref(v)) == -4


WORKER = r'''
import os, sys, json
sys.path.insert(0, sys.argv[1])
import torch, torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
inst, run = bench.replica_instance(0, rank)             # config 0, one independent seeded replica per rank
ms = bench.max_over_ranks(100.0 + 50.0 * rank, world, device="cpu")
sig = float(inst.J.sum())
sigs = [None] * world
dist.all_gather_object(sigs, sig)
if rank == 0:
    print(json.dumps({"ms": ms, "value": bench.whole_job_value(ms, 1, world), "sigs": sigs}))
dist.destroy_process_group()
'''


def test_replicas_plumbing_gloo_world2(tmp_path):
    """bench.py --gpus N = N independent replicas: different seeds per rank, device time =
    max over ranks, value = seconds per instance over the whole job."""
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29577", WORLD_SIZE="2")
    procs = []
    for r in range(2):
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    import json
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["ms"] == 150.0                            # max over ranks
    assert abs(res["value"] - 0.150 / 2) < 1e-15         # two instances solved in 0.150 s
    assert res["sigs"][0] != res["sigs"][1]              # the replicas are different instances


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
