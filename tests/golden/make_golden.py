"""Writes tests/golden/cfg1_bruteforce.txt.  Calls ONLY oracle/ (+ the seeded generator).

The paper prints no worked numerical example, so the stored values are the
plain definition -- enumeration of all 2^24 states of BASELINE.json config 1, Eq. (1) PAPER.md:53,
Eq. (6)/(10) PAPER.md:90,119 -- evaluated by oracle.brute.  Run:  python tests/golden/make_golden.py
"""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import instances  # noqa: E402
from oracle import brute  # noqa: E402

inst, run = instances.config(0)
E = brute.all_energies(inst)
idx, El = brute.lowest(E, 16)
with open(os.path.join(os.path.dirname(__file__), "cfg1_bruteforce.txt"), "w") as f:
    f.write("# BASELINE.json config 1 (2x3 cells of 4 spins, seed 0, beta = 1): brute force over 2^24 states\n")
    f.write("# Eq. (1) PAPER.md:53, Eq. (10) PAPER.md:119; written by tests/golden/make_golden.py\n")
    f.write("log_z %.17g\n" % brute.log_z(E, run["beta"][0]))
    for k, e in zip(idx.tolist(), El.tolist()):
        f.write("state %d energy %.17g\n" % (k, e))
