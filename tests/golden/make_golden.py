"""Writes tests/golden/tiny_oracle_sample.txt: a few oracle outputs of the `tiny` config.

Calls ONLY oracle/ and synthetic/ (never the CUDA path).  It is a regression anchor for the
oracle itself (so a later edit to bf_oracle.c that changes its arithmetic is noticed), not a
value from the paper -- the paper prints no beam powers (Figs. 5-7 are images).
Run:  python tests/golden/make_golden.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import synthetic  # noqa: E402

w = synthetic.make_workload("tiny")
P = oracle.beamform(w.ant_xyz, w.freqs, w.beam_dir, w.make_voltages(), w.nint)
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_oracle_sample.txt")
with open(out, "w") as fh:
    fh.write("# oracle.beamform on synthetic.make_workload('tiny') (numpy default_rng([0,0,0])), written by make_golden.py\n")
    fh.write("# chan beam bin power(fp64)\n")
    for (c, b, j) in [(0, 0, 0), (0, 15, 63), (31, 7, 20), (63, 8, 1), (63, 15, 63), (17, 3, 42)]:
        fh.write(f"{c} {b} {j} {float(P[c, b, j])!r}\n")
print("wrote", out)
