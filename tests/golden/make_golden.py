"""Writes tests/golden/cfg1_oracle.txt: the CPU oracle's result for BASELINE.json config 1
(10,000 alphas, T = 1e-3 s) -- loss flags, loss fraction and accepted-step total.

Calls only oracle/ and the seeded input generator; nothing here comes from the CUDA path.
Takes ~10 minutes on 8 cores.  Usage: python tests/golden/make_golden.py
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import catapult_oracle as O  # noqa: E402
from paper_2604_07617_b200 import workloads as W  # noqa: E402


def main():
    cfg = W.config(1)
    f, p = O.Field(cfg["field"]), O.make_params(cfg["params"])
    t0 = time.time()
    r = O.trace(f, p, cfg["x0"])
    dt = time.time() - t0
    lost = (r["status"] == 1).astype(int)
    with open(os.path.join(HERE, "cfg1_oracle.txt"), "w") as fh:
        fh.write("# oracle result for BASELINE.json configs[1] (PAPER.md:25 g = 1[lost], PAPER.md:29 Eq. 2)\n")
        fh.write("# written by tests/golden/make_golden.py from oracle/catapult_oracle.c only\n")
        fh.write(f"# oracle wall time {dt:.1f} s on {O.max_threads()} threads\n")
        fh.write(f"n = {len(lost)}\n")
        fh.write(f"loss_fraction = {lost.mean():.10f}\n")
        fh.write(f"nacc_sum = {int(r['nacc'].sum())}\n")
        fh.write(f"nrej_sum = {int(r['nrej'].sum())}\n")
        fh.write(f"status_counts = {np.bincount(r['status'], minlength=4).tolist()}\n")
        fh.write(f"tstop_lost_median = {float(np.median(r['tstop'][lost == 1])):.10e}\n")
        fh.write("lost_bits = " + "".join(str(b) for b in lost) + "\n")
    print("done in", dt, "s; loss fraction", lost.mean())


if __name__ == "__main__":
    main()
