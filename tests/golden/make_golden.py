"""Writes tests/golden/cfg{1,2,3,4}_oracle.txt: the CPU oracle's result for BASELINE.json configs 1-4 on
the first 10,000 particles of each seeded ensemble -- loss flags, loss fraction, accepted / rejected totals
and the quartiles of the loss times (PAPER.md:25 g = 1[lost], Eq. 2; north_star: "loss fraction
within 3 binomial standard deviations at n >= 1e4").

Config 1 is traced to its own T = 1e-3 s.  Configs 2, 3 and 4 (T = 1e-2 s, 1e5-1e6 particles) are traced
to T = 1e-3 s on their first 10,000 particles: that is what the oracle finishes in minutes on 8 cores
(BASELINE.md section 3); the T used is written into each file and the GPU test traces to the same T.

Calls only oracle/ and the seeded input generator; nothing here comes from the CUDA path.
Usage: python tests/golden/make_golden.py [1 2 3 4]      (default: all four; ~20 minutes on 8 cores)
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import catapult_oracle as O  # noqa: E402
from paper_2604_07617_b200 import workloads as W  # noqa: E402

N_GOLD = 10_000
T_GOLD = {1: 1e-3, 2: 1e-3, 3: 1e-3, 4: 1e-3}


def quartiles(v):
    return [float(q) for q in np.quantile(v, [0.25, 0.5, 0.75])] if len(v) else [float("nan")] * 3


def write_one(idx: int):
    cfg = W.config(idx, n=N_GOLD, T=T_GOLD[idx])
    f, p = O.Field(cfg["field"]), O.make_params(cfg["params"])
    t0 = time.time()
    r = O.trace(f, p, cfg["x0"])
    dt = time.time() - t0
    lost = (r["status"] == 1).astype(int)
    path = os.path.join(HERE, f"cfg{idx}_oracle.txt")
    with open(path, "w") as fh:
        fh.write(f"# oracle result for BASELINE.json configs[{idx}], first {N_GOLD} particles, traced to T below\n")
        fh.write("# (PAPER.md:25 g = 1[lost], PAPER.md:29 Eq. 2); written by tests/golden/make_golden.py from\n")
        fh.write("# oracle/catapult_oracle.c only\n")
        fh.write(f"# oracle wall time {dt:.1f} s on {O.max_threads()} threads\n")
        fh.write(f"n = {len(lost)}\n")
        fh.write(f"T = {T_GOLD[idx]:.10e}\n")
        fh.write(f"loss_fraction = {lost.mean():.10f}\n")
        fh.write(f"nacc_sum = {int(r['nacc'].sum())}\n")
        fh.write(f"nrej_sum = {int(r['nrej'].sum())}\n")
        fh.write(f"status_counts = {np.bincount(r['status'], minlength=4).tolist()}\n")
        q = quartiles(r["tstop"][lost == 1])
        fh.write(f"tstop_lost_median = {q[1]:.10e}\n")
        fh.write("tstop_lost_quartiles = " + " ".join(f"{v:.10e}" for v in q) + "\n")
        alive = r["status"] == 0
        fh.write(f"nacc_alive_median = {float(np.median(r['nacc'][alive])) if alive.any() else float('nan'):.1f}\n")
        fh.write("lost_bits = " + "".join(str(b) for b in lost) + "\n")
    print(f"cfg{idx}: done in {dt:.1f} s; loss fraction {lost.mean():.4f}; accepted {int(r['nacc'].sum())}", flush=True)


def main():
    which = [int(a) for a in sys.argv[1:]] or [1, 2, 3, 4]
    for idx in which:
        write_one(idx)


if __name__ == "__main__":
    main()
