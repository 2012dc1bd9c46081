#!/usr/bin/env python
"""Writes tests/golden/cfg4_200step_oracle.txt: the ORACLE's long-run diagnostics of BASELINE.json
config 4 exactly as specified (16384 cells x 4000 ppc x 2 species = 1.31e8 particles, 200 free-running
steps, seed 7).  Calls only oracle/ and the seeded input generator (paper_1104_3998_b200/workloads.py,
which holds none of the method's arithmetic); nothing from the CUDA path is imported or run.

    python tests/golden/make_long_run_golden.py [--config 4] [--steps 200] [--every 10]

Takes ~20 min of one core and ~8 GB of RAM.  The stored quantities are the ones north_star's long-run
bar names: time-averaged n_e(x), n_i(x) (sampled every `every` steps) and phi(x) (same samples), and the
series of particle counts, <v^2> and <v^4> per species at the sampled steps.  tests/test_gpu_parity.py
runs the GPU alone and compares against this file (relative L2 <= 1 %).
"""
import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import oracle as O  # noqa: E402
from paper_1104_3998_b200 import workloads as W  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--every", type=int, default=10)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    out = a.out or os.path.join(HERE, "cfg%d_%dstep_oracle.txt" % (a.config, a.steps))
    p = W.make_params(a.config)
    parts = W.make_particles(p)
    o = O.Oracle(p)
    for s, arr in enumerate(parts):
        o.load_particles(s, *arr)
    del parts
    acc = [0.0, 0.0, 0.0]
    series = []
    t0 = time.time()
    n_samples = 0
    for n in range(1, a.steps + 1):
        rc = o.step(1)
        assert rc == 0, rc
        if n % a.every == 0:
            m = [o.moments(s) for s in range(2)]
            acc[0] = acc[0] + m[0]["density"]
            acc[1] = acc[1] + m[1]["density"]
            acc[2] = acc[2] + o.get_rho_phi_E()[1]
            n_samples += 1
            row = [n]
            for s in range(2):
                row += [m[s]["count"], m[s]["sum_v2"] / m[s]["count"], m[s]["sum_v4"] / m[s]["count"]]
            series.append(row)
            print("step %d  %.0f s  N_e %d  N_i %d" % (n, time.time() - t0, m[0]["count"], m[1]["count"]), flush=True)
    with open(out, "w") as f:
        f.write("# oracle long-run diagnostics; written by tests/golden/make_long_run_golden.py (calls only oracle/)\n")
        f.write("# workload: BASELINE.json config %d, %s: %d cells x %d ppc x 2 species, seed %d, %d steps, sampled every %d\n"
                % (a.config, p["name"], p["n_cells"], p["ppc"], p["seed"], a.steps, a.every))
        f.write("# quantities: north_star long-run bar (200-step density, potential, energy-distribution moments)\n")
        f.write("series %d  # step N_e <v2>_e <v4>_e N_i <v2>_i <v4>_i\n" % len(series))
        for row in series:
            f.write("%d %d %.12e %.12e %d %.12e %.12e\n" % tuple(row))
        for name, arr in zip(("mean_n_e", "mean_n_i", "mean_phi"), acc):
            arr = np.asarray(arr) / n_samples
            f.write("%s %d\n" % (name, arr.shape[0]))
            for i in range(0, arr.shape[0], 8):
                f.write(" ".join("%.9e" % v for v in arr[i:i + 8]) + "\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
