"""Writes tests/golden/*.txt.  Calls ONLY oracle/ (and ensembles/ for the seeded inputs): no value here comes from the
CUDA path.  The paper prints no worked example or number for this method (PAPER.md:49 is an absent figure), so there
are no paper values to store; these files freeze the pinned oracle's own trajectories so that a later change to the
oracle's arithmetic shows up as a diff that its commit message has to justify.

    python tests/golden/make_golden.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import numpy as np

import ensembles as E
import oracle

ALPHA, TOL = 0.08, 1e-15


def trajectory(name, fft_mode):
    U, cfg = E.make_config(name)
    o = oracle.Oracle(cfg["dims"], cfg["storage"], fft_mode=fft_mode)
    o.load(U)
    r = o.fix(ALPHA, TOL, 1000, history=True)
    return cfg, r


def main():
    for name, fft_mode in (("C0", 0), ("C1", 1)):
        cfg, r = trajectory(name, fft_mode)
        path = os.path.join(HERE, f"oracle_{name}_trajectory.txt")
        with open(path, "w") as f:
            f.write(f"# oracle.fix(alpha=0.08, theta_tol=1e-15) on ensembles.make_config('{name}'): dims {cfg['dims']}, "
                    f"{cfg['storage']}-real, fft_mode {fft_mode} ({'naive DFT' if fft_mode == 0 else 'radix-2 FFT'})\n")
            f.write("# source: BASELINE.json configs / PAPER.md:47 (alpha, stopping rule); written by tests/golden/make_golden.py\n")
            f.write(f"# n_iter {r['n_iter']} status {r['status']}\n# k F_k theta_k\n")
            for k, (F, th) in enumerate(r["history"]):
                f.write(f"{k} {F:.17e} {th:.17e}\n")
        print(path, r["n_iter"])


if __name__ == "__main__":
    main()
