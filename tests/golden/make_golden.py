"""Writes tests/golden/*.txt.  Calls ONLY oracle/ and workloads/ (never the CUDA path).

The paper (arXiv:1510.04068) prints no worked numerical example (all timings are in figures,
no force values anywhere), so there is no paper value to store.  The fixtures here are
  ring_sums.txt   closed-form inward acceleration of a regular n-gon (textbook; pure math below)
  cfg1_n64.txt    the oracle's outputs for a 64-particle scaled-down config 1 (regression pin so
                  that a later change to the oracle's arithmetic is noticed)
Run:  python tests/golden/make_golden.py
"""
import math
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from workloads import make_config  # noqa: E402


def main():
    with open(os.path.join(HERE, "ring_sums.txt"), "w") as f:
        f.write("# n  sum_{k=1}^{n-1} 1/sin(pi k/n)   (inward acc of a unit n-gon = m/4 * this; SURVEY sec 8(c) ring pin)\n")
        for n in (2, 3, 4, 6, 8, 17, 64):
            f.write(f"{n} {math.fsum(1 / math.sin(math.pi * k / n) for k in range(1, n))!r}\n")
    w = make_config(1, N=64)
    xp, vp, ap = oracle.predict(4, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk)
    r = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, w.ident, w.eps2, h2_i=w.h2 * 0.4, ngb_cap=16)
    with open(os.path.join(HERE, "cfg1_n64.txt"), "w") as f:
        f.write("# oracle output, config 1 recipe scaled to N=64 (seed 1510040681), 4th order, eps2=1e-6, t=1-2^-13\n")
        f.write("# i ax ay az jx jy jz pot nn_addr nn_d2 ngb_count   (hex floats)\n")
        for i in range(w.N):
            vals = list(r.acc[i]) + list(r.jerk[i]) + [r.pot[i]]
            f.write(f"{i} " + " ".join(float(v).hex() for v in vals)
                    + f" {r.nn_addr[i]} {float(r.nn_d2[i]).hex()} {r.ngb_count[i]}\n")


if __name__ == "__main__":
    main()
