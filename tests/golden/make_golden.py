"""Writes tests/golden/oracle_regression.txt.  Calls ONLY oracle/ (and the input
generator); never the CUDA path.

The paper (arXiv 1204.6367) prints no numeric value of P(u) or of a line
integral, so there is no paper-printed fixture to store.  This file freezes a
few oracle outputs on C0 and C1 so that an accidental change to the oracle's
arithmetic is noticed; it is a regression guard, not an independent pin (the
independent pins are in tests/test_oracle_pins.py).

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from workloads import make_workload  # noqa: E402

PIXELS = {"C0": [(32, 24), (20, 17), (40, 30), (0, 0), (31, 9)],
          "C1": [(128, 96), (10, 10), (200, 150), (77, 33), (255, 191)]}


def main():
    lines = ["# workload p i j j0 n signal LI_0 [LI_1 ...]   (oracle/gdrr_oracle.c, fp64)"]
    for name, pix in PIXELS.items():
        w = make_workload(name)
        arr = np.array([[0, i, j] for i, j in pix])
        out = oracle.project(w, pixels=arr)
        for q, (i, j) in enumerate(pix):
            li = " ".join(f"{x:.17g}" for x in out["line_integrals"][q])
            lines.append(f"{name} 0 {i} {j} {out['ray_table'][q, 0]} {out['ray_table'][q, 1]} "
                         f"{out['signal'][q]:.17g} {li}")
    with open(os.path.join(os.path.dirname(__file__), "oracle_regression.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")

    # the Siddon option on the same pixels, and the denoiser on a seeded image
    lines = ["# siddon: workload p i j n_segments signal LI_0 [LI_1 ...]   (oracle ray_siddon, fp64)"]
    for name, pix in PIXELS.items():
        w = make_workload(name)
        arr = np.array([[0, i, j] for i, j in pix])
        out = oracle.project(w, pixels=arr, method="siddon")
        for q, (i, j) in enumerate(pix):
            li = " ".join(f"{x:.17g}" for x in out["line_integrals"][q])
            lines.append(f"{name} 0 {i} {j} {out['n_segments'][q]} {out['signal'][q]:.17g} {li}")
    with open(os.path.join(os.path.dirname(__file__), "oracle_siddon_regression.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")

    rng = np.random.default_rng(12046367)
    img = rng.poisson(30.0, size=(6, 8)).astype(np.float64) + 1.0
    out = oracle.denoise(img, beta=0.25, n_iter=7)
    lines = ["# denoise: rng default_rng(12046367).poisson(30, (6, 8)) + 1, beta 0.25, 7 sweeps, omega 0.8; rows of S(7)"]
    lines += [" ".join(f"{x:.17g}" for x in row) for row in out]
    with open(os.path.join(os.path.dirname(__file__), "oracle_denoise_regression.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
