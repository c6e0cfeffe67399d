#!/usr/bin/env python
"""Writes tests/golden/config1_sigma.txt - the FTLM stochastic error bar of BASELINE config 1.

    python tests/golden/make_config1_sigma.py            (about 6 minutes on 8 cores; calls only oracle/)

PAPER.md L213 and Eq. 22 (L225-L230): the statistical error of an FTLM estimate is the spread of the estimate over
independent sets of R random start vectors; reading 29 takes sigma_emp = sample standard deviation over
>= 10 seed sets.  Here: N = 16 ring, J = 1, all sectors N_up = 8..16 (M_z > 0 weighted twice), R = 20, N_L = 60,
200-point T grid, seeds SEED_VECTORS + 0..9, FP64 oracle only (oracle.ftlm_oracle.ftlm_run).  The GPU parity test
(tests/test_gpu_parity.py::test_config1_full_size_thermodynamics) requires |X_gpu - X_oracle| at the SAME seed to be
below sigma_emp(T) for X = C, chi at every T - on top of the 1e-4 relative criterion.
Columns: i  T  C_mean  C_sigma  chi_mean  chi_sigma.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import ftlm_oracle as fo  # noqa: E402
from paper_2605_26261_b200 import workloads as W  # noqa: E402  (seeded inputs only: bond list, T grid, seed)

N_SETS, R, N_L = 10, 20, 60


def main():
    w = W.baseline_config(1)
    T = W.temperature_grid(200)
    C, X = [], []
    for k in range(N_SETS):
        out, _, _ = fo.ftlm_run(w.N, w.bond_i, w.bond_j, w.J, 0.0, w.sectors, R, N_L, W.SEED_VECTORS + k, T)
        C.append(out["C"]); X.append(out["chi"])
        print(f"seed set {k}: C(T=1) = {np.interp(1.0, T, out['C']):.6f}", file=sys.stderr)
    C, X = np.array(C), np.array(X)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_sigma.txt")
    with open(path, "w") as f:
        f.write("# sigma_emp of C(T), chi(T) for BASELINE config 1 (PAPER.md L213, Eq. 22 L225-L230; DESIGN.md reading 29)\n")
        f.write(f"# written by tests/golden/make_config1_sigma.py: FP64 oracle, {N_SETS} seed sets (SEED_VECTORS + k), R = {R}, N_L = {N_L}\n")
        f.write("# i T C_mean C_sigma chi_mean chi_sigma\n")
        for i in range(T.shape[0]):
            f.write(f"{i} {T[i]:.12e} {C[:, i].mean():.10e} {C[:, i].std(ddof=1):.6e} {X[:, i].mean():.10e} {X[:, i].std(ddof=1):.6e}\n")
    print(path)


if __name__ == "__main__":
    main()
