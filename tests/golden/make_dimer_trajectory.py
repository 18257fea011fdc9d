"""Writes tests/golden/dimer_trajectory.txt from the CPU oracle ONLY (never the CUDA path).

BASELINE.json config 1 (dimer, K=1, D=4, dt = 1 fs): rho_11, rho_12, sum_u |sigma_u|_F^2 at
steps 1, 10, 100, 1000.  Regression fixture; the independent pins are in tests/test_oracle_*.py.
Run:  python tests/golden/make_dimer_trajectory.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import workloads                      # noqa: E402
from oracle.oracle import Oracle      # noqa: E402


def main():
    w = workloads.dimer()
    o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D)
    o.set_state(w.sigma0())
    rows, done = [], 0
    for s in (1, 10, 100, 1000):
        o.rk4_steps(w.dt_fs, s - done); done = s
        st = o.get_full_state()
        rows.append((s, st[0][0, 0].real, st[0][0, 1].real, st[0][0, 1].imag, (np.abs(st) ** 2).sum()))
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "dimer_trajectory.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_dimer_trajectory.py from oracle/ only\n")
        f.write("# step rho11 re(rho12) im(rho12) sum_frobenius_sq\n")
        for r in rows:
            f.write("%d %.17g %.17g %.17g %.17g\n" % r)
    print(open(out).read())


if __name__ == "__main__":
    main()
