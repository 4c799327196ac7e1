"""Writes the stored oracle results under tests/golden/ (calls only oracle/ through tests/oracle_jobs.py).

  python tests/golden/make_golden.py            # ~10 minutes on one core

poiseuille_config2.txt: BASELINE.json configs[1] exactly as DESIGN.md fixes it (4x128x4, walls in y, tau_A = 1.0,
tau_B = 0.1 i.e. viscosity ratio 10, density ratio 1, g_x = 1e-6, fp64) run by the oracle until
max|u(t) - u(t-1)| < 1e-10; columns j, phi(y_j), u_x(y_j) (x,z-averaged; the fields are x,z-invariant).
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import numpy as np  # noqa: E402

import oracle_jobs  # noqa: E402


def main():
    r = oracle_jobs.poiseuille_steady(ny=128, tau_a=1.0, tau_b=0.1, visc_interp=0, tol=1e-10, check_every=1000)
    with open(os.path.join(HERE, "poiseuille_config2.txt"), "w") as fh:
        fh.write("# written by tests/golden/make_golden.py from oracle/clip_oracle.c (no CUDA code involved)\n")
        fh.write("# BASELINE.json configs[1]: 4x128x4, y walls, tau_A=1.0 tau_B=0.1, rho ratio 1, gx=1e-6, fp64\n")
        fh.write(f"# steps={r['steps']} last_du={r['du']:.3e} ux_spread={r['ux_spread']:.3e} uyz_max={r['uyz_max']:.3e}\n")
        for j, (a, b) in enumerate(zip(r["phi"], r["ux"])):
            fh.write(f"{j} {a:.17e} {b:.17e}\n")


if __name__ == "__main__":
    main()
