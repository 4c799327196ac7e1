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


def shear():
    """shear_interface.txt: PAPER.md:675-713 (Sec. 5.4, Table 4) run by the oracle in phase_only mode on 200 x 200 x 1 for both
    readings of the period T in Eq. 48 (T = T_f and T = 2 T_f), 10 000 steps each (~4 min each on one core)."""
    with open(os.path.join(HERE, "shear_interface.txt"), "w") as fh:
        fh.write("# written by tests/golden/make_golden.py from oracle/clip_oracle.c (phase_only mode; no CUDA code involved)\n")
        fh.write("# PAPER.md:675-713: L0=200, U0=0.04, M=0.0002, xi=3, Pe=600, circle R=40 at (100,60), run to 2 T_f = 10000 steps\n")
        fh.write("# columns: period_factor (T / T_f)  err_eq50 (phi = 1 inside the circle)  err at t = T_f  mass drift  sum(phi0^2)  sum((1-phi0)^2)\n")
        for pf in (1.0, 2.0):
            r = oracle_jobs.shear_interface(L0=200, period_factor=pf)
            fh.write(f"{pf} {r['err']:.9e} {r['stretch']:.9e} {r['mass']:.3e} {r['s_in']:.9e} {r['s_out']:.9e}\n")


def main():
    r = oracle_jobs.poiseuille_steady(ny=128, tau_a=1.0, tau_b=0.1, visc_interp=0, tol=1e-10, check_every=1000)
    with open(os.path.join(HERE, "poiseuille_config2.txt"), "w") as fh:
        fh.write("# written by tests/golden/make_golden.py from oracle/clip_oracle.c (no CUDA code involved)\n")
        fh.write("# BASELINE.json configs[1]: 4x128x4, y walls, tau_A=1.0 tau_B=0.1, rho ratio 1, gx=1e-6, fp64\n")
        fh.write(f"# steps={r['steps']} last_du={r['du']:.3e} ux_spread={r['ux_spread']:.3e} uyz_max={r['uyz_max']:.3e}\n")
        for j, (a, b) in enumerate(zip(r["phi"], r["ux"])):
            fh.write(f"{j} {a:.17e} {b:.17e}\n")


if __name__ == "__main__":
    if "--shear" in sys.argv:
        shear()
    else:
        main()
