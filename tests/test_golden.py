"""Stored values: the paper's Table 3 (cited fixture) and the oracle's config-2 steady state (written by
tests/golden/make_golden.py, which calls only oracle/).  No CUDA code is touched."""
import os

import numpy as np

import closed_forms as cf

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_paper_table3_trend_brackets_oracle_error():
    """Table 3: the printed Laplace errors at sigma = 0.01 fall as ~c/R.  The oracle's own error
    on configs[0] (R_eff = 8.39, measured 1.98 %, test_oracle_physics.test_laplace_law_P5) must sit on the same
    trend: within a factor 1.5 of c/R_eff with c fitted to the table."""
    t = np.loadtxt(os.path.join(GOLD, "paper_table3_laplace.txt"))
    R, E = t[:, 0], t[:, 3]
    c = float((E * R).mean())                # E ~ c / R
    assert 13.0 < c < 17.0                   # ~15, SURVEY.md section 4
    assert np.all(np.abs(E * R / c - 1) < 0.25)
    predicted = c / 8.3915
    assert predicted / 1.5 < 1.975 < predicted * 1.5


def test_poiseuille_config2_golden():
    """BASELINE configs[1] proper (tau_A = 1.0, tau_B = 0.1; 147 000 oracle steps to |du| < 1e-10, stored):
    L2 error (Eq. 47) against the quadrature of Eq. 45 with the smooth mu(y) < 1 %; against the sharp piecewise
    parabola ~4 % (linear tau, reading on P6)."""
    path = os.path.join(GOLD, "poiseuille_config2.txt")
    d = np.loadtxt(path)
    head = open(path).read().split("\n")[2]
    assert "last_du=" in head and float(head.split("last_du=")[1].split()[0]) < 1e-10
    phi, ux = d[:, 1], d[:, 2]
    assert len(phi) == 128 and ux.max() > 0.02
    ta, tb = 1.0, 0.1
    ref = cf.poiseuille_quadrature(phi, lambda f: np.ones_like(f), lambda f: (tb + f * (ta - tb)) / 3.0, 1e-6)
    assert cf.l2_rel(ux, ref) < 0.01
    sharp = cf.poiseuille_sharp(128, ta / 3, tb / 3, 1e-6)
    assert cf.l2_rel(ux, sharp) < 0.06
    # interface stays where it was put and keeps the tanh shape (no drift at density ratio 1)
    fits = cf.tanh_width_fit(phi)
    assert len(fits) == 1 and abs(fits[0][0] / 4.0 - 1) < 0.05


def test_shear_interface_table4():
    """Table 4 prints 8.58e-3 for the error of Eq. 50 after the circular interface has been sheared
    and restored (Sec. 5.4).  The text is ambiguous about the period T of Eq. 48 (T_f or 2 T_f) and
    about which phase carries phi = 1; Eq. 8 is symmetric under phi -> 1 - phi, so the two choices differ only in the
    denominator of Eq. 50.  The oracle's four values (stored, phase_only mode, 200 x 200, 10 000 steps) bracket the
    printed one, and the reading (T = T_f, phi = 1 outside the circle) reproduces it to ~15 %: a WEAK pin of the g path
    (Eq. 33-36 + streaming) -- order of magnitude and mass conservation only."""
    d = np.loadtxt(os.path.join(GOLD, "shear_interface.txt"))
    paper = 8.58e-3
    vals = {}
    for pf, err, at_tf, mass, s_in, s_out in d:
        vals[(pf, "in")] = err
        vals[(pf, "out")] = err * np.sqrt(s_in / s_out)
        assert abs(mass) < 1e-11                      # "excellent mass conservation"
    assert min(vals.values()) < paper < max(vals.values())
    best = vals[(1.0, "out")]
    assert 0.5 * paper < best < 2.0 * paper, best
    assert vals[(2.0, "in")] > vals[(1.0, "in")]      # twice the stretching costs accuracy
