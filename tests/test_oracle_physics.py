"""Pins of the CPU oracle, part 3: the physics the paper fixes.

The long oracle runs are started together in a process pool at the first use (tests/oracle_jobs.py), one run per
host core, so that the whole CPU suite stays within a few minutes.  Thresholds are the ones BASELINE.json's
north_star names (Laplace within 2 %, Poiseuille L2 < 1 %, relative drift of sum(phi) < 1e-12 per 1000 steps);
where the paper is silent the measured value is noted next to the bound.  No CUDA code is touched.
"""
import os
from concurrent.futures import ProcessPoolExecutor

import numpy as np
import pytest

import closed_forms as cf
import oracle_jobs


class _Pool:
    def __init__(self):
        self.ex = None
        self.fut = {}

    def get(self, name):
        if self.ex is None:
            from oracle import clip_oracle
            clip_oracle.build()  # compile once before the workers start
            self.ex = ProcessPoolExecutor(max_workers=max(1, min(len(oracle_jobs.JOBS), os.cpu_count() or 1)))
            self.fut = {k: self.ex.submit(oracle_jobs.run_job, k) for k in oracle_jobs.JOBS}
        return self.fut[name].result()

    def close(self):
        if self.ex is not None:
            self.ex.shutdown(wait=False, cancel_futures=True)


@pytest.fixture(scope="module")
def runs():
    p = _Pool()
    yield p
    p.close()


# ------------------------------------------------------------------------------------------------ P8: viscosity
@pytest.mark.parametrize("name", ["wave_xy", "wave_yz", "wave_zx", "wave_diag", "wave_diag_bgk"])
def test_shear_wave_decay_P8(runs, name):
    """P8: a small shear wave in a single-phase fluid decays as exp(-nu k^2 t) with nu = tau c_s^2 (Eq. 23,
    PAPER.md:209) and relaxation rate s_nu = 1/(tau + 1/2) (G3) on the 5 traceless second-order moments (G2); the
    diagonal wave exercises the (e_x^2 - e_y^2) moment, which a reading with only the 3 off-diagonal moments at
    s_nu would get wrong.  Lattice dispersion error is O(k^2) ~ 1e-3 here."""
    r = runs.get(name)
    amp, k2, tau = r["amp"], r["k2"], r["tau"]
    t = np.arange(len(amp))
    sel = slice(100, len(amp))
    slope = np.polyfit(t[sel], np.log(amp[sel]), 1)[0]
    nu = -slope / k2
    assert abs(nu / (tau / 3.0) - 1) < 0.01, (name, nu, tau / 3.0)


# ------------------------------------------------------------------------------------------------ P5 + P2: drop
def test_laplace_law_P5(runs):
    """P5 (north_star; Eq. 44 PAPER.md:614 in its 3-D form dp = 2 sigma / R, reading G5; Table 3):
    stationary drop of BASELINE configs[0]; dp = mean p (r < R/2) - mean p (r > R + 2W); R_eff from the drop volume.
    Measured 1.0198 (the continuum value of an unrelaxed tanh drop at R = 8, W = 4 is already 1.022, and the
    paper's own errors run ~15/R %, 1.04 % at R = 15)."""
    r = runs.get("laplace")
    R_eff = (3 * r["sum1"] / (4 * np.pi)) ** (1 / 3)
    ratio = r["dp"] / (2 * 0.01 / R_eff)
    assert abs(ratio - 1) < 0.02, ratio
    assert abs(r["dp"] / r["dp_prev"] - 1) < 1e-6          # stationary
    assert r["umax"] < 1e-4                                  # spurious currents (measured 2.7e-5)
    assert r["dp"] > 0                                       # higher pressure inside (sign of F_s, G4)


def test_phi_conservation_P2(runs):
    """P2 (north_star): relative drift of total phi < 1e-12 per 1000 steps in fp64 on configs[0]."""
    r = runs.get("laplace")
    assert r["steps"] == 1000
    assert abs(r["sum1"] - r["sum0"]) / r["sum0"] < 1e-12
    assert -1e-3 < r["phi_min"] and r["phi_max"] < 1 + 1e-3


def test_drop_interface_width(runs):
    """PAPER.md:618 / Eq. 5: the relaxed drop keeps a tanh interface of width ~W (4-5 cells)."""
    r = runs.get("laplace")
    fits = cf.tanh_width_fit(r["phi_line"])
    assert len(fits) == 2
    for W, res in fits:
        assert abs(W / 4.0 - 1) < 0.10 and res < 0.02, (W, res)


# ------------------------------------------------------------------------------------------------ P3: tanh profile
@pytest.mark.parametrize("name", ["tanh_wide", "tanh_narrow"])
def test_tanh_equilibrium_profile_P3(runs, name):
    """P3 (north_star; Eq. 5): a flat interface started at width 2W or W/2 relaxes to the tanh
    profile of width W; the column stays 1-D, at rest, and conserves phi."""
    r = runs.get(name)
    fits = cf.tanh_width_fit(r["phi"])
    assert len(fits) == 2
    for W, res in fits:
        assert abs(W / 4.0 - 1) < 0.05, (name, W)      # measured within ~2 %
        assert res < 1e-2, (name, res)
    assert r["spread"] < 1e-13 and r["umax"] < 1e-6
    assert abs(r["sum1"] - r["sum0"]) / r["sum0"] < 1e-11


# ------------------------------------------------------------------------------------------------ P6, P7: Poiseuille
def _mu_rho(params):
    ta, tb, ra, rb = params["tau_a"], params["tau_b"], params["rho_a"], params["rho_b"]
    rho_of = lambda phi: rb + phi * (ra - rb)
    if params["visc_interp"] == 2:  # Eq. 25 / 46b: the dynamic viscosity itself is linear in phi
        return rho_of, (lambda phi: rb * tb / 3.0 + phi * (ra * ta / 3.0 - rb * tb / 3.0))
    if params["visc_interp"] == 1:
        tau_of = lambda phi: 1.0 / (1.0 / tb + phi * (1.0 / ta - 1.0 / tb))
    else:
        tau_of = lambda phi: tb + phi * (ta - tb)
    return rho_of, (lambda phi: rho_of(phi) * tau_of(phi) / 3.0)


def test_poiseuille_vs_eq45_P6(runs):
    """P6-(i): steady layered Poiseuille (configs[1] family: 4x128x4, walls in y, viscosity ratio 10, density ratio 1,
    g = 1e-6) against the quadrature of Eq. 45 with the smooth mu(y) the method itself uses
    (linear tau(phi), Eq. 24) -- the comparison the paper makes: L2 (Eq. 47) < 1 %."""
    r = runs.get("pois_linear")
    assert r["du"] < 1e-10
    rho_of, mu_of = _mu_rho(r["params"])
    ref = cf.poiseuille_quadrature(r["phi"], rho_of, mu_of, r["params"]["gx"])
    err = cf.l2_rel(r["ux"], ref)
    assert err < 0.01, err
    assert r["ux_spread"] < 1e-12 and r["uyz_max"] < 1e-10


def test_poiseuille_sharp_closed_form_P6ii(runs):
    """P6-(ii) (north_star: closed-form piecewise-parabolic profile, L2 < 1 %): with harmonic interpolation of tau
    (visc_interp = 1, not in the paper) the diffuse-interface solution sits within 1 % of the sharp two-layer
    parabola; with the paper's linear tau (Eq. 24) the smooth-mu solution of Eq. 45 itself differs from the sharp
    one by ~4 % (a property of the interpolation), so that case is bounded at 6 % and reported."""
    rh, rl = runs.get("pois_harmonic"), runs.get("pois_linear")
    for r, bound in ((rh, 0.01), (rl, 0.06)):
        pr = r["params"]
        sharp = cf.poiseuille_sharp(pr["ny"], pr["rho_a"] * pr["tau_a"] / 3, pr["rho_b"] * pr["tau_b"] / 3, pr["rho_a"] * pr["gx"])
        err = cf.l2_rel(r["ux"], sharp)
        print("sharp-form L2:", "harmonic" if pr["visc_interp"] else "linear", err)
        assert err < bound, (pr["visc_interp"], err)


def test_poiseuille_density_ratio_bgk(runs):
    """SURVEY 8(f) NEXT-1, BGK mode (Eq. 26 with the viscous force of Eq. 29): the same
    rho* = 10, mu* = 100 Poiseuille case against the quadrature of Eq. 45 -- Eq. 29's prefactor nu / ((tau + 1/2) c_s^2)
    is what makes the stress in F_mu the physical one when every moment relaxes at 1 / (tau + 1/2)."""
    r = runs.get("pois_rho10_bgk")
    assert r["du"] < 1e-12
    rho_of, mu_of = _mu_rho(r["params"])
    ref = cf.poiseuille_quadrature(r["phi"], rho_of, mu_of, r["params"]["gx"])
    err = cf.l2_rel(r["ux"], ref)
    assert err < 0.02, err


def test_poiseuille_linear_mu_eq25(runs):
    """SURVEY 8(f) NEXT-6, visc_interp = 2 (Eq. 25): mu, not tau, is linear in phi -- exactly the
    viscosity field of the paper's Poiseuille comparison, Eq. 46b.  The rho* = 10, mu* = 100 case
    against the quadrature of Eq. 45 with mu(y) = mu_L + phi (mu_H - mu_L); the same run must NOT fit the
    quadrature with the linear-tau viscosity of Eq. 24 (the two differ by ~10 % at this density ratio), so a mode
    that silently fell back to Eq. 24 fails."""
    r = runs.get("pois_rho10_mu")
    assert r["du"] < 1e-12
    rho_of, mu_of = _mu_rho(r["params"])
    ref = cf.poiseuille_quadrature(r["phi"], rho_of, mu_of, r["params"]["gx"])
    err = cf.l2_rel(r["ux"], ref)
    print("Eq. 25 Poiseuille L2:", err)
    assert err < 0.01, err
    other = dict(r["params"]); other["visc_interp"] = 0
    rho0, mu0 = _mu_rho(other)
    err0 = cf.l2_rel(r["ux"], cf.poiseuille_quadrature(r["phi"], rho0, mu0, r["params"]["gx"]))
    assert err0 > 5 * err and err0 > 0.02, (err, err0)


def test_poiseuille_density_ratio_P7(runs):
    """P7: the paper's Fig. 11a case family (rho* = 10, mu* = 100, F_b = rho g) against the
    quadrature of Eq. 45 with smooth rho(y), mu(y): the one pin that exercises F_mu (Eq. 30) and F_p (Eq. 21)
    under shear (both vanish at density ratio 1)."""
    r = runs.get("pois_rho10")
    assert r["du"] < 1e-12
    rho_of, mu_of = _mu_rho(r["params"])
    ref = cf.poiseuille_quadrature(r["phi"], rho_of, mu_of, r["params"]["gx"])
    err = cf.l2_rel(r["ux"], ref)
    assert err < 0.02, err


# ------------------------------------------------------------------------------------------------ P14: advection
def test_galilean_drift_P14(runs):
    """P14: with sigma = 0, equal densities and uniform u0, F == 0 and uniform translation is an exact solution of
    Eq. 8-9: u stays u0, p stays 0, phi is conserved and its centre of mass moves by u0 t."""
    r = runs.get("galilean")
    assert r["du"] < 1e-13 and r["pmax"] < 1e-13
    phi0, phi = r["phi0"], r["phi"]
    assert abs(phi.sum() - phi0.sum()) / phi0.sum() < 1e-12
    n = phi.shape[0]
    ang = 2 * np.pi * np.arange(n) / n
    for c, ax in ((0, 2), (1, 1), (2, 0)):   # component c lives on array axis ax
        other = tuple(a for a in range(3) if a != ax)
        def com(f):
            m = f.sum(axis=other)
            return np.angle((m * np.exp(1j * ang)).sum()) * n / (2 * np.pi)
        shift = (com(phi) - com(phi0)) % n
        expect = r["u0"][c] * r["steps"]
        assert abs(shift - expect) < 0.05, (c, shift, expect)
