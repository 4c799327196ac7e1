"""Long oracle runs used by test_oracle_physics.py (and by tests/golden/make_golden.py), as picklable top-level
functions so that a process pool can run them side by side on the host cores.  Each returns a small dict of numpy
arrays / floats.  Only oracle/ and the seeded input generators are used here -- never the CUDA path.
"""
from __future__ import annotations

import numpy as np

from oracle.clip_oracle import Oracle
from paper_2505_12205_b200 import inputs


def laplace_drop(n=32, R=8.0, W=4.0, sigma=0.01, steps=1000):
    """BASELINE configs[0] run to stationarity; returns pressure jump pieces (Eq. 44 as read in G5), drift of
    sum(phi) (P2) and the spurious velocity."""
    case = inputs.drop(n=n, R=R, W=W, sigma=sigma)
    z, y, x = np.meshgrid(*[np.arange(n, dtype=float)] * 3, indexing="ij")
    c = 0.5 * (n - 1)
    r = np.sqrt((x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2)
    inside, outside = r < R / 2, r > R + 2 * W
    o = Oracle.from_case(case)
    s0 = float(np.sum(case["phi0"], dtype=np.longdouble))
    hist = []
    done = 0
    for chunk in (steps - 100, 100):
        o.step(chunk); done += chunk
        phi, p, u = o.get()
        hist.append(float(p[inside].mean() - p[outside].mean()))
    s1 = float(np.sum(phi, dtype=np.longdouble))
    return dict(dp=hist[-1], dp_prev=hist[-2], sum0=s0, sum1=s1, steps=done, umax=float(np.abs(u).max()),
                phi_line=phi[n // 2, n // 2, :].copy(), phi_min=float(phi.min()), phi_max=float(phi.max()))


def poiseuille_steady(ny=128, tau_a=5.0, tau_b=0.5, rho_a=1.0, rho_b=1.0, gx=1e-6, visc_interp=0, tol=1e-10,
                      max_steps=400000, check_every=500, collision=0):
    """Layered Poiseuille (BASELINE configs[1] family) run until max|u(t) - u(t-1)| < tol."""
    case = inputs.poiseuille(nx=4, ny=ny, nz=4, tau_a=tau_a, tau_b=tau_b, rho_a=rho_a, rho_b=rho_b, gx=gx,
                             visc_interp=visc_interp)
    case["params"]["collision"] = collision
    o = Oracle.from_case(case)
    du = np.inf
    while o.time < max_steps:
        o.step(check_every - 1)
        u_prev = o.get()[2]
        o.step(1)
        phi, p, u = o.get()
        du = float(np.abs(u - u_prev).max())
        if du < tol:
            break
    return dict(phi=phi.mean(axis=(0, 2)), ux=u[0].mean(axis=(0, 2)), steps=o.time, du=du,
                ux_spread=float(np.ptp(u[0], axis=(0, 2)).max()), uyz_max=float(max(np.abs(u[1]).max(), np.abs(u[2]).max())),
                params=dict(ny=ny, tau_a=tau_a, tau_b=tau_b, rho_a=rho_a, rho_b=rho_b, gx=gx, visc_interp=visc_interp))


def shear_wave(orient="xy", tau=0.8, n=64, steps=1000, A=1e-4, rho=1.0, collision=0):
    """P8: single-phase (phi = 1) decaying shear wave; returns the projected amplitude history.

    orient: "xy" u_x(y), "yz" u_y(z), "zx" u_z(x) on a 4-thick slab; "diag" u along (1,-1,0)/sqrt2 varying along
    (1,1,0) on n x n x 2.
    """
    if orient == "diag":
        nx, ny, nz = n, n, 2
    else:
        nx, ny, nz = {"xy": (4, n, 4), "yz": (4, 4, n), "zx": (n, 4, 4)}[orient]
    z, y, x = np.meshgrid(np.arange(nz, dtype=float), np.arange(ny, dtype=float), np.arange(nx, dtype=float), indexing="ij")
    k0 = 2 * np.pi / n
    u0 = np.zeros((3, nz, ny, nx))
    if orient == "xy":
        mode = np.sin(k0 * y); comp = np.array([1.0, 0, 0]); k2 = k0 ** 2
    elif orient == "yz":
        mode = np.sin(k0 * z); comp = np.array([0, 1.0, 0]); k2 = k0 ** 2
    elif orient == "zx":
        mode = np.sin(k0 * x); comp = np.array([0, 0, 1.0]); k2 = k0 ** 2
    else:
        mode = np.sin(k0 * (x + y)); comp = np.array([1.0, -1.0, 0]) / np.sqrt(2); k2 = 2 * k0 ** 2
    for c in range(3):
        u0[c] = A * comp[c] * mode
    p = inputs.default_params(rho_h=rho, rho_l=rho, tau_h=tau, tau_l=tau, sigma=0.0, collision=collision)
    o = Oracle(nx, ny, nz, p)
    o.init(np.ones((nz, ny, nx)), u0)
    amp = []
    norm = (mode ** 2).sum()
    for t in range(steps + 1):
        if t:
            o.step(1)
        u = o.get()[2]
        amp.append(float(sum(comp[c] * (u[c] * mode).sum() for c in range(3)) / norm))
    return dict(amp=np.array(amp), k2=k2, tau=tau)


def tanh_relax(W=4.0, W0_factor=2.0, nz=64, steps=20000, sigma=0.01):
    """P3: two flat interfaces on a 4 x 4 x nz periodic column, started with width W0 = W0_factor * W."""
    nx = ny = 4
    zc = np.arange(nz, dtype=float)
    W0 = W * W0_factor
    prof = 0.5 * (np.tanh(2 * (zc - (nz / 4 - 0.5)) / W0) - np.tanh(2 * (zc - (3 * nz / 4 - 0.5)) / W0))
    phi0 = np.broadcast_to(prof[:, None, None], (nz, ny, nx)).copy()
    p = inputs.default_params(rho_h=1.0, rho_l=0.1, sigma=sigma, W=W, M=0.1)
    o = Oracle(nx, ny, nz, p)
    o.init(phi0, np.zeros((3, nz, ny, nx)))
    o.step(steps)
    phi, pr, u = o.get()
    return dict(phi=phi[:, 0, 0].copy(), spread=float(np.ptp(phi, axis=(1, 2)).max()), umax=float(np.abs(u).max()),
                sum0=float(phi0.sum()), sum1=float(phi.sum()))


def galilean_drift(n=24, steps=400, u0=(0.01, 0.02, 0.005)):
    """P14: drop advected by a uniform velocity, sigma = 0, equal densities: uniform translation is exact."""
    case = inputs.drop(n=n, R=6.0, W=4.0, sigma=0.0, rho_ratio=1.0)
    for c in range(3):
        case["u0"][c] = u0[c]
    o = Oracle.from_case(case)
    o.step(steps)
    phi, p, u = o.get()
    return dict(phi0=case["phi0"], phi=phi, du=float(max(np.abs(u[c] - u0[c]).max() for c in range(3))),
                pmax=float(np.abs(p).max()), steps=steps, u0=u0)


def shear_interface(L0=200, U0=0.04, W=3.0, Pe=600.0, center=(0.5, 0.3), period_factor=2.0):
    """Sec. 5.4: circular interface of radius L0/5 in the reversing shear flow of Eq. 48 on a periodic
    L0 x L0 (x 1) lattice, phase-field equation only (u prescribed), M = U0 W / Pe (Eq. 49).  The velocity carries
    cos(pi t / T) with T = period_factor * T_f, T_f = L0 / U0 (Eq. 51): it reverses at t = T_f and the run ends at 2 T_f
    (PAPER.md:705), which fixes period_factor = 2 (the text's bare "T" is ambiguous).
    Returns the error of Eq. 50 and the mass drift."""
    M = U0 * W / Pe
    p = inputs.default_params(W=W, M=M, sigma=0.0, rho_h=1.0, rho_l=1.0, phase_only=1)
    y, x = np.meshgrid(np.arange(L0, dtype=float), np.arange(L0, dtype=float), indexing="ij")
    r = np.sqrt((x - center[0] * L0) ** 2 + (y - center[1] * L0) ** 2)
    phi0 = 0.5 + 0.5 * np.tanh(2.0 * (L0 / 5.0 - r) / W)
    Tf = L0 / U0
    T = period_factor * Tf
    sx, sy = np.sin(np.pi * x / L0) ** 2 * np.sin(2 * np.pi * y / L0), -np.sin(np.pi * y / L0) ** 2 * np.sin(2 * np.pi * x / L0)

    def vel(t):
        c = U0 * np.cos(np.pi * t / T)
        return np.stack([c * sx, c * sy, np.zeros_like(sx)])[:, None]

    o = Oracle(L0, L0, 1, p)
    o.init(phi0[None], vel(0))
    n = int(round(2 * Tf))
    phi_half = None
    for k in range(n):
        o.set_u(vel(k))
        o.step(1)
        if k + 1 == n // 2:
            phi_half = o.get()[0][0].copy()
    phi = o.get()[0][0]
    err = float(np.sqrt(((phi - phi0) ** 2).sum() / (phi0 ** 2).sum()))
    return dict(err=err, mass=float(phi.sum() / phi0.sum() - 1.0), steps=n, L0=L0, s_in=float((phi0 ** 2).sum()),
                s_out=float(((1 - phi0) ** 2).sum()),
                stretch=float(np.sqrt(((phi_half - phi0) ** 2).sum() / (phi0 ** 2).sum())))


JOBS = {
    "laplace": (laplace_drop, {}),
    "pois_linear": (poiseuille_steady, dict(visc_interp=0)),
    "pois_harmonic": (poiseuille_steady, dict(visc_interp=1)),
    "pois_rho10": (poiseuille_steady, dict(ny=64, tau_a=5.0, tau_b=0.5, rho_a=10.0, rho_b=1.0, gx=1e-7, tol=1e-12)),
    "wave_xy": (shear_wave, dict(orient="xy")),
    "wave_yz": (shear_wave, dict(orient="yz", tau=0.3)),
    "wave_zx": (shear_wave, dict(orient="zx", tau=1.5)),
    "wave_diag": (shear_wave, dict(orient="diag", n=64, steps=600)),
    "tanh_wide": (tanh_relax, dict(W0_factor=2.0)),
    "tanh_narrow": (tanh_relax, dict(W0_factor=0.5)),
    "galilean": (galilean_drift, {}),
    "wave_diag_bgk": (shear_wave, dict(orient="diag", n=64, steps=600, tau=0.6, collision=1)),
    "pois_rho10_mu": (poiseuille_steady, dict(ny=64, tau_a=5.0, tau_b=0.5, rho_a=10.0, rho_b=1.0, gx=1e-7, tol=1e-12, visc_interp=2)),
    "pois_rho10_bgk": (poiseuille_steady, dict(ny=64, tau_a=5.0, tau_b=0.5, rho_a=10.0, rho_b=1.0, gx=1e-7, tol=1e-12, collision=1)),
}


def run_job(name):
    fn, kw = JOBS[name]
    return fn(**kw)
