"""Closed-form / semi-analytic references the oracle is pinned against (numpy only; no oracle, no CUDA code).

Each function states the passage of PAPER.md it restates.
"""
from __future__ import annotations

import numpy as np


def poiseuille_sharp(ny, mu_a, mu_b, rho_g):
    """Sharp two-layer solution of Eq. 45: d/dy(mu du/dy) + rho g = 0 with constant rho g = G,
    fluid A (mu_a) in 0 <= y < H/2, fluid B (mu_b) above, no-slip at y = 0 and y = H = ny (halfway bounce-back puts
    the wall half a cell outside the last node), nodes at y_j = j + 1/2.
    Continuity of u and of the shear stress at y = H/2 gives the integration constant T = mu u'(0)."""
    H = float(ny)
    y = np.arange(ny) + 0.5
    G = rho_g
    T = G * H / 4 * (3 * mu_a + mu_b) / (mu_a + mu_b)
    ua = -G * y ** 2 / (2 * mu_a) + T * y / mu_a
    ub = G * (H ** 2 - y ** 2) / (2 * mu_b) - T * (H - y) / mu_b
    return np.where(y < H / 2, ua, ub)


def poiseuille_quadrature(phi_nodes, rho_of, mu_of, g, sub=200):
    """Eq. 45 integrated for smooth rho(y), mu(y) -- the paper's own comparison is against a
    finite-difference solution of Eq. 45 with the smoothed fields of Eq. 46.

    phi_nodes: steady phi at the nodes y_j = j + 1/2; extended to the walls y = 0, H by the clamp rule (R9) and
    interpolated linearly.  First integral: mu u' = T - B(y), B = int_0^y rho g; u(0) = u(H) = 0 fixes T.
    """
    ny = len(phi_nodes)
    yn = np.concatenate([[0.0], np.arange(ny) + 0.5, [float(ny)]])
    pn = np.concatenate([[phi_nodes[0]], phi_nodes, [phi_nodes[-1]]])
    y = np.linspace(0.0, float(ny), ny * sub + 1)
    phi = np.interp(y, yn, pn)
    mu, b = mu_of(phi), rho_of(phi) * g
    dy = y[1] - y[0]

    def cumtrapz(v):
        return np.concatenate([[0.0], np.cumsum(0.5 * (v[1:] + v[:-1]) * dy)])

    B = cumtrapz(b)
    I1, I2 = cumtrapz(1.0 / mu), cumtrapz(B / mu)
    T = I2[-1] / I1[-1]
    u = T * I1 - I2
    return np.interp(np.arange(ny) + 0.5, y, u)


def l2_rel(u, ref):
    """Eq. 47."""
    return float(np.sqrt(((u - ref) ** 2).sum() / (ref ** 2).sum()))


def tanh_width_fit(phi_line, lo=0.05, hi=0.95):
    """Width of an equilibrium profile phi = 1/2 + 1/2 tanh(2 z / W) (Eq. 5): least-squares slope of
    atanh(2 phi - 1) against the node index over one monotone crossing; returns (W_fit, max residual of phi)."""
    idx = np.where((phi_line > lo) & (phi_line < hi))[0]
    # split into contiguous runs, one per interface
    runs = np.split(idx, np.where(np.diff(idx) > 1)[0] + 1)
    out = []
    for r in runs:
        if len(r) < 3:
            continue
        t = np.arctanh(2 * phi_line[r] - 1)
        A = np.vstack([r.astype(float), np.ones(len(r))]).T
        (s, c), *_ = np.linalg.lstsq(A, t, rcond=None)
        W = 2.0 / abs(s)
        fit = 0.5 + 0.5 * np.tanh(s * r + c)
        out.append((W, float(np.abs(fit - phi_line[r]).max())))
    return out


def prosperetti_capillary_wave(t, nu, k, sigma, rho_h, rho_l):
    """Eq. 41-42 (Prosperetti 1981): eta(t)/eta0 of a small-amplitude capillary wave between two
    fluids of equal kinematic viscosity nu, no gravity.  omega0^2 = sigma k^3 / (rho_h + rho_l), gamma = rho_h rho_l /
    (rho_h + rho_l)^2, z_i the four roots of Eq. 42, Z_i = prod_{j != i} (z_j - z_i).  As printed, Eq. 41's first term reads
    ".../(8(1-4 gamma) nu^2 k^4 + omega0)" and Eq. 42's constant term "(1-4 gamma) nu k^2 + omega0^2": dimensionally both
    need omega0^2 and (nu k^2)^2 (Prosperetti's Eq. 21-22), which is what is evaluated here; eta(0) = 1 and the inviscid
    limit cos(omega0 t) pin that reading (tests/test_oracle_pins.py).  erfc of a complex argument through the Faddeeva
    function: erfc(x) = exp(-x^2) w(i x)."""
    from scipy.special import wofz
    t = np.maximum(np.asarray(t, dtype=np.float64), 1e-12)
    w0sq = sigma * k ** 3 / (rho_h + rho_l)
    gam = rho_h * rho_l / (rho_h + rho_l) ** 2
    nk2 = nu * k * k
    erfc = lambda x: np.exp(-x * x) * wofz(1j * x)
    z = np.roots([1.0, -4 * gam * np.sqrt(nk2), 2 * (1 - 6 * gam) * nk2, 4 * (1 - 3 * gam) * nk2 ** 1.5,
                  (1 - 4 * gam) * nk2 ** 2 + w0sq])
    out = 4 * (1 - 4 * gam) * nk2 ** 2 / (8 * (1 - 4 * gam) * nk2 ** 2 + w0sq) * erfc(np.sqrt(nk2 * t) + 0j)
    for i in range(4):
        Z = np.prod([z[j] - z[i] for j in range(4) if j != i])
        out = out + z[i] / Z * w0sq / (z[i] ** 2 - nk2) * np.exp((z[i] ** 2 - nk2) * t) * erfc(z[i] * np.sqrt(t))
    return out.real
