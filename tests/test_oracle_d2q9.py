"""Pins of the D2Q9 build of the oracle (oracle/clip_oracle.c with -DCLIPO_D2Q9; the lattice of the paper's 2-D benchmarks,
PAPER.md:568).  Same equations, so the pins are the 2-D versions of P1, P2, P5, P7, P8, P11, P15 -- plus one
that ties the two builds together: a z-invariant D3Q19 run of the phase-field equation IS the D2Q9 run (the D3Q19 weights project
onto 4/9, 1/9, 1/36 and Eq. 33 is linear in g; SURVEY.md:541-544)."""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import closed_forms as cf  # noqa: E402

from oracle.clip_oracle import Oracle  # noqa: E402
from paper_2505_12205_b200 import inputs  # noqa: E402

P_, WL, FS = inputs.PERIODIC, inputs.WALL, inputs.FREESLIP


def test_lattice_constants_and_basis_d2q9():
    """Weights 4/9, 1/9, 1/36; isotropy to 4th order with c_s^2 = 1/3; opposite pairs adjacent; M W M^T diagonal;
    dense M^-1 S M = I - (1 - s_nu) P with P built on the TWO-dimensional deviator (2 shear moments at s_nu, 7 at rate 1, G2)."""
    o = Oracle(4, 4, 1, inputs.default_params(lattice=1))
    e, w = o.lattice()
    assert o.Q == 9 and e.shape == (9, 3) and np.all(e[:, 2] == 0)
    assert sorted(np.round(w * 36).astype(int)) == [1, 1, 1, 1, 4, 4, 4, 4, 16] and abs(w.sum() - 1) < 1e-15
    assert len({tuple(v) for v in e.astype(int)}) == 9
    for a in range(1, 9, 2):
        assert np.all(e[a] == -e[a + 1])
    e2 = e[:, :2]
    assert np.abs(w @ e2).max() < 1e-16
    assert np.abs(np.einsum("a,ai,aj->ij", w, e2, e2) - np.eye(2) / 3).max() < 1e-16
    d = np.eye(2)
    iso4 = (np.einsum("ij,kl->ijkl", d, d) + np.einsum("ik,jl->ijkl", d, d) + np.einsum("il,jk->ijkl", d, d)) / 9
    assert np.abs(np.einsum("a,ai,aj,ak,al->ijkl", w, e2, e2, e2, e2) - iso4).max() < 1e-16
    M, Mi = o.basis()
    G = M @ np.diag(w) @ M.T
    assert np.abs(G - np.diag(np.diag(G))).max() < 1e-15 and np.abs(M @ Mi - np.eye(9)).max() < 1e-14
    Qa = np.einsum("ai,aj->aij", e2, e2) - np.eye(2) / 3
    dev = Qa - np.trace(Qa, axis1=1, axis2=2)[:, None, None] / 2 * np.eye(2)
    Pm = w[:, None] / (2 / 9) * np.einsum("aij,bij->ab", Qa, dev)
    for s in (0.3, 1.0, 1.9):
        A = o.collision_matrix(s)
        assert np.abs(A - (np.eye(9) - (1 - s) * Pm)).max() < 1e-15
        r = np.random.default_rng(1).normal(size=9)
        Pi = np.einsum("a,ai,aj->ij", r, e2, e2)
        out = np.einsum("a,ai,aj->ij", A @ r, e2, e2)
        assert np.abs(out - (s * (Pi - np.trace(Pi) / 2 * np.eye(2)) + np.trace(Pi) / 2 * np.eye(2))).max() < 1e-14   # stress identity
        assert abs((A @ r).sum() - r.sum()) < 1e-14 and np.abs((A @ r) @ e2 - r @ e2).max() < 1e-14                 # conserved moments


def test_stencils_exact_on_quadratics_d2q9():
    """Eq. 40a/b with the D2Q9 weights: exact gradient and Laplacian of any quadratic in x, y (interior nodes)."""
    n = 12
    o = Oracle(n, n, 1, inputs.default_params(lattice=1, bc=(WL,) * 4 + (P_, P_)))
    y, x = np.meshgrid(np.arange(n, dtype=float), np.arange(n, dtype=float), indexing="ij")
    phi = 0.3 + 0.1 * x - 0.2 * y + 0.05 * x * x - 0.03 * y * y + 0.07 * x * y
    G, L, mu = o.stencil_field(phi[None])
    inner = (slice(0, 1), slice(1, n - 1), slice(1, n - 1))
    assert np.abs(G[0][inner] - (0.1 + 0.1 * x + 0.07 * y)[None][inner]).max() < 1e-13
    assert np.abs(G[1][inner] - (-0.2 - 0.06 * y + 0.07 * x)[None][inner]).max() < 1e-13
    assert np.abs(G[2]).max() == 0.0 and np.abs(L[inner] - (0.1 - 0.06)).max() < 1e-13


def test_uniform_rest_and_conservation_d2q9():
    """P1: phi == 1 at rest: f == 0, u == 0, p == 0 bitwise.  P2: sum(phi) conserved to round-off over 1000 steps in a periodic box,
    a walled box and a free-slip box (R11: edges and corners)."""
    o = Oracle(8, 8, 1, inputs.default_params(lattice=1))
    o.init(np.ones((1, 8, 8)), np.zeros((3, 1, 8, 8)))
    o.step(200)
    phi, p, u = o.get()
    assert np.abs(u).max() == 0.0 and np.abs(p).max() == 0.0 and np.abs(phi - 1).max() < 1e-13
    for bc in ((P_,) * 6, (WL,) * 4 + (P_, P_), (FS, FS, WL, FS, P_, P_)):
        case = inputs.sweep2d(nx=24, ny=20, ndrops=3, rmin=3, rmax=5, precision=64, bc=bc)
        case["params"].update(rho_l=0.1, g=(1e-5, -2e-5, 0.0))
        o = Oracle.from_case(case)
        s0 = float(np.sum(case["phi0"], dtype=np.longdouble))
        o.step(1000)
        phi, p, u = o.get()
        assert np.isfinite(u).all() and abs(float(np.sum(phi, dtype=np.longdouble)) - s0) / s0 < 1e-12, bc
        assert np.abs(u[2]).max() == 0.0


@pytest.mark.parametrize("orient,tau,coll", [("xy", 0.8, 0), ("diag", 0.3, 0), ("diag", 0.6, 1)])
def test_shear_wave_decay_d2q9(orient, tau, coll):
    """P8 in two dimensions: nu = tau / 3 (Eq. 23) from the decay of a shear wave along y and along the (1,1) diagonal (both
    shear moments), WMRT and BGK."""
    n = 48
    y, x = np.meshgrid(np.arange(n, dtype=float), np.arange(n, dtype=float), indexing="ij")
    k0 = 2 * np.pi / n
    if orient == "xy":
        mode, comp, k2 = np.sin(k0 * y), np.array([1.0, 0.0]), k0 ** 2
    else:
        mode, comp, k2 = np.sin(k0 * (x + y)), np.array([1.0, -1.0]) / np.sqrt(2), 2 * k0 ** 2
    u0 = np.zeros((3, 1, n, n))
    u0[0, 0], u0[1, 0] = 1e-4 * comp[0] * mode, 1e-4 * comp[1] * mode
    o = Oracle(n, n, 1, inputs.default_params(lattice=1, rho_h=1.0, rho_l=1.0, tau_h=tau, tau_l=tau, sigma=0.0, collision=coll))
    o.init(np.ones((1, n, n)), u0)
    amp = []
    for t in range(601):
        if t:
            o.step(1)
        u = o.get()[2]
        amp.append(float(((comp[0] * u[0, 0] + comp[1] * u[1, 0]) * mode).sum() / (mode ** 2).sum()))
    amp = np.array(amp)
    t = np.arange(601)
    slope = np.polyfit(t[100:], np.log(amp[100:]), 1)[0]
    assert abs(-slope / (tau / 3 * k2) - 1) < 0.01, -slope / (tau / 3 * k2)


def test_laplace_law_2d():
    """Eq. 44 AS PRINTED, dp = sigma / R, is the two-dimensional law: stationary disc of radius 16 on 64 x 64,
    rho ratio 1000; R_eff from the disc area."""
    case = inputs.drop2d(n=64, R=16.0)
    n, R, W = 64, 16.0, 4.0
    o = Oracle.from_case(case)
    y, x = np.meshgrid(np.arange(n, dtype=float), np.arange(n, dtype=float), indexing="ij")
    r = np.sqrt((x - 31.5) ** 2 + (y - 31.5) ** 2)
    inside, outside = r < R / 2, r > R + 2 * W
    o.step(11900)
    p0 = o.get()[1][0]
    o.step(100)
    phi, p, u = o.get()
    dp_prev, dp = p0[inside].mean() - p0[outside].mean(), p[0][inside].mean() - p[0][outside].mean()
    R_eff = np.sqrt(phi.sum() / np.pi)
    ratio = dp / (0.01 / R_eff)
    print(f"2-D Laplace: ratio {ratio:.4f}, R_eff {R_eff:.3f}, stationarity {abs(dp / dp_prev - 1):.1e}, spurious u {np.abs(u).max():.1e}")
    assert abs(ratio - 1) < 0.02 and abs(dp / dp_prev - 1) < 5e-5 and np.abs(u).max() < 1e-4


def test_poiseuille_64_nodes_density_ratio_d2q9():
    """The paper's Sec. 5.3 set-up itself (2-D, 64 nodes across, rho* = 10, mu* = 100, F_b = rho g) against the
    quadrature of Eq. 45 with the smoothed rho(y), mu(y): exercises F_mu (Eq. 30) and F_p (Eq. 21) on D2Q9."""
    case = inputs.poiseuille2d(nx=4, ny=64, tau_a=5.0, tau_b=0.5, rho_a=10.0, rho_b=1.0, gx=1e-7)
    o = Oracle.from_case(case)
    du = 1.0
    while o.time < 200000 and du > 1e-12:
        o.step(499)
        prev = o.get()[2]
        o.step(1)
        phi, p, u = o.get()
        du = float(np.abs(u - prev).max())
    assert du <= 1e-12, (o.time, du)
    pr = case["params"]
    rho_of = lambda f: pr["rho_l"] + f * (pr["rho_h"] - pr["rho_l"])                      # noqa: E731
    mu_of = lambda f: rho_of(f) * (pr["tau_l"] + f * (pr["tau_h"] - pr["tau_l"])) / 3       # noqa: E731
    ref = cf.poiseuille_quadrature(phi[0].mean(axis=1), rho_of, mu_of, pr["g"][0])
    err = cf.l2_rel(u[0, 0].mean(axis=1), ref)
    print(f"D2Q9 Poiseuille rho* = 10: L2 = {err:.2e} after {o.time} steps")
    assert err < 0.02 and np.abs(u[1]).max() < 1e-9


def test_z_invariant_d3q19_phase_field_run_is_the_d2q9_run():
    """The D3Q19 weights project onto the D2Q9 ones along z (1/3 + 2/18 = 4/9, 1/18 + 2/36 = 1/9, 1/36) and Eq. 33 is linear in g with
    an equilibrium that projects too: with nz = 1 (periodic) and a prescribed in-plane velocity, the heavily pinned D3Q19 oracle and
    the D2Q9 build must give the same phi to round-off -- reversing shear flow of Sec. 5.4 at reduced size, 300 steps."""
    n, U0, W = 48, 0.04, 3.0
    y, x = np.meshgrid(np.arange(n, dtype=float), np.arange(n, dtype=float), indexing="ij")
    phi0 = 0.5 + 0.5 * np.tanh(2.0 * (n / 5 - np.sqrt((x - 0.5 * n) ** 2 + (y - 0.3 * n) ** 2)) / W)

    def vel(t):
        c = U0 * np.cos(np.pi * t / 600.0)
        return np.stack([c * np.sin(np.pi * x / n) ** 2 * np.sin(2 * np.pi * y / n), -c * np.sin(np.pi * y / n) ** 2 * np.sin(2 * np.pi * x / n),
                         np.zeros_like(x)])[:, None]
    out = []
    for lattice in (0, 1):
        p = inputs.default_params(W=W, M=U0 * W / 600.0, sigma=0.0, rho_h=1.0, rho_l=1.0, phase_only=1, lattice=lattice)
        o = Oracle(n, n, 1, p)
        o.init(phi0[None], vel(0))
        for k in range(300):
            o.set_u(vel(k)); o.step(1)
        out.append(o.get()[0])
    assert np.abs(out[0] - phi0).max() > 0.3               # the interface really moved
    assert np.abs(out[0] - out[1]).max() < 1e-13
