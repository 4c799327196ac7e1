"""Pins of the CPU oracle (oracle/clip_oracle.c) against what the paper and the mathematics fix -- algebraic part.

Every test here checks the oracle against something other than itself: closed forms, invariants, symmetry,
special cases (SURVEY.md 8(c) pins P1, P2, P4, P9-P15 and the readings G2, G4, G6, R8, R11, R12).  The slower
physics pins (Laplace law, Poiseuille, tanh profile, shear-wave viscosity) live in test_oracle_physics.py.
None of these tests touches the CUDA path.
"""
import numpy as np
import pytest

from oracle.clip_oracle import Oracle
from paper_2505_12205_b200 import inputs


# ------------------------------------------------------------------------------------------------ lattice
def test_lattice_constants():
    """Eq. 14-15: 19 velocities, weights 1/3, 1/18, 1/36; isotropy up to 4th order."""
    o = Oracle(4, 4, 4, inputs.default_params())
    e, w = o.lattice()
    assert e.shape == (19, 3) and len({tuple(v) for v in e.astype(int)}) == 19
    n2 = (e ** 2).sum(1)
    assert sorted(n2.tolist()) == [0] + [1] * 6 + [2] * 12
    assert np.allclose(w[n2 == 0], 1 / 3) and np.allclose(w[n2 == 1], 1 / 18) and np.allclose(w[n2 == 2], 1 / 36)
    assert abs(w.sum() - 1) < 1e-15
    assert np.abs(w @ e).max() < 1e-16
    assert np.allclose(np.einsum("a,ai,aj->ij", w, e, e), np.eye(3) / 3, atol=1e-16)          # c_s^2 = 1/3 (:172)
    d = np.eye(3)
    iso4 = (np.einsum("ij,kl->ijkl", d, d) + np.einsum("ik,jl->ijkl", d, d) + np.einsum("il,jk->ijkl", d, d)) / 9
    assert np.allclose(np.einsum("a,ai,aj,ak,al->ijkl", w, e, e, e, e), iso4, atol=1e-16)
    # opposite pairs adjacent; +x-pointing set is {1,7,9,11,13}
    for a in range(1, 19, 2):
        assert (e[a] == -e[a + 1]).all()
    assert [a for a in range(19) if e[a, 0] > 0] == [1, 7, 9, 11, 13]


def test_basis_and_collision_matrix_G2_P15():
    """G2/P15: M W M^T diagonal, M^-1 M = I, and dense M^-1 S M = I - (1 - s_nu) P with
    P_ab = w_a/(2 c_s^4) Q_a : dev(Q_b); second moment of (M^-1 S M r) = s_nu dev(Pi) + tr(Pi)/3 I; conserved
    moments untouched."""
    o = Oracle(4, 4, 4, inputs.default_params())
    e, w = o.lattice()
    M, Mi = o.basis()
    D = M @ np.diag(w) @ M.T
    assert np.abs(D - np.diag(np.diag(D))).max() < 1e-14
    assert np.abs(Mi @ M - np.eye(19)).max() < 1e-13
    Qa = np.einsum("ai,aj->aij", e, e) - np.eye(3) / 3
    dev = Qa - np.trace(Qa, axis1=1, axis2=2)[:, None, None] * np.eye(3) / 3
    P = 4.5 * w[:, None] * np.einsum("aij,bij->ab", Qa, dev)
    rng = np.random.default_rng(1)
    for s in (0.3, 1.0, 1.7, 1.0 / (0.8 + 0.5)):
        A = o.collision_matrix(s)
        assert np.abs(A - (np.eye(19) - (1 - s) * P)).max() < 2e-15
        r = rng.normal(size=19)
        t = A @ r
        Pi = np.einsum("a,ai,aj->ij", r, e, e)
        devPi = Pi - np.trace(Pi) / 3 * np.eye(3)
        assert np.abs(np.einsum("a,ai,aj->ij", t, e, e) - (s * devPi + np.trace(Pi) / 3 * np.eye(3))).max() < 1e-14
        assert abs(t.sum() - r.sum()) < 1e-14 and np.abs(t @ e - r @ e).max() < 1e-14
    assert np.abs(o.collision_matrix(1.0) - np.eye(19)).max() < 1e-14


def test_moment_identities_P12():
    """P12: sum feq_bar = p*, sum e feq_bar = u - F/(2 rho), sum e e feq = p* c_s^2 I + u u (Eq. 16-19);
    sum geq_bar = phi, sum F_a = sum F^phi_a = 0, sum e F^phi_a = c_s^2 [1-4(phi-1/2)^2]/W n (Eq. 34-36)."""
    p = inputs.default_params(rho_h=2.0, rho_l=0.5, W=3.0)
    o = Oracle(4, 4, 4, p)
    e, w = o.lattice()
    rng = np.random.default_rng(2)
    for _ in range(5):
        ps, phi = rng.normal() * 0.01, rng.uniform(0, 1)
        u, F = rng.normal(size=3) * 0.05, rng.normal(size=3) * 1e-3
        nv = rng.normal(size=3); nv /= np.linalg.norm(nv)
        rho = 0.5 + phi * 1.5
        feqb, Fa, geqb, Fphi = o.node_terms(ps, u, phi, F, nv)
        assert abs(feqb.sum() - ps) < 1e-16
        assert np.abs(feqb @ e - (u - F / (2 * rho))).max() < 1e-16
        feq = feqb + 0.5 * Fa
        assert np.abs(np.einsum("a,ai,aj->ij", feq, e, e) - (ps / 3 * np.eye(3) + np.outer(u, u))).max() < 1e-16
        assert abs(Fa.sum()) < 1e-17 and np.abs(Fa @ e - F / rho).max() < 1e-16
        pref = (1 - 4 * (phi - 0.5) ** 2) / 3.0
        assert abs(geqb.sum() - phi) < 1e-15 and abs(Fphi.sum()) < 1e-16
        assert np.abs(Fphi @ e - pref * nv / 3).max() < 1e-16
        assert np.abs(geqb @ e - (phi * u - 0.5 * pref * nv / 3)).max() < 1e-16


@pytest.mark.parametrize("coll", [0, 1])  # 1 = BGK: Eq. 29, every moment (the trace of Pi too) carries 1/(tau + 1/2)
def test_viscous_force_closed_form(coll):
    """Eq. 30 with Eq. 32 evaluated through the dense M^-1 S M must equal the closed form
    F_mu = -tau (rho_h-rho_l) [s_nu dev(Pi) + tr(Pi)/3 I] grad phi, Pi = sum e e (f - feq); F_p = -p* c_s^2 grad rho
    (Eq. 21); F_s = mu_phi grad phi (Eq. 10); F_b = (rho - rho_ref) g."""
    p = inputs.default_params(rho_h=3.0, rho_l=1.0, tau_h=0.3, tau_l=0.9, sigma=0.02, W=4.0, g=(1e-4, -2e-4, 3e-4),
                              rho_ref=0.7, collision=coll)
    o = Oracle(4, 4, 4, p)
    e, w = o.lattice()
    rng = np.random.default_rng(3)
    for _ in range(4):
        phi, ps = rng.uniform(0, 1), rng.normal() * 0.01
        u, G, L = rng.normal(size=3) * 0.03, rng.normal(size=3) * 0.2, rng.normal() * 0.05
        eu = e @ u
        feq = ps * w + w * (1 + 3 * eu + 4.5 * eu ** 2 - 1.5 * u @ u) - w
        f = feq + rng.normal(size=19) * 1e-3
        f += (ps - f.sum()) * w  # keep sum f = p*
        tau = 0.9 + phi * (0.3 - 0.9); s = 1 / (tau + 0.5); rho = 1 + 2 * phi
        Pi = np.einsum("a,ai,aj->ij", f - feq, e, e)
        S = s * Pi if coll == 1 else s * (Pi - np.trace(Pi) / 3 * np.eye(3)) + np.trace(Pi) / 3 * np.eye(3)
        beta, kappa = 12 * 0.02 / 4, 1.5 * 0.02 * 4
        mu = 4 * beta * phi * (phi - 1) * (phi - 0.5) - kappa * L
        F_expect = mu * G + (rho - 0.7) * np.array(p["g"]) - ps / 3 * 2.0 * G - tau * 2.0 * (S @ G)
        F = o.total_force(f, ps, u, phi, G, L)
        assert np.abs(F - F_expect).max() < 1e-15


# ------------------------------------------------------------------------------------------------ stencils
def test_stencil_exactness_P11():
    """P11: Eq. 40a/b are exact for polynomials up to second degree (interior nodes; 3 sum w e e = I, lap prefactor 6)."""
    p = inputs.default_params(bc=(inputs.WALL,) * 6)
    nx, ny, nz = 9, 8, 7
    o = Oracle(nx, ny, nz, p)
    z, y, x = np.meshgrid(np.arange(nz, dtype=float), np.arange(ny, dtype=float), np.arange(nx, dtype=float), indexing="ij")
    phi = 0.3 + 0.1 * x - 0.2 * y + 0.05 * z + 0.01 * x * x - 0.02 * y * y + 0.03 * z * z + 0.015 * x * y - 0.01 * y * z + 0.02 * x * z
    G, L, mu = o.stencil_field(phi)
    I = (slice(1, -1),) * 3
    gx = 0.1 + 0.02 * x + 0.015 * y + 0.02 * z
    gy = -0.2 - 0.04 * y + 0.015 * x - 0.01 * z
    gz = 0.05 + 0.06 * z - 0.01 * y + 0.02 * x
    assert np.abs(G[0][I] - gx[I]).max() < 1e-14 and np.abs(G[1][I] - gy[I]).max() < 1e-14
    assert np.abs(G[2][I] - gz[I]).max() < 1e-14
    assert np.abs(L[I] - 2 * (0.01 - 0.02 + 0.03)).max() < 1e-13


def test_stencil_periodic_fourier_symbol():
    """On a periodic box the stencils act on a Fourier mode by their symbols: grad -> i*3 sum_a w_a e_a sin(k.e_a),
    lap -> 6 sum_a w_a (cos(k.e_a) - 1) (Eq. 40 with the B.7 wrap).  Pins weights, signs and the wrap."""
    n = 8
    o = Oracle(n, n, n, inputs.default_params())
    e, w = o.lattice()
    z, y, x = np.meshgrid(*[np.arange(n, dtype=float)] * 3, indexing="ij")
    k = 2 * np.pi / n * np.array([1.0, 2.0, 3.0])
    arg = k[0] * x + k[1] * y + k[2] * z
    G, L, _ = o.stencil_field(np.sin(arg))
    ke = e @ k
    gsym = 3 * (w * np.sin(ke)) @ e
    lsym = 6 * (w * (np.cos(ke) - 1)).sum()
    for c in range(3):
        assert np.abs(G[c] - gsym[c] * np.cos(arg)).max() < 1e-14
    assert np.abs(L - lsym * np.sin(arg)).max() < 1e-14


def test_ghost_rule_R9():
    """R9: non-periodic faces clamp the index (mirror across the halfway wall): a field depending on y only has
    zero normal gradient contribution from the ghost, i.e. G_y(0) = 3*(1/18+4/36)*(phi(1)-phi(0)) = (phi1-phi0)/2."""
    p = inputs.default_params(bc=(0, 0, 1, 1, 0, 0))
    o = Oracle(4, 6, 4, p)
    prof = np.array([0.1, 0.4, 0.2, 0.9, 0.5, 0.3])
    phi = np.broadcast_to(prof[None, :, None], (4, 6, 4)).copy()
    G, L, _ = o.stencil_field(phi)
    assert np.allclose(G[1][:, 0, :], (prof[1] - prof[0]) / 2, atol=1e-15)
    assert np.allclose(G[1][:, 5, :], (prof[5] - prof[4]) / 2, atol=1e-15)
    assert np.allclose(G[1][:, 2, :], (prof[3] - prof[1]) / 2, atol=1e-15)
    assert np.allclose(L[:, 0, :], prof[1] - prof[0], atol=1e-15)          # 6*(1/18+4/36)*(phi1-phi0)
    assert np.abs(G[0]).max() < 1e-16 and np.abs(G[2]).max() < 1e-16


def test_chemical_potential_on_tanh_P4_G4():
    """P4/G4: mu_phi (Eq. 11 with the corrected sign) vanishes on the planar equilibrium profile Eq. 5 up to the
    discretisation error of Eq. 40b; with the printed sign it would be O(beta/8).  Also kappa * int phi'^2 = sigma
    (Eq. 12), which fixes beta, kappa against sigma."""
    W, sigma = 4.0, 0.01
    p = inputs.default_params(sigma=sigma, W=W, bc=(0, 0, 0, 0, 1, 1))
    nz = 64
    o = Oracle(4, 4, nz, p)
    zc = np.arange(nz) - 31.5
    prof = 0.5 + 0.5 * np.tanh(2 * zc / W)
    phi = np.broadcast_to(prof[:, None, None], (nz, 4, 4)).copy()
    G, L, mu = o.stencil_field(phi)
    beta = 12 * sigma / W
    assert np.abs(mu).max() < 0.05 * beta            # discretisation only (measured: ~0.03 beta at W = 4)
    wrong = 4 * beta * prof * (1 - prof) * (prof - 0.5) - 1.5 * sigma * W * L[:, 0, 0]
    assert np.abs(wrong).max() > 0.15 * beta          # the printed sign is far from equilibrium
    # kappa * int phi'^2 dz = sigma on a well-resolved profile (W = 10: central differences are then within 1.5 %)
    W2 = 10.0
    o2 = Oracle(4, 4, 128, inputs.default_params(sigma=sigma, W=W2, bc=(0, 0, 0, 0, 1, 1)))
    prof2 = 0.5 + 0.5 * np.tanh(2 * (np.arange(128) - 63.5) / W2)
    G2, _, mu2 = o2.stencil_field(np.broadcast_to(prof2[:, None, None], (128, 4, 4)).copy())
    assert abs(1.5 * sigma * W2 * (G2[2][:, 0, 0] ** 2).sum() / sigma - 1) < 0.015
    assert np.abs(mu2).max() < 0.01 * (12 * sigma / W2)


def test_prosperetti_closed_form_limits():
    """The capillary-wave reference of Eq. 41-42 as restated in closed_forms.py: eta(0) = eta0; for
    nu -> 0 it tends to the inviscid standing wave cos(omega0 t); for weak damping the envelope decays at about
    2 nu k^2 (Lamb) -- fixes the two places where the printed formulas are dimensionally garbled."""
    import closed_forms as cf
    k, sigma, rh, rl = 2 * np.pi / 256, 1e-4, 1.0, 0.1
    w0 = np.sqrt(sigma * k ** 3 / (rh + rl))
    t = np.linspace(0.0, 3 * 2 * np.pi / w0, 400)
    assert abs(cf.prosperetti_capillary_wave(np.array([0.0]), 0.005, k, sigma, rh, rl)[0] - 1.0) < 1e-6
    inviscid = cf.prosperetti_capillary_wave(t, 1e-9, k, sigma, rh, rl)
    assert np.abs(inviscid - np.cos(w0 * t)).max() < 2e-3
    weak = cf.prosperetti_capillary_wave(t, 2e-4, k, sigma, rh, rl)
    peaks = [i for i in range(1, len(t) - 1) if weak[i] > weak[i - 1] and weak[i] > weak[i + 1]]
    rate = -np.log(weak[peaks[-1]] / weak[peaks[0]]) / (t[peaks[-1]] - t[peaks[0]])
    assert 0.8 * 2 * 2e-4 * k * k < rate < 2.5 * 2 * 2e-4 * k * k, (rate, 2 * 2e-4 * k * k)
