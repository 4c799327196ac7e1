"""Pins of the oracle's convective outlet (App. B.5; SURVEY.md:454-455; reading R12).

What the paper and the mathematics fix, independent of the oracle's code:
  * B.25 with a constant lambda is the implicit first-order upwind scheme of B.21: driven by the values of layer N-1 it has the
    closed-form response chi_N(n) = chi_N(0) (1+lam)^-n + sum_k lam (1+lam)^-(n-k+1) chi_{N-1}(k).  A phase-field pulse carried by a
    uniform velocity U is a travelling wave phi0(z - U t) of Eq. 8 (the tanh kernel of Eq. 5 is its equilibrium profile), so the
    response of the outlet layer can be written down without running anything.
  * chi(N, t) in B.26-B.27 is the value the layer held at time t (pre-collision); a disturbance of layer N that layer N-1 never
    sees therefore changes by exactly 1/(1+lam) per step: decay for outflow, GROWTH for lam < 0 (backflow) -- which is why
    `outlet_clamp = 1` exists -- and no change at all with the clamp.
  * B.22's three schemes and the two time levels of U the text mentions (PAPER.md:1107 vs :1117) are both implemented; the black-box
    recurrence on the returned fields tells them apart.
"""
import numpy as np
import pytest

from oracle.clip_oracle import Oracle
from paper_2505_12205_b200 import inputs

P, W_, I_, O_ = inputs.PERIODIC, inputs.WALL, inputs.INLET, inputs.OUTLET


def _upwind_response(chi0, driver, lam):
    """chi_N(n), n = 0..len(driver): closed form of B.25 with constant lam; driver[k-1] = chi_{N-1}(k)."""
    out = [chi0]
    for n in range(1, len(driver) + 1):
        k = np.arange(1, n + 1)
        out.append(chi0 * (1 + lam) ** (-n) + float(np.sum(lam * (1 + lam) ** (-(n - k + 1.0)) * driver[:n])))
    return np.array(out)


def test_advected_pulse_leaves_through_the_outlet_as_first_order_upwind():
    """SURVEY.md:454-455.  Thin z column, phase-field equation alone (phase_only), uniform prescribed u = (0, 0, U): a slab of
    phi = 1 with two tanh faces of width W travels to +z and leaves through the convective outlet.  phi(N, t) must follow the
    closed-form upwind response driven by the ANALYTIC travelling profile at layer N-1 (tolerance: the lattice's own advection
    error of a W = 4 interface), and -- to round-off, on the returned fields only -- the one driven by phi(N-1, t)."""
    nz, U, W = 96, 0.05, 4.0
    p = inputs.default_params(W=W, M=0.02, sigma=0.0, rho_h=1.0, rho_l=1.0, phase_only=1, bc=(P, P, P, P, W_, O_))
    z = np.arange(nz, dtype=float)
    z1, z2 = 50.0, 74.0
    prof = lambda s: 0.5 * (np.tanh(2 * (s - z1) / W) - np.tanh(2 * (s - z2) / W))   # noqa: E731
    phi0 = np.broadcast_to(prof(z)[:, None, None], (nz, 2, 2)).copy()
    u = np.zeros((3, nz, 2, 2)); u[2] = U
    o = Oracle(2, 2, nz, p)
    o.init(phi0, u)
    steps = 1200                                   # the trailing face (z1 = 50) reaches z = N after 45 / U = 900 steps
    hist = [o.get()[0][:, 0, 0].copy()]
    for _ in range(steps):
        o.set_u(u); o.step(1)
        hist.append(o.get()[0][:, 0, 0].copy())
    hist = np.array(hist)
    N = nz - 1
    # (i) exact, black box: phi_N(t+1) (1 + lam) = phi_N(t) + lam phi_{N-1}(t+1) with lam = U (B.25 summed over a, Eq. 38)
    res = hist[1:, N] * (1 + U) - hist[:-1, N] - U * hist[1:, N - 1]
    assert np.abs(res).max() < 1e-15
    own = _upwind_response(hist[0, N], hist[1:, N - 1], U)
    assert np.abs(own - hist[:, N]).max() < 1e-13
    # (ii) the pin: driver = the travelling wave phi0(z - U t) evaluated at z = N-1, nothing taken from the oracle
    t = np.arange(1, steps + 1)
    ana = _upwind_response(prof(float(N)), prof(N - 1 - U * t), U)
    err = np.abs(ana - hist[:, N]).max()
    peak = hist[:, N].max()
    print(f"outlet pulse: max |phi_N - upwind(analytic driver)| = {err:.2e}, peak {peak:.3f}, residual phi at the end {hist[-1, N]:.1e}")
    assert peak > 0.95                             # the slab really went through the outlet layer
    assert err < 3e-2                              # measured 1.6e-2: the lattice's own advection error of the W = 4 faces (900 steps)
    assert abs(hist[-1, N]) < 1e-3 and np.abs(hist[-1, 40:]).max() < 1e-3   # ... and left: no reflection back into the column
    # a wrong lambda (2 U, or U of the wrong sign) is far outside the tolerance
    for bad in (2 * U, 0.5 * U):
        assert np.abs(_upwind_response(prof(float(N)), prof(N - 1 - U * t), bad) - hist[:, N]).max() > 5 * err


@pytest.mark.parametrize("U,clamp,factor", [(0.02, 0, 1 / 1.02), (-0.02, 0, 1 / 0.98), (-0.02, 1, 1.0), (0.02, 1, 1 / 1.02)])
def test_outlet_layer_disturbance_changes_by_one_over_one_plus_lambda(U, clamp, factor):
    """A disturbance of the outlet layer's populations that leaves phi(N) and the populations layer N-1 pulls (e_z = -1)
    untouched -- + d on direction (0,0,1), - d/4 on the four (+-1,0,1), (0,+-1,1) diagonals, uniform phi = 1, prescribed uniform u --
    is invisible to the rest of the lattice, so B.27 alone acts on it: factor 1/(1 + lambda) per step.  lambda < 0 (backflow)
    GROWS without the clamp (the instability DESIGN.md R12 records) and is frozen with it.  Also pins that chi(N, t) of B.25 is the
    PRE-collision value of the layer (a post-collision value would bring in a factor 1 - omega_phi)."""
    nz = 40
    p = inputs.default_params(W=4.0, M=0.1, sigma=0.0, rho_h=1.0, rho_l=1.0, phase_only=1, bc=(P, P, P, P, W_, O_), outlet_clamp=clamp)
    o = Oracle(2, 2, nz, p)
    u = np.zeros((3, nz, 2, 2)); u[2] = U
    o.init(np.ones((nz, 2, 2)), u)
    e, w = o.lattice()
    f, g = o.populations()
    d = 1e-3
    pert = np.where(e[:, 2] == 1, np.where((e[:, 0] == 0) & (e[:, 1] == 0), d, -d / 4), 0.0)
    assert abs(pert.sum()) < 1e-18 and np.count_nonzero(pert) == 5
    base = g[-1].copy()
    g[-1] += pert
    o.set_populations(f, g)
    n = 15                                           # the wall's own transient at z = 0 travels one layer per step: far away
    for _ in range(n):
        o.set_u(u); o.step(1)
    g1 = o.populations()[1]
    got = g1[-1] - base
    assert np.abs(got - pert * factor ** n).max() < 1e-15
    assert np.abs(g1[-2] - base).max() < 1e-15       # layer N-1 never noticed
    if U < 0 and not clamp:
        assert factor ** n > 1.3                     # growth


@pytest.mark.parametrize("when", [0, 1])
@pytest.mark.parametrize("clamp", [0, 1])
def test_recurrence_tells_the_two_time_levels_of_U_apart(when, clamp):
    """Full two-phase run (jet replica with in- AND outflow over the outlet layer).  On the returned fields:
    chi(N,t+1) (1 + lam) - chi(N,t) - lam chi(N-1,t+1) = 0 holds for lam built from u_z(N-1, t) with outlet_u_time = 0
    ("from the previous time step") and from sum_a e_az f_a(N-1, t+1) with outlet_u_time = 1 (PAPER.md:1117
    "U(t + dt) ... after the streaming step in the (N-1)th layer") -- and NOT the other way round; with and without the clamp."""
    case = inputs.jet(nxy=12, nz=16, r_nozzle=3.0)
    case["params"].update(outlet_clamp=clamp, outlet_u_time=when)
    rng = np.random.default_rng(11)
    case["u0"][2] += 0.01 + 0.03 * rng.uniform(-1.0, 1.0, size=case["u0"][2].shape)   # outflow and backflow over the layer
    o = Oracle.from_case(case)
    e, _ = o.lattice()
    o.step(2)
    seen_back = False
    for _ in range(3):
        f0, g0 = o.populations()
        uz_t = o.get()[2][2][-2]
        o.step(1)
        f1, g1 = o.populations()
        U = {0: uz_t, 1: f1[-2] @ e[:, 2]}
        seen_back = seen_back or bool((U[when] < 0).any())
        for k in (0, 1):
            lam = (np.maximum(U[k], 0.0) if clamp else U[k])[..., None]
            res = max(np.abs(a1[-1] * (1 + lam) - a0[-1] - lam * a1[-2]).max() for a0, a1 in ((f0, f1), (g0, g1)))
            if k == when:
                assert res < 1e-15
            else:
                assert res > 1e-7
    assert seen_back


def _sens_run(kw):
    """One oracle run of the jet replica with parameter overrides (top level: runs in a process pool)."""
    case = inputs.jet(nxy=24, nz=48, r_nozzle=4.0)
    case["params"].update(kw)
    o = Oracle.from_case(case)
    o.step(200)
    phi, p, u = o.get()
    return phi, u / case["params"]["inlet_u"][2]


def test_sensitivity_of_the_unpinned_readings_on_the_jet_replica():
    """What the readings the paper cannot pin are worth (recorded in DESIGN.md, readings R9, R12, R13): jet replica 24 x 24 x 48,
    nozzle radius 4, 200 steps; max |d phi| and max |d u| / U_in against the default readings for
      (a) R9 at the open faces: linear extrapolation of phi through the inlet disc / outlet instead of the clamp (oracle only);
      (b) R12: U of B.22 from the post-stream moment at t + dt instead of the stored u(t);
      (c) R12: B.25 as printed (no clamp) instead of lambda = max(0, U);
      (d) R13: F_mu of the macro update re-evaluated once with the new u instead of the lagged one alone (oracle only).
    Not a pin: the differences are reported and only bounded loosely (each reading changes the fields near the face it acts on)."""
    from concurrent.futures import ProcessPoolExecutor
    variants = (("R9 open faces: linear extrapolation", dict(open_ghost=1)),
                ("R12: U(t+dt) from the post-stream moment", dict(outlet_u_time=1)),
                ("R12: B.25 without the clamp", dict(outlet_clamp=0)),
                ("R13: one refinement of u in the macro update", dict(macro_u_refine=1)))
    with ProcessPoolExecutor(max_workers=5) as ex:
        runs = list(ex.map(_sens_run, [dict()] + [kw for _, kw in variants]))
    base = runs[0]
    out = {}
    for (name, kw), (phi, u) in zip(variants, runs[1:]):
        dphi, du = np.abs(phi - base[0]), np.abs(u - base[1]).max(axis=0)
        zphi, zu = np.unravel_index(dphi.argmax(), dphi.shape)[0], np.unravel_index(du.argmax(), du.shape)[0]
        out[name] = (dphi.max(), du.max())
        print(f"{name}: max |d phi| = {dphi.max():.2e} (plane z = {zphi}), max |d u| / U_in = {du.max():.2e} (plane z = {zu})")
        assert np.isfinite(phi).all() and np.isfinite(u).all()
        assert dphi.max() < 0.1 and du.max() < 0.1
    assert all(v[0] > 0 or v[1] > 0 for v in out.values())   # every switch really changes the computation
