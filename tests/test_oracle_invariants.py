"""Pins of the CPU oracle, part 2: invariants of whole time steps (SURVEY.md 8(c) P1, P2, P9, P10, P13 and the
readings R8, R11, R12, G6).  No CUDA code is touched.
"""
import numpy as np
import pytest

from oracle.clip_oracle import Oracle
from paper_2505_12205_b200 import inputs

P, Wl, IN, OUT = inputs.PERIODIC, inputs.WALL, inputs.INLET, inputs.OUTLET


def _run(case, steps):
    o = Oracle.from_case(case)
    o.step(steps)
    return o.get()


def test_uniform_rest_P1():
    """P1 (north_star): a uniform single-phase field at rest shows zero spurious change: f == 0, p == 0, u == 0
    bitwise (feq = p* w + (Gamma - w) vanishes identically, Eq. 17), phi stays within round-off of sum_a w_a."""
    for val in (1.0, 0.0):
        for bc in ((P,) * 6, (Wl,) * 6):
            p = inputs.default_params(bc=bc, g=(0.0, 0.0, 0.0))
            o = Oracle(6, 5, 7, p)
            o.init(np.full((7, 5, 6), val), np.zeros((3, 7, 5, 6)))
            o.step(300)
            phi, pr, u = o.get()
            f, g = o.populations()
            assert np.abs(f).max() == 0.0 and np.abs(pr).max() == 0.0 and np.abs(u).max() == 0.0
            assert np.abs(phi - val).max() <= 1e-13


def test_initial_state_R8():
    """R8: the barred-equilibrium initial state reproduces the inputs: sum g = phi0, sum f = p* = 0,
    sum f e + F/(2 rho) = u0 with F = F_s + F_b (Eq. 31, 38)."""
    case = inputs.walled_box()
    o = Oracle.from_case(case)
    f, g = o.populations()
    e, w = o.lattice()
    assert np.abs(g.sum(-1) - case["phi0"]).max() < 1e-15
    assert np.abs(f.sum(-1)).max() < 1e-15
    G, L, mu = o.stencil_field(case["phi0"])
    pp = case["params"]
    rho = pp["rho_l"] + case["phi0"] * (pp["rho_h"] - pp["rho_l"])
    for c in range(3):
        F = mu * G[c] + (rho - pp["rho_ref"]) * pp["g"][c]
        assert np.abs((f * e[:, c]).sum(-1) + F / (2 * rho) - case["u0"][c]).max() < 1e-15
    phi, p, u = o.get()
    assert np.array_equal(phi, case["phi0"]) and np.array_equal(u, case["u0"]) and np.abs(p).max() == 0.0


def test_phi_conservation_P2_walls_R11():
    """P2 + R11: total phi is conserved to round-off by collision (sum F^phi_a = 0), periodic streaming and halfway
    bounce-back including edge and corner links (B.10-B.11): relative drift < 1e-12 over 1000 steps."""
    case = inputs.walled_box()
    phi, p, u = _run(case, 1000)
    s0 = float(np.sum(case["phi0"], dtype=np.longdouble)); s1 = float(np.sum(phi, dtype=np.longdouble))
    assert abs(s1 - s0) / s0 < 1e-12
    assert np.isfinite(u).all()


def test_no_slip_momentum_sink_and_periodic_momentum():
    """Halfway bounce-back (B.10-B.11): with equal densities, sigma = 0 and no body force, a periodic box conserves
    total momentum sum(u) to round-off, while a walled box can only lose kinetic energy."""
    rng = np.random.default_rng(5)
    n = 10
    u0 = rng.uniform(-0.01, 0.01, size=(3, n, n, n))
    base = dict(rho_h=1.0, rho_l=1.0, sigma=0.0, tau_h=0.5, tau_l=0.5)
    o = Oracle(n, n, n, inputs.default_params(**base))
    o.init(np.ones((n, n, n)), u0); o.step(50)
    u = o.get()[2]
    assert np.abs(u.sum(axis=(1, 2, 3)) - u0.sum(axis=(1, 2, 3))).max() < 1e-14
    o = Oracle(n, n, n, inputs.default_params(bc=(Wl,) * 6, **base))
    o.init(np.ones((n, n, n)), u0)
    ke = [(u0 ** 2).sum()]
    for _ in range(5):
        o.step(10); ke.append((o.get()[2] ** 2).sum())
    assert all(b < a for a, b in zip(ke, ke[1:]))


def test_translation_invariance_P10():
    """P10: shifting a periodic input by (3, 5, 7) nodes shifts the output, bit for bit (B.5-B.7)."""
    case = inputs.sweep_drops(shape=(16, 12, 20), ndrops=3, rmin=3, rmax=5, W=3.0, precision=64)
    a = _run(case, 30)
    sh = dict(case)
    roll = lambda v: np.roll(v, (7, 5, 3), axis=(-3, -2, -1))
    sh["phi0"], sh["u0"] = roll(case["phi0"]).copy(), roll(case["u0"]).copy()
    b = _run(sh, 30)
    for x, y in zip(a, b):
        assert np.array_equal(roll(x), y)


def test_lattice_symmetry_P9():
    """P9: D3Q19 is invariant under axis permutations and mirrors (Eq. 14-15): permuted / mirrored inputs give the
    permuted / mirrored fields (round-off only: the summation order over a changes)."""
    case = inputs.sweep_drops(shape=(16, 12, 20), ndrops=3, rmin=3, rmax=5, W=3.0, precision=64)
    case["params"]["g"] = (1e-5, -2e-5, 3e-5); case["params"]["rho_ref"] = 0.3
    phi, p, u = _run(case, 40)
    # cyclic permutation: new (x, y, z) = old (y, z, x): arrays [z,y,x] -> transpose so that new z = old x ...
    perm = dict(case)
    perm["nx"], perm["ny"], perm["nz"] = case["ny"], case["nz"], case["nx"]
    tr = lambda v: np.ascontiguousarray(np.transpose(v, (2, 0, 1)))   # [z,y,x] -> [x,z,y] = new [z',y',x']
    perm["phi0"] = tr(case["phi0"])
    perm["u0"] = np.stack([tr(case["u0"][1]), tr(case["u0"][2]), tr(case["u0"][0])])
    perm["params"] = dict(case["params"]); g = case["params"]["g"]; perm["params"]["g"] = (g[1], g[2], g[0])
    phi2, p2, u2 = _run(perm, 40)
    assert np.abs(phi2 - tr(phi)).max() < 1e-13 and np.abs(p2 - tr(p)).max() < 1e-13
    assert np.abs(u2 - np.stack([tr(u[1]), tr(u[2]), tr(u[0])])).max() < 1e-13
    # mirror in x
    mir = dict(case)
    fl = lambda v: np.ascontiguousarray(v[..., ::-1])
    mir["phi0"] = fl(case["phi0"])
    mir["u0"] = np.stack([-fl(case["u0"][0]), fl(case["u0"][1]), fl(case["u0"][2])])
    mir["params"] = dict(case["params"]); mir["params"]["g"] = (-g[0], g[1], g[2])
    phi3, p3, u3 = _run(mir, 40)
    assert np.abs(phi3 - fl(phi)).max() < 1e-13 and np.abs(p3 - fl(p)).max() < 1e-13
    assert np.abs(u3 - np.stack([-fl(u[0]), fl(u[1]), fl(u[2])])).max() < 1e-13


def _mirror_extend(v, axes, sign_axis=None):
    """Even (or, for the vector component normal to the mirror, odd) extension of v[z, y, x] across the halfway planes
    of the given axes: index n + k <- n - 1 - k."""
    for ax in axes:
        m = np.flip(v, axis=ax)
        if sign_axis is not None and ax == sign_axis:
            m = -m
        v = np.concatenate([v, m], axis=ax)
    return v


@pytest.mark.parametrize("faces", ["y", "xyz"])
def test_free_slip_is_a_mirror_plane(faces):
    """SURVEY 8(f) NEXT-3, free-slip faces (B.8-B.9): specular reflection half a cell outside the
    last node makes the face a symmetry plane, so a box with free-slip faces must evolve exactly like one octant of
    the mirror-extended PERIODIC box (phi, p, tangential u even; normal u odd) -- a run that never enters the
    free-slip branch.  'y': free-slip on the two y faces, x / z periodic; 'xyz': all six faces (edges and corners
    reflect two / three components).  Round-off only (the order of the sums over a changes)."""
    nx, ny, nz = 10, 8, 6
    case = inputs.sweep_drops(shape=(nx, ny, nz), ndrops=2, rmin=2.5, rmax=3.5, W=3.0, precision=64, u_amp=0.01)
    FS, PE = inputs.FREESLIP, inputs.PERIODIC
    axes = {"y": (1,), "xyz": (0, 1, 2)}[faces]              # numpy axes of [z, y, x] arrays
    case["params"]["bc"] = tuple(FS if (2 - d) in axes else PE for d in (0, 0, 1, 1, 2, 2))
    case["params"]["g"] = (2e-5, 0.0, 0.0) if faces == "y" else (0.0, 0.0, 0.0)   # gravity only along a tangential, unmirrored axis
    phi, p, u = _run(case, 40)
    big = dict(case)
    big["params"] = dict(case["params"]); big["params"]["bc"] = (PE,) * 6
    big["phi0"] = _mirror_extend(case["phi0"], axes)
    big["u0"] = np.stack([_mirror_extend(case["u0"][c], axes, sign_axis=2 - c) for c in range(3)])
    big["nz"], big["ny"], big["nx"] = big["phi0"].shape
    phi2, p2, u2 = _run(big, 40)
    sub = (slice(0, nz), slice(0, ny), slice(0, nx))
    assert np.abs(phi2[sub] - phi).max() < 1e-13 and np.abs(p2[sub] - p).max() < 1e-13
    assert np.abs(u2[(slice(None),) + sub] - u).max() < 1e-13
    assert np.abs(phi - case["phi0"]).max() > 1e-3          # the run did something
    # the normal velocity at the node next to the face stays small but the tangential one is free
    assert np.abs(u).max() > 1e-3


def test_free_slip_keeps_tangential_momentum():
    """Free-slip y faces exert no tangential stress: with x / z periodic and no body force the total x- and z-momentum
    sum rho u stays constant, whereas the same box with halfway bounce-back (B.10) loses it."""
    FS, PE, WA = inputs.FREESLIP, inputs.PERIODIC, inputs.WALL
    out = {}
    for name, wall in (("slip", FS), ("noslip", WA)):
        case = inputs.sweep_drops(shape=(8, 10, 6), ndrops=1, rmin=2.5, rmax=3.0, W=3.0, precision=64, u_amp=0.0)
        case["params"].update(bc=(PE, PE, wall, wall, PE, PE), rho_h=1.0, rho_l=1.0, sigma=0.0)
        case["u0"][0] += 0.02
        case["u0"][2] -= 0.01
        phi, p, u = _run(case, 60)
        out[name] = (u[0].sum(), u[2].sum())
        m0 = (0.02 * 480, -0.01 * 480)
        if name == "slip":
            assert abs(out[name][0] - m0[0]) < 1e-12 and abs(out[name][1] - m0[1]) < 1e-12
        else:
            assert out[name][0] < 0.95 * m0[0]


def test_inlet_invariants_P13_G6():
    """P13: after the velocity-inlet rule (B.12-B.20 as read in G6) a node satisfies the two conditions the paper
    says it must: sum_a f_a e_a = u_in (B.12; F = 0 at the inlet, :1088) and sum_a g_a = phi_in
    (B.16), for arbitrary incoming populations; known populations are untouched."""
    uin, phin = (0.003, -0.002, 0.05), 0.9
    p = inputs.default_params(bc=(Wl, Wl, Wl, Wl, IN, OUT), inlet_u=uin, inlet_phi=phin, inlet_c=(2.0, 2.0), inlet_r=1.5)
    o = Oracle(5, 5, 6, p)
    e, w = o.lattice()
    rng = np.random.default_rng(11)
    for _ in range(5):
        f = rng.normal(size=19) * 0.01
        g = w * phin + rng.normal(size=19) * 0.01
        f2, g2 = o.inlet_node(f, g)
        assert np.abs(f2 @ e - np.array(uin)).max() < 1e-15
        assert abs(g2.sum() - phin) < 1e-15
        known = e[:, 2] <= 0
        assert np.array_equal(f2[known], f[known]) and np.array_equal(g2[known], g[known])


def _jet_case():
    return inputs.jet(nxy=10, nz=14, r_nozzle=2.6)


def test_inlet_nodes_in_a_run():
    """Step 8 + step 10 on a running case: on disc nodes phi == phi_in, u == u_in and the populations satisfy
    B.12 / B.16; plate nodes outside the disc behave as no-slip wall nodes (populations bounce back)."""
    case = _jet_case()
    o = Oracle.from_case(case)
    o.step(25)
    phi, p, u = o.get()
    f, g = o.populations()
    e, w = o.lattice()
    pp = case["params"]
    yy, xx = np.meshgrid(np.arange(case["ny"]), np.arange(case["nx"]), indexing="ij")
    disc = (xx - pp["inlet_c"][0]) ** 2 + (yy - pp["inlet_c"][1]) ** 2 <= pp["inlet_r"] ** 2
    assert disc.sum() >= 9
    assert np.all(phi[0][disc] == pp["inlet_phi"])
    for c in range(3):
        assert np.all(u[c, 0][disc] == pp["inlet_u"][c])
        assert np.abs((f[0] * e[:, c]).sum(-1)[disc] - pp["inlet_u"][c]).max() < 1e-15
    assert np.abs(g[0].sum(-1)[disc] - pp["inlet_phi"]).max() < 1e-15


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_outlet_recurrence_R12(mode):
    """B.26-B.27: chi(N,t+1) (1 + lam) - chi(N,t) = lam chi(N-1,t+1) for all 38 populations,
    with lam = max(0, U) and U one of the three schemes of B.22 evaluated on u_z(N-1, t) (reading R12):
    0 = U_local (per column), 1 = U_ave (mean over the layer), 2 = U_max."""
    case = _jet_case()
    case["params"]["outlet_u_mode"] = mode
    rng = np.random.default_rng(5)
    case["u0"][2] += 0.02 + 0.015 * rng.uniform(-1.0, 1.0, size=case["u0"][2].shape)   # outflow that varies over the layer
    o = Oracle.from_case(case)
    o.step(2)
    for _ in range(3):
        f0, g0 = o.populations()
        uz = o.get()[2][2]
        o.step(1)
        f1, g1 = o.populations()
        U = uz[-2] if mode == 0 else (np.full_like(uz[-2], uz[-2].mean()) if mode == 1 else np.full_like(uz[-2], uz[-2].max()))
        lam = np.maximum(U, 0.0)[..., None]
        for a0, a1 in ((f0, f1), (g0, g1)):
            assert np.abs(a1[-1] * (1 + lam) - a0[-1] - lam * a1[-2]).max() < 1e-15
    assert np.isfinite(f1).all() and np.isfinite(g1).all()
    assert uz[-2].max() > 1.2 * uz[-2].mean() > 0 and np.ptp(uz[-2]) > 0.3 * uz[-2].mean()   # the three schemes really differ here


def test_phase_only_mode():
    """Prescribed-velocity mode (PAPER.md:675-713 set-up, small): f stays 0, p = 0, u is returned as prescribed, total
    phi is conserved to round-off, and the reversed flow brings the interface back (Eq. 50 error small)."""
    import sys, os
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    import oracle_jobs
    r = oracle_jobs.shear_interface(L0=40)
    assert abs(r["mass"]) < 1e-12
    assert r["err"] < 0.1 and r["stretch"] > 0.5     # strongly deformed at t = T_f, restored at 2 T_f
