"""GPU parity on the D2Q9 lattice (clip_params.lattice = 1): libclip through the C ABI against
the D2Q9 build of the oracle, element by element on the same seeded inputs, north_star tolerances."""
import numpy as np
import pytest

from paper_2505_12205_b200 import inputs

pytestmark = pytest.mark.gpu

FP64_ABS, FP32_PHI, FP32_U = 1e-10, 1e-4, 1e-3
P_, WL, FS = inputs.PERIODIC, inputs.WALL, inputs.FREESLIP


def _with(case, **kw):
    case["params"].update(kw)
    return case


def _capwave2d():
    case = inputs.capillary_wave(L0=32, sigma=5e-3)     # Sec. 5.1 set-up at reduced size: free-slip sides, no-slip top / bottom
    case["params"]["lattice"] = 1
    return case


# The cases avoid ONE thing on purpose: a drop at rest at density ratio 1000.  The interface normal n = grad phi / |grad phi| (Eq. 34) is
# ill-conditioned on the plateau inside a drop, where phi overshoots 1 by ~1e-3 during the start-up transient; in two dimensions this
# amplifies round-off so strongly that two fp64 runs of the ORACLE whose inputs differ by 6e-8 relative are 6e-5 .. 1e-3 apart in phi
# after 100 steps (drop2d R = 16, rho* = 1000; 3-D configs[0]: 3e-9) -- DESIGN.md reading G21.  The cases below have that factor <= 2e-7.
CASES = {
    "sweep2d_periodic": (lambda: _with(inputs.sweep2d(nx=128, ny=96), rho_l=0.01), 100),       # seeded discs, rho ratio 100
    "sweep2d_walls": (lambda: _with(inputs.sweep2d(nx=67, ny=50, ndrops=4), bc=(WL,) * 4 + (P_, P_), g=(1e-5, -2e-5, 0.0), rho_l=0.05, sigma=0.002), 100),
    "sweep2d_freeslip_mixed": (lambda: _with(inputs.sweep2d(nx=40, ny=36, ndrops=3, rmin=4, rmax=6), bc=(FS, WL, FS, FS, P_, P_), rho_l=0.1), 100),
    "poiseuille2d": (lambda: inputs.poiseuille2d(nx=4, ny=32), 1000),
    "poiseuille2d_rho10_mu": (lambda: inputs.poiseuille2d(nx=4, ny=64, tau_a=5.0, tau_b=0.5, rho_a=10.0, rho_b=1.0, gx=1e-7, visc_interp=2), 500),
    "capwave2d": (_capwave2d, 200),
    "sweep2d_bgk": (lambda: _with(inputs.sweep2d(nx=64, ny=48, ndrops=3), rho_l=0.01, collision=1, tau_l=0.3), 100),
    "drop2d_rho1000_20_steps": (lambda: inputs.drop2d(n=64, R=16.0), 20),       # the resting drop itself, before the amplification sets in
}
_ref = {}


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("precision", [64, 32])
def test_parity_d2q9(name, precision):
    import torch
    from oracle.clip_oracle import Oracle
    from paper_2505_12205_b200 import clip
    mk, steps = CASES[name]
    if name not in _ref:
        case = mk()
        o = Oracle.from_case(case)
        assert o.Q == 9
        o.step(steps)
        _ref[name] = (case, o.get())
    case, (rphi, rp, ru) = _ref[name]
    sim = clip.Clip.from_case(case, precision=precision)
    sim.step(steps)
    phi, p, u = (t.double().cpu().numpy() for t in sim.get())
    torch.cuda.synchronize()
    sim.close()
    assert np.isfinite(phi).all() and np.isfinite(p).all() and np.isfinite(u).all() and np.abs(u[2]).max() == 0.0
    if precision == 64:
        e = [np.abs(a - b).max() for a, b in ((phi, rphi), (p, rp), (u, ru))]
        print(f"{name} fp64: max-abs phi {e[0]:.2e} p {e[1]:.2e} u {e[2]:.2e}")
        assert max(e) <= FP64_ABS
    else:
        ephi = np.abs(phi - rphi).max() / np.abs(rphi).max()
        eu = np.abs(u - ru).max() / max(np.abs(ru).max(), 1e-30)
        print(f"{name} fp32: field-rel phi {ephi:.2e} u {eu:.2e}")
        assert ephi <= FP32_PHI and eu <= FP32_U


@pytest.mark.parametrize("precision", [64, 32])
def test_phase_only_d2q9(precision):
    """The set-up of Sec. 5.4 (2-D, D2Q9, prescribed reversing shear flow) at reduced size: clip_set_u + clip_step
    against the D2Q9 oracle.  The GPU stores post-collision populations, so it takes u(k+1) before step k+1."""
    import torch
    from oracle.clip_oracle import Oracle
    from paper_2505_12205_b200 import clip
    n, U0, W, steps = 48, 0.04, 3.0, 150
    p = inputs.default_params(W=W, M=U0 * W / 600.0, sigma=0.0, rho_h=1.0, rho_l=1.0, phase_only=1, lattice=1, precision=precision)
    y, x = np.meshgrid(np.arange(n, dtype=float), np.arange(n, dtype=float), indexing="ij")
    phi0 = (0.5 + 0.5 * np.tanh(2.0 * (n / 5 - np.sqrt((x - 0.5 * n) ** 2 + (y - 0.3 * n) ** 2)) / W))[None]

    def vel(t):
        c = U0 * np.cos(np.pi * t / 300.0)
        return np.stack([c * np.sin(np.pi * x / n) ** 2 * np.sin(2 * np.pi * y / n), -c * np.sin(np.pi * y / n) ** 2 * np.sin(2 * np.pi * x / n),
                         np.zeros_like(x)])[:, None]
    o = Oracle(n, n, 1, p)
    o.init(phi0, vel(0))
    for k in range(steps):
        o.set_u(vel(k)); o.step(1)
    rphi = o.get()[0]
    sim = clip.Clip(n, n, 1, p)
    sim.init(torch.as_tensor(phi0), torch.as_tensor(vel(0)))
    for k in range(steps):
        sim.set_u(torch.as_tensor(vel(k + 1))); sim.step(1)
    phi, pr, u = (t.double().cpu().numpy() for t in sim.get())
    sim.close()
    err = np.abs(phi - rphi).max()
    assert np.abs(pr).max() == 0.0 and np.abs(rphi - phi0).max() > 0.2
    assert err <= (FP64_ABS if precision == 64 else FP32_PHI), err


def test_d2q9_abi():
    from paper_2505_12205_b200 import clip
    p = inputs.default_params(lattice=1)
    n2 = clip.clip_workspace_bytes(64, 64, 1, clip.make_params(p))
    n3 = clip.clip_workspace_bytes(64, 64, 1, clip.make_params(dict(p, lattice=0)))
    assert 0 < n2 < n3 and n2 >= (4 * 9 + 4) * 64 * 64 * 8
    assert clip.clip_workspace_bytes(64, 64, 2, clip.make_params(p)) == 0 and "D2Q9" in clip.clip_last_error(None)
    assert clip.clip_workspace_bytes(64, 64, 1, clip.make_params(dict(p, bc=(0, 0, 0, 0, 1, 1)))) == 0
    assert clip.clip_workspace_bytes(64, 64, 1, clip.make_params(dict(p, lattice=2))) == 0


@pytest.mark.parametrize("precision", [64, 32])
def test_d2q9_pair_kernels_match_the_scalar_kernels(precision):
    """k_phi9p + k_step9p (node pair per thread, packed arithmetic, address-selected pulls; even nx) against the thread-per-node
    k_phi9 + k_step9 (path = 1): round-off only; periodic, walls, free-slip mixed with walls, BGK, Eq. 25, a narrow lattice (nx = 2)."""
    import torch
    from paper_2505_12205_b200 import clip
    cases = [_with(inputs.sweep2d(nx=128, ny=96), rho_l=0.01),
             _with(inputs.sweep2d(nx=66, ny=50, ndrops=4), bc=(WL,) * 4 + (P_, P_), g=(1e-5, -2e-5, 0.0), rho_l=0.05, sigma=0.002),
             _with(inputs.sweep2d(nx=40, ny=36, ndrops=3, rmin=4, rmax=6), bc=(FS, WL, FS, FS, P_, P_), rho_l=0.1),
             _with(inputs.sweep2d(nx=40, ny=36, ndrops=3, rmin=4, rmax=6), bc=(WL, FS, WL, WL, P_, P_), rho_l=0.1, collision=1, tau_l=0.3),
             inputs.poiseuille2d(nx=2, ny=32, tau_a=5.0, tau_b=0.5, rho_a=10.0, rho_b=1.0, gx=1e-7, visc_interp=2)]
    tol = 1e-12 if precision == 64 else 3e-5
    for case in cases:
        outs = []
        for path in (1, 0):
            c = dict(case, params=dict(case["params"], path=path))
            sim = clip.Clip.from_case(c, precision=precision)
            sim.step(60)
            outs.append([t.double().cpu().numpy() for t in sim.get()])
            torch.cuda.synchronize()
            sim.close()
        for a, b in zip(*outs):
            assert np.isfinite(b).all()
            assert np.abs(a - b).max() <= tol * max(1.0, np.abs(a).max()), case["name"]


def test_shear_interface_table4_on_the_gpu():
    """The paper's Sec. 5.4 run itself (Table 4: L0 = 200, U0 = 0.04, M = 2e-4, xi = 3, circle of radius 40 at (100, 60),
    reversing shear flow of Eq. 48 with T = T_f, 2 T_f = 10 000 steps) ON THE PRODUCT, on the paper's lattice (D2Q9, phase_only, fp64):
    the error of Eq. 50 must reproduce the oracle's stored value (tests/golden/shear_interface.txt, written by the D3Q19 oracle with nz = 1 --
    the same run by the projection pin of test_oracle_d2q9) and total phi must be conserved.  In the normalisation with
    phi = 1 outside the circle this is 7.35e-3 against the 8.58e-3 the paper prints (weak pin)."""
    import os
    import torch
    from paper_2505_12205_b200 import clip
    gold = np.loadtxt(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "shear_interface.txt"))
    pf, err_gold, _, _, s_in, s_out = gold[0]
    assert pf == 1.0
    L0, U0, W = 200, 0.04, 3.0
    p = inputs.default_params(W=W, M=U0 * W / 600.0, sigma=0.0, rho_h=1.0, rho_l=1.0, phase_only=1, lattice=1, precision=64)
    y, x = np.meshgrid(np.arange(L0, dtype=float), np.arange(L0, dtype=float), indexing="ij")
    phi0 = 0.5 + 0.5 * np.tanh(2.0 * (L0 / 5.0 - np.sqrt((x - 0.5 * L0) ** 2 + (y - 0.3 * L0) ** 2)) / W)
    Tf = L0 / U0
    dev = torch.device("cuda:0")
    sx = torch.as_tensor(np.sin(np.pi * x / L0) ** 2 * np.sin(2 * np.pi * y / L0), device=dev)
    sy = torch.as_tensor(-np.sin(np.pi * y / L0) ** 2 * np.sin(2 * np.pi * x / L0), device=dev)
    u = torch.zeros((3, 1, L0, L0), dtype=torch.float64, device=dev)

    def vel(t):
        c = U0 * np.cos(np.pi * t / Tf)
        u[0, 0] = c * sx; u[1, 0] = c * sy
        return u
    sim = clip.Clip(L0, L0, 1, p)
    sim.init(torch.as_tensor(phi0[None]), vel(0).clone())
    n = int(round(2 * Tf))
    for k in range(n):
        sim.set_u(vel(k + 1)); sim.step(1)     # post-collision storage: the collision of step k+1 wants u(k+1)
    phi = sim.get()[0][0].cpu().numpy()
    sim.close()
    err = float(np.sqrt(((phi - phi0) ** 2).sum() / (phi0 ** 2).sum()))
    mass = float(phi.sum() / phi0.sum() - 1.0)
    print(f"shear interface on the GPU (D2Q9, 200^2, 10 000 steps): Eq. 50 error {err:.6e} (oracle {err_gold:.6e}); phi = 1 outside: {err * np.sqrt(s_in / s_out):.3e} (paper 8.58e-3); mass drift {mass:.1e}")
    assert abs(err / err_gold - 1) < 1e-6 and abs(mass) < 1e-11


@pytest.mark.parametrize("rho_ratio", [10.0, 1000.0])
def test_poiseuille_paper_cases_on_the_gpu(rho_ratio):
    """The paper's own two-phase Poiseuille cases (Sec. 5.3, Fig. 11a / 11b: 2-D, 64 nodes across, rho* = 10 and 1000,
    mu* = 100, F_b = rho g) ON THE PRODUCT (D2Q9, fp64) to steady state, against the quadrature of Eq. 45 with the smoothed rho(y), mu(y)
    of the run (the paper compares with a finite-difference solution of the same equation, :655-660).  rho* = 1000 is beyond what the
    oracle pins (rho* = 10): reported and gated at 3 %."""
    import os
    import sys
    import torch
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    import closed_forms as cf
    from paper_2505_12205_b200 import clip
    tau_b = 0.5                                        # the light fluid (Fig. 11c: tau_L = 0.5)
    tau_a = tau_b * 100.0 / rho_ratio                  # mu* = rho* tau_A / tau_B = 100
    case = inputs.poiseuille2d(nx=4, ny=64, tau_a=tau_a, tau_b=tau_b, rho_a=rho_ratio, rho_b=1.0, gx=1e-7 / rho_ratio * 10.0)
    sim = clip.Clip.from_case(case, precision=64)
    du, steps = 1.0, 0
    while steps < 600000 and du > 1e-13:
        sim.step(1999); prev = sim.get()[2].clone(); sim.step(1); steps += 2000
        du = float((sim.get()[2] - prev).abs().max())
    phi, p, u = (t.cpu().numpy() for t in sim.get())
    torch.cuda.synchronize()
    sim.close()
    pr = case["params"]
    rho_of = lambda f: pr["rho_l"] + f * (pr["rho_h"] - pr["rho_l"])                    # noqa: E731
    mu_of = lambda f: rho_of(f) * (pr["tau_l"] + f * (pr["tau_h"] - pr["tau_l"])) / 3     # noqa: E731
    ref = cf.poiseuille_quadrature(phi[0].mean(axis=1), rho_of, mu_of, pr["g"][0])
    err = cf.l2_rel(u[0, 0].mean(axis=1), ref)
    print(f"D2Q9 Poiseuille rho* = {rho_ratio:g}, mu* = 100 on the GPU: L2 (Eq. 47) = {err:.2e} after {steps} steps (du {du:.1e}), u_max {u[0].max():.2e}")
    assert np.isfinite(u).all() and du <= 1e-13 and err < 0.03


@pytest.mark.parametrize("precision", [64, 32])
def test_single_pass_d2q9_against_the_pair_kernels(precision):
    """k_fused9 + k_fix9 (path = 3: one pass over f and g, phi(t+2) scattered on chip in a ring of four rows, chunk halos through partial
    rows) against k_phi9p + k_step9p: the same arithmetic up to the association of phi's nine-term sum -> round-off only; periodic,
    walled, mixed free-slip / wall faces, BGK; the default chunking, one chunk, one row per chunk, five chunks."""
    import torch
    from paper_2505_12205_b200 import clip

    def run(case, **over):
        sim = clip.Clip(case["nx"], case["ny"], case["nz"], dict(case["params"], precision=precision, **over))
        sim.init(torch.as_tensor(case["phi0"]), torch.as_tensor(case["u0"]))
        sim.step(30)
        out = [t.double().cpu().numpy() for t in sim.get()]
        ran = {k for k, (ms, cnt) in sim.step_profiled(1).items() if cnt}
        sim.close()
        return out, ran

    cases = [_with(inputs.sweep2d(nx=128, ny=96), rho_l=0.01),
             _with(inputs.sweep2d(nx=64, ny=50, ndrops=4), bc=(WL,) * 4 + (P_, P_), rho_l=0.05, g=(1e-5, -2e-5, 0.0)),
             _with(inputs.sweep2d(nx=64, ny=36, ndrops=3, rmin=4, rmax=6), bc=(FS, WL, FS, FS, P_, P_), rho_l=0.1),
             _with(inputs.sweep2d(nx=192, ny=40, ndrops=3, rmin=4, rmax=6), bc=(WL, FS, WL, FS, P_, P_), rho_l=0.1, collision=1, tau_l=0.3),
             _with(inputs.sweep2d(nx=512, ny=24, ndrops=4, rmin=4, rmax=6), rho_l=0.1)]      # two sweeps of 256 threads per row
    tol = 1e-12 if precision == 64 else 3e-5
    for case in cases:
        ref, r0 = run(case, path=2)
        assert "k_fused" not in r0
        for over in ({}, {"tile_chunks": 1}, {"tile_chunks": case["ny"]}, {"tile_chunks": 5}):
            out, ran = run(case, path=3, **over)
            assert "k_fused" in ran and "k_fix" in ran
            for a, b in zip(ref, out):
                assert np.isfinite(b).all()
                assert np.abs(a - b).max() <= tol * max(1.0, np.abs(a).max()), (case["name"], over)
