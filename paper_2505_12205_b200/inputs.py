"""Seeded synthetic inputs for the CLIP hot path (shared by the oracle tests, the GPU tests and bench.py).

This module holds *no* arithmetic of the method: it only builds initial fields phi0 / u0 and parameter
dictionaries.  Recipes are the ones stated in DESIGN.md ("Input recipe") and SURVEY.md section 8(d); the initial
interface profile is the paper's equilibrium kernel, PAPER.md:118 (Eq. 5), and the Rayleigh-Taylor perturbation
is PAPER.md:729 (Eq. 53) as restated by BASELINE.json configs[2].

Layout everywhere: phi0[z, y, x] (x fastest), u0[c, z, y, x].  Node j sits at coordinate j (cell index); walls
(halfway bounce-back) sit half a cell outside the first / last node.

Parameter dictionary keys (both the oracle binding and the CUDA binding marshal these into their own structs):
  precision (32|64), rho_h, rho_l, tau_h, tau_l, sigma, W, M, g (3), rho_ref, bc (6: -x,+x,-y,+y,-z,+z),
  inlet_u (3), inlet_phi, inlet_c (2), inlet_r, outlet_u_mode, visc_interp, collision (0 WMRT, 1 BGK), phase_only (1: prescribed u),
  outlet_clamp (0: lambda of B.25 as printed; 1: max(0, lambda)), outlet_u_time (0: stored u(t); 1: post-stream moment at t+dt),
  lattice (0: D3Q19, 1: D2Q9)
"""
from __future__ import annotations

import numpy as np

PERIODIC, WALL, INLET, OUTLET, FREESLIP = 0, 1, 2, 3, 4


def default_params(**kw) -> dict:
    p = dict(
        precision=64,
        rho_h=1.0, rho_l=1.0e-3,
        tau_h=0.8, tau_l=0.8,
        sigma=0.01, W=4.0, M=0.1,
        g=(0.0, 0.0, 0.0), rho_ref=0.0,
        bc=(PERIODIC,) * 6,
        inlet_u=(0.0, 0.0, 0.0), inlet_phi=1.0,
        inlet_c=(0.0, 0.0), inlet_r=0.0,
        outlet_u_mode=0, visc_interp=0, collision=0, phase_only=0,
        outlet_clamp=0, outlet_u_time=0,
        lattice=0,  # 0 = D3Q19; 1 = D2Q9 (nz = 1, z faces PERIODIC): the lattice of the paper's 2-D benchmarks
        path=0, tile_ty=0, tile_chunks=0, runtime_nx=0, cluster_y=0,  # libclip only: kernel path / tiling (include/clip.h); the oracle ignores them
    )
    p.update(kw)
    return p


def _grid(nx, ny, nz):
    z, y, x = np.meshgrid(np.arange(nz, dtype=np.float64), np.arange(ny, dtype=np.float64),
                          np.arange(nx, dtype=np.float64), indexing="ij")
    return x, y, z


def _case(nx, ny, nz, params, phi0, u0, name):
    return dict(name=name, nx=int(nx), ny=int(ny), nz=int(nz), params=params,
                phi0=np.ascontiguousarray(phi0, dtype=np.float64),
                u0=np.ascontiguousarray(u0, dtype=np.float64))


def drop(n=32, R=8.0, W=4.0, sigma=0.01, rho_ratio=1000.0, tau=0.8, M=0.1, precision=64):
    """BASELINE.json configs[0]: stationary drop in a periodic cube, centred at ((n-1)/2,)*3, u0 = 0."""
    x, y, z = _grid(n, n, n)
    c = 0.5 * (n - 1)
    r = np.sqrt((x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2)
    phi0 = 0.5 + 0.5 * np.tanh(2.0 * (R - r) / W)
    u0 = np.zeros((3, n, n, n))
    p = default_params(precision=precision, rho_h=1.0, rho_l=1.0 / rho_ratio, tau_h=tau, tau_l=tau,
                       sigma=sigma, W=W, M=M)
    return _case(n, n, n, p, phi0, u0, f"drop{n}")


def poiseuille(nx=4, ny=128, nz=4, tau_a=1.0, tau_b=0.1, rho_a=1.0, rho_b=1.0, gx=1.0e-6, W=4.0, M=0.1,
               visc_interp=0, precision=64):
    """BASELINE.json configs[1]: layered two-phase Poiseuille; fluid A (phi=1) below y = ny/2, walls in y."""
    x, y, z = _grid(nx, ny, nz)
    yc = y + 0.5
    phi0 = 0.5 - 0.5 * np.tanh(2.0 * (yc - 0.5 * ny) / W)
    u0 = np.zeros((3, nz, ny, nx))
    p = default_params(precision=precision, rho_h=rho_a, rho_l=rho_b, tau_h=tau_a, tau_l=tau_b, sigma=0.0,
                       W=W, M=M, g=(gx, 0.0, 0.0), rho_ref=0.0,
                       bc=(PERIODIC, PERIODIC, WALL, WALL, PERIODIC, PERIODIC), visc_interp=visc_interp)
    return _case(nx, ny, nz, p, phi0, u0, f"poiseuille{nx}x{ny}x{nz}")


def rayleigh_taylor(L=128, W=5.0, precision=32):
    """BASELINE.json configs[2] at scale L (L=128 is the named lattice L x 4L x L; L=16 the parity replica).

    At = 0.5 (rho_h=3, rho_l=1); U0 = sqrt(g L) = 0.04; Re = 3000; mu ratio 1; Pe = 1000; Ca = 0.26
    (Table 5; Eq. 54-57).  Heavy fluid on top, gravity along -y, walls in y.
    """
    nx, ny, nz = L, 4 * L, L
    x, y, z = _grid(nx, ny, nz)
    y0 = 2.0 * L + 0.05 * L * (np.cos(2 * np.pi * x / L) + np.cos(2 * np.pi * z / L))
    phi0 = 0.5 + 0.5 * np.tanh(2.0 * (y - y0) / W)
    u0 = np.zeros((3, nz, ny, nx))
    U0 = 0.04
    gy = U0 * U0 / L
    rho_h, rho_l = 3.0, 1.0
    nu_h = U0 * L / 3000.0
    tau_h = 3.0 * nu_h
    tau_l = tau_h * rho_h / rho_l          # equal dynamic viscosity
    Mob = U0 * L / 1000.0
    sigma = rho_h * nu_h * U0 / 0.26
    p = default_params(precision=precision, rho_h=rho_h, rho_l=rho_l, tau_h=tau_h, tau_l=tau_l, sigma=sigma,
                       W=W, M=Mob, g=(0.0, -gy, 0.0), rho_ref=0.5 * (rho_h + rho_l),
                       bc=(PERIODIC, PERIODIC, WALL, WALL, PERIODIC, PERIODIC))
    return _case(nx, ny, nz, p, phi0, u0, f"rt{L}")


def jet(nxy=192, nz=1536, r_nozzle=12.0, We=2.2, W=4.0, U=0.05, precision=32):
    """BASELINE.json configs[3] (nxy=192, nz=1536, r=12) or its parity replica (24, 96, 4).

    -z face: INLET disc (plug inflow U along +z, phi_in = 1; wall outside the disc); +z face: convective OUTLET;
    x and y faces: no-slip walls.  Re = 200, mu ratio 100, rho ratio 1000 (Table 6).
    """
    nx = ny = nxy
    x, y, z = _grid(nx, ny, nz)
    c = 0.5 * (nxy - 1)
    rxy = np.sqrt((x - c) ** 2 + (y - c) ** 2)
    d = np.minimum(r_nozzle - rxy, r_nozzle - z)
    phi0 = 0.5 + 0.5 * np.tanh(2.0 * d / W)
    u0 = np.zeros((3, nz, ny, nx))
    D = 2.0 * r_nozzle
    rho_h, rho_l = 1.0, 1.0e-3
    nu_h = U * D / 200.0
    nu_l = nu_h * (rho_h / rho_l) / 100.0
    sigma = rho_h * U * U * D / We
    p = default_params(precision=precision, rho_h=rho_h, rho_l=rho_l, tau_h=3 * nu_h, tau_l=3 * nu_l,
                       sigma=sigma, W=W, M=0.1,
                       bc=(WALL, WALL, WALL, WALL, INLET, OUTLET),
                       inlet_u=(0.0, 0.0, U), inlet_phi=1.0, inlet_c=(c, c), inlet_r=r_nozzle,
                       outlet_clamp=1)   # quiescent gas at the outlet: u_z < 0 occurs, B.25 as printed then amplifies (R12)
    return _case(nx, ny, nz, p, phi0, u0, f"jet{nxy}x{nz}")


# Table 6: Re, We, Fr of the paper's twelve jet cases; rho* = 814, mu* = 55, Oh = sqrt(We) / Re = 4.4e-3
JET_TABLE6 = {"a": (151, 0.44, 2.60), "b": (211, 0.88, 3.65), "c": (228, 1.03, 3.94), "d": (302, 1.79, 5.22), "e": (332, 2.17, 5.74),
              "f": (340, 2.27, 5.87), "g": (347, 2.37, 6.01), "h": (362, 2.58, 6.26), "i": (397, 3.10, 6.86), "j": (408, 3.27, 7.05),
              "k": (423, 3.52, 7.31), "l": (454, 4.05, 7.84)}


def jet_paper(case="l", D=32, W=4.0, precision=32, nz=None, M=0.1, U=0.05):
    """The paper's own jet set-up (Sec. 6.1, Fig. 18; Eq. 58-59; Table 6): domain 6 D x 6 D x 20 D, circular inlet of
    diameter D with uniform velocity u_j = 0.05 and rho_j = 1 (:849), FREE-SLIP side walls, convective outlet, gravity along the jet
    with F_g = (rho - rho_L) g (Eq. 58: rho_ref = rho_l), rho* = 814, mu* = 55, and (Re, We, Fr) of the named row of Table 6
    (Eq. 59: sigma = rho_j u_j^2 D / We, nu_j = u_j D / Re, g = u_j^2 / (Fr^2 D)).  The jet runs along +z here (the paper's y).
    D = 32 gives 192 x 192 x 640; D = 4 the parity replica 24 x 24 x 80.  The paper states neither the interface width nor the mobility of
    these runs: W and M are free here; U = u_j is the paper's 0.05 unless a run needs a smaller lattice velocity (same Re, We, Fr)."""
    Re, We, Fr = JET_TABLE6[case]
    nxy, nz = 6 * D, (20 * D if nz is None else nz)
    x, y, z = _grid(nxy, nxy, nz)
    c = 0.5 * (nxy - 1)
    r_n = 0.5 * D
    rxy = np.sqrt((x - c) ** 2 + (y - c) ** 2)
    phi0 = 0.5 + 0.5 * np.tanh(2.0 * np.minimum(r_n - rxy, r_n - z) / W)          # a liquid stub in front of the nozzle
    u0 = np.zeros((3, nz, nxy, nxy))
    rho_h, rho_l = 1.0, 1.0 / 814.0
    nu_h = U * D / Re
    nu_l = nu_h * 814.0 / 55.0                                                    # mu* = 55
    p = default_params(precision=precision, rho_h=rho_h, rho_l=rho_l, tau_h=3 * nu_h, tau_l=3 * nu_l, sigma=rho_h * U * U * D / We, W=W, M=M,
                       g=(0.0, 0.0, U * U / (Fr * Fr * D)), rho_ref=rho_l,
                       bc=(FREESLIP,) * 4 + (INLET, OUTLET), inlet_u=(0.0, 0.0, U), inlet_phi=1.0, inlet_c=(c, c), inlet_r=r_n, outlet_clamp=1)
    return _case(nxy, nxy, nz, p, phi0, u0, f"jet_paper_{case}_D{D}")


def capillary_wave(L0=256, nu=0.005, sigma=1.0e-4, W=4.0, M=0.02, rho_h=1.0, rho_l=0.1, eta0_rel=0.02, precision=64):
    """PAPER.md Sec. 5.1 (:559-595, Fig. 7): L0 x 2 L0 (x 1) box, free-slip faces in x, no-slip walls in y; heavy fluid
    below the interface y = L0 + eta0 cos(2 pi x / L0), eta0 = 0.02 L0; equal kinematic viscosity nu in both fluids;
    sigma = 1e-4, xi = 4, M = 0.02 as printed.  The paper does not print the densities: rho_h / rho_l = 10 here.
    Quasi-2D: nz = 1, periodic in z (D3Q19 with no z dependence)."""
    nx, ny, nz = L0, 2 * L0, 1
    x, y, z = _grid(nx, ny, nz)
    yi = L0 + eta0_rel * L0 * np.cos(2 * np.pi * (x + 0.5) / L0)      # nodes at j + 1/2, faces at 0 and n
    phi0 = 0.5 - 0.5 * np.tanh(2.0 * (y + 0.5 - yi) / W)
    u0 = np.zeros((3, nz, ny, nx))
    p = default_params(precision=precision, rho_h=rho_h, rho_l=rho_l, tau_h=3.0 * nu, tau_l=3.0 * nu, sigma=sigma, W=W, M=M,
                       bc=(FREESLIP, FREESLIP, WALL, WALL, PERIODIC, PERIODIC))
    return _case(nx, ny, nz, p, phi0, u0, f"capwave{L0}")


def sweep_drops(n=64, seed=2505, ndrops=20, rmin=6.0, rmax=20.0, W=4.0, u_amp=0.01, precision=32,
                shape=None, z_planes=None):
    """BASELINE.json configs[4]: periodic box with `ndrops` seeded spherical drops and i.i.d. uniform u0.

    phi0 = max_k [0.5 + 0.5 tanh(2 (R_k - d_k)/W)] with d_k the periodic minimum-image distance.
    `shape=(nx,ny,nz)` gives a non-cubic box (used by the odd-size parity case).
    `z_planes` (list of global z indices; the z-slab bench of a lattice too large to build whole on every rank) returns only those
    planes of phi0 / u0 (nz of the case stays the global one); u0 is then drawn plane by plane from PCG64([seed, z]) -- a different
    but equally seeded field, the same on whichever rank asks for the plane.
    """
    nx, ny, nz = (n, n, n) if shape is None else shape
    rng = np.random.Generator(np.random.PCG64(seed))
    cen = rng.uniform(0.0, 1.0, size=(ndrops, 3)) * np.array([nx, ny, nz], dtype=np.float64)
    rad = rng.uniform(rmin, rmax, size=ndrops)
    x = np.arange(nx, dtype=np.float64)[None, None, :]
    y = np.arange(ny, dtype=np.float64)[None, :, None]
    z = (np.arange(nz, dtype=np.float64) if z_planes is None else np.asarray(z_planes, dtype=np.float64))[:, None, None]
    phi0 = np.zeros((z.shape[0], ny, nx))
    for k in range(ndrops):
        dz = np.abs(z - cen[k, 2]); dz = np.minimum(dz, nz - dz)
        near = dz[:, 0, 0] <= rad[k] + 10.0 * W      # beyond that tanh(2 (R - d) / W) == -1 exactly in fp64: the drop adds exactly 0
        if not near.any():
            continue
        dx = np.abs(x - cen[k, 0]); dx = np.minimum(dx, nx - dx)
        dy = np.abs(y - cen[k, 1]); dy = np.minimum(dy, ny - dy)
        d = np.sqrt(dx * dx + dy * dy + dz[near] * dz[near])
        phi0[near] = np.maximum(phi0[near], 0.5 + 0.5 * np.tanh(2.0 * (rad[k] - d) / W))
    if z_planes is None:
        u0 = rng.uniform(-u_amp, u_amp, size=(3, nz, ny, nx))
    else:
        u0 = np.stack([np.random.Generator(np.random.PCG64([seed, int(zz)])).uniform(-u_amp, u_amp, size=(3, ny, nx))
                       for zz in z_planes], axis=1)
    p = default_params(precision=precision, rho_h=1.0, rho_l=1.0e-3, tau_h=0.8, tau_l=0.8, sigma=0.01,
                       W=W, M=0.1)
    return _case(nx, ny, nz, p, phi0, u0, f"sweep{nx}x{ny}x{nz}")


def walled_box(nx=12, ny=10, nz=14, seed=7, precision=64):
    """A small all-walls box with one off-centre drop and a random u0 (exercises edges and corners, R11)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    x, y, z = _grid(nx, ny, nz)
    r = np.sqrt((x - 0.45 * nx) ** 2 + (y - 0.5 * ny) ** 2 + (z - 0.4 * nz) ** 2)
    phi0 = 0.5 + 0.5 * np.tanh(2.0 * (0.28 * min(nx, ny, nz) - r) / 3.0)
    u0 = rng.uniform(-0.005, 0.005, size=(3, nz, ny, nx))
    p = default_params(precision=precision, rho_h=1.0, rho_l=0.1, tau_h=0.6, tau_l=0.3, sigma=0.005, W=3.0,
                       M=0.05, g=(0.0, 0.0, -1.0e-5), bc=(WALL,) * 6)
    return _case(nx, ny, nz, p, phi0, u0, f"walled{nx}x{ny}x{nz}")


# ---- two-dimensional cases on the D2Q9 lattice ("For 2D problems, the D2Q9 lattice model is utilized"): nz = 1
def drop2d(n=64, R=16.0, W=4.0, sigma=0.01, rho_ratio=1000.0, tau=0.8, M=0.1, precision=64):
    """Stationary 2-D drop (a cylinder) in a periodic square: the 2-D Laplace law dp = sigma / R (Eq. 44 as printed)."""
    x, y, z = _grid(n, n, 1)
    c = 0.5 * (n - 1)
    r = np.sqrt((x - c) ** 2 + (y - c) ** 2)
    phi0 = 0.5 + 0.5 * np.tanh(2.0 * (R - r) / W)
    p = default_params(precision=precision, rho_h=1.0, rho_l=1.0 / rho_ratio, tau_h=tau, tau_l=tau, sigma=sigma, W=W, M=M, lattice=1)
    return _case(n, n, 1, p, phi0, np.zeros((3, 1, n, n)), f"drop2d_{n}")


def poiseuille2d(nx=4, ny=64, **kw):
    """The paper's own layered Poiseuille set-up (Sec. 5.3: 2-D, 64 nodes across) on D2Q9; arguments as poiseuille()."""
    case = poiseuille(nx=nx, ny=ny, nz=1, **kw)
    case["params"]["lattice"] = 1
    case["name"] = f"poiseuille2d_{nx}x{ny}"
    return case


def sweep2d(nx=128, ny=96, seed=2505, ndrops=8, rmin=5.0, rmax=12.0, W=4.0, u_amp=0.01, precision=32, bc=(PERIODIC,) * 6):
    """2-D analogue of configs[4]: seeded discs in a box, i.i.d. uniform in-plane u0 (u_z = 0), density ratio 1000, D2Q9."""
    case = sweep_drops(shape=(nx, ny, 1), seed=seed, ndrops=ndrops, rmin=rmin, rmax=rmax, W=W, u_amp=u_amp, precision=precision)
    case["u0"][2] = 0.0
    case["params"].update(lattice=1, bc=tuple(bc))
    case["name"] = f"sweep2d_{nx}x{ny}"
    return case


RANDOM_LATTICE_SEEDS = range(96)   # the seeds tests/test_fuzz_gpu.py runs


def random_lattice(seed, nx_choices=(8, 12, 20, 34, 64, 128, 192, 66, 40, 256), ny_choices=(4, 7, 8, 10, 12, 16, 20),
                   nz_choices=(4, 5, 8, 9, 12, 17, 33)):
    """Seeded random small lattice for the path fuzz (tests/test_fuzz_gpu.py): sizes, faces (every combination the ABI admits in x / y;
    PERIODIC, WALL, FREESLIP, INLET + OUTLET, WALL + OUTLET, INLET + WALL in z), material parameters, collision operator, viscosity
    interpolation, gravity, outlet scheme / clamp / time level, three seeded drops (minimum-image distance across PERIODIC faces) and an
    i.i.d. uniform u0.  An inlet gets the liquid stub of jet() in front of its disc and a density ratio <= 50: a bare phi = 1 disc
    next to gas under a random velocity field is not a start the method runs from (oracle and kernels alike diverge within ten
    steps), and neither is a drop cut off sharply at a periodic seam."""
    rng = np.random.Generator(np.random.PCG64([2505, int(seed)]))
    pick = lambda a: a[int(rng.integers(len(a)))]   # noqa: E731
    nx, ny, nz = pick(nx_choices), pick(ny_choices), pick(nz_choices)
    xf = pick([(PERIODIC, PERIODIC), (WALL, WALL), (FREESLIP, FREESLIP), (FREESLIP, WALL), (WALL, FREESLIP)])
    yf = pick([(PERIODIC, PERIODIC), (WALL, WALL), (FREESLIP, FREESLIP), (FREESLIP, WALL), (WALL, FREESLIP)])
    zf = pick([(PERIODIC, PERIODIC), (WALL, WALL), (INLET, OUTLET), (WALL, OUTLET), (INLET, WALL), (FREESLIP, FREESLIP), (INLET, OUTLET)])
    inlet = zf[0] == INLET
    W = 3.0
    p = default_params(
        rho_l=pick([0.02, 0.1, 1.0] if inlet else [1.0e-3, 0.1, 1.0]), tau_l=pick([0.8, 0.3, 0.1]), tau_h=pick([0.8, 0.6]),
        visc_interp=pick([0, 1, 2]), collision=pick([0, 0, 1]), g=pick([(0.0, 0.0, 0.0), (1.0e-5, -2.0e-5, 3.0e-5)]),
        rho_ref=pick([0.0, 1.0]), sigma=pick([0.01, 0.002]), M=pick([0.1, 0.05]), W=W,
        inlet_u=(0.0, 0.0, 0.03), inlet_c=(nx / 2 - 0.5, ny / 2 - 0.5), inlet_r=min(nx, ny) / 4,
        outlet_clamp=pick([0, 1]), outlet_u_mode=pick([0, 1, 2]), outlet_u_time=pick([0, 1]), bc=xf + yf + zf)
    x, y, z = _grid(nx, ny, nz)
    phi0 = np.zeros((nz, ny, nx))
    for _ in range(3):
        c = rng.uniform(0.0, 1.0, 3) * np.array([nx, ny, nz], dtype=np.float64)
        R = rng.uniform(2.0, max(2.5, min(nx, ny, nz) / 3))
        d = [np.abs(q - c[k]) for k, q in enumerate((x, y, z))]
        d = [np.minimum(dk, n - dk) if f[0] == PERIODIC else dk for dk, n, f in zip(d, (nx, ny, nz), (xf, yf, zf))]
        phi0 = np.maximum(phi0, 0.5 + 0.5 * np.tanh(2.0 * (R - np.sqrt(d[0] ** 2 + d[1] ** 2 + d[2] ** 2)) / W))
    if inlet:
        rxy = np.sqrt((x - p["inlet_c"][0]) ** 2 + (y - p["inlet_c"][1]) ** 2)
        phi0 = np.maximum(phi0, 0.5 + 0.5 * np.tanh(2.0 * np.minimum(p["inlet_r"] - rxy, p["inlet_r"] - z) / W))
    u0 = rng.uniform(-0.01, 0.01, size=(3, nz, ny, nx))
    return _case(nx, ny, nz, p, phi0, u0, f"random{seed}_{nx}x{ny}x{nz}")


def random_lattice2d(seed):
    """random_lattice on the D2Q9 lattice (nz = 1, z faces PERIODIC): x / y faces PERIODIC, WALL, FREESLIP and the mixed pairs, seeded
    discs, in-plane u0."""
    rng = np.random.Generator(np.random.PCG64([2509, int(seed)]))
    pick = lambda a: a[int(rng.integers(len(a)))]   # noqa: E731
    nx, ny = pick((8, 12, 20, 34, 64, 66, 128, 250, 256, 21)), pick((4, 7, 8, 16, 33, 64))
    faces = [(PERIODIC, PERIODIC), (WALL, WALL), (FREESLIP, FREESLIP), (FREESLIP, WALL), (WALL, FREESLIP)]
    xf, yf = pick(faces), pick(faces)
    W = 3.0
    p = default_params(
        rho_l=pick([1.0e-3, 0.1, 1.0]), tau_l=pick([0.8, 0.3, 0.1]), tau_h=pick([0.8, 0.6]), visc_interp=pick([0, 1, 2]),
        collision=pick([0, 0, 1]), g=pick([(0.0, 0.0, 0.0), (1.0e-5, -2.0e-5, 0.0)]), rho_ref=pick([0.0, 1.0]),
        sigma=pick([0.01, 0.002]), M=pick([0.1, 0.05]), W=W, bc=xf + yf + (PERIODIC, PERIODIC), lattice=1)
    x, y, _ = _grid(nx, ny, 1)
    phi0 = np.zeros((1, ny, nx))
    for _k in range(3):
        c = rng.uniform(0.0, 1.0, 2) * np.array([nx, ny], dtype=np.float64)
        R = rng.uniform(2.0, max(2.5, min(nx, ny) / 3))
        d = [np.abs(q - c[k]) for k, q in enumerate((x, y))]
        d = [np.minimum(dk, n - dk) if f[0] == PERIODIC else dk for dk, n, f in zip(d, (nx, ny), (xf, yf))]
        phi0 = np.maximum(phi0, 0.5 + 0.5 * np.tanh(2.0 * (R - np.sqrt(d[0] ** 2 + d[1] ** 2)) / W))
    u0 = rng.uniform(-0.01, 0.01, size=(3, 1, ny, nx))
    u0[2] = 0.0
    return _case(nx, ny, 1, p, phi0, u0, f"random2d_{seed}_{nx}x{ny}")
