"""ctypes binding of oracle/clip_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports the CUDA package's binding or sources.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "clip_oracle.c")
_LIB = os.path.join(_HERE, "libclip_oracle.so")
_LIB9 = os.path.join(_HERE, "libclip_oracle_d2q9.so")


def build(force: bool = False, lattice: str = "d3q19") -> str:
    """Compile the oracle with gcc (fp64, no FMA contraction): the D3Q19 library and the D2Q9 one (same source, -DCLIPO_D2Q9)."""
    for target, extra in ((_LIB, []), (_LIB9, ["-DCLIPO_D2Q9"])):
        if force or not os.path.exists(target) or os.path.getmtime(target) < os.path.getmtime(_SRC):
            tmp = target + f".tmp{os.getpid()}"
            subprocess.check_call(["gcc", "-O3", "-ffp-contract=off", "-shared", "-fPIC", *extra, "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, target)
    return _LIB9 if lattice == "d2q9" else _LIB


class _Params(C.Structure):
    _fields_ = [
        ("rho_h", C.c_double), ("rho_l", C.c_double),
        ("tau_h", C.c_double), ("tau_l", C.c_double),
        ("sigma", C.c_double), ("W", C.c_double), ("M", C.c_double),
        ("g", C.c_double * 3), ("rho_ref", C.c_double),
        ("bc", C.c_int * 6),
        ("inlet_u", C.c_double * 3), ("inlet_phi", C.c_double), ("inlet_c", C.c_double * 2),
        ("inlet_r", C.c_double),
        ("outlet_u_mode", C.c_int), ("visc_interp", C.c_int), ("collision", C.c_int), ("phase_only", C.c_int),
        ("outlet_clamp", C.c_int), ("outlet_u_time", C.c_int), ("macro_u_refine", C.c_int), ("open_ghost", C.c_int),
    ]


def _marshal(p: dict) -> _Params:
    s = _Params()
    for k in ("rho_h", "rho_l", "tau_h", "tau_l", "sigma", "W", "M", "rho_ref", "inlet_phi", "inlet_r"):
        setattr(s, k, float(p[k]))
    s.g = (C.c_double * 3)(*[float(v) for v in p["g"]])
    s.bc = (C.c_int * 6)(*[int(v) for v in p["bc"]])
    s.inlet_u = (C.c_double * 3)(*[float(v) for v in p["inlet_u"]])
    s.inlet_c = (C.c_double * 2)(*[float(v) for v in p["inlet_c"]])
    s.outlet_u_mode = int(p["outlet_u_mode"])
    s.visc_interp = int(p["visc_interp"])
    s.collision = int(p.get("collision", 0))
    s.phase_only = int(p.get("phase_only", 0))
    s.outlet_clamp = int(p.get("outlet_clamp", 0))
    s.outlet_u_time = int(p.get("outlet_u_time", 0))
    s.open_ghost = int(p.get("open_ghost", 0))   # oracle only (sensitivity of reading R9)
    s.macro_u_refine = int(p.get("macro_u_refine", 0))   # oracle only (sensitivity of reading R13)
    return s


_libs = {}


def lib(lattice: str = "d3q19"):
    if lattice not in _libs:
        _lib = C.CDLL(build(lattice=lattice))
        _libs[lattice] = _lib
        d = C.POINTER(C.c_double)
        _lib.clipo_create.restype = C.c_void_p
        _lib.clipo_create.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(_Params)]
        _lib.clipo_destroy.argtypes = [C.c_void_p]
        _lib.clipo_init.argtypes = [C.c_void_p, d, d]
        _lib.clipo_step.argtypes = [C.c_void_p, C.c_int]
        _lib.clipo_set_u.argtypes = [C.c_void_p, d]
        _lib.clipo_get.argtypes = [C.c_void_p, d, d, d]
        _lib.clipo_get_populations.argtypes = [C.c_void_p, d, d]
        _lib.clipo_set_populations.argtypes = [C.c_void_p, d, d]
        _lib.clipo_lattice.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), d]
        _lib.clipo_basis.argtypes = [C.c_void_p, d, d]
        _lib.clipo_collision_matrix.argtypes = [C.c_void_p, C.c_double, d]
        _lib.clipo_stencil_field.argtypes = [C.c_void_p, d, d, d, d]
        _lib.clipo_node_terms.argtypes = [C.c_void_p, C.c_double, d, C.c_double, d, d, d, d, d, d]
        _lib.clipo_inlet_node.argtypes = [C.c_void_p, d, d]
        _lib.clipo_total_force.argtypes = [C.c_void_p, d, C.c_double, d, C.c_double, d, C.c_double, d]
        _lib.clipo_time.restype = C.c_long
        _lib.clipo_time.argtypes = [C.c_void_p]
        _lib.clipo_q.restype = C.c_int
    return _libs[lattice]


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Oracle:
    """One oracle simulation.  Fields are numpy fp64 arrays, phi[z,y,x], u[3,z,y,x]."""

    def __init__(self, nx: int, ny: int, nz: int, params: dict):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.n = self.nx * self.ny * self.nz
        self._p = _marshal(params)
        self.lattice_name = "d2q9" if int(params.get("lattice", 0)) == 1 else "d3q19"   # params["lattice"]: 0 = D3Q19, 1 = D2Q9
        self._lib = lib(self.lattice_name)
        self.Q = int(self._lib.clipo_q())
        self._h = self._lib.clipo_create(self.nx, self.ny, self.nz, C.byref(self._p))
        if not self._h:
            raise ValueError("clipo_create failed")

    @classmethod
    def from_case(cls, case: dict) -> "Oracle":
        o = cls(case["nx"], case["ny"], case["nz"], case["params"])
        o.init(case["phi0"], case["u0"])
        return o

    def close(self):
        if self._h:
            self._lib.clipo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init(self, phi0, u0):
        phi0 = np.ascontiguousarray(phi0, dtype=np.float64).reshape(self.nz, self.ny, self.nx)
        u0 = np.ascontiguousarray(u0, dtype=np.float64).reshape(3, self.nz, self.ny, self.nx)
        self._lib.clipo_init(self._h, _dp(phi0), _dp(u0))

    def set_u(self, u):
        u = np.ascontiguousarray(u, dtype=np.float64).reshape(3, self.nz, self.ny, self.nx)
        self._lib.clipo_set_u(self._h, _dp(u))

    def step(self, n: int = 1):
        if self._lib.clipo_step(self._h, int(n)) != 0:
            raise RuntimeError("clipo_step failed")

    def get(self):
        phi = np.empty((self.nz, self.ny, self.nx)); p = np.empty_like(phi)
        u = np.empty((3, self.nz, self.ny, self.nx))
        self._lib.clipo_get(self._h, _dp(phi), _dp(p), _dp(u))
        return phi, p, u

    @property
    def time(self) -> int:
        return int(self._lib.clipo_time(self._h))

    # ---- introspection (pins only)
    def populations(self):
        f = np.empty((self.nz, self.ny, self.nx, self.Q)); g = np.empty_like(f)
        self._lib.clipo_get_populations(self._h, _dp(f), _dp(g))
        return f, g

    def set_populations(self, f, g):
        f = np.ascontiguousarray(f, dtype=np.float64); g = np.ascontiguousarray(g, dtype=np.float64)
        self._lib.clipo_set_populations(self._h, _dp(f), _dp(g))

    def lattice(self):
        ex = (C.c_int * self.Q)(); ey = (C.c_int * self.Q)(); ez = (C.c_int * self.Q)(); w = np.empty(self.Q)
        self._lib.clipo_lattice(self._h, ex, ey, ez, _dp(w))
        e = np.stack([np.array(ex[:]), np.array(ey[:]), np.array(ez[:])], axis=1).astype(np.float64)
        return e, w

    def basis(self):
        M = np.empty((self.Q, self.Q)); Mi = np.empty((self.Q, self.Q))
        self._lib.clipo_basis(self._h, _dp(M), _dp(Mi))
        return M, Mi

    def collision_matrix(self, s_nu: float):
        A = np.empty((self.Q, self.Q))
        self._lib.clipo_collision_matrix(self._h, float(s_nu), _dp(A))
        return A

    def stencil_field(self, phi):
        phi = np.ascontiguousarray(phi, dtype=np.float64).reshape(self.nz, self.ny, self.nx)
        G = np.empty((3,) + phi.shape); L = np.empty_like(phi); mu = np.empty_like(phi)
        self._lib.clipo_stencil_field(self._h, _dp(phi), _dp(G), _dp(L), _dp(mu))
        return G, L, mu

    def node_terms(self, pstar, u, phi, F, nvec):
        u = np.ascontiguousarray(u, dtype=np.float64); F = np.ascontiguousarray(F, dtype=np.float64)
        nvec = np.ascontiguousarray(nvec, dtype=np.float64)
        out = [np.empty(self.Q) for _ in range(4)]
        self._lib.clipo_node_terms(self._h, float(pstar), _dp(u), float(phi), _dp(F), _dp(nvec), *[_dp(o) for o in out])
        return out  # feqbar, Fa, geqbar, Fphi

    def inlet_node(self, f, g):
        f = np.array(f, dtype=np.float64); g = np.array(g, dtype=np.float64)
        self._lib.clipo_inlet_node(self._h, _dp(f), _dp(g))
        return f, g

    def total_force(self, f, pstar, u, phi, G, L):
        f = np.ascontiguousarray(f, dtype=np.float64); u = np.ascontiguousarray(u, dtype=np.float64)
        G = np.ascontiguousarray(G, dtype=np.float64)
        F = np.empty(3)
        self._lib.clipo_total_force(self._h, _dp(f), float(pstar), _dp(u), float(phi), _dp(G), float(L), _dp(F))
        return F
