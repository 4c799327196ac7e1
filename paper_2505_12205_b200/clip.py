"""Thin Python binding of libclip (include/clip.h): argument marshalling only -- every step of the path runs in
the CUDA kernels of csrc/.  PyTorch is used for device memory and streams, nothing else.

Same names as the C ABI: clip_workspace_bytes, clip_create, clip_init, clip_step, clip_get, clip_destroy,
clip_last_error (+ clip_launch_count), plus the convenience class `Clip` and the host-buffer entry point
`run_host` used by bench.py's e2e leg.  There is NO CPU fallback: a missing libclip.so raises.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libclip.so")

CLIP_OK, CLIP_EINVAL, CLIP_ENOMEM, CLIP_ESTATE, CLIP_ECUDA = 0, -1, -2, -3, -4


class clip_params(C.Structure):
    """Mirror of `struct clip_params` in include/clip.h."""
    _fields_ = [
        ("precision", C.c_int),
        ("rho_h", C.c_double), ("rho_l", C.c_double),
        ("tau_h", C.c_double), ("tau_l", C.c_double),
        ("sigma", C.c_double), ("W", C.c_double), ("M", C.c_double),
        ("g", C.c_double * 3), ("rho_ref", C.c_double),
        ("bc", C.c_int * 6),
        ("inlet_u", C.c_double * 3), ("inlet_phi", C.c_double),
        ("inlet_c", C.c_double * 2), ("inlet_r", C.c_double),
        ("outlet_u_mode", C.c_int), ("visc_interp", C.c_int), ("collision", C.c_int), ("phase_only", C.c_int),
        ("outlet_clamp", C.c_int), ("outlet_u_time", C.c_int),
        ("path", C.c_int), ("tile_ty", C.c_int), ("tile_chunks", C.c_int), ("runtime_nx", C.c_int),
        ("lattice", C.c_int),
        ("cluster_y", C.c_int),
    ]


def make_params(p: dict) -> clip_params:
    s = clip_params()
    s.precision = int(p["precision"])
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
    for k in ("outlet_clamp", "outlet_u_time", "path", "tile_ty", "tile_chunks", "runtime_nx", "lattice", "cluster_y"):
        setattr(s, k, int(p.get(k, 0)))
    return s


_lib = None


def lib():
    """Load libclip.so (built in-tree by __graft_entry__.build()); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.clip_workspace_bytes.restype = C.c_size_t
        L.clip_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(clip_params)]
        L.clip_create.restype = C.c_int
        L.clip_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.POINTER(clip_params),
                                  C.c_void_p, C.c_size_t, C.c_void_p]
        L.clip_init.restype = C.c_int
        L.clip_init.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.clip_step.restype = C.c_int
        L.clip_step.argtypes = [C.c_void_p, C.c_int]
        L.clip_set_u.restype = C.c_int
        L.clip_set_u.argtypes = [C.c_void_p, C.c_void_p]
        L.clip_get.restype = C.c_int
        L.clip_get.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.clip_destroy.restype = C.c_int
        L.clip_destroy.argtypes = [C.c_void_p]
        L.clip_last_error.restype = C.c_char_p
        L.clip_last_error.argtypes = [C.c_void_p]
        L.clip_launch_count.restype = C.c_longlong
        L.clip_launch_count.argtypes = [C.c_void_p]
        L.clip_graph_steps.restype = C.c_longlong
        L.clip_graph_steps.argtypes = [C.c_void_p]
        L.clip_step_profiled.restype = C.c_int
        L.clip_step_profiled.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.clip_kernel_kinds.restype = C.c_int
        L.clip_halo_bytes.restype = C.c_size_t
        L.clip_halo_bytes.argtypes = [C.c_void_p]
        L.clip_halo_pack.restype = C.c_int
        L.clip_halo_pack.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.clip_halo_unpack.restype = C.c_int
        L.clip_halo_unpack.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.clip_halo_stream.restype = C.c_int
        L.clip_halo_stream.argtypes = [C.c_void_p, C.c_void_p]
        L.clip_step_halo_begin.restype = C.c_int
        L.clip_step_halo_begin.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.clip_step_halo_end.restype = C.c_int
        L.clip_step_halo_end.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.clip_kernel_name.restype = C.c_char_p
        L.clip_kernel_name.argtypes = [C.c_int]
        L.clip_outlet_lambda_static.restype = C.c_int
        L.clip_outlet_lambda_static.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.clip_static_last_error.restype = C.c_char_p
        L.clip_static_last_error.argtypes = []
        _lib = L
    return _lib


# ---- the C ABI, same names ------------------------------------------------------------------------------
def clip_workspace_bytes(nx, ny, nz, params: clip_params) -> int:
    return int(lib().clip_workspace_bytes(nx, ny, nz, C.byref(params)))


def clip_create(nx, ny, nz, params: clip_params, d_workspace: int, nbytes: int, cuda_stream: int):
    h = C.c_void_p()
    rc = lib().clip_create(C.byref(h), nx, ny, nz, C.byref(params), C.c_void_p(d_workspace), nbytes,
                           C.c_void_p(cuda_stream))
    return rc, h


def clip_init(h, d_phi0: int, d_u0: int) -> int:
    return lib().clip_init(h, C.c_void_p(d_phi0), C.c_void_p(d_u0))


def clip_step(h, n: int) -> int:
    return lib().clip_step(h, int(n))


def clip_set_u(h, d_u: int) -> int:
    return lib().clip_set_u(h, C.c_void_p(d_u))


def clip_get(h, d_phi: int, d_p: int, d_u: int) -> int:
    return lib().clip_get(h, C.c_void_p(d_phi), C.c_void_p(d_p), C.c_void_p(d_u))


def clip_destroy(h) -> int:
    return lib().clip_destroy(h)


def clip_last_error(h=None) -> str:
    s = lib().clip_last_error(h)
    return s.decode() if s else ""


def clip_launch_count(h) -> int:
    return int(lib().clip_launch_count(h))


def clip_graph_steps(h) -> int:
    return int(lib().clip_graph_steps(h))


def clip_halo_bytes(h) -> int:
    return int(lib().clip_halo_bytes(h))


def clip_halo_pack(h, d_lo: int, d_hi: int) -> int:
    return lib().clip_halo_pack(h, C.c_void_p(d_lo), C.c_void_p(d_hi))


def clip_halo_unpack(h, d_recv_lo: int, d_recv_hi: int, d_sent_lo: int, d_sent_hi: int) -> int:
    return lib().clip_halo_unpack(h, C.c_void_p(d_recv_lo), C.c_void_p(d_recv_hi), C.c_void_p(d_sent_lo), C.c_void_p(d_sent_hi))


def clip_halo_stream(h, cuda_stream: int) -> int:
    return lib().clip_halo_stream(h, C.c_void_p(cuda_stream))


def clip_step_halo_begin(h, d_lo: int, d_hi: int) -> int:
    return lib().clip_step_halo_begin(h, C.c_void_p(d_lo), C.c_void_p(d_hi))


def clip_step_halo_end(h, d_recv_lo: int, d_recv_hi: int, d_sent_lo: int, d_sent_hi: int) -> int:
    return lib().clip_step_halo_end(h, C.c_void_p(d_recv_lo), C.c_void_p(d_recv_hi), C.c_void_p(d_sent_lo), C.c_void_p(d_sent_hi))


def clip_step_profiled(h, n: int):
    """Returns {kernel name: (total ms, launches)} for n steps (host-synchronous instrumentation)."""
    k = lib().clip_kernel_kinds()
    ms = (C.c_double * k)()
    cnt = (C.c_longlong * k)()
    rc = lib().clip_step_profiled(h, int(n), ms, cnt)
    return rc, {lib().clip_kernel_name(i).decode(): (ms[i], cnt[i]) for i in range(k)}


CLIP_STATIC_MAX_PLANE_NODES = 262144


def clip_outlet_lambda_static(d_u: int, nx, ny, nz, precision, outlet_u_mode, outlet_clamp, d_lambda: int, cuda_stream: int) -> int:
    """No-allocation entry point (include/clip.h): lambda of the convective outlet from u(t), scratch in a static device array."""
    return lib().clip_outlet_lambda_static(C.c_void_p(d_u), int(nx), int(ny), int(nz), int(precision), int(outlet_u_mode),
                                           int(outlet_clamp), C.c_void_p(d_lambda), C.c_void_p(cuda_stream))


def clip_static_last_error() -> str:
    s = lib().clip_static_last_error()
    return s.decode() if s else ""


class ClipError(RuntimeError):
    def __init__(self, rc, msg):
        super().__init__(f"libclip error {rc}: {msg}")
        self.rc = rc


# ---- convenience wrapper --------------------------------------------------------------------------------
class Clip:
    """One simulation on one GPU.  Owns the workspace tensor; fields are torch CUDA tensors phi[z,y,x], u[3,z,y,x]."""

    def __init__(self, nx, ny, nz, params: dict, device="cuda:0", stream=None):
        import torch
        self.torch = torch
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.device = torch.device(device)
        self.dtype = torch.float32 if int(params["precision"]) == 32 else torch.float64
        self._p = make_params(params)
        nbytes = clip_workspace_bytes(self.nx, self.ny, self.nz, self._p)
        if nbytes == 0:
            raise ClipError(CLIP_EINVAL, clip_last_error(None))
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self._ws.data_ptr()
            self._ws_ptr = (base + 255) // 256 * 256
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            rc, self._h = clip_create(self.nx, self.ny, self.nz, self._p, self._ws_ptr, nbytes, self.stream.cuda_stream)
        if rc != CLIP_OK:
            raise ClipError(rc, clip_last_error(None))

    @classmethod
    def from_case(cls, case: dict, device="cuda:0", precision=None):
        import torch
        params = dict(case["params"])
        if precision is not None:
            params["precision"] = precision
        c = cls(case["nx"], case["ny"], case["nz"], params, device=device)
        c.init(torch.as_tensor(case["phi0"]), torch.as_tensor(case["u0"]))
        return c

    def _check(self, rc):
        if rc != CLIP_OK:
            raise ClipError(rc, clip_last_error(self._h))

    def _on_stream(self, x, shape):
        """Copy / cast `x` to the device ON the handle's stream (which first waits for the caller's current stream, where
        `x` may still be being produced)."""
        t = self.torch
        self.stream.wait_stream(t.cuda.current_stream(self.device))
        with t.cuda.stream(self.stream):
            y = x.to(device=self.device, dtype=self.dtype).contiguous().reshape(shape)
        if y.is_cuda:
            y.record_stream(self.stream)
        return y

    def init(self, phi0, u0):
        t = self.torch
        with t.cuda.device(self.device):
            phi0 = self._on_stream(phi0, (self.nz, self.ny, self.nx))
            u0 = self._on_stream(u0, (3, self.nz, self.ny, self.nx))
            with t.cuda.stream(self.stream):
                self._check(clip_init(self._h, phi0.data_ptr(), u0.data_ptr()))

    def set_u(self, u):
        t = self.torch
        with t.cuda.device(self.device):
            u = self._on_stream(u, (3, self.nz, self.ny, self.nx))
            with t.cuda.stream(self.stream):
                self._check(clip_set_u(self._h, u.data_ptr()))

    def step(self, n=1):
        with self.torch.cuda.device(self.device):
            self._check(clip_step(self._h, n))

    def get(self, phi=True, p=True, u=True):
        t = self.torch
        with t.cuda.device(self.device), t.cuda.stream(self.stream):
            o_phi = t.empty((self.nz, self.ny, self.nx), dtype=self.dtype, device=self.device) if phi else None
            o_p = t.empty((self.nz, self.ny, self.nx), dtype=self.dtype, device=self.device) if p else None
            o_u = t.empty((3, self.nz, self.ny, self.nx), dtype=self.dtype, device=self.device) if u else None
            self._check(clip_get(self._h, o_phi.data_ptr() if phi else 0, o_p.data_ptr() if p else 0,
                                 o_u.data_ptr() if u else 0))
        return o_phi, o_p, o_u

    def get_into(self, phi, p, u):
        with self.torch.cuda.device(self.device):
            self._check(clip_get(self._h, phi.data_ptr() if phi is not None else 0,
                                 p.data_ptr() if p is not None else 0, u.data_ptr() if u is not None else 0))

    def halo_buffer(self):
        """Device buffer for one face's halo record, [12, ny, nx] in the handle's precision (clip_halo_pack / clip_halo_unpack)."""
        assert clip_halo_bytes(self._h) == 12 * self.ny * self.nx * (4 if self.dtype == self.torch.float32 else 8)
        return self.torch.empty((12, self.ny, self.nx), dtype=self.dtype, device=self.device)

    def halo_pack(self, lo, hi):
        with self.torch.cuda.device(self.device):
            self._check(clip_halo_pack(self._h, lo.data_ptr() if lo is not None else 0, hi.data_ptr() if hi is not None else 0))

    def halo_unpack(self, recv_lo, recv_hi, sent_lo, sent_hi):
        ptr = lambda t: t.data_ptr() if t is not None else 0  # noqa: E731
        with self.torch.cuda.device(self.device):
            self._check(clip_halo_unpack(self._h, ptr(recv_lo), ptr(recv_hi), ptr(sent_lo), ptr(sent_hi)))

    def halo_stream(self, stream):
        """Second (torch) stream of the overlapped slab step (clip_halo_stream); kept alive by the object."""
        self._halo_stream = stream
        with self.torch.cuda.device(self.device):
            self._check(clip_halo_stream(self._h, stream.cuda_stream if stream is not None else 0))

    def step_halo_begin(self, lo, hi):
        with self.torch.cuda.device(self.device):
            self._check(clip_step_halo_begin(self._h, lo.data_ptr() if lo is not None else 0, hi.data_ptr() if hi is not None else 0))

    def step_halo_end(self, recv_lo, recv_hi, sent_lo, sent_hi):
        ptr = lambda t: t.data_ptr() if t is not None else 0  # noqa: E731
        with self.torch.cuda.device(self.device):
            self._check(clip_step_halo_end(self._h, ptr(recv_lo), ptr(recv_hi), ptr(sent_lo), ptr(sent_hi)))

    def step_profiled(self, n=1):
        with self.torch.cuda.device(self.device):
            rc, d = clip_step_profiled(self._h, n)
        self._check(rc)
        return d

    @property
    def launches(self) -> int:
        return clip_launch_count(self._h)

    @property
    def graph_steps(self) -> int:
        return clip_graph_steps(self._h)

    def close(self):
        if getattr(self, "_h", None):
            try:
                self.stream.synchronize()   # kernels of this stream may still use the workspace the allocator is about to reuse
            except Exception:
                pass
            clip_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def run_host(case_or_sim, phi0_host, u0_host, nsteps, out_phi_host, out_p_host, out_u_host, dev_bufs=None):
    """Host-buffer entry point (bench.py e2e): pinned host phi0/u0 -> H2D -> init -> n steps -> get -> D2H.

    `case_or_sim` is an existing Clip (its workspace is reused).  Returns (h2d_bytes, d2h_bytes).
    """
    sim = case_or_sim
    t = sim.torch
    with t.cuda.device(sim.device), t.cuda.stream(sim.stream):
        if dev_bufs is None:
            dev_bufs = (t.empty_like(phi0_host, device=sim.device), t.empty_like(u0_host, device=sim.device),
                        t.empty_like(out_phi_host, device=sim.device), t.empty_like(out_p_host, device=sim.device),
                        t.empty_like(out_u_host, device=sim.device))
        d_phi0, d_u0, d_phi, d_p, d_u = dev_bufs
        d_phi0.copy_(phi0_host, non_blocking=True)
        d_u0.copy_(u0_host, non_blocking=True)
        sim._check(clip_init(sim._h, d_phi0.data_ptr(), d_u0.data_ptr()))
        sim._check(clip_step(sim._h, nsteps))
        sim._check(clip_get(sim._h, d_phi.data_ptr(), d_p.data_ptr(), d_u.data_ptr()))
        out_phi_host.copy_(d_phi, non_blocking=True)
        out_p_host.copy_(d_p, non_blocking=True)
        out_u_host.copy_(d_u, non_blocking=True)
    h2d = phi0_host.numel() * phi0_host.element_size() + u0_host.numel() * u0_host.element_size()
    d2h = sum(x.numel() * x.element_size() for x in (out_phi_host, out_p_host, out_u_host))
    return h2d, d2h
