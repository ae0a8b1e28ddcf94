"""Thin ctypes binding of libah_b200.so (include/ah_b200.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used for
device buffers and streams.  There is no CPU fallback: if the library is missing, or there
is no CUDA device, the calls raise.

    sim = Simulation(nx=64, s=0.0, p=1.0)          # allocates 20 torch device buffers
    sim.init_fields(seed=1)                          # ah_init_fields
    sim.step(160, tau=1.0, dt=0.1)                   # ah_step
    d = sim.diagnostics(tau=17.0, dt=0.1)            # ah_diagnostics -> dict
    f = sim.get_fields()                             # ah_get_fields -> numpy (10, nz, ny, nx)
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libah_b200.so"

AH_OK, AH_EINVAL, AH_ECUDA, AH_ESTATE = 0, -1, -2, -3
AH_NFIELDS = 10
KERNEL_AUTO, KERNEL_SITE, KERNEL_TILED = 0, 1, 2

FIELD_NAMES = ("phi_re", "phi_im", "pi_re", "pi_im", "th_x", "th_y", "th_z", "ep_x", "ep_y", "ep_z")

# every symbol include/ah_b200.h declares (checked by tests/test_abi.py)
EXPORTS = (
    "ah_create", "ah_destroy", "ah_init_fields", "ah_set_fields", "ah_get_fields", "ah_current_bufs",
    "ah_step", "ah_step_cooling", "ah_diagnostics", "ah_step_diag", "ah_winding_field", "ah_set_kernel", "ah_get_kernel",
    "ah_launch_count", "ah_tiled_launch_info", "ah_coeffs", "ah_test_trig", "ah_test_trig_fast", "ah_last_error", "ah_version",
)


class AhError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"ah_b200 error {code}: {msg}")
        self.code = code


class Params(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("dx", C.c_double),
        ("lambda0", C.c_double), ("e0", C.c_double), ("sigma", C.c_double),
        ("s", C.c_double), ("p", C.c_double), ("tau_ref", C.c_double), ("alpha", C.c_double),
        ("compact", C.c_int32), ("fp64", C.c_int32),
    ]


class Diag(C.Structure):
    _fields_ = [
        ("tau", C.c_double),
        ("n_wind", C.c_int64), ("n_wind_xy", C.c_int64), ("n_wind_xz", C.c_int64),
        ("n_wind_yz", C.c_int64), ("n_near_branch", C.c_int64), ("n_big_plaq", C.c_int64),
        ("string_length", C.c_double), ("xi_w", C.c_double),
        ("sum_pi2_L", C.c_double), ("sum_grad2_L", C.c_double), ("sum_L", C.c_double),
        ("v2_phi", C.c_double),
        ("gauss_max", C.c_double), ("gauss_l2", C.c_double), ("gauss_rel", C.c_double),
        ("gauss_div_l2", C.c_double), ("gauss_charge_l2", C.c_double),
        ("xi_l", C.c_double),
    ]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def lib():
    """Load libah_b200.so; raise loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise ImportError(
            f"{LIB_PATH} not found: build it with `python -m paper_2005_14454_b200.build` "
            "(nvcc, sm_100a).  There is no CPU fallback.")
    L = C.CDLL(str(LIB_PATH))
    vp, ip, dp = C.c_void_p, C.c_int, C.c_double
    L.ah_last_error.restype = C.c_char_p
    L.ah_version.restype = C.c_char_p
    L.ah_create.argtypes = [C.POINTER(vp), C.POINTER(Params), C.POINTER(vp), ip, C.c_size_t, vp]
    L.ah_destroy.argtypes = [vp]
    L.ah_init_fields.argtypes = [vp, C.c_uint64]
    L.ah_set_fields.argtypes = [vp, vp]
    L.ah_get_fields.argtypes = [vp, vp]
    L.ah_current_bufs.argtypes = [vp, C.POINTER(vp)]
    L.ah_step.argtypes = [vp, ip, dp, dp]
    L.ah_step_cooling.argtypes = [vp, ip, dp, dp]
    L.ah_diagnostics.argtypes = [vp, dp, dp, C.POINTER(Diag)]
    L.ah_step_diag.argtypes = [vp, ip, dp, dp, ip, C.POINTER(Diag), ip, C.POINTER(ip)]
    L.ah_winding_field.argtypes = [vp, vp, vp]
    L.ah_set_kernel.argtypes = [vp, ip]
    L.ah_get_kernel.argtypes = [vp]
    L.ah_launch_count.argtypes = [vp]
    L.ah_tiled_launch_info.argtypes = [ip, ip, ip, C.POINTER(ip), C.POINTER(ip)]
    L.ah_launch_count.restype = C.c_int64
    L.ah_coeffs.argtypes = [C.POINTER(Params), dp, dp] + [C.POINTER(dp)] * 4
    L.ah_test_trig.argtypes = [vp, vp, vp, vp, C.c_size_t, vp]
    L.ah_test_trig_fast.argtypes = [vp, vp, vp, vp, C.c_size_t, vp]
    for name in EXPORTS:
        if name not in ("ah_last_error", "ah_version", "ah_launch_count"):
            getattr(L, name).restype = ip
    _lib = L
    return L


def _check(rc):
    if rc != AH_OK:
        raise AhError(rc, lib().ah_last_error().decode())


def make_params(nx, ny=None, nz=None, dx=0.5, lambda0=2.0, e0=1.0, sigma=1.0, s=0.0, p=1.0,
                tau_ref=1.0, alpha=2.0, compact=1, fp64=False) -> Params:
    ny = nx if ny is None else ny
    nz = nx if nz is None else nz
    return Params(int(nx), int(ny), int(nz), float(dx), float(lambda0), float(e0), float(sigma),
                  float(s), float(p), float(tau_ref), float(alpha), int(compact), int(bool(fp64)))


def tiled_launch_info(nx, ny, nz):
    """(planes per CTA, number of CTAs) of the tiled kernel for this lattice; host logic, no device needed."""
    zc, n = C.c_int(0), C.c_int(0)
    _check(lib().ah_tiled_launch_info(int(nx), int(ny), int(nz), C.byref(zc), C.byref(n)))
    return zc.value, n.value


def coeffs(P: Params, tau: float, dt: float):
    a, q, d, w = (C.c_double() for _ in range(4))
    _check(lib().ah_coeffs(C.byref(P), tau, dt, C.byref(a), C.byref(q), C.byref(d), C.byref(w)))
    return a.value, q.value, d.value, w.value


class Simulation:
    """One periodic lattice resident in one GPU's HBM (20 torch-owned SoA buffers)."""

    def __init__(self, nx=None, params: Params | None = None, device="cuda:0", stream=None, **kw):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2005_14454_b200 needs a CUDA device (B200); there is no CPU fallback")
        self.P = params if params is not None else make_params(nx, **kw)
        P = self.P
        self.torch = torch
        self.device = torch.device(device)
        self.dtype = torch.float64 if P.fp64 else torch.float32
        self.np_dtype = np.float64 if P.fp64 else np.float32
        self.n = P.nx * P.ny * P.nz
        self.shape = (AH_NFIELDS, P.nz, P.ny, P.nx)
        with torch.cuda.device(self.device):
            # 20 separate 1-D allocations: each scalar array is its own buffer (SoA, ping-pong)
            self.bufs = [torch.empty(self.n, dtype=self.dtype, device=self.device) for _ in range(2 * AH_NFIELDS)]
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            ptrs = (C.c_void_p * (2 * AH_NFIELDS))(*[b.data_ptr() for b in self.bufs])
            self._ctx = C.c_void_p()
            _check(lib().ah_create(C.byref(self._ctx), C.byref(P), ptrs, 2 * AH_NFIELDS,
                                   self.n * self.bufs[0].element_size(),
                                   C.c_void_p(self.stream.cuda_stream)))

    # -- lifetime
    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            lib().ah_destroy(self._ctx)
            self._ctx = C.c_void_p()
        self.bufs = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _dev(self):
        return self.torch.cuda.device(self.device)

    # -- C ABI, same names
    def init_fields(self, seed: int):
        with self._dev():
            _check(lib().ah_init_fields(self._ctx, C.c_uint64(seed)))

    def set_fields(self, host):
        """host: array-like (10, nz, ny, nx); cast to the context's dtype, C-contiguous."""
        a = np.ascontiguousarray(host, dtype=self.np_dtype)
        if a.shape != self.shape:
            raise ValueError(f"fields must have shape {self.shape}, got {a.shape}")
        with self._dev():
            _check(lib().ah_set_fields(self._ctx, a.ctypes.data))

    def set_fields_ptr(self, host_ptr: int):
        with self._dev():
            _check(lib().ah_set_fields(self._ctx, C.c_void_p(host_ptr)))

    def get_fields(self, out=None) -> np.ndarray:
        if out is None:
            out = np.empty(self.shape, dtype=self.np_dtype)
        assert out.dtype == self.np_dtype and out.flags["C_CONTIGUOUS"] and out.shape == self.shape
        with self._dev():
            _check(lib().ah_get_fields(self._ctx, out.ctypes.data))
        return out

    def get_fields_ptr(self, host_ptr: int):
        with self._dev():
            _check(lib().ah_get_fields(self._ctx, C.c_void_p(host_ptr)))

    def current_bufs(self):
        """The 10 torch tensors holding the current state (ping-pong parity resolved)."""
        ptrs = (C.c_void_p * AH_NFIELDS)()
        _check(lib().ah_current_bufs(self._ctx, ptrs))
        by_ptr = {b.data_ptr(): b for b in self.bufs}
        return [by_ptr[p] for p in ptrs]

    def step(self, n: int, tau: float, dt: float):
        with self._dev():
            _check(lib().ah_step(self._ctx, int(n), float(tau), float(dt)))

    def step_cooling(self, n: int, delta: float, dt: float):
        with self._dev():
            _check(lib().ah_step_cooling(self._ctx, int(n), float(delta), float(dt)))

    def diagnostics(self, tau: float, dt: float) -> dict:
        d = Diag()
        with self._dev():
            _check(lib().ah_diagnostics(self._ctx, float(tau), float(dt), C.byref(d)))
        return d.asdict()

    def step_diag(self, n: int, tau: float, dt: float, every: int):
        cap = max(1, (n + every - 1) // every) if every >= 1 else 1
        recs = (Diag * cap)()
        nw = C.c_int(0)
        with self._dev():
            _check(lib().ah_step_diag(self._ctx, int(n), float(tau), float(dt), int(every), recs, cap, C.byref(nw)))
        return [recs[i].asdict() for i in range(nw.value)]

    def winding_field(self):
        P = self.P
        w = np.zeros((3, P.nz, P.ny, P.nx), dtype=np.int8)
        near = np.zeros((3, P.nz, P.ny, P.nx), dtype=np.uint8)
        with self._dev():
            _check(lib().ah_winding_field(self._ctx, w.ctypes.data, near.ctypes.data))
        return w, near

    def set_kernel(self, kernel: int):
        _check(lib().ah_set_kernel(self._ctx, int(kernel)))

    def get_kernel(self) -> int:
        k = lib().ah_get_kernel(self._ctx)
        if k < 0:
            _check(k)
        return int(k)

    def launch_count(self) -> int:
        return int(lib().ah_launch_count(self._ctx))

    def synchronize(self):
        self.stream.synchronize()


def test_trig(x):
    """Evaluate the library's fp32 link sin/cos and plaquette sine on a torch cuda float32 tensor."""
    import torch

    assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()
    s, c, ps = torch.empty_like(x), torch.empty_like(x), torch.empty_like(x)
    with torch.cuda.device(x.device):
        st = torch.cuda.current_stream(x.device).cuda_stream
        _check(lib().ah_test_trig(x.data_ptr(), s.data_ptr(), c.data_ptr(), ps.data_ptr(), x.numel(), C.c_void_p(st)))
    return s, c, ps


def test_trig_fast(x):
    """The tiled kernel's own link sin/cos (pi-reduced polynomials) and small-angle sine on a cuda float32 tensor."""
    import torch

    assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()
    s, c, ss = torch.empty_like(x), torch.empty_like(x), torch.empty_like(x)
    with torch.cuda.device(x.device):
        st = torch.cuda.current_stream(x.device).cuda_stream
        _check(lib().ah_test_trig_fast(x.data_ptr(), s.data_ptr(), c.data_ptr(), ss.data_ptr(), x.numel(), C.c_void_p(st)))
    return s, c, ss
