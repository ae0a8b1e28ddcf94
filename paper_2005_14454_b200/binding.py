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
AH_NHALO, AH_NDIAG_INT, AH_NDIAG_FLT = 6, 5, 9
HALO_FIELDS = (0, 1, 4, 5, 6, 9)          # phi_re, phi_im, th_x, th_y, th_z, ep_z (include/ah_b200.h)
KERNEL_AUTO, KERNEL_SITE, KERNEL_TILED = 0, 1, 2
PRECISION_FP32, PRECISION_FP64, PRECISION_MIXED = 0, 1, 2

FIELD_NAMES = ("phi_re", "phi_im", "pi_re", "pi_im", "th_x", "th_y", "th_z", "ep_x", "ep_y", "ep_z")

# every symbol include/*.h declares (checked by tests/test_abi.py)
EXPORTS = (
    "ah_create_slab", "ah_slab_step", "ah_slab_halo_ptrs", "ah_slab_exchange_done", "ah_slab_diagnostics",
    "ah_slab_diag_partial", "ah_diag_finish", "ah_diag_combine", "ah_step_diag_sums", "ah_readout_noalloc",
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
        ("sum_p_L", C.c_double), ("sum_rho_L", C.c_double), ("v2_omega", C.c_double),
        ("xi_w_corr", C.c_double),
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
    L.ah_create_slab.argtypes = [C.POINTER(vp), C.POINTER(Params), ip, ip, C.POINTER(vp), ip, C.c_size_t, vp]
    L.ah_slab_step.argtypes = [vp, dp, dp, ip, vp]
    L.ah_slab_halo_ptrs.argtypes = [vp] + [C.POINTER(vp)] * 4 + [C.POINTER(C.c_size_t)]
    L.ah_slab_exchange_done.argtypes = [vp, vp]
    L.ah_slab_diagnostics.argtypes = [vp, dp, dp]
    L.ah_slab_diag_partial.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(dp)]
    L.ah_diag_finish.argtypes = [C.POINTER(Params), C.POINTER(C.c_int64), C.POINTER(dp), dp, C.POINTER(Diag)]
    L.ah_diag_combine.argtypes = [ip, C.POINTER(C.c_int64), C.POINTER(dp), C.POINTER(C.c_int64), C.POINTER(dp)]
    L.ah_readout_noalloc.argtypes = [C.POINTER(Params), C.POINTER(vp), dp, dp, vp, vp]
    L.ah_destroy.argtypes = [vp]
    L.ah_init_fields.argtypes = [vp, C.c_uint64]
    L.ah_set_fields.argtypes = [vp, vp]
    L.ah_get_fields.argtypes = [vp, vp]
    L.ah_current_bufs.argtypes = [vp, C.POINTER(vp)]
    L.ah_step.argtypes = [vp, ip, dp, dp]
    L.ah_step_cooling.argtypes = [vp, ip, dp, dp]
    L.ah_diagnostics.argtypes = [vp, dp, dp, C.POINTER(Diag)]
    L.ah_step_diag.argtypes = [vp, ip, dp, dp, ip, C.POINTER(Diag), ip, C.POINTER(ip)]
    L.ah_step_diag_sums.argtypes = [vp, ip, dp, dp, ip, C.POINTER(Diag), ip, C.POINTER(ip)]
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
    # fp64: False / True, or one of PRECISION_FP32 / PRECISION_FP64 / PRECISION_MIXED
    return Params(int(nx), int(ny), int(nz), float(dx), float(lambda0), float(e0), float(sigma),
                  float(s), float(p), float(tau_ref), float(alpha), int(compact), int(fp64))


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
        self.dtype = torch.float64 if P.fp64 == PRECISION_FP64 else torch.float32
        self.np_dtype = np.float64 if P.fp64 == PRECISION_FP64 else np.float32
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

    def step_diag(self, n: int, tau: float, dt: float, every: int, winding: bool = True):
        """ah_step_diag (winding=True) or ah_step_diag_sums (winding=False: no winding read-out in the records)."""
        cap = max(1, (n + every - 1) // every) if every >= 1 else 1
        recs = (Diag * cap)()
        nw = C.c_int(0)
        fn = lib().ah_step_diag if winding else lib().ah_step_diag_sums
        with self._dev():
            _check(fn(self._ctx, int(n), float(tau), float(dt), int(every), recs, cap, C.byref(nw)))
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


def diag_finish(P: Params, counts, sums, tau: float) -> dict:
    """ah_diag_finish: totals of a whole lattice -> the ah_diag record (host side of the library)."""
    ci = (C.c_int64 * AH_NDIAG_INT)(*[int(v) for v in counts])
    cf = (C.c_double * AH_NDIAG_FLT)(*[float(v) for v in sums])
    d = Diag()
    _check(lib().ah_diag_finish(C.byref(P), ci, cf, float(tau), C.byref(d)))
    return d.asdict()


NOALLOC_MAX_PARTIALS = 65536                 # AH_NOALLOC_MAX_PARTIALS: blocks of 64 x 4 x 8 sites (512^3 at most)
NOALLOC_TOTALS_WORDS = AH_NDIAG_INT + AH_NDIAG_FLT   # dev_totals: that many 8-byte words


def readout_noalloc(P: Params, dev_fields, tau: float, dt: float, dev_totals, stream=None):
    """ah_readout_noalloc: read-outs of the snapshot in the 10 device tensors dev_fields, for callers that may not
    allocate (see include/ah_b200.h): no context, no cudaMalloc; the partial sums use the library's fixed device array
    (shared by all calls on a device: keep them on one stream).  dev_totals is the caller's own device tensor of
    NOALLOC_TOTALS_WORDS int64; it receives the raw totals asynchronously on `stream` (default: torch's current one).
    Nothing is allocated here either: turn the totals into a record later with noalloc_totals_to_diag."""
    import torch

    if len(dev_fields) != AH_NFIELDS:
        raise ValueError(f"need {AH_NFIELDS} field tensors")
    if dev_totals.dtype != torch.int64 or dev_totals.numel() < NOALLOC_TOTALS_WORDS or not dev_totals.is_cuda:
        raise ValueError(f"dev_totals must be a CUDA int64 tensor of {NOALLOC_TOTALS_WORDS} elements")
    st = stream if stream is not None else torch.cuda.current_stream(dev_totals.device)
    ptrs = (C.c_void_p * AH_NFIELDS)(*[t.data_ptr() for t in dev_fields])
    with torch.cuda.device(dev_totals.device):
        _check(lib().ah_readout_noalloc(C.byref(P), ptrs, float(tau), float(dt), C.c_void_p(dev_totals.data_ptr()),
                                        C.c_void_p(st.cuda_stream)))


def noalloc_totals_to_diag(P: Params, host_totals, tau: float) -> dict:
    """The 14 words ah_readout_noalloc left in dev_totals, copied to the host (numpy int64), -> the ah_diag record
    (ah_diag_finish).  Words 0..4 are the int64 counts, words 5..13 hold the bit patterns of the double sums."""
    a = np.ascontiguousarray(host_totals, dtype=np.int64)
    return diag_finish(P, a[:AH_NDIAG_INT], a[AH_NDIAG_INT:NOALLOC_TOTALS_WORDS].view(np.float64), tau)


def slab_planes(nz: int, nslabs: int, r: int):
    """(first own plane, number of own planes) of slab r when nz planes are cut into nslabs nearly equal slabs."""
    if not (1 <= nslabs <= nz and 0 <= r < nslabs):
        raise ValueError("need 1 <= nslabs <= nz and 0 <= r < nslabs")
    base, rem = divmod(nz, nslabs)
    first = r * base + min(r, rem)
    return first, base + (1 if r < rem else 0)


class SlabSimulation:
    """One z slab of a periodic lattice (ah_create_slab): own planes [z_first, z_first + nz_own) plus one ghost plane
    on each side, 20 torch-owned buffers of nx*ny*(nz_own+2) elements.  Marshalling and stream plumbing only; the
    exchange of the boundary planes is done by a SlabGroup (slabs of one process) or a DistributedSlab (one slab per
    rank, torch.distributed)."""

    def __init__(self, params: Params, nz_own: int, z_first: int, device="cuda:0", stream=None, comm_stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2005_14454_b200 needs a CUDA device (B200); there is no CPU fallback")
        self.P, self.nz_own, self.z_first = params, int(nz_own), int(z_first)
        P = params
        self.torch = torch
        self.device = torch.device(device)
        self.dtype = torch.float64 if P.fp64 == PRECISION_FP64 else torch.float32
        self.np_dtype = np.float64 if P.fp64 == PRECISION_FP64 else np.float32
        self.nza = self.nz_own + 2
        self.n = P.nx * P.ny * self.nza
        self.shape = (AH_NFIELDS, self.nza, P.ny, P.nx)
        with torch.cuda.device(self.device):
            self.bufs = [torch.empty(self.n, dtype=self.dtype, device=self.device) for _ in range(2 * AH_NFIELDS)]
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.comm_stream = comm_stream if comm_stream is not None else self.stream
            ptrs = (C.c_void_p * (2 * AH_NFIELDS))(*[b.data_ptr() for b in self.bufs])
            self._ctx = C.c_void_p()
            _check(lib().ah_create_slab(C.byref(self._ctx), C.byref(P), self.nz_own, self.z_first, ptrs, 2 * AH_NFIELDS,
                                        self.n * self.bufs[0].element_size(), C.c_void_p(self.stream.cuda_stream)))

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

    def _dev(self):
        return self.torch.cuda.device(self.device)

    def init_fields(self, seed: int):
        with self._dev():
            _check(lib().ah_init_fields(self._ctx, C.c_uint64(seed)))

    def set_fields(self, host):
        a = np.ascontiguousarray(host, dtype=self.np_dtype)
        if a.shape != self.shape:
            raise ValueError(f"fields must have shape {self.shape}, got {a.shape}")
        with self._dev():
            _check(lib().ah_set_fields(self._ctx, a.ctypes.data))

    def get_fields(self) -> np.ndarray:
        out = np.empty(self.shape, dtype=self.np_dtype)
        with self._dev():
            _check(lib().ah_get_fields(self._ctx, out.ctypes.data))
        return out

    def step(self, tau: float, dt: float, want_diag: bool = False):
        with self._dev():
            _check(lib().ah_slab_step(self._ctx, float(tau), float(dt), int(bool(want_diag)),
                                      C.c_void_p(self.comm_stream.cuda_stream)))

    def halo_planes(self):
        """(send_lo, send_hi, recv_lo, recv_hi): four lists of AH_NHALO torch views (one plane each) into the buffers
        of the current state, found from the device pointers ah_slab_halo_ptrs returns."""
        arrs = [(C.c_void_p * AH_NHALO)() for _ in range(4)]
        nbytes = C.c_size_t(0)
        _check(lib().ah_slab_halo_ptrs(self._ctx, *arrs, C.byref(nbytes)))
        by_ptr = {b.data_ptr(): b for b in self.bufs}
        plane = self.P.nx * self.P.ny
        es = self.bufs[0].element_size()
        assert nbytes.value == plane * es
        out = []
        for arr in arrs:
            views = []
            for p in arr:
                base = max(q for q in by_ptr if q <= p)          # the buffer this plane lies in
                off = (p - base) // es
                views.append(by_ptr[base][off:off + plane])
            out.append(views)
        return out

    def exchange_done(self):
        with self._dev():
            _check(lib().ah_slab_exchange_done(self._ctx, C.c_void_p(self.comm_stream.cuda_stream)))

    def diagnostics_partial(self, tau: float, dt: float):
        with self._dev():
            _check(lib().ah_slab_diagnostics(self._ctx, float(tau), float(dt)))
        return self.diag_partial()

    def diag_partial(self):
        ci = (C.c_int64 * AH_NDIAG_INT)()
        cf = (C.c_double * AH_NDIAG_FLT)()
        with self._dev():
            _check(lib().ah_slab_diag_partial(self._ctx, ci, cf))
        return list(ci), list(cf)

    def launch_count(self) -> int:
        return int(lib().ah_launch_count(self._ctx))

    def get_kernel(self) -> int:
        return int(lib().ah_get_kernel(self._ctx))


def combine_partials(parts):
    """ah_diag_combine: totals of per-slab (counts, sums) — marshalling only, the adding is done behind the C ABI."""
    n = len(parts)
    ci = (C.c_int64 * (AH_NDIAG_INT * n))(*[int(v) for p in parts for v in p[0]])
    cf = (C.c_double * (AH_NDIAG_FLT * n))(*[float(v) for p in parts for v in p[1]])
    co, so = (C.c_int64 * AH_NDIAG_INT)(), (C.c_double * AH_NDIAG_FLT)()
    _check(lib().ah_diag_combine(n, ci, cf, co, so))
    return list(co), list(so)


class SlabGroup:
    """All slabs of one lattice in ONE process (one GPU, or several GPUs of one process): the boundary planes are
    exchanged by device-to-device copies on each slab's comm stream.  This is how the multi-GPU path is exercised
    with a single GPU: the slabs' kernels are launched one after the other and never wait on one another."""

    def __init__(self, params: Params, nslabs: int, devices=None, overlap=True):
        import torch

        self.P = params
        devices = devices or ["cuda:0"] * nslabs
        self.slabs = []
        for r in range(nslabs):
            first, own = slab_planes(params.nz, nslabs, r)
            with torch.cuda.device(devices[r]):
                comm = torch.cuda.Stream(device=devices[r]) if overlap else None
            self.slabs.append(SlabSimulation(params, own, first, device=devices[r], comm_stream=comm))
        self.torch = torch

    def close(self):
        for s in self.slabs:
            s.close()

    def init_fields(self, seed: int):
        for s in self.slabs:
            s.init_fields(seed)

    def set_fields(self, host):
        """host: the whole lattice (10, nz, ny, nx); every slab gets its own planes and its two ghost planes."""
        nz = self.P.nz
        for s in self.slabs:
            idx = [(s.z_first - 1 + k) % nz for k in range(s.nza)]
            s.set_fields(np.ascontiguousarray(np.asarray(host)[:, idx]))

    def get_fields(self) -> np.ndarray:
        out = np.empty((AH_NFIELDS, self.P.nz, self.P.ny, self.P.nx), dtype=self.slabs[0].np_dtype)
        for s in self.slabs:
            out[:, s.z_first:s.z_first + s.nz_own] = s.get_fields()[:, 1:-1]
        return out

    def _exchange(self):
        R = len(self.slabs)
        planes = [s.halo_planes() for s in self.slabs]
        for r, s in enumerate(self.slabs):
            lo, hi = (r - 1) % R, (r + 1) % R
            with self.torch.cuda.stream(s.comm_stream):
                # the copies run on the SENDER's comm stream (it waits for the sender's boundary planes); the
                # receiver's compute stream is made to wait for them in exchange_done below
                for a in range(AH_NHALO):
                    planes[lo][3][a].copy_(planes[r][0][a], non_blocking=True)     # my first own plane -> lower's upper ghost
                    planes[hi][2][a].copy_(planes[r][1][a], non_blocking=True)     # my last own plane  -> upper's lower ghost
        # a slab's next step must see the ghost planes its neighbours wrote: wait on their comm streams too
        for r, s in enumerate(self.slabs):
            for nb in {(r - 1) % R, (r + 1) % R, r}:
                ev = self.torch.cuda.Event()
                ev.record(self.slabs[nb].comm_stream)
                s.stream.wait_event(ev)
            s.exchange_done()

    def step(self, n: int, tau: float, dt: float, diag_every: int = 0):
        """n steps; diag_every > 0 returns the records of the entry snapshots of steps 0, diag_every, ..."""
        recs = []
        for j in range(n):
            tj = tau + j * dt
            want = diag_every > 0 and j % diag_every == 0
            # a slab's step reads its ghost planes, which the neighbours' comm streams wrote: ordering is in _exchange
            for s in self.slabs:
                s.step(tj, dt, want)
            if want:
                counts, sums = combine_partials([s.diag_partial() for s in self.slabs])
                recs.append(diag_finish(self.P, counts, sums, tj))
            self._exchange()
        return recs

    def diagnostics(self, tau: float, dt: float) -> dict:
        counts, sums = combine_partials([s.diagnostics_partial(tau, dt) for s in self.slabs])
        return diag_finish(self.P, counts, sums, tau)


def halo_schedule(rank: int, world: int):
    """Point-to-point operations of one boundary exchange for `rank` of `world` slabs (periodic in z), per exchanged
    field: (kind, which plane list of SlabSimulation.halo_planes(), peer).  plane lists: 0 send_lo (first own plane),
    1 send_hi (last own plane), 2 recv_lo (ghost below), 3 recv_hi (ghost above).  My first own plane is my lower
    neighbour's upper ghost; my last own plane is my upper neighbour's lower ghost.  The order pairs every send with the
    receive the peer posts at the same position (a rank's "send down / receive from above" meets the neighbour's),
    so the schedule also works with blocking transports."""
    if not (world >= 1 and 0 <= rank < world):
        raise ValueError("need world >= 1 and 0 <= rank < world")
    lo, hi = (rank - 1) % world, (rank + 1) % world
    return [("send", 0, lo), ("recv", 3, hi), ("send", 1, hi), ("recv", 2, lo)]


class DistributedSlab:
    """One slab per rank (one process per GPU): boundary planes travel by torch.distributed point-to-point calls
    (NCCL over NVLink on GPUs) on the comm stream, overlapped with the update of the interior; read-outs are combined
    by two all-reduces (sum, max).  Host plumbing only."""

    def __init__(self, params: Params, dist, device="cuda:0", overlap=True):
        import torch

        self.P, self.dist, self.torch = params, dist, torch
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        first, own = slab_planes(params.nz, self.world, self.rank)
        with torch.cuda.device(device):
            comm = torch.cuda.Stream(device=device) if overlap else None
        self.slab = SlabSimulation(params, own, first, device=device, comm_stream=comm)

    def exchange_ops(self, planes):
        """The 4 * AH_NHALO point-to-point operations of one exchange, as (kind, tensor, peer) tuples; with world == 1
        the slab is its own neighbour and the list is empty (plain copies are used instead)."""
        ops = []
        for a in range(AH_NHALO):
            ops += [(kind, planes[which][a], peer) for kind, which, peer in halo_schedule(self.rank, self.world)]
        return ops if self.world > 1 else []

    def _exchange(self):
        s, dist = self.slab, self.dist
        planes = s.halo_planes()
        with self.torch.cuda.stream(s.comm_stream):
            if self.world == 1:
                for a in range(AH_NHALO):
                    planes[3][a].copy_(planes[0][a], non_blocking=True)
                    planes[2][a].copy_(planes[1][a], non_blocking=True)
            else:
                reqs = dist.batch_isend_irecv([dist.P2POp(dist.isend if k == "send" else dist.irecv, t, peer)
                                               for k, t, peer in self.exchange_ops(planes)])
                for r in reqs:
                    r.wait()
        s.exchange_done()

    def step(self, n: int, tau: float, dt: float, diag_every: int = 0):
        recs = []
        for j in range(n):
            tj = tau + j * dt
            want = diag_every > 0 and j % diag_every == 0
            self.slab.step(tj, dt, want)
            if want:
                recs.append(self._reduce(self.slab.diag_partial(), tj))
            self._exchange()
        return recs

    def _reduce(self, part, tau):
        torch, dist = self.torch, self.dist
        counts, sums = part
        dev = self.slab.device if dist.get_backend() == "nccl" else "cpu"
        add = torch.tensor([float(c) for c in counts] + sums[:-1], dtype=torch.float64, device=dev)   # counts < 2^53
        mx = torch.tensor([sums[-1]], dtype=torch.float64, device=dev)
        if self.world > 1:
            dist.all_reduce(add, op=dist.ReduceOp.SUM)
            dist.all_reduce(mx, op=dist.ReduceOp.MAX)
        add = add.tolist()
        return diag_finish(self.P, [int(round(v)) for v in add[:AH_NDIAG_INT]], add[AH_NDIAG_INT:] + [float(mx.item())], tau)

    def diagnostics(self, tau: float, dt: float) -> dict:
        return self._reduce(self.slab.diagnostics_partial(tau, dt), tau)


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
