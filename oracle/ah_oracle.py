"""ORACLE binding (test infrastructure, NOT the product).

ctypes wrapper around oracle/ah_oracle.c (fp64, plain loops; see that file's
header for the citations).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports
nothing from paper_2005_14454_b200 and shares no code with the CUDA path.

Field block layout: numpy float64 array of shape (10, nz, ny, nx), x fastest, in
the order phi_re, phi_im, pi_re, pi_im, th_x, th_y, th_z, ep_x, ep_y, ep_z.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "ah_oracle.c"
_LIB = _HERE / "libah_oracle.so"

FIELD_NAMES = ("phi_re", "phi_im", "pi_re", "pi_im", "th_x", "th_y", "th_z", "ep_x", "ep_y", "ep_z")


class Params(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("dx", C.c_double),
        ("lambda0", C.c_double), ("e0", C.c_double), ("sigma", C.c_double),
        ("s", C.c_double), ("p", C.c_double), ("tau_ref", C.c_double), ("alpha", C.c_double),
        ("compact", C.c_int32),
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
    ]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (plain -O2, OpenMP on the outer z loop only)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", str(_LIB), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        dp = C.POINTER(C.c_double)
        L.ahref_num_threads.restype = C.c_int
        L.ahref_uniform.restype = C.c_double
        L.ahref_uniform.argtypes = [C.c_uint64, C.c_uint64]
        L.ahref_coeffs.restype = None
        L.ahref_coeffs.argtypes = [C.POINTER(Params), C.c_double, C.c_double, dp, dp, dp, dp]
        L.ahref_init_fields.argtypes = [C.POINTER(Params), C.c_uint64, C.c_void_p]
        L.ahref_step.argtypes = [C.POINTER(Params), C.c_void_p, C.c_int, C.c_double, C.c_double]
        L.ahref_diagnostics.argtypes = [C.POINTER(Params), C.c_void_p, C.c_double, C.c_double, C.POINTER(Diag)]
        L.ahref_winding.argtypes = [C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def make_params(nx, ny=None, nz=None, dx=0.5, lambda0=2.0, e0=1.0, sigma=1.0, s=0.0, p=1.0,
                tau_ref=1.0, alpha=2.0, compact=1) -> Params:
    ny = nx if ny is None else ny
    nz = nx if nz is None else nz
    return Params(int(nx), int(ny), int(nz), float(dx), float(lambda0), float(e0), float(sigma),
                  float(s), float(p), float(tau_ref), float(alpha), int(compact))


def num_threads() -> int:
    return int(lib().ahref_num_threads())


def uniform(seed: int, idx: int) -> float:
    return float(lib().ahref_uniform(C.c_uint64(seed), C.c_uint64(idx)))


def coeffs(P: Params, tau: float, dt: float):
    a, q, d, w = C.c_double(), C.c_double(), C.c_double(), C.c_double()
    lib().ahref_coeffs(C.byref(P), tau, dt, C.byref(a), C.byref(q), C.byref(d), C.byref(w))
    return a.value, q.value, d.value, w.value


def _check(P: Params, f: np.ndarray):
    assert f.dtype == np.float64 and f.flags["C_CONTIGUOUS"], "fields must be C-contiguous float64"
    assert f.shape == (10, P.nz, P.ny, P.nx), f"fields must have shape (10,{P.nz},{P.ny},{P.nx})"


def empty_fields(P: Params) -> np.ndarray:
    return np.zeros((10, P.nz, P.ny, P.nx), dtype=np.float64)


def init_fields(P: Params, seed: int) -> np.ndarray:
    f = empty_fields(P)
    rc = lib().ahref_init_fields(C.byref(P), C.c_uint64(seed), f.ctypes.data)
    assert rc == 0
    return f


def step(P: Params, f: np.ndarray, n: int, tau: float, dt: float) -> np.ndarray:
    """Advance f in place by n steps starting at tau (step j at tau + j*dt)."""
    _check(P, f)
    rc = lib().ahref_step(C.byref(P), f.ctypes.data, int(n), float(tau), float(dt))
    if rc != 0:
        raise ValueError("ahref_step: invalid arguments")
    return f


def diagnostics(P: Params, f: np.ndarray, tau: float, dt: float) -> dict:
    _check(P, f)
    d = Diag()
    rc = lib().ahref_diagnostics(C.byref(P), f.ctypes.data, float(tau), float(dt), C.byref(d))
    assert rc == 0
    return d.asdict()


def winding(P: Params, f: np.ndarray):
    """Per-plaquette winding integers W[3, nz, ny, nx] (xy, xz, yz) and near-branch flags."""
    _check(P, f)
    w = np.zeros((3, P.nz, P.ny, P.nx), dtype=np.int8)
    near = np.zeros((3, P.nz, P.ny, P.nx), dtype=np.uint8)
    rc = lib().ahref_winding(C.byref(P), f.ctypes.data, w.ctypes.data, near.ctypes.data)
    assert rc == 0
    return w, near
