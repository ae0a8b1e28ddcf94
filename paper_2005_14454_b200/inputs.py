"""Seeded synthetic input generators shared by the oracle tests and the CUDA tests.

This module holds NONE of the method's arithmetic (no link variables, no stencils,
no coefficients): it only draws seeded random / smooth arrays with numpy.  Both
sides consume its output: the oracle as float64, the CUDA path after a cast to
float32.  The paper's own initial condition (random phase) is part
of the method (step I0) and is implemented independently on each side from the
counter-based generator specified in DESIGN.md; it is not generated here.

Field block layout everywhere: (10, nz, ny, nx), x fastest, order
phi_re, phi_im, pi_re, pi_im, th_x, th_y, th_z, ep_x, ep_y, ep_z.
"""
from __future__ import annotations

import numpy as np

FIELD_NAMES = ("phi_re", "phi_im", "pi_re", "pi_im", "th_x", "th_y", "th_z", "ep_x", "ep_y", "ep_z")


def random_state(nx, ny, nz, seed, phi_amp=1.0, pi_amp=0.3, th_amp=0.5, ep_amp=0.3,
                 round_to_f32=True):
    """Generic dense random state: every field non-zero so every term of the step is exercised.

    With round_to_f32 the values are exactly representable in float32, so the fp64
    oracle and the fp32 CUDA path start from bit-identical numbers.
    """
    rng = np.random.default_rng(seed)
    f = np.empty((10, nz, ny, nx), dtype=np.float64)
    f[0:2] = phi_amp * rng.standard_normal((2, nz, ny, nx))
    f[2:4] = pi_amp * rng.standard_normal((2, nz, ny, nx))
    f[4:7] = th_amp * rng.standard_normal((3, nz, ny, nx))
    f[7:10] = ep_amp * rng.standard_normal((3, nz, ny, nx))
    if round_to_f32:
        f = f.astype(np.float32).astype(np.float64)
    return f


def smooth_state(nx, ny, nz, seed, nmodes=12, kmax=2, phi_amp=0.6, th_amp=0.3, round_to_f32=False):
    """Smooth state made of a dozen low-k Fourier modes, |phi| <= ~sigma, zero momenta."""
    rng = np.random.default_rng(seed)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    f = np.zeros((10, nz, ny, nx), dtype=np.float64)
    for comp in (0, 1, 4, 5, 6):
        amp = phi_amp if comp < 2 else th_amp
        acc = np.zeros((nz, ny, nx))
        for _ in range(nmodes):
            k = rng.integers(-kmax, kmax + 1, size=3)
            ph = rng.uniform(0, 2 * np.pi)
            acc += rng.standard_normal() * np.cos(
                2 * np.pi * (k[0] * x / nx + k[1] * y / ny + k[2] * z / nz) + ph)
        f[comp] = amp * acc / np.sqrt(nmodes)
    f[0] += 0.5  # keep phi away from zero on average
    if round_to_f32:
        f = f.astype(np.float32).astype(np.float64)
    return f


def random_gauge_function(nx, ny, nz, seed, amp=20.0):
    """chi(x) uniform in [-amp, amp] (large transforms included)."""
    rng = np.random.default_rng(seed)
    return rng.uniform(-amp, amp, size=(nz, ny, nx))
