"""Independent numpy restatements used ONLY to pin the oracle (tests, not gpu).

Written with whole-array np.roll arithmetic and complex numbers — a different
formulation from oracle/ah_oracle.c's per-site loops — so that a wrong sign,
index or factor in either one shows up as a disagreement.  Nothing here is
imported by the oracle or by the CUDA path.

Arrays have shape (nz, ny, nx); direction i = 0,1,2 (x,y,z) lives on axis 2-i.
"""
import numpy as np


def up(a, i):
    """a(x + k_i)"""
    return np.roll(a, -1, axis=2 - i)


def dn(a, i):
    """a(x - k_i)"""
    return np.roll(a, +1, axis=2 - i)


def unpack(f):
    phi = f[0] + 1j * f[1]
    Pi = f[2] + 1j * f[3]
    th = [f[4], f[5], f[6]]
    ep = [f[7], f[8], f[9]]
    return phi, Pi, th, ep


def plaquette(th, i, j):
    return th[i] + up(th[j], i) - up(th[i], j) - th[j]


def energy(f, dx, lambda0, e0, sigma, q=1.0, Pi=None, ep=None):
    """Total energy (a=1 form): sum dx^3 [ |Pi|^2 + |D+ phi|^2 + V + (E^2 + B^2)/(2 e0^2 q) ]."""
    phi, Pi0, th, ep0 = unpack(f)
    Pi = Pi0 if Pi is None else Pi
    ep = ep0 if ep is None else ep
    grad2 = sum(np.abs(np.exp(-1j * th[i]) * up(phi, i) - phi) ** 2 for i in range(3)) / dx**2
    pot = 0.25 * lambda0 * q * (np.abs(phi) ** 2 - sigma**2) ** 2
    e2 = sum(ep[i] ** 2 for i in range(3)) / dx**2
    b2 = sum(2.0 * (1.0 - np.cos(plaquette(th, i, j))) for i, j in ((0, 1), (0, 2), (1, 2))) / dx**4
    dens = np.abs(Pi) ** 2 + grad2 + pot + (e2 + b2) / (2.0 * e0**2 * q)
    return float(dens.sum() * dx**3)


def lagrangian_sums(f, dx, lambda0, e0, sigma, q):
    """Naive evaluation of sum |Pi|^2 L, sum (sum_i |D+_i phi|^2) L, sum L — term by term."""
    phi, Pi, th, ep = unpack(f)
    pi2 = Pi.real**2 + Pi.imag**2
    grad2 = np.zeros_like(pi2)
    for i in range(3):
        link = np.cos(th[i]) - 1j * np.sin(th[i])
        diff = link * up(phi, i) - phi
        grad2 = grad2 + (diff.real**2 + diff.imag**2) / dx**2
    pot = 0.25 * lambda0 * q * (phi.real**2 + phi.imag**2 - sigma**2) ** 2
    e2 = (ep[0] ** 2 + ep[1] ** 2 + ep[2] ** 2) / dx**2
    b2 = np.zeros_like(pi2)
    for i, j in ((0, 1), (0, 2), (1, 2)):
        b2 = b2 + 2.0 * (1.0 - np.cos(plaquette(th, i, j))) / dx**4
    L = pi2 - grad2 - pot + (e2 - b2) / (2.0 * e0**2 * q)
    return float((pi2 * L).sum()), float((grad2 * L).sum()), float(L.sum())


def gauss_residual(f, dx, e0, kappa):
    phi, Pi, th, ep = unpack(f)
    div = sum(ep[i] - dn(ep[i], i) for i in range(3)) / dx**2
    charge = 2.0 * e0**2 * kappa * (np.conj(phi) * Pi).imag
    return div - charge, div, charge


def winding_bruteforce(f):
    """Winding from explicit integer link shifts.

    Delta_i(x) = arg phi(x+i) - arg phi(x) - th_i(x); n_i(x) is the integer with
    Delta_i - 2 pi n_i in (-pi, pi].  Around a plaquette the Delta's sum to -Phi_ij exactly,
    so W_ij(x) = -( n_i(x) + n_j(x+i) - n_i(x+j) - n_j(x) ): pure integer arithmetic.
    """
    phi, _, th, _ = unpack(f)
    arg = np.angle(phi)
    n = []
    for i in range(3):
        delta = up(arg, i) - arg - th[i]
        n.append(np.ceil((delta - np.pi) / (2 * np.pi)).astype(np.int64))
    W = []
    for i, j in ((0, 1), (0, 2), (1, 2)):
        W.append(-(n[i] + up(n[j], i) - up(n[i], j) - n[j]))
    return np.stack(W)


def gauge_transform(f, chi):
    """phi -> e^{i chi} phi, Pi -> e^{i chi} Pi, th_i -> th_i + chi(x+i) - chi(x), ep unchanged."""
    g = f.copy()
    phi, Pi, th, ep = unpack(f)
    ph = np.exp(1j * chi)
    g[0], g[1] = (ph * phi).real, (ph * phi).imag
    g[2], g[3] = (ph * Pi).real, (ph * Pi).imag
    for i in range(3):
        g[4 + i] = th[i] + up(chi, i) - chi
    return g
