"""Pins for the oracle from closed forms and independent formulations (CPU only).

 * Plane-wave dispersion on the vacuum (Higgs mode, transverse gauge mode): exact
   solution of the linearised discrete equations, m^2 = lambda0 sigma^2 resp.
   2 e0^2 sigma^2 (beta = 1) — fixes every dx and dt factor of Eqs. 7-10, 12-15.
 * Leapfrog is O(dt^2): time-centred Minkowski energy, written
   independently in numpy (tests/indep.py), oscillates ∝ dt^2 without drift.
 * Vortex-antivortex pair: relaxes to a static solution with windings {+1,-1},
   energy -> 2 mu L_z with mu = 2 pi sigma^2 at O(dx^2), <v^2> = 0.
 * Winding (Eq. 16): brute-force integer formulation, flux
   conservation, zero net flux through periodic planes, 1/3 density for random phases.
 * Lagrangian-weighted sums (Eqs. 17-18): naive numpy evaluation, and CLOSED FORMS on
   uniform states (every |Pi|^2, ep^2, potential, gradient and plaquette term of L_x fixed by arithmetic,
   <v^2>_phi = 2R/(1+R) away from its static limit).
"""
import numpy as np
import pytest

from tests import indep
from paper_2005_14454_b200 import inputs


# ------------------------------------------------------------------ dispersion

def _omega_hat(kvec, dx, dt, m2):
    lap = sum(4.0 / dx**2 * np.sin(0.5 * k * dx) ** 2 for k in kvec)
    return 2.0 / dt * np.arcsin(0.5 * dt * np.sqrt(lap + m2))


def test_dispersion_closed_form_value():
    """The helper itself: k = (1,2,0)·2π/8, dx=.5, dt=.1, m²=2 gives 2.229951 (continuum 2.254828)."""
    k = 2 * np.pi / 8.0 * np.array([1, 2, 0])
    assert np.sqrt((k**2).sum() + 2.0) == pytest.approx(2.254828, abs=1e-6)
    assert _omega_hat(k, 0.5, 0.1, 2.0) == pytest.approx(2.229951, abs=1e-6)


@pytest.mark.parametrize("mode", ["higgs", "gauge"])
def test_plane_wave_dispersion(oracle, mode):
    o = oracle
    nx, ny, nz, dx, dt, nsteps, amp = 8, 8, 4, 0.5, 0.1, 200, 1e-7
    lam, e0, sig = 2.0, 1.0, 1.0
    P = o.make_params(nx, ny, nz, dx=dx, lambda0=lam, e0=e0, sigma=sig, p=0.0, s=0.0)
    kvec = 2 * np.pi / (np.array([nx, ny, nz]) * dx) * np.array([1, 2, 0])
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    kx = (kvec[0] * x + kvec[1] * y + kvec[2] * z) * dx
    m2 = lam * sig**2 if mode == "higgs" else 2 * e0**2 * sig**2
    w = _omega_hat(kvec, dx, dt, m2)

    def wave(t):
        return amp * np.cos(kx - w * t)

    f = o.empty_fields(P)
    f[0] = sig
    comp, mom = (0, 2) if mode == "higgs" else (6, 9)     # gauge: polarisation z ⟂ k
    f[comp] += wave(0.0)
    f[mom] = (wave(0.0) - wave(-dt)) / dt                  # exact half-step momentum
    o.step(P, f, nsteps, 1.0, dt)
    got = f[comp] - (sig if mode == "higgs" else 0.0)
    err = np.abs(got - wave(nsteps * dt)).max() / amp
    assert err < (5e-6 if mode == "higgs" else 1e-9)       # Higgs: O(amp) nonlinearity
    # a wrong mass (factor 2 in the current or the potential) dephases by O(1)
    w_bad = _omega_hat(kvec, dx, dt, 2 * m2)
    assert np.abs(got - amp * np.cos(kx - w_bad * nsteps * dt)).max() / amp > 0.1


# ---------------------------------------------------------------------- energy

def _centred_energy_track(o, P, f, nsteps, dt):
    E = []
    for _ in range(nsteps):
        pi_old, ep_old = f[2:4].copy(), f[7:10].copy()
        g = f.copy()
        o.step(P, g, 1, 1.0, dt)
        Pi_c = 0.5 * ((pi_old[0] + g[2]) + 1j * (pi_old[1] + g[3]))
        ep_c = [0.5 * (ep_old[i] + g[7 + i]) for i in range(3)]
        E.append(indep.energy(f, P.dx, P.lambda0, P.e0, P.sigma, 1.0, Pi=Pi_c, ep=ep_c))
        f[...] = g
    return np.array(E)


def test_minkowski_energy_second_order(oracle):
    o = oracle
    n = 12
    P = o.make_params(n, dx=0.5, p=0.0, s=0.0)
    dev = []
    for dt in (0.1, 0.05, 0.025):
        f = inputs.smooth_state(n, n, n, seed=4)
        E = _centred_energy_track(o, P, f, int(round(8.0 / dt)), dt)
        dev.append(np.abs(E / E[0] - 1).max())
        # no secular drift: last quarter's mean equals first quarter's mean to within the oscillation
        q4 = len(E) // 4
        assert abs(E[-q4:].mean() - E[:q4].mean()) / E[0] < dev[-1]
    assert dev[0] < 2e-2
    assert 3.0 < dev[0] / dev[1] < 5.0
    assert 3.0 < dev[1] / dev[2] < 5.0


# ----------------------------------------------------------------- vortex pair

def _vortex_pair(o, nxy, dx, relax_steps):
    P_relax = o.make_params(nxy, nxy, 1, dx=dx, p=1.0, s=0.0)   # delta = omega = dt/tau, q = 1
    f = o.empty_fields(P_relax)
    y, x = np.meshgrid(np.arange(nxy), np.arange(nxy), indexing="ij")
    c1 = (nxy / 4 + 0.5, nxy / 2 + 0.5)
    c2 = (3 * nxy / 4 + 0.5, nxy / 2 + 0.5)
    r1 = np.hypot(x - c1[0], y - c1[1]) * dx
    r2 = np.hypot(x - c2[0], y - c2[1]) * dx
    a1 = np.arctan2(y - c1[1], x - c1[0])
    a2 = np.arctan2(y - c2[1], x - c2[0])
    phi = np.tanh(r1 / 1.2) * np.tanh(r2 / 1.2) * np.exp(1j * (a1 - a2))
    f[0, 0], f[1, 0] = phi.real, phi.imag
    dt = 0.2 * dx
    delta = 0.15
    for _ in range(relax_steps):
        o.step(P_relax, f, 1, dt / delta, dt)                    # constant damping
    return f, dt


def _pair_energy(o, nxy, dx, relax_steps):
    f, dt = _vortex_pair(o, nxy, dx, relax_steps)
    P = o.make_params(nxy, nxy, 1, dx=dx, p=0.0, s=0.0)
    d = o.diagnostics(P, f, 1.0, dt)
    return P, f, dt, d


def test_vortex_pair_static_and_tension(oracle):
    o = oracle
    P, f, dt, d = _pair_energy(o, 48, 0.5, 3000)
    w, near = o.winding(P, f)
    assert sorted(w[0].ravel()[w[0].ravel() != 0].tolist()) == [-1, 1]
    assert not w[1].any() and not w[2].any()
    assert d["n_wind"] == 2 and d["n_wind_xy"] == 2 and d["n_near_branch"] == 0 and d["n_big_plaq"] == 0
    assert d["string_length"] == pytest.approx(2 * 0.5)
    assert d["xi_w"] == pytest.approx(np.sqrt(48 * 48 * 0.5**3 / 1.0))
    # relaxed: momenta tiny, Gauss holds, v^2 = 0
    eps_relax = max(np.abs(f[2:4]).max(), np.abs(f[7:10]).max())
    assert eps_relax < 1e-5
    assert d["gauss_max"] < 1e-12
    assert d["v2_phi"] < 1e-8
    # energy = -sum L dx^3 = 2 mu Lz (1 - O(dx^2)), mu = 2 pi sigma^2
    mu, Lz = 2 * np.pi, 0.5
    deficit_coarse = 1 - (-d["sum_L"] * 0.5**3) / (2 * mu * Lz)
    assert 0.005 < deficit_coarse < 0.02
    # Eq. 16 left: xi_L = sqrt(-mu V / int L) must agree with the winding estimator for two straight strings of
    # length Lz (the paper finds the two "fully consistent"), up to the same O(dx^2) deficit
    assert d["xi_l"] == pytest.approx(np.sqrt(mu * 48 * 48 * 0.5**3 / (-d["sum_L"] * 0.5**3)), rel=1e-12)
    assert d["xi_l"] == pytest.approx(d["xi_w"] * (1 + 0.5 * deficit_coarse), rel=1e-3)
    # energy from the independent numpy expression agrees
    assert indep.energy(f, 0.5, 2.0, 1.0, 1.0) == pytest.approx(-d["sum_L"] * 0.5**3, rel=1e-6)
    # stays static under undamped Minkowski evolution
    g = f.copy()
    o.step(P, g, 100, 1.0, dt)
    assert np.abs(g[0:2] - f[0:2]).max() < 1e-3
    w2, _ = o.winding(P, g)
    assert np.array_equal(w, w2)


def test_vortex_pair_tension_converges_second_order(oracle):
    o = oracle
    mu = 2 * np.pi
    _, _, _, d1 = _pair_energy(o, 32, 0.5, 2500)
    _, _, _, d2 = _pair_energy(o, 64, 0.25, 5000)
    def1 = 1 - (-d1["sum_L"] * 0.5**3) / (2 * mu * 0.5)
    def2 = 1 - (-d2["sum_L"] * 0.25**3) / (2 * mu * 0.25)
    assert 0 < def2 < def1
    assert 3.0 < def1 / def2 < 5.5


# --------------------------------------------------------------------- winding

@pytest.mark.parametrize("shape", [(4, 4, 4), (6, 5, 4), (8, 8, 8), (7, 3, 5)])
def test_winding_bruteforce(oracle, shape):
    o = oracle
    nx, ny, nz = shape
    P = o.make_params(nx, ny, nz)
    for seed in range(3):
        f = inputs.random_state(nx, ny, nz, seed=100 + seed, th_amp=0.4, round_to_f32=False)
        w, near = o.winding(P, f)
        wb = indep.winding_bruteforce(f)
        assert near.sum() == 0
        assert np.array_equal(w.astype(np.int64), wb)
        assert np.abs(w).sum() > 0
        d = o.diagnostics(P, f, 1.0, 0.1)
        assert d["n_wind"] == np.abs(wb).sum()
        assert (d["n_wind_xy"], d["n_wind_xz"], d["n_wind_yz"]) == tuple(np.abs(wb[k]).sum() for k in range(3))


@pytest.mark.parametrize("shape", [(4, 4, 4), (6, 5, 4), (8, 8, 8)])
def test_winding_bruteforce_large_plaquette_angles(oracle, shape):
    """Reading #13 (un-wrapped Phi_ij in Eq. 16 right): with link angles of order 1.5 rad many
    plaquettes have |Phi| > pi, where the `+ Phi` term decides the integer.  The brute-force formulation never
    forms Phi at all (pure integer link shifts), so dropping or wrapping the term in the oracle fails here."""
    o = oracle
    nx, ny, nz = shape
    P = o.make_params(nx, ny, nz)
    n_big = 0
    for seed in range(3):
        f = inputs.random_state(nx, ny, nz, seed=300 + seed, th_amp=1.6, round_to_f32=False)
        th = [f[4], f[5], f[6]]
        Phi = np.stack([indep.plaquette(th, i, j) for i, j in ((0, 1), (0, 2), (1, 2))])
        big = np.abs(Phi) > np.pi
        assert big.sum() > 0.1 * big.size          # the branch is really exercised
        w, near = o.winding(P, f)
        wb = indep.winding_bruteforce(f)
        ok = near == 0
        assert np.array_equal(w.astype(np.int64)[ok], wb[ok])
        assert ok.mean() > 0.999
        # the term matters: without it the integers differ on the big plaquettes
        assert np.abs(wb[big & ok]).sum() > 0
        d = o.diagnostics(P, f, 1.0, 0.1)
        assert d["n_big_plaq"] == (np.abs(Phi) > np.pi - 1e-5).sum()
        assert abs(d["n_wind"] - np.abs(wb).sum()) <= (~ok).sum()
        n_big += int(big.sum())
    assert n_big > 0


def test_winding_flux_conservation_and_planes(oracle):
    o = oracle
    n = 16
    P = o.make_params(n, dx=0.5, p=1.0, s=0.0)
    f = o.init_fields(P, seed=7)
    o.step(P, f, 25, 1.0, 0.1)
    w, _ = o.winding(P, f)
    w = w.astype(np.int64)
    wxy, wxz, wyz = w
    up = indep.up
    div = (up(wxy, 2) - wxy) + (up(wyz, 0) - wyz) - (up(wxz, 1) - wxz)
    assert not div.any()
    assert np.abs(w).sum() > 50
    assert not wxy.sum(axis=(1, 2)).any()     # each z-plane
    assert not wxz.sum(axis=(0, 2)).any()     # each y-plane
    assert not wyz.sum(axis=(0, 1)).any()     # each x-plane


def test_winding_random_phase_density(oracle):
    o = oracle
    n = 32
    P = o.make_params(n)
    f = o.init_fields(P, seed=1)
    d = o.diagnostics(P, f, 1.0, 0.1)
    frac = d["n_wind"] / (3 * n**3)
    assert abs(frac - 1 / 3) < 4 * np.sqrt((1 / 3) * (2 / 3) / (3 * n**3)) * 2


def test_winding_near_branch_flag(oracle):
    o = oracle
    P = o.make_params(4)
    f = o.empty_fields(P)
    f[0] = 1.0
    f[0, 1, 2, 3] = -1.0                      # phase difference exactly pi on its 6 links
    d = o.diagnostics(P, f, 1.0, 0.1)
    assert d["n_near_branch"] == 12           # the 12 plaquettes that have this site as a corner
    f[4] = 3.2                                # |Phi| stays 0 for uniform theta
    assert o.diagnostics(P, f, 1.0, 0.1)["n_big_plaq"] == 0
    f[4, 0, 0, 0] = 0.0
    assert o.diagnostics(P, f, 1.0, 0.1)["n_big_plaq"] > 0


# -------------------------------------------------------------------- <v^2>_phi

@pytest.mark.parametrize("case", [dict(p=0.0, s=0.0), dict(p=1.0, s=1.0, tau_ref=3.0), dict(p=2.0, s=0.5, tau_ref=2.0)])
def test_lagrangian_sums_naive(oracle, case):
    o = oracle
    P = o.make_params(6, 5, 4, dx=0.5, lambda0=1.7, e0=0.8, sigma=1.1, **case)
    f = inputs.random_state(6, 5, 4, seed=21, round_to_f32=False)
    tau, dt = 1.7, 0.1
    a, q, dl, om = o.coeffs(P, tau, dt)
    d = o.diagnostics(P, f, tau, dt)
    s_pi, s_gr, s_L = indep.lagrangian_sums(f, P.dx, P.lambda0, P.e0, P.sigma, q)
    assert d["sum_pi2_L"] == pytest.approx(s_pi, rel=1e-11)
    assert d["sum_grad2_L"] == pytest.approx(s_gr, rel=1e-11)
    assert d["sum_L"] == pytest.approx(s_L, rel=1e-11)
    R = s_pi / s_gr
    assert d["v2_phi"] == pytest.approx(2 * R / (1 + R), rel=1e-11)
    # Gauss residual of a generic (non-constraint-satisfying) state vs the numpy form
    G, div, ch = indep.gauss_residual(f, P.dx, P.e0, q * (1 - dl) / (1 - om))
    assert d["gauss_max"] == pytest.approx(np.abs(G).max(), rel=1e-12)
    assert d["gauss_l2"] == pytest.approx(np.sqrt((G**2).sum()), rel=1e-12)
    assert d["gauss_rel"] == pytest.approx(
        np.sqrt((G**2).sum()) / (np.sqrt((div**2).sum()) + np.sqrt((ch**2).sum())), rel=1e-12)


# ------------------------------------------------- closed forms for the Lagrangian density (reading #15)

UNIFORM_MODELS = [dict(p=1.0, s=1.0, tau_ref=3.0), dict(p=2.0, s=0.5, tau_ref=2.0), dict(p=0.0, s=0.0)]


@pytest.mark.parametrize("model", UNIFORM_MODELS)
def test_lagrangian_closed_form_uniform_state(oracle, model):
    """phi = rho e^{i beta}, th_i = t_i, Pi = c, ep_i = e_i, all uniform in space (Eqs. 17-18):
    every plaquette angle vanishes, U_i phi(x+i) - phi = (e^{-i t_i} - 1) phi, so per site

        |Pi|^2 = |c|^2,   sum_i |D_i phi|^2 = sum_i 2 (1 - cos t_i) rho^2 / dx^2,
        L = |c|^2 - sum_i|D_i phi|^2 - (lambda0 q / 4)(rho^2 - sigma^2)^2 + sum_i e_i^2 / (2 e0^2 q dx^2),

    with q = a^{2s} != 1.  Pins sign and factor of the kinetic, electric, potential and gradient terms and
    <v^2>_phi = 2R/(1+R), R = |c|^2 / sum_i|D_i phi|^2, away from the static limit."""
    o = oracle
    nx, ny, nz = 5, 4, 3
    dx, lam, e0, sig = 0.5, 1.7, 0.8, 1.1
    P = o.make_params(nx, ny, nz, dx=dx, lambda0=lam, e0=e0, sigma=sig, **model)
    tau, dt = 1.7, 0.1
    _, q, _, _ = o.coeffs(P, tau, dt)
    if model["s"] != 0.0:
        assert abs(q - 1.0) > 0.1
    rho, beta = 0.9, 0.4
    t = (0.3, -0.7, 1.9)
    c = 0.35 - 0.2j
    e = (0.21, -0.4, 0.13)
    f = o.empty_fields(P)
    f[0], f[1] = rho * np.cos(beta), rho * np.sin(beta)
    f[2], f[3] = c.real, c.imag
    for i in range(3):
        f[4 + i] = t[i]
        f[7 + i] = e[i]
    N = nx * ny * nz
    pi2 = abs(c) ** 2
    grad2 = sum(2.0 * (1.0 - np.cos(ti)) * rho**2 for ti in t) / dx**2
    L = pi2 - grad2 - 0.25 * lam * q * (rho**2 - sig**2) ** 2 + sum(ei**2 for ei in e) / (2.0 * e0**2 * q * dx**2)
    d = o.diagnostics(P, f, tau, dt)
    assert d["sum_L"] == pytest.approx(N * L, rel=1e-12)
    assert d["sum_pi2_L"] == pytest.approx(N * pi2 * L, rel=1e-12)
    assert d["sum_grad2_L"] == pytest.approx(N * grad2 * L, rel=1e-12)
    R = pi2 / grad2
    assert d["v2_phi"] == pytest.approx(2 * R / (1 + R), rel=1e-12)
    assert d["n_wind"] == 0 and d["n_big_plaq"] == 0
    # Eq. 17 right with reading #17: rho and p of the same five pieces, weight W = L
    pot = 0.25 * lam * q * (rho**2 - sig**2) ** 2
    E2 = sum(ei**2 for ei in e) / (2.0 * e0**2 * q * dx**2)
    rho_x = pi2 + grad2 + pot + E2
    p_x = pi2 - grad2 / 3.0 - pot + E2 / 3.0
    assert d["sum_rho_L"] == pytest.approx(N * rho_x * L, rel=1e-12)
    assert d["sum_p_L"] == pytest.approx(N * p_x * L, rel=1e-12)
    assert d["v2_omega"] == pytest.approx(0.5 * (1.0 + 3.0 * p_x / rho_x), rel=1e-12)
    # the electric and kinetic terms enter with a PLUS sign: L grows with |c| and with |e|
    g = f.copy()
    g[2:4] *= 2.0
    assert o.diagnostics(P, g, tau, dt)["sum_L"] == pytest.approx(N * (L + 3.0 * pi2), rel=1e-12)
    g = f.copy()
    g[7:10] *= 2.0
    assert o.diagnostics(P, g, tau, dt)["sum_L"] == pytest.approx(
        N * (L + 3.0 * sum(ei**2 for ei in e) / (2.0 * e0**2 * q * dx**2)), rel=1e-12)


@pytest.mark.parametrize("compact", [1, 0])
def test_lagrangian_closed_form_uniform_magnetic_field(oracle, compact):
    """th_x = B*y on the vacuum phi = sigma, Pi = ep = 0: Phi_xy = th_x(y) - th_x(y+1) = -B on every plaquette
    except the periodic seam y = ny-1, where it is +B(ny-1); Phi_xz = Phi_yz = 0.  The magnetic energy
    2(1 - cos Phi)/dx^4 (compact; Phi^2/dx^4 non-compact, reading #10) enters L with a MINUS sign and the factor
    1/(2 e0^2 q); the gradient term is 2(1 - cos(B y)) sigma^2/dx^2 on the x links."""
    o = oracle
    nx, ny, nz = 4, 6, 3
    dx, lam, e0, sig = 0.5, 2.0, 0.8, 1.0
    P = o.make_params(nx, ny, nz, dx=dx, lambda0=lam, e0=e0, sigma=sig, p=1.0, s=1.0, tau_ref=2.5, compact=compact)
    tau, dt = 1.3, 0.1
    _, q, _, _ = o.coeffs(P, tau, dt)
    B = 0.37
    f = o.empty_fields(P)
    f[0] = sig
    f[4] = B * np.arange(ny)[None, :, None]
    en = (lambda ph: 2.0 * (1.0 - np.cos(ph))) if compact else (lambda ph: ph * ph)
    b2_rows = np.array([en(-B)] * (ny - 1) + [en(B * (ny - 1))]) / dx**4
    g2_rows = 2.0 * (1.0 - np.cos(B * np.arange(ny))) * sig**2 / dx**2
    L_rows = -g2_rows - b2_rows / (2.0 * e0**2 * q)
    d = o.diagnostics(P, f, tau, dt)
    assert d["sum_L"] == pytest.approx(nx * nz * L_rows.sum(), rel=1e-12)
    assert d["sum_grad2_L"] == pytest.approx(nx * nz * (g2_rows * L_rows).sum(), rel=1e-12)
    assert d["sum_pi2_L"] == 0.0 and d["v2_phi"] == 0.0


# ------------------------------------------------------ <v^2>_omega, the equation-of-state estimator (Eq. 17 right)

def test_v2_omega_limits(oracle):
    """<v^2>_omega = (1 + 3 sum p W / sum rho W) / 2 on states whose equation of state is known
    whatever the weight: pure kinetic energy p = rho (v^2 = 2 by the formula), pure potential p = -rho (v^2 = -1),
    pure electric field p = rho/3 (radiation: v^2 = 1), a uniform magnetic field p = rho/3 as well."""
    o = oracle
    P = o.make_params(4, 5, 3, dx=0.5, lambda0=2.0, e0=0.9, sigma=1.0, p=1.0, s=1.0, tau_ref=2.0)
    tau, dt = 1.4, 0.1
    vac = o.empty_fields(P)
    vac[0] = 1.0                               # phi = sigma: no gradient, no potential
    f = vac.copy(); f[2] = 0.3; f[3] = -0.1    # only |Pi|^2
    assert o.diagnostics(P, f, tau, dt)["v2_omega"] == pytest.approx(2.0, rel=1e-12)
    f = vac.copy(); f[0] = 0.6                 # only the potential
    assert o.diagnostics(P, f, tau, dt)["v2_omega"] == pytest.approx(-1.0, rel=1e-12)
    f = vac.copy(); f[7] = 0.2; f[9] = -0.3    # only the electric field; phi = sigma, th = 0: no current either
    assert o.diagnostics(P, f, tau, dt)["v2_omega"] == pytest.approx(1.0, rel=1e-12)
    f = o.empty_fields(P)                      # phi = 0, th_x = B y: only the magnetic energy (and the constant potential)
    f[4] = 0.37 * np.arange(P.ny)[None, :, None]
    d = o.diagnostics(P, f, tau, dt)
    _, q, _, _ = o.coeffs(P, tau, dt)
    N = P.nx * P.ny * P.nz
    b2 = np.array([2 * (1 - np.cos(0.37))] * (P.ny - 1) + [2 * (1 - np.cos(0.37 * (P.ny - 1)))]) / 0.5**4 / (2 * 0.9**2 * q)
    V = 0.25 * 2.0 * q
    L, rho, prs = -V - b2, V + b2, -V + b2 / 3.0
    assert d["sum_rho_L"] == pytest.approx(P.nx * P.nz * (rho * L).sum(), rel=1e-12)
    assert d["sum_p_L"] == pytest.approx(P.nx * P.nz * (prs * L).sum(), rel=1e-12)


def test_v2_omega_vanishes_on_the_static_critical_string(oracle):
    """At critical coupling (beta = 1) the in-plane stresses of a static straight string vanish point by
    point (Bogomolnyi), so p = T_zz/3 = -rho/3 everywhere and <v^2>_omega = 0 for ANY weight: the relaxed vortex pair
    must give 0 up to the lattice's O(dx^2) and the relaxation residual, and <v^2>_phi = 0 with it."""
    o = oracle
    _, _, _, d = _pair_energy(o, 32, 0.5, 3000)
    print("static pair, dx = 0.5 :", d["v2_omega"], d["v2_phi"])
    assert abs(d["v2_omega"]) < 0.02, d["v2_omega"]
    assert abs(d["v2_phi"]) < 1e-6
    _, _, _, d2 = _pair_energy(o, 64, 0.25, 5000)
    print("static pair, dx = 0.25:", d2["v2_omega"], d2["v2_phi"])
    assert abs(d2["v2_omega"]) < 0.5 * abs(d["v2_omega"]) + 1e-4, (d["v2_omega"], d2["v2_omega"])   # -> 0 with dx
