"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the fp64 oracle
element by element on the same seeded inputs.

Tolerances:
  * fp64 site kernel vs oracle: 1e-12 relative to the field's max (same algebra, rounding order only).
  * fp32 kernels, ONE step from identical (fp32-representable) inputs: 2e-6 of the field's max
    (a few fp32 ulps through ~30 operations; 1/dx^2 = 4 amplifies the Laplacian's rounding).
  * north_star: after 100 steps at 64^3, max|d phi|/max|phi| and max|d ep|/max|ep| <= 1e-4.
  * winding: per-plaquette integers identical to the oracle's on the downloaded fp32 snapshot
    promoted to fp64, except plaquettes the oracle flags near-branch.
  * Sigma-type diagnostics on the same snapshot: 1e-5 relative to the sum of |terms| scale.
"""
import numpy as np
import pytest

from paper_2005_14454_b200 import inputs

pytestmark = pytest.mark.gpu

MODEL_KEYS = ("dx", "lambda0", "e0", "sigma", "s", "p", "tau_ref", "alpha", "compact")


@pytest.fixture(scope="module")
def ah():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2005_14454_b200 import build
    build.build()
    from paper_2005_14454_b200 import binding
    return binding


def both(ah, oracle, shape, fp64=False, kernel=None, **model):
    nx, ny, nz = shape
    Po = oracle.make_params(nx, ny, nz, **model)
    sim = ah.Simulation(params=ah.make_params(nx, ny, nz, fp64=fp64, **model))
    if kernel is not None:
        sim.set_kernel(kernel)
    return sim, Po


def rel_max(a, b):
    """max |a-b| / max |b| per field group: phi, Pi, th, ep."""
    out = {}
    for name, sl in (("phi", slice(0, 2)), ("pi", slice(2, 4)), ("th", slice(4, 7)), ("ep", slice(7, 10))):
        den = np.abs(b[sl]).max()
        out[name] = float(np.abs(a[sl].astype(np.float64) - b[sl]).max() / (den if den > 0 else 1.0))
    return out


def kernels_for(ah, nx):
    ks = [ah.KERNEL_SITE]
    if nx % 64 == 0:
        ks.append(ah.KERNEL_TILED)
    return ks


# ------------------------------------------------------------------------------------- trig

def test_trig_against_fp64(ah):
    import torch
    rng = np.random.default_rng(5)
    parts = [rng.uniform(-s, s, 400_000) for s in (1e-3, 0.5, 4.0, 100.0, 3.0e4, 1.0e6)]
    parts.append(np.array([0.0, -0.0, np.pi, -np.pi, np.pi / 2, 32767.9, 32768.0, -32768.5, 1e-30]))
    x = np.concatenate(parts).astype(np.float32)
    s, c, ps = ah.test_trig(torch.from_numpy(x).cuda())
    s, c, ps = s.cpu().numpy(), c.cpu().numpy(), ps.cpu().numpy()
    xd = x.astype(np.float64)
    assert np.abs(s - np.sin(xd)).max() <= 1.5e-7
    assert np.abs(c - np.cos(xd)).max() <= 1.5e-7
    assert np.abs(ps - np.sin(xd)).max() <= 2.0e-7
    small = np.abs(xd) < 1.0
    rel = np.abs(ps[small] - np.sin(xd[small])) / np.maximum(np.abs(np.sin(xd[small])), 1e-30)
    assert rel.max() <= 2.0e-7   # plaquette sines keep RELATIVE accuracy for small angles


def test_tiled_kernel_trig_against_fp64(ah):
    """The tiled kernel's polynomial pair (reduction by multiples of pi) over its whole domain |th| < 2^16 and up
    to the 2^18 its plaquette angles can reach, and its Taylor sine for |Phi| < 0.5."""
    import torch
    rng = np.random.default_rng(6)
    parts = [rng.uniform(-s, s, 400_000) for s in (1e-3, 0.5, 4.0, 100.0, 6.5e4, 2.6e5)]
    parts.append(np.array([0.0, -0.0, np.pi, -np.pi, np.pi / 2, -np.pi / 2, 65535.9, -65535.9, 1e-30]))
    x = np.concatenate(parts).astype(np.float32)
    s, c, ss = ah.test_trig_fast(torch.from_numpy(x).cuda())
    s, c, ss = s.cpu().numpy(), c.cpu().numpy(), ss.cpu().numpy()
    xd = x.astype(np.float64)
    assert np.abs(s - np.sin(xd)).max() <= 1.6e-7
    assert np.abs(c - np.cos(xd)).max() <= 1.6e-7
    small = np.abs(xd) < 0.5
    rel = np.abs(ss[small] - np.sin(xd[small])) / np.maximum(np.abs(np.sin(xd[small])), 1e-30)
    assert rel.max() <= 1.5e-7   # relative accuracy: these feed the gauge force directly


# ------------------------------------------------------------------------------------- I0

@pytest.mark.parametrize("fp64", [False, True])
def test_init_fields_matches_oracle(ah, oracle, fp64):
    sim, Po = both(ah, oracle, (20, 12, 7), fp64=fp64, sigma=1.5)
    sim.init_fields(12345)
    g = sim.get_fields()
    o = oracle.init_fields(Po, 12345)
    # a few ulp of sigma: device sincospi vs the oracle's libm cos/sin of 2*pi*u
    tol = 4 * 2.3e-16 * 1.5 if fp64 else 1.2e-7 * 1.5
    assert np.abs(g[:2] - o[:2]).max() <= tol
    assert not g[2:].any()
    assert np.allclose(np.hypot(g[0], g[1]), 1.5, rtol=2e-7)
    sim.close()


# ------------------------------------------------------------------------------- single step

ONE_STEP_CASES = [
    dict(p=0.0, s=0.0),
    dict(p=1.0, s=0.0),
    dict(p=1.0, s=1.0, tau_ref=3.0),
    dict(p=2.0, s=1.0, tau_ref=3.0),
    dict(p=1.0, s=0.5, tau_ref=2.0, lambda0=1.3, e0=0.7, sigma=1.2, dx=0.4, alpha=1.5),
    dict(p=1.0, s=1.0, tau_ref=3.0, compact=0),
    dict(p=1.0, s=-0.5, tau_ref=3.0),      # s < 0: the core-growth phase of PAPER.md:57
]


@pytest.mark.parametrize("case", ONE_STEP_CASES)
@pytest.mark.parametrize("shape", [(20, 12, 7), (33, 5, 9), (64, 64, 3)])
def test_one_step_fp64_site_kernel(ah, oracle, case, shape):
    """fp64 instantiation of the site kernel = the oracle's algebra up to rounding order."""
    sim, Po = both(ah, oracle, shape, fp64=True, **case)
    f0 = inputs.random_state(*shape, seed=11)
    sim.set_fields(f0)
    sim.step(3, 1.7, 0.1)
    g = sim.get_fields()
    o = oracle.step(Po, f0.copy(), 3, 1.7, 0.1)
    r = rel_max(g, o)
    assert max(r.values()) <= 1e-12, r
    sim.close()


@pytest.mark.parametrize("case", ONE_STEP_CASES)
@pytest.mark.parametrize("shape", [(20, 12, 7), (128, 9, 6), (256, 16, 11), (128, 8, 1), (128, 1, 5), (384, 3, 2),
                                   (64, 9, 6), (192, 7, 5), (64, 1, 1)])    # the last three: 64-site warp rows
def test_one_step_fp32(ah, oracle, case, shape):
    f0 = inputs.random_state(*shape, seed=7)
    for kern in kernels_for(ah, shape[0]):
        sim, Po = both(ah, oracle, shape, kernel=kern, **case)
        sim.set_fields(f0)
        sim.step(1, 1.7, 0.1)
        g = sim.get_fields()
        o = oracle.step(Po, f0.copy(), 1, 1.7, 0.1)
        r = rel_max(g, o)
        assert max(r.values()) <= 2e-6, (kern, r)
        sim.close()


@pytest.mark.parametrize("shape", [(1, 1, 1), (1, 6, 5), (7, 1, 1), (2, 2, 2), (5, 4, 1)])
def test_degenerate_lattices(ah, oracle, shape):
    """Extent-1 and extent-2 directions: a site is its own neighbour; the oracle's modulo indexing decides."""
    f0 = inputs.random_state(*shape, seed=3)
    for fp64, tol in ((True, 1e-12), (False, 3e-6)):
        sim, Po = both(ah, oracle, shape, fp64=fp64, p=1.0, s=1.0, tau_ref=2.0)
        sim.set_fields(f0)
        sim.step(2, 1.0, 0.1)
        r = rel_max(sim.get_fields(), oracle.step(Po, f0.copy(), 2, 1.0, 0.1))
        assert max(r.values()) <= tol, (fp64, r)
        sim.close()


def test_large_link_angles(ah, oracle):
    """th is never wrapped (Eq. 10): angles of a few hundred radians must still give the right links."""
    shape = (128, 6, 5)
    f0 = inputs.random_state(*shape, seed=21, th_amp=150.0)
    for kern in kernels_for(ah, shape[0]):
        sim, Po = both(ah, oracle, shape, kernel=kern, p=1.0, s=0.0)
        sim.set_fields(f0)
        sim.step(1, 2.0, 0.1)
        r = rel_max(sim.get_fields(), oracle.step(Po, f0.copy(), 1, 2.0, 0.1))
        # th itself is ~150 rad: one fp32 ulp of it is 1.5e-5 rad, which enters every plaquette angle
        assert r["phi"] <= 3e-6 and r["pi"] <= 3e-5 and r["th"] <= 1e-6 and r["ep"] <= 3e-4, (kern, r)
        sim.close()


def test_link_angles_beyond_the_tiled_domain_are_redone(ah, oracle):
    """|th| >= 2^16 rad is outside the tiled kernel's polynomial range: it must raise its overflow flag and the
    step must come out of the libm-based redo (identical to the site kernel), then the next, in-range step must
    run on the fast path again with a cleared flag."""
    shape = (128, 9, 6)
    f0 = inputs.random_state(*shape, seed=22, th_amp=0.5)
    f0[5, 3, 4, 77] = 7.0e4     # one th_y link beyond 2^16
    f0[4, 0, 0, 0] = -2.5e5     # one th_x link at a tile corner
    got = {}
    for kern in kernels_for(ah, shape[0]):
        sim, Po = both(ah, oracle, shape, kernel=kern, p=1.0, s=0.0)
        sim.set_fields(f0)
        sim.step(1, 2.0, 0.1)
        got[kern] = sim.get_fields()
        sim.close()
    assert np.array_equal(got[ah.KERNEL_SITE], got[ah.KERNEL_TILED])
    ref = oracle.step(Po, f0.copy(), 1, 2.0, 0.1)
    r = rel_max(got[ah.KERNEL_TILED], ref)
    # th ~ 1e5 rad carries an fp32 ulp of 8e-3 rad into its plaquettes; fields are compared to their max
    assert r["phi"] <= 1e-5 and r["th"] <= 1e-6, r
    # in-range state after an out-of-range one: the flag of the previous step must not leak
    f1 = inputs.random_state(*shape, seed=23, th_amp=0.5)
    sim, Po = both(ah, oracle, shape, kernel=ah.KERNEL_TILED, p=1.0, s=0.0)
    sim.set_fields(f0)
    sim.step(1, 2.0, 0.1)
    sim.set_fields(f1)
    sim.step(3, 2.0, 0.1)
    r = rel_max(sim.get_fields(), oracle.step(Po, f1.copy(), 3, 2.0, 0.1))
    assert max(r.values()) <= 5e-6, r
    sim.close()


# ------------------------------------------------------------------------ north_star parity

def test_parity_config1_64cubed_100_and_160_steps(ah, oracle):
    """BASELINE config 1: 64^3, dx=0.5, dt=0.1, radiation, s=0, random-phase IC from seed 1.
    north_star: max rel |d phi|, |d ep| <= 1e-4 after 100 steps."""
    n, dt, tau0 = 64, 0.1, 1.0
    sim, Po = both(ah, oracle, (n, n, n), p=1.0, s=0.0)
    assert sim.get_kernel() == ah.KERNEL_TILED            # the product kernel (64-site warp rows), not the site kernel
    f = oracle.init_fields(Po, 1)
    sim.set_fields(f)                      # identical ICs: cos/sin values rounded once to fp32
    f = sim.get_fields().astype(np.float64)
    sim.step(100, tau0, dt)
    g100 = sim.get_fields()
    oracle.step(Po, f, 100, tau0, dt)
    r100 = rel_max(g100, f)
    print("64^3 100 steps rel err:", r100)
    assert r100["phi"] <= 1e-4 and r100["ep"] <= 1e-4, r100
    assert r100["pi"] <= 1e-4 and r100["th"] <= 1e-4, r100
    sim.step(60, tau0 + 100 * dt, dt)
    oracle.step(Po, f, 60, tau0 + 100 * dt, dt)
    r160 = rel_max(sim.get_fields(), f)
    print("64^3 160 steps rel err:", r160)
    assert max(r160.values()) <= 1e-3, r160
    sim.close()


@pytest.mark.parametrize("model", [dict(p=1.0, s=0.0), dict(p=1.0, s=1.0, tau_ref=1.0 + 160 * 0.1)])
def test_parity_north_star_gate_on_the_tiled_kernel(ah, oracle, model):
    """north_star's gate (max rel |d phi|, |d ep| <= 1e-4 after 100 steps) on the PRODUCT kernel: 64^3 is below
    the tiled kernel's 128-site rows, so the gate is run at 128^3, the smallest cube it takes, for s = 0
    (BASELINE config 1's model) and s = 1 (configs 2-5), from oracle initial conditions, 100 and 160 steps."""
    n, dt, tau0 = 128, 0.1, 1.0
    sim, Po = both(ah, oracle, (n, n, n), **model)
    assert sim.get_kernel() == ah.KERNEL_TILED
    f = oracle.init_fields(Po, 1)
    sim.set_fields(f)
    f = sim.get_fields().astype(np.float64)
    sim.step(100, tau0, dt)
    g100 = sim.get_fields()
    oracle.step(Po, f, 100, tau0, dt)
    r100 = rel_max(g100, f)
    print("tiled 128^3 100 steps rel err:", model, r100)
    assert r100["phi"] <= 1e-4 and r100["ep"] <= 1e-4, r100
    assert r100["pi"] <= 1e-4 and r100["th"] <= 1e-4, r100
    sim.step(60, tau0 + 100 * dt, dt)
    oracle.step(Po, f, 60, tau0 + 100 * dt, dt)
    r160 = rel_max(sim.get_fields(), f)
    print("tiled 128^3 160 steps rel err:", model, r160)
    assert max(r160.values()) <= 1e-3, r160
    sim.close()


def test_tiled_step_repeats_bit_identically(ah):
    """Race detector for the tiled kernel's shared-memory protocol (ring slots and the per-warp Pi, ep row are
    refilled by async-proxy bulk copies after generic-proxy reads, ordered by the CTA barrier / program order):
    a timing-dependent overwrite would change Pi, ep by O(1) at the sites of the clobbered row, so the same state
    advanced several times must come out bit-identical, under the plain and under the DIAG instantiation.
    256 x 66 x 200 covers full 64-plane chunks, a partial last chunk and a ragged y tail (66 = 11 x 6)."""
    shape = (256, 66, 200)
    f0 = inputs.random_state(*shape, seed=77, th_amp=0.4)
    sim = ah.Simulation(params=ah.make_params(*shape, p=1.0, s=1.0, tau_ref=3.0))
    assert sim.get_kernel() == ah.KERNEL_TILED
    outs = []
    for rep in range(4):
        sim.set_fields(f0)
        if rep < 3:
            sim.step(6, 1.0, 0.1)
        else:
            sim.step_diag(6, 1.0, 0.1, 1)          # every step through the DIAG instantiation
        outs.append(sim.get_fields())
    for o_ in outs[1:]:
        assert np.array_equal(outs[0], o_)
    # and against the independent site kernel (different code path, same fp32 algebra up to rounding order)
    sim.set_kernel(ah.KERNEL_SITE)
    sim.set_fields(f0)
    sim.step(6, 1.0, 0.1)
    r = rel_max(sim.get_fields(), outs[0].astype(np.float64))
    assert max(r.values()) <= 1e-5, r
    sim.close()


def test_parity_tiled_128cubed_physical_width(ah, oracle):
    """Config-2-like (radiation, s=1, tau_ref = end time) at 128^3 for 40 steps, tiled kernel vs oracle,
    and tiled vs site kernel."""
    n, dt, tau0, steps = 128, 0.1, 1.0, 40
    model = dict(p=1.0, s=1.0, tau_ref=tau0 + 640 * dt)
    sim, Po = both(ah, oracle, (n, n, n), **model)
    f = oracle.init_fields(Po, 2)
    sim.set_fields(f)
    f = sim.get_fields().astype(np.float64)
    sim.step(steps, tau0, dt)
    g = sim.get_fields()
    oracle.step(Po, f, steps, tau0, dt)
    r = rel_max(g, f)
    print("128^3 40 steps rel err:", r)
    assert max(r.values()) <= 2e-5, r
    sim.close()


# ------------------------------------------------------------------------------ diagnostics

def test_parity_config2_256cubed_winding_every_20(ah, oracle):
    """BASELINE configs[1] (256^3, radiation, s=1, winding every 20 steps), first 40 of its 640 steps: the fused
    step+diagnostics path on the tiled kernel against the oracle advanced from the same device-generated I0."""
    n, nsteps, every, tau0, dt = 256, 40, 20, 1.0, 0.1
    model = dict(p=1.0, s=1.0, tau_ref=tau0 + 640 * dt)
    sim, Po = both(ah, oracle, (n, n, n), **model)
    assert sim.get_kernel() == ah.KERNEL_TILED
    sim.init_fields(1)
    ref = sim.get_fields().astype(np.float64)
    assert np.abs(ref - oracle.init_fields(Po, 1)).max() <= 1.2e-7
    recs = sim.step_diag(nsteps, tau0, dt, every)
    assert [r["tau"] for r in recs] == pytest.approx([1.0, 3.0])
    got = sim.get_fields()
    # record 0 is the initial condition: winding of random phases with th = 0, exact integers
    od = oracle.diagnostics(Po, ref, tau0, dt)
    assert abs(recs[0]["n_wind"] - od["n_wind"]) <= recs[0]["n_near_branch"] + od["n_near_branch"]
    assert recs[0]["n_wind"] / (3.0 * n ** 3) == pytest.approx(1.0 / 3.0, abs=2e-3)
    oracle.step(Po, ref, every, tau0, dt)
    od = oracle.diagnostics(Po, ref, tau0 + every * dt, dt)
    # different snapshots here (fp32-evolved vs fp64-evolved): counts agree statistically, not bit for bit
    assert recs[1]["n_wind"] == pytest.approx(od["n_wind"], rel=2e-3)
    assert recs[1]["gauss_rel"] <= 2e-5
    oracle.step(Po, ref, nsteps - every, tau0 + every * dt, dt)
    r = rel_max(got, ref)
    assert r["phi"] <= 1e-4 and r["ep"] <= 1e-4 and r["pi"] <= 1e-4 and r["th"] <= 1e-4, r
    sim.close()


def test_parity_config3_512cubed_matter_fused_record(ah, oracle):
    """BASELINE configs[2] at its own size (512^3, matter era, s = 1, tau_ref = 129, all three read-outs), first 21
    of its 1280 steps: the record the fused DIAG instantiation writes for step 20 against oracle.diagnostics of the
    snapshot downloaded at that step.  Sigma-type sums 1e-5; the Gauss residual is truncation-level in the matter
    era with s != 0 (reading #18), so it is COMPARED with the oracle's value, not asserted to be round-off."""
    import torch
    n, tau0, dt, every = 512, 1.0, 0.1, 20
    model = dict(p=2.0, s=1.0, tau_ref=tau0 + 1280 * dt)
    sim, Po = both(ah, oracle, (n, n, n), **model)
    assert sim.get_kernel() == ah.KERNEL_TILED
    sim.init_fields(1)
    sim.step(every, tau0, dt)
    tau = tau0 + every * dt
    snap = sim.get_fields()
    rec = sim.step_diag(1, tau, dt, 1)[0]
    sim.close()
    torch.cuda.empty_cache()
    od = oracle.diagnostics(Po, snap.astype(np.float64), tau, dt)
    del snap
    slack = rec["n_near_branch"] + od["n_near_branch"]
    for key in ("n_wind", "n_wind_xy", "n_wind_xz", "n_wind_yz"):
        assert abs(rec[key] - od[key]) <= slack, (key, rec[key], od[key], slack)
    assert rec["n_wind"] > 1000
    assert rec["n_big_plaq"] == od["n_big_plaq"]
    for key in ("sum_pi2_L", "sum_grad2_L", "sum_L", "sum_p_L", "sum_rho_L"):
        assert rec[key] == pytest.approx(od[key], rel=1e-5), (key, rec[key], od[key])
    assert rec["v2_phi"] == pytest.approx(od["v2_phi"], abs=1e-5)
    assert rec["v2_omega"] == pytest.approx(od["v2_omega"], abs=1e-5)
    assert rec["xi_l"] == pytest.approx(od["xi_l"], rel=1e-5)
    for key in ("gauss_max", "gauss_l2", "gauss_div_l2", "gauss_charge_l2"):
        assert rec[key] == pytest.approx(od[key], rel=1e-9), (key, rec[key], od[key])
    assert rec["gauss_rel"] == pytest.approx(od["gauss_rel"], rel=1e-8)
    print("config 3 record at step 20:", {k: rec[k] for k in ("n_wind", "xi_w", "xi_l", "v2_phi", "gauss_rel")})


def _evolved_snapshot(ah, oracle, n, steps, seed, **model):
    sim, Po = both(ah, oracle, (n, n, n), **model)
    sim.init_fields(seed)
    sim.step(steps, 1.0, 0.1)
    return sim, Po, 1.0 + steps * 0.1


@pytest.mark.parametrize("model", [dict(p=1.0, s=0.0), dict(p=2.0, s=1.0, tau_ref=9.0)])
def test_winding_bit_exact_on_snapshot(ah, oracle, model):
    sim, Po, tau = _evolved_snapshot(ah, oracle, 48, 60, 4, **model)
    snap = sim.get_fields().astype(np.float64)
    w_gpu, near_gpu = sim.winding_field()
    w_or, near_or = oracle.winding(Po, snap)
    differ = w_gpu != w_or
    assert np.abs(w_or).sum() > 50, "vacuous without strings"
    assert not (differ & (near_or == 0)).any(), "winding differs on a plaquette that is not near-branch"
    d_gpu = sim.diagnostics(tau, 0.1)
    d_or = oracle.diagnostics(Po, snap, tau, 0.1)
    for key in ("n_wind", "n_wind_xy", "n_wind_xz", "n_wind_yz"):
        assert abs(d_gpu[key] - d_or[key]) <= d_or["n_near_branch"], key
    assert d_gpu["n_wind"] == int(np.abs(w_gpu).sum())
    assert d_gpu["n_big_plaq"] == d_or["n_big_plaq"] == 0
    assert abs(d_gpu["n_near_branch"] - d_or["n_near_branch"]) <= 2
    assert d_gpu["xi_w"] == pytest.approx(np.sqrt(48**3 * 0.5**3 / (0.5 * d_gpu["n_wind"])), rel=1e-14)
    # Eq. 16 left from the returned sum (mu = 2 pi sigma^2), and against the oracle's own evaluation
    if d_gpu["sum_L"] < 0:
        assert d_gpu["xi_l"] == pytest.approx(np.sqrt(-2 * np.pi * 48**3 / d_gpu["sum_L"]), rel=1e-14)
        assert d_gpu["xi_l"] == pytest.approx(d_or["xi_l"], rel=1e-5)
    else:
        assert np.isinf(d_gpu["xi_l"]) and np.isinf(d_or["xi_l"])
    sim.close()


def test_static_vortex_pair_cooling_on_the_tiled_kernel(ah, oracle):
    """north_star's static Nielsen-Olesen string on the CUDA path: a vortex-antivortex pair (a single winding cannot
    live on a periodic lattice) relaxed with ah_step_cooling (the paper's artificial damping) on the
    tiled kernel, against the oracle doing the same sequence; then evolved undamped in Minkowski space."""
    nx, ny, dx = 128, 128, 0.5      # square: a flatter box puts a spurious second pair on the y seam
    Pr = oracle.make_params(nx, ny, 1, dx=dx, p=1.0, s=0.0)          # the oracle's constant damping: tau = dt/delta
    f = oracle.empty_fields(Pr)
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    c1, c2 = (nx / 4 + 0.5, ny / 2 + 0.5), (3 * nx / 4 + 0.5, ny / 2 + 0.5)
    r1, r2 = np.hypot(x - c1[0], y - c1[1]) * dx, np.hypot(x - c2[0], y - c2[1]) * dx
    a1, a2 = np.arctan2(y - c1[1], x - c1[0]), np.arctan2(y - c2[1], x - c2[0])
    phi = np.tanh(r1 / 1.2) * np.tanh(r2 / 1.2) * np.exp(1j * (a1 - a2))
    f[0, 0], f[1, 0] = phi.real, phi.imag
    f = f.astype(np.float32).astype(np.float64)
    dt, delta, nrelax = 0.1, 0.15, 1500
    sim = ah.Simulation(params=ah.make_params(nx, ny, 1, dx=dx, p=0.0, s=0.0))   # Minkowski context
    assert sim.get_kernel() == ah.KERNEL_TILED
    sim.set_fields(f)
    sim.step_cooling(nrelax, delta, dt)
    for _ in range(nrelax):
        oracle.step(Pr, f, 1, dt / delta, dt)
    g = sim.get_fields()
    r = rel_max(g, f)
    # a contraction: fp32 errors do not grow (Pi, ep relax to the fp32 noise floor and are not compared)
    assert r["phi"] <= 5e-5 and r["th"] <= 1e-4, r
    d = sim.diagnostics(1.0, dt)
    assert d["n_wind"] == 2 and d["n_wind_xy"] == 2 and d["n_near_branch"] == 0
    w, _ = sim.winding_field()
    assert sorted(w[0][w[0] != 0].tolist()) == [-1, 1] and not w[1].any() and not w[2].any()
    # tension: -sum L dx^3 = 2 mu Lz (1 - O(dx^2)), mu = 2 pi sigma^2, Lz = dx; and xi_L ~ xi_W
    deficit = 1 - (-d["sum_L"] * dx**3) / (2 * 2 * np.pi * dx)
    assert 0.005 < deficit < 0.02, deficit
    assert d["xi_l"] == pytest.approx(d["xi_w"] * (1 + 0.5 * deficit), rel=2e-3)
    assert d["v2_phi"] < 1e-6
    assert abs(d["v2_omega"]) < 0.02          # p = -rho/3 on the static critical-coupling string (O(dx^2) on the lattice)
    # static: 300 undamped Minkowski steps move nothing beyond the relaxation residual
    eps = max(np.abs(g[2:4]).max(), np.abs(g[7:10]).max())
    sim.step(300, 1.0, dt)
    h = sim.get_fields()
    assert np.abs(h[0:2] - g[0:2]).max() <= 10 * (delta / dt) * eps * (300 * dt) ** 2 + 2e-5
    w2, _ = sim.winding_field()
    assert np.array_equal(w, w2)
    sim.close()


def test_winding_with_exactly_zero_phi_sites(ah, oracle):
    """The library takes link phases as wrapped differences of site phases alpha = Arg(phi); a site with phi == 0
    has none, and the oracle's convention (Arg of a zero link product := 0) must still come out, on both kernels
    and on the fused path."""
    shape = (128, 7, 5)
    f0 = inputs.random_state(*shape, seed=41, th_amp=0.6)
    rng = np.random.default_rng(42)
    for _ in range(60):
        x, y, z = rng.integers(shape[0]), rng.integers(shape[1]), rng.integers(shape[2])
        f0[0:2, z, y, x] = 0.0
    f0[0:2, 0, 0, 0] = 0.0
    f0[0:2, 4, 6, 127] = 0.0
    f0[0, 2, 3, 64] = -0.0                                  # signed zeros are zeros too
    f0[1, 2, 3, 64] = 0.0
    Po = oracle.make_params(*shape, p=1.0, s=0.0)
    w_ref, near_ref = oracle.winding(Po, f0)
    od = oracle.diagnostics(Po, f0, 1.0, 0.1)
    for kern in kernels_for(ah, shape[0]):
        sim, _ = both(ah, oracle, shape, kernel=kern, p=1.0, s=0.0)
        sim.set_fields(f0)
        w, near = sim.winding_field()
        ok = (w == w_ref) | (near_ref != 0) | (near != 0)
        assert ok.all(), (kern, int((~ok).sum()))
        rec = sim.step_diag(1, 1.0, 0.1, 1)[0]               # fused on the tiled kernel
        assert abs(rec["n_wind"] - od["n_wind"]) <= rec["n_near_branch"] + od["n_near_branch"]
        assert rec["sum_L"] == pytest.approx(od["sum_L"], rel=1e-5)
        sim.close()


def test_winding_random_phase_snapshot(ah, oracle):
    """Uncorrelated random phases: a third of all plaquettes wind (oracle pin (v)); bit-exact vs oracle."""
    sim, Po = both(ah, oracle, (40, 24, 10), p=0.0)
    sim.init_fields(9)
    snap = sim.get_fields().astype(np.float64)
    w_gpu, _ = sim.winding_field()
    w_or, near_or = oracle.winding(Po, snap)
    assert not ((w_gpu != w_or) & (near_or == 0)).any()
    assert abs(np.abs(w_gpu).mean() - 1 / 3) < 0.02
    sim.close()


@pytest.mark.parametrize("model", [dict(p=1.0, s=0.0), dict(p=1.0, s=1.0, tau_ref=9.0),
                                   dict(p=2.0, s=1.0, tau_ref=9.0), dict(p=1.0, s=1.0, tau_ref=9.0, compact=0)])
def test_sigma_diagnostics_on_snapshot(ah, oracle, model):
    sim, Po, tau = _evolved_snapshot(ah, oracle, 40, 50, 6, **model)
    snap = sim.get_fields().astype(np.float64)
    d_gpu = sim.diagnostics(tau, 0.1)
    d_or = oracle.diagnostics(Po, snap, tau, 0.1)
    for key in ("sum_pi2_L", "sum_grad2_L", "sum_L", "sum_p_L", "sum_rho_L"):
        assert d_gpu[key] == pytest.approx(d_or[key], rel=1e-5), (key, d_gpu[key], d_or[key])
    assert d_gpu["v2_phi"] == pytest.approx(d_or["v2_phi"], abs=1e-5)
    assert d_gpu["v2_omega"] == pytest.approx(d_or["v2_omega"], abs=1e-5)      # Eq. 17 right
    # Gauss: evaluated in fp64 from the same stored values on both sides
    for key in ("gauss_max", "gauss_l2", "gauss_div_l2", "gauss_charge_l2"):
        assert d_gpu[key] == pytest.approx(d_or[key], rel=1e-9), (key, d_gpu[key], d_or[key])
    assert d_gpu["gauss_rel"] == pytest.approx(d_or["gauss_rel"], rel=1e-8)
    sim.close()


def test_gauss_residual_is_fp32_roundoff(ah):
    """the scheme keeps Gauss's law; in fp32 the residual is fp32 round-off (reported)."""
    sim = ah.Simulation(nx=64, p=1.0, s=0.0)
    sim.init_fields(1)
    sim.step(100, 1.0, 0.1)
    d = sim.diagnostics(11.0, 0.1)
    print("gauss_rel after 100 fp32 steps:", d["gauss_rel"])
    assert d["gauss_div_l2"] > 1.0
    assert d["gauss_rel"] < 2e-5
    sim.close()


def test_gauss_residual_fp64_kernel_roundoff(ah):
    sim = ah.Simulation(nx=24, p=1.0, s=1.0, tau_ref=5.0, fp64=True)
    sim.init_fields(1)
    sim.step(40, 1.0, 0.1)
    d = sim.diagnostics(5.0, 0.1)
    assert d["gauss_rel"] < 1e-12
    sim.close()


def test_step_diag_equals_diagnostics_before_step(ah):
    """D-fuse contract: the record for step j is ah_diagnostics(tau_j) of the ENTRY snapshot."""
    a = ah.Simulation(nx=32, p=1.0, s=1.0, tau_ref=4.0)
    b = ah.Simulation(nx=32, p=1.0, s=1.0, tau_ref=4.0)
    a.init_fields(5)
    b.init_fields(5)
    recs = a.step_diag(25, 1.0, 0.1, 10)
    assert [r["tau"] for r in recs] == pytest.approx([1.0, 2.0, 3.0])
    for r in recs:
        nsteps = int(round((r["tau"] - 1.0) / 0.1))
        b.init_fields(5)
        b.step(nsteps, 1.0, 0.1)
        d = b.diagnostics(1.0 + nsteps * 0.1, 0.1)
        for key, val in d.items():
            assert r[key] == val or (np.isnan(val) and np.isnan(r[key])), key
    b.init_fields(5)
    b.step(25, 1.0, 0.1)
    assert np.array_equal(a.get_fields(), b.get_fields())
    a.close()
    b.close()


@pytest.mark.parametrize("shape,model", [((128, 20, 9), dict(p=1.0, s=1.0, tau_ref=4.0)),
                                         ((256, 13, 70), dict(p=2.0, s=1.0, tau_ref=5.0)),
                                         ((128, 6, 3), dict(p=0.0, s=0.0, compact=0))])
def test_fused_step_diag_tiled_kernel(ah, oracle, shape, model):
    """Row D-fuse on the tiled kernel: the DIAG instantiation (read-outs from the staged planes, inside the step
    pass) must give, for the entry snapshot of step j, the integers of the standalone kernel exactly (same
    per-site arithmetic) and its fp64 sums up to the order of summation; the fields it leaves are those of the
    plain step; and the whole record agrees with the oracle on the downloaded snapshot."""
    nx, ny, nz = shape
    a = ah.Simulation(params=ah.make_params(nx, ny, nz, **model))
    b = ah.Simulation(params=ah.make_params(nx, ny, nz, **model))
    assert a.get_kernel() == ah.KERNEL_TILED
    f0 = inputs.random_state(nx, ny, nz, seed=31, th_amp=0.4)
    a.set_fields(f0)
    b.set_fields(f0)
    every, nsteps, tau0, dt = 4, 10, 1.5, 0.1
    recs = a.step_diag(nsteps, tau0, dt, every)
    assert len(recs) == 3
    ints = ("n_wind", "n_wind_xy", "n_wind_xz", "n_wind_yz", "n_near_branch", "n_big_plaq")
    sums = ("sum_pi2_L", "sum_grad2_L", "sum_L", "sum_p_L", "sum_rho_L", "gauss_l2", "gauss_div_l2", "gauss_charge_l2",
            "v2_phi", "v2_omega", "gauss_rel")
    Po = oracle.make_params(nx, ny, nz, **model)
    done = 0
    for r in recs:
        j = int(round((r["tau"] - tau0) / dt))
        b.step(j - done, tau0 + done * dt, dt)
        done = j
        d = b.diagnostics(r["tau"], dt)
        for key in ints:
            assert r[key] == d[key], (key, r[key], d[key])
        assert r["gauss_max"] == d["gauss_max"]
        for key in sums:
            assert r[key] == pytest.approx(d[key], rel=1e-11, abs=1e-300), key
        od = oracle.diagnostics(Po, b.get_fields().astype(np.float64), r["tau"], dt)
        assert abs(r["n_wind"] - od["n_wind"]) <= r["n_near_branch"] + od["n_near_branch"]
        assert r["sum_L"] == pytest.approx(od["sum_L"], rel=1e-5, abs=1e-5 * abs(od["sum_pi2_L"]) + 1e-6)
    b.step(nsteps - done, tau0 + done * dt, dt)
    assert np.array_equal(a.get_fields(), b.get_fields())
    a.close()
    b.close()


def test_fused_and_plain_steps_agree_bitwise_in_the_physical_regime(ah):
    """The DIAG instantiation cuts the lattice into tiles of 5 rows, the plain one into tiles of 6: the fields a
    diagnostic step leaves must still be those of a plain step bit for bit, also where plaquette angles are small and
    the warp-wide choice of the sine polynomial comes into play (random-phase IC, th = 0 at the start)."""
    a = ah.Simulation(nx=128, ny=31, nz=24, p=1.0, s=1.0, tau_ref=4.0)
    b = ah.Simulation(nx=128, ny=31, nz=24, p=1.0, s=1.0, tau_ref=4.0)
    a.init_fields(3)
    b.init_fields(3)
    a.step_diag(12, 1.0, 0.1, 1)
    b.step(12, 1.0, 0.1)
    assert np.array_equal(a.get_fields(), b.get_fields())
    a.close()
    b.close()


@pytest.mark.parametrize("case", [dict(p=1.0, s=1.0, tau_ref=3.0), dict(p=0.0, s=0.0, compact=0)])
@pytest.mark.parametrize("shape", [(20, 12, 7), (128, 9, 6)])
def test_one_step_mixed_precision(ah, oracle, case, shape):
    """SURVEY 8(f)4, mixed precision: fp32 storage, every operation of the step in fp64.  One step from
    fp32-representable inputs is the oracle's result rounded once to fp32: half an ulp of each value, i.e. 6e-8 of
    the field's scale (the fp32 build needs 2e-6)."""
    f0 = inputs.random_state(*shape, seed=7)
    sim, Po = both(ah, oracle, shape, fp64=ah.PRECISION_MIXED, **case)
    assert sim.get_kernel() == ah.KERNEL_SITE and sim.np_dtype == np.float32
    sim.set_fields(f0)
    sim.step(1, 1.7, 0.1)
    g = sim.get_fields()
    o = oracle.step(Po, f0.copy(), 1, 1.7, 0.1)
    assert np.array_equal(g, o.astype(np.float32)) or max(rel_max(g, o).values()) <= 6.1e-8, rel_max(g, o)
    # over 40 steps the only rounding is the one store per value and step
    sim.set_fields(f0)
    sim.step(40, 1.7, 0.1)
    ref = oracle.step(Po, f0.copy(), 40, 1.7, 0.1)
    r = rel_max(sim.get_fields(), ref)
    print("mixed precision, 40 steps:", r)
    assert max(r.values()) <= 1e-5, r
    d = sim.diagnostics(1.7 + 4.0, 0.1)                     # read-outs run on the fp32 snapshot
    assert d["n_wind"] >= 0
    sim.close()


@pytest.mark.parametrize("shape", [(128, 20, 9), (64, 7, 6), (20, 12, 7)])
def test_step_diag_sums_equals_step_diag_without_the_winding(ah, shape):
    """ah_step_diag_sums (the read-outs the paper's timed runs evaluate): every field of its records
    except the winding ones is bit-identical to ah_step_diag's, the winding fields say "not computed", and the steps
    leave the same fields — on the tiled kernel (both row widths) and on the site kernel."""
    nx, ny, nz = shape
    a = ah.Simulation(params=ah.make_params(nx, ny, nz, p=1.0, s=1.0, tau_ref=4.0))
    b = ah.Simulation(params=ah.make_params(nx, ny, nz, p=1.0, s=1.0, tau_ref=4.0))
    f0 = inputs.random_state(nx, ny, nz, seed=33, th_amp=0.3)
    a.set_fields(f0)
    b.set_fields(f0)
    ra = a.step_diag(9, 1.5, 0.1, 4)
    rb = b.step_diag(9, 1.5, 0.1, 4, winding=False)
    assert len(ra) == len(rb) == 3
    wind = ("n_wind", "n_wind_xy", "n_wind_xz", "n_wind_yz", "n_near_branch", "n_big_plaq")
    for x, y in zip(ra, rb):
        for key, val in x.items():
            if key in wind:
                assert y[key] == -1 and val >= 0, key
            elif key in ("string_length", "xi_w", "xi_w_corr"):
                assert np.isnan(y[key]), key
            else:
                assert y[key] == val, (key, y[key], val)
    assert np.array_equal(a.get_fields(), b.get_fields())
    a.close()
    b.close()


def test_diagnostics_deterministic(ah):
    sim = ah.Simulation(nx=48, p=1.0, s=0.0)
    sim.init_fields(8)
    sim.step(30, 1.0, 0.1)
    d1 = sim.diagnostics(4.0, 0.1)
    d2 = sim.diagnostics(4.0, 0.1)
    assert d1 == d2
    sim.close()


# ---------------------------------------------------------------------------- ABI behaviour

def test_error_codes_on_device(ah):
    sim = ah.Simulation(nx=16)
    with pytest.raises(ah.AhError) as ei:
        sim.step(1, 1.0, 0.1)                      # no fields yet
    assert ei.value.code == ah.AH_ESTATE
    sim.init_fields(1)
    for args in ((-1, 1.0, 0.1), (1, 0.0, 0.1), (1, 1.0, 0.0), (1, 1.0, float("nan"))):
        with pytest.raises(ah.AhError) as ei:
            sim.step(*args)
        assert ei.value.code == ah.AH_EINVAL
    before = sim.get_fields()
    sim.step(0, 1.0, 0.1)                          # n = 0 is a no-op
    assert np.array_equal(before, sim.get_fields())
    import ctypes as C
    recs = (ah.Diag * 1)()
    nw = C.c_int(7)
    rc = ah.lib().ah_step_diag(sim._ctx, 30, 1.0, 0.1, 10, recs, 1, C.byref(nw))   # cap too small
    assert rc == ah.AH_EINVAL and nw.value == 0
    assert np.array_equal(before, sim.get_fields())   # ... and it did not step
    with pytest.raises(ah.AhError):
        sim.set_kernel(ah.KERNEL_TILED)            # nx = 16 is not a multiple of 128
    sim.close()


def test_ping_pong_parity_and_current_bufs(ah):
    sim = ah.Simulation(nx=16)
    sim.init_fields(3)
    first = [b.data_ptr() for b in sim.current_bufs()]
    sim.step(1, 1.0, 0.1)
    second = [b.data_ptr() for b in sim.current_bufs()]
    assert set(first).isdisjoint(second)
    sim.step(1, 1.1, 0.1)
    assert [b.data_ptr() for b in sim.current_bufs()] == first
    cur = sim.current_bufs()
    got = sim.get_fields()
    assert np.array_equal(got[0].ravel(), cur[0].cpu().numpy())
    assert sim.launch_count() == 3
    sim.close()


def test_step_n_equals_n_single_steps(ah):
    """tau_j = tau + j*dt as a product: one call of n steps == n calls at those times."""
    a = ah.Simulation(nx=24, p=1.0, s=1.0, tau_ref=3.0)
    b = ah.Simulation(nx=24, p=1.0, s=1.0, tau_ref=3.0)
    a.init_fields(2)
    b.init_fields(2)
    a.step(7, 1.3, 0.1)
    for j in range(7):
        b.step(1, 1.3 + j * 0.1, 0.1)
    assert np.array_equal(a.get_fields(), b.get_fields())
    a.close()
    b.close()


# ------------------------------------------------------------------ the paper's printed values (soft, but guarded)

def _table1():
    from pathlib import Path
    rows = {}
    for ln in (Path(__file__).parent / "golden" / "table1.txt").read_text().splitlines():
        if ln.strip() and not ln.startswith("#"):
            t = ln.split()
            rows[t[0]] = dict(p=float(t[1]), xi_l=(float(t[2]), float(t[3])), xi_w=(float(t[4]), float(t[5])),
                              v2_omega=(float(t[6]), float(t[7])), v2_phi=(float(t[8]), float(t[9])))
    return rows


def table1_run(ah, n, era_p, steps, every, fit_from, seed=1):
    """One s = 0 run of n^3 sites from tau = 1 with all read-outs every `every` steps: the slopes of xi_L and of the
    library's corrected xi_W (xi_w_corr, reading #13; no factor is applied in the tests) and the mean velocity
    estimators over the records with tau >= fit_from, plus the worst relative Gauss residual."""
    dt, tau0 = 0.1, 1.0
    sim = ah.Simulation(params=ah.make_params(n, s=0.0, p=era_p, tau_ref=tau0 + steps * dt))
    assert sim.get_kernel() == ah.KERNEL_TILED
    sim.init_fields(seed)
    recs = sim.step_diag(steps, tau0, dt, every)
    sim.close()
    tau = np.array([r["tau"] for r in recs])
    m = tau >= fit_from
    col = lambda key: np.array([r[key] for r in recs])[m]
    return dict(size=n, seed=seed, steps=steps, every=every, fit_range=[float(tau[m][0]), float(tau[-1])],
                xi_l_dot=float(np.polyfit(tau[m], col("xi_l"), 1)[0]), xi_w_dot=float(np.polyfit(tau[m], col("xi_w_corr"), 1)[0]),
                v2_phi=float(col("v2_phi").mean()), v2_omega=float(col("v2_omega").mean()),
                gauss_rel_max=float(max(r["gauss_rel"] for r in recs)))


def record_table1(got):
    """Printed, and written to gpurun_out/ when that directory exists (copied to profiles/ by hand)."""
    import json
    from pathlib import Path
    print(json.dumps(got))
    out = Path(__file__).resolve().parent.parent / "gpurun_out"
    if out.is_dir():
        (out / f"table1_{got['size']}_{got['era']}.json").write_text(json.dumps(got, indent=1) + "\n")


@pytest.mark.parametrize("era", ["radiation", "matter"])
def test_network_estimators_against_table1(ah, era):
    """End to end on the CUDA path, quick version: a 512^3, s = 0 run to half the light-crossing time (1270 steps,
    PAPER.md:63), read-outs every 10 steps, fit range [80, 128].

    Which printed row?  Table 1 has a 512^3 row (PAPER.md:153 / :160), but it is the EARLIER single-GPU code's
    (Correia & Martins 2020b, twelve runs), and it sits 0.03-0.04 above every row of this paper's own code in <v^2>
    (0.31 against 0.272 / 0.283 / 0.282 for 1024^3 ... 4096^3).  This build lands on this paper's own rows (the 1024^3
    run is compared like for like, within 3 printed sigma, in tests/test_gpu_fullsize.py) and NOT on the 2020b row: at
    512^3 it gives <v^2>_phi = 0.257 / 0.200 (radiation / matter) against 0.31 / 0.25 +- 0.01 printed, i.e. 5 sigma
    low, which this repository cannot resolve (the 2020b set-up is not in PAPER.md).  So this test keeps the bands of
    an unlike-box comparison with this paper's 1024^3 rows (one seed at half the box size: 0.035 on the velocities,
    0.08 on the slopes), bounds the distance to the 2020b row only loosely (0.07 / 0.09), and records both distances
    (profiles/r03_table1.md)."""
    rows = _table1()
    ref, ref512 = rows[era], rows[era + "_512"]
    got = table1_run(ah, 512, ref["p"], 1270, 10, 80.0)
    got.update(era=era, paper_1024=ref, paper_512_2020b=ref512)
    record_table1(got)
    for key, band, band512 in (("v2_phi", 0.035, 0.07), ("v2_omega", 0.035, 0.07), ("xi_l", 0.08, 0.09), ("xi_w", 0.08, 0.09)):
        mine = got[key if key.startswith("v2") else key + "_dot"]
        assert abs(mine - ref[key][0]) <= band, (key, mine, ref[key])
        assert abs(mine - ref512[key][0]) <= band512, (key, mine, ref512[key])
    assert got["v2_omega"] > got["v2_phi"]                  # as in every row of Table 1
    assert abs(got["xi_l_dot"] - got["xi_w_dot"]) <= 0.04   # "fully consistent" estimators
    assert got["gauss_rel_max"] < 1e-4                      # Gauss's law at fp32 round-off throughout (s = 0)
