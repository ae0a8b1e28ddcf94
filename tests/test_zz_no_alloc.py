"""ah_readout_noalloc: the read-outs for callers that may not allocate (include/ah_b200.h).

Every other read-out goes through an ah_ctx whose scratch comes from cudaMalloc.  A host that gave all device memory
to its own pool, a steering loop that must not pay cudaMalloc's device-wide synchronisation, or code inside someone
else's no-allocation region cannot make that call; for them the library keeps the per-block partial sums in a fixed
7 MiB device array of its own (65536 partials: lattices up to 512^3) and writes the totals to a caller-owned buffer.

What is checked here:
  * on the GPU: the totals equal what ah_diagnostics gives for the same snapshot — integers exactly, fp64 sums within
    the 1e-11 the fused-vs-standalone read-out tests use — on calls made one after the other WITHOUT clearing anything in
    between (the array is shared and keeps the previous call's contents: a large lattice first, then smaller ones, then
    a lattice that fills the array to its last entry);
  * without a GPU: sizes beyond the limit and bad arguments are refused with AH_EINVAL before any CUDA call.

The file name sorts after the other test files on purpose: pytest -x stops at the first failure, and a failure in this
add-on must not hide the parity tests.  The GPU test passes alone in a fresh process (its first call is then also the
first use of the library on the device) and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2005_14454_b200 import inputs

INTS = ("n_wind", "n_wind_xy", "n_wind_xz", "n_wind_yz", "n_near_branch", "n_big_plaq")
FLOATS = ("string_length", "xi_w", "xi_w_corr", "sum_pi2_L", "sum_grad2_L", "sum_L", "v2_phi", "gauss_max", "gauss_l2", "gauss_rel",
          "gauss_div_l2", "gauss_charge_l2", "xi_l", "sum_p_L", "sum_rho_L", "v2_omega")


@pytest.fixture(scope="module")
def ah():
    from paper_2005_14454_b200 import build
    build.build()
    from paper_2005_14454_b200 import binding
    return binding


def same_record(got, want):
    assert got["tau"] == want["tau"]
    for key in INTS:
        assert got[key] == want[key], (key, got[key], want[key])
    for key in FLOATS:
        assert got[key] == pytest.approx(want[key], rel=1e-11, abs=1e-300), (key, got[key], want[key])


def noalloc_record(ah, sim, tau, dt, dev_totals):
    """One call of the entry point on the simulation's current device arrays; the totals tensor is the caller's and is
    deliberately NOT cleared between calls."""
    ah.readout_noalloc(sim.P, sim.current_bufs(), tau, dt, dev_totals, stream=sim.stream)
    sim.synchronize()
    return ah.noalloc_totals_to_diag(sim.P, dev_totals.cpu().numpy(), tau)


@pytest.mark.gpu
def test_noalloc_readout_equals_diagnostics_on_calls_in_a_row(ah):
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    dt = 0.1
    dev_totals = torch.full((ah.NOALLOC_TOTALS_WORDS,), -1, dtype=torch.int64, device="cuda:0")

    # call 1 and call 2: one fp32 lattice of several blocks with ragged y and z, two snapshots three steps apart
    big = ah.Simulation(params=ah.make_params(128, 38, 21, s=1.0, p=1.0, tau_ref=3.0))
    big.set_fields(inputs.random_state(128, 38, 21, seed=41, th_amp=0.4))
    big.step(5, 1.0, dt)
    tau = 1.0 + 5 * dt
    first = noalloc_record(ah, big, tau, dt, dev_totals)
    same_record(first, big.diagnostics(tau, dt))
    assert first["n_wind"] > 0 and first["sum_L"] != 0.0
    big.step(3, tau, dt)
    tau += 3 * dt
    second = noalloc_record(ah, big, tau, dt, dev_totals)
    same_record(second, big.diagnostics(tau, dt))
    assert second["sum_L"] != first["sum_L"]          # a different snapshot, not a stale result

    # call 3: a much smaller fp64 lattice, so most of the shared array still holds call 2's partial sums
    small = ah.Simulation(params=ah.make_params(20, 12, 7, s=0.0, p=2.0, fp64=True))
    small.set_fields(inputs.random_state(20, 12, 7, seed=42, th_amp=0.4))
    small.step(4, 2.0, dt)
    third = noalloc_record(ah, small, 2.0 + 4 * dt, dt, dev_totals)
    same_record(third, small.diagnostics(2.0 + 4 * dt, dt))

    # call 4: a lattice that needs exactly the 65536 partial sums the array holds; one more plane is refused
    ny, nz = 4 * 256, 8 * 256
    full = ah.Simulation(params=ah.make_params(1, ny, nz, s=1.0, p=1.0, tau_ref=2.0))
    full.init_fields(9)
    full.step(2, 1.0, dt)
    fourth = noalloc_record(ah, full, 1.0 + 2 * dt, dt, dev_totals)
    same_record(fourth, full.diagnostics(1.0 + 2 * dt, dt))
    bufs = full.current_bufs()
    with pytest.raises(ah.AhError, match="65536") as err:
        ah.readout_noalloc(ah.make_params(1, ny, nz + 1), bufs, 1.0, dt, dev_totals, stream=full.stream)
    assert err.value.code == ah.AH_EINVAL

    # and the first lattice once more, after the array was filled to the brim by another one
    again = noalloc_record(ah, big, tau, dt, dev_totals)
    same_record(again, second)
    for sim in (big, small, full):
        sim.close()


def fake_fields(step=0x1000):
    return (C.c_void_p * 10)(*[0x10000 + step * i for i in range(10)])


def test_noalloc_readout_refuses_sizes_beyond_the_fixed_array(ah):
    """No GPU needed: the size limit and the argument checks come before the first CUDA call."""
    L = ah.lib()
    out = C.c_void_p(0x20000)
    for shape in ((1024, 1024, 1024), (513, 512, 512), (512, 516, 512), (1, 1024, 2049)):
        P = ah.make_params(*shape)
        assert L.ah_readout_noalloc(C.byref(P), fake_fields(), 1.0, 0.1, out, None) == ah.AH_EINVAL
        msg = L.ah_last_error().decode()
        assert "65536" in msg and "ah_diagnostics" in msg, msg
    assert ah.NOALLOC_MAX_PARTIALS == 65536 and ah.NOALLOC_TOTALS_WORDS * 8 == 112
    header = (ah._PKG.parent / "include" / "ah_b200.h").read_text()
    assert "#define AH_NOALLOC_MAX_PARTIALS 65536" in header


def test_noalloc_readout_argument_checks(ah):
    L = ah.lib()
    P = ah.make_params(64, 8, 8)
    out = C.c_void_p(0x20000)
    assert L.ah_readout_noalloc(None, fake_fields(), 1.0, 0.1, out, None) == ah.AH_EINVAL
    assert L.ah_readout_noalloc(C.byref(P), None, 1.0, 0.1, out, None) == ah.AH_EINVAL
    assert L.ah_readout_noalloc(C.byref(P), fake_fields(), 1.0, 0.1, None, None) == ah.AH_EINVAL
    holes = fake_fields()
    holes[3] = None
    assert L.ah_readout_noalloc(C.byref(P), holes, 1.0, 0.1, out, None) == ah.AH_EINVAL
    assert "dev_fields[3]" in L.ah_last_error().decode()
    odd = fake_fields()
    odd[6] = 0x10002
    assert L.ah_readout_noalloc(C.byref(P), odd, 1.0, 0.1, out, None) == ah.AH_EINVAL
    assert L.ah_readout_noalloc(C.byref(P), fake_fields(), 1.0, 0.1, C.c_void_p(0x20004), None) == ah.AH_EINVAL
    assert L.ah_readout_noalloc(C.byref(P), fake_fields(), 1.0, 0.0, out, None) == ah.AH_EINVAL     # dt
    assert L.ah_readout_noalloc(C.byref(P), fake_fields(), 0.0, 0.1, out, None) == ah.AH_EINVAL     # tau with p = 1
    # omega = (1 - s) delta = 1: s = 0, p = 1, alpha = 2 -> delta = dt / tau
    assert L.ah_readout_noalloc(C.byref(ah.make_params(64, 8, 8, s=0.0, p=1.0)), fake_fields(), 0.1, 0.1, out,
                                None) == ah.AH_EINVAL
    assert "omega" in L.ah_last_error().decode()
