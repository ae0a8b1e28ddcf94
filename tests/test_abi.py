"""CPU-side checks of the C-ABI library: it builds, loads without a GPU, exports every symbol
include/ah_b200.h declares, and its argument validation / host coefficient code behave as the
header says.  No compute call is made here (those are the -m gpu tests)."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def ahlib():
    from paper_2005_14454_b200 import build
    build.build()
    from paper_2005_14454_b200 import binding
    return binding


def test_header_symbols_all_exported(ahlib):
    headers = sorted((ROOT / "include").glob("*.h"))
    assert [h.name for h in headers] == ["ah_b200.h", "ah_b200_test.h"]
    declared = set()
    for h in headers:
        declared |= set(re.findall(r"\b(ah_[a-z0-9_]+)\s*\(", h.read_text()))
    declared -= {"ah_ctx"}
    # the product interface holds no test hooks
    public = set(re.findall(r"\b(ah_[a-z0-9_]+)\s*\(", headers[0].read_text()))
    assert not public & {"ah_test_trig", "ah_test_trig_fast", "ah_set_kernel", "ah_get_kernel", "ah_launch_count",
                         "ah_tiled_launch_info"}
    assert declared == set(ahlib.EXPORTS), f"header/binding mismatch: {declared ^ set(ahlib.EXPORTS)}"
    L = C.CDLL(str(ahlib.LIB_PATH))
    for name in declared:
        assert hasattr(L, name), f"libah_b200.so does not export {name}"


def test_no_torch_types_in_abi():
    header = (ROOT / "include" / "ah_b200.h").read_text()
    assert "torch" not in header.lower().replace("pytorch tensors", "")
    assert "at::" not in header and "std::" not in header


def test_version_and_last_error(ahlib):
    L = ahlib.lib()
    assert b"sm_100a" in L.ah_version()
    assert L.ah_last_error() is not None


def test_struct_layouts_match_header(ahlib):
    # int32 x3, double x8, int32 x2 -> 4*3 (+4 pad) + 8*8 + 4*2 = 88 bytes
    assert C.sizeof(ahlib.Params) == 88
    # double + 6 int64 + 16 double
    assert C.sizeof(ahlib.Diag) == 8 * 23


def test_tiled_launch_geometry(ahlib):
    """Host logic of the tiled kernel's launch: the z extent is covered, chunks are at most 64 planes, small
    lattices fill whole waves of 148 SMs x 2 resident CTAs, and unsupported lattices are refused."""
    resident = 148 * 2
    for n in (128, 256, 384, 512, 768, 1024):
        zc, ctas = ahlib.tiled_launch_info(n, n, n)
        cols = (n // 128) * -(-n // 6)
        assert 1 <= zc <= 64 and ctas == cols * -(-n // zc)
        if ctas < 6 * resident:                       # few waves: the last one must not be mostly empty
            waves = -(-ctas // resident)
            assert ctas / (waves * resident) >= 0.85, (n, zc, ctas)
    assert ahlib.tiled_launch_info(128, 128, 128) == (10, 286)      # one wave
    assert ahlib.tiled_launch_info(1024, 1024, 1024)[0] == 64
    zc, ctas = ahlib.tiled_launch_info(128, 1, 1)
    assert (zc, ctas) == (1, 1)
    zc, ctas = ahlib.tiled_launch_info(256, 16, 11)
    assert zc * -(-11 // zc) >= 11 and ctas == 2 * 3 * -(-11 // zc)
    # 64-site warp rows when nx is a multiple of 64 but not of 128: one x tile per 64 sites
    zc, ctas = ahlib.tiled_launch_info(64, 64, 64)
    assert ctas == 1 * 11 * -(-64 // zc) and 4 <= zc <= 64
    zc, ctas = ahlib.tiled_launch_info(192, 6, 4)
    assert ctas == 3 * 1 * -(-4 // zc)
    with pytest.raises(ahlib.AhError):
        ahlib.tiled_launch_info(32, 64, 64)
    with pytest.raises(ahlib.AhError):
        ahlib.tiled_launch_info(200, 8, 8)


def test_coeffs_closed_forms(ahlib):
    """delta = (alpha/2) p dt/tau, omega = (1-s) delta, a = (tau/tau_ref)^p, q = a^{2s}."""
    P = ahlib.make_params(8, s=1.0, p=2.0, tau_ref=129.0, alpha=2.0)
    a, q, d, w = ahlib.coeffs(P, 12.9, 0.1)
    assert a == pytest.approx(0.01, rel=1e-14)
    assert q == pytest.approx(1e-4, rel=1e-14)
    assert d == pytest.approx(2.0 * 0.1 / 12.9, rel=1e-14)
    assert w == 0.0
    P = ahlib.make_params(8, s=0.0, p=1.0)
    a, q, d, w = ahlib.coeffs(P, 4.0, 0.1)
    assert q == 1.0 and d == pytest.approx(0.025) and w == pytest.approx(0.025)
    P = ahlib.make_params(8, s=0.25, p=0.0)
    assert ahlib.coeffs(P, -3.0, 0.1) == (1.0, 1.0, 0.0, 0.0)
    # s < 0, the core-growth phase of PAPER.md:57: q = a^{2s} > 1 for a < 1, omega = (1-s) delta > delta
    P = ahlib.make_params(8, s=-0.5, p=1.0, tau_ref=8.0)
    a, q, d, w = ahlib.coeffs(P, 2.0, 0.1)
    assert a == pytest.approx(0.25, rel=1e-14) and q == pytest.approx(4.0, rel=1e-14)
    assert d == pytest.approx(0.05, rel=1e-14) and w == pytest.approx(0.075, rel=1e-14)
    with pytest.raises(ahlib.AhError) as ei:
        ahlib.coeffs(ahlib.make_params(8, p=1.0), 0.0, 0.1)
    assert ei.value.code == ahlib.AH_EINVAL


def test_create_validates_before_touching_cuda(ahlib):
    L = ahlib.lib()
    ctx = C.c_void_p()
    fake = (C.c_void_p * 20)(*[0x1000 * (i + 1) for i in range(20)])

    def create(P, ptrs=fake, nbufs=20, bytes_each=None):
        be = P.nx * P.ny * P.nz * (8 if P.fp64 else 4) if bytes_each is None else bytes_each
        return L.ah_create(C.byref(ctx), C.byref(P), ptrs, nbufs, be, None)

    assert create(ahlib.make_params(0)) == ahlib.AH_EINVAL
    assert create(ahlib.make_params(8, dx=0.0)) == ahlib.AH_EINVAL
    assert create(ahlib.make_params(8, s=1.0, p=1.0, tau_ref=0.0)) == ahlib.AH_EINVAL
    assert create(ahlib.make_params(8), nbufs=10) == ahlib.AH_EINVAL
    assert create(ahlib.make_params(8), bytes_each=17) == ahlib.AH_EINVAL
    assert b"bytes_each" in L.ah_last_error()
    nullbuf = (C.c_void_p * 20)(*[0x1000 * (i + 1) for i in range(19)] + [None])
    assert create(ahlib.make_params(8), ptrs=nullbuf) == ahlib.AH_EINVAL
    misaligned = (C.c_void_p * 20)(*[0x1000 * (i + 1) + 4 for i in range(20)])
    assert create(ahlib.make_params(8), ptrs=misaligned) == ahlib.AH_EINVAL
    dup = (C.c_void_p * 20)(*[0x1000] * 20)
    assert create(ahlib.make_params(8), ptrs=dup) == ahlib.AH_EINVAL
    assert not ctx.value
    # null context / null pointers
    assert L.ah_step(None, 1, 1.0, 0.1) == ahlib.AH_EINVAL
    assert L.ah_destroy(None) == ahlib.AH_OK
    assert L.ah_launch_count(None) == 0


def test_no_cpu_fallback_without_gpu(ahlib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        ahlib.Simulation(nx=8)


def test_product_does_not_import_oracle():
    """The product path must not route through oracle/ (only tests, smoke and bench's CPU legs may)."""
    bad = re.compile(r"(import\s+oracle|from\s+oracle|ah_oracle|ahref_|libah_oracle)")
    for path in (ROOT / "paper_2005_14454_b200").rglob("*"):
        if path.suffix in (".py", ".cu", ".cuh", ".h"):
            assert not bad.search(path.read_text()), f"{path} refers to the oracle"


def test_diag_combine_adds_counts_and_sums_and_takes_the_maximum(ahlib):
    """ah_diag_combine (host arithmetic of the z-slab read-outs): counts and the first eight sums add in the order
    given, the last sum (max |G|) takes the maximum; bad arguments are refused."""
    parts = [([1, 2, 3, 4, 5], [1.0, 2.0, 3.0, 4.0, 5.0, 6.0, 7.0, 8.0, 0.5]),
             ([10, 20, 30, 40, 50], [0.5] * 8 + [0.9]),
             ([2 ** 40, 0, 0, 0, 1], [1e-20] * 8 + [0.7])]
    counts, sums = ahlib.combine_partials(parts)
    assert counts == [11 + 2 ** 40, 22, 33, 44, 56]
    assert sums[:8] == [(a + 0.5) + 1e-20 for a in (1.0, 2.0, 3.0, 4.0, 5.0, 6.0, 7.0, 8.0)]
    assert sums[8] == 0.9
    assert ahlib.combine_partials(parts[:1]) == (parts[0][0], parts[0][1])
    L = ahlib.lib()
    ci, cf = (C.c_int64 * 5)(), (C.c_double * 9)()
    assert L.ah_diag_combine(0, ci, cf, ci, cf) == ahlib.AH_EINVAL
    assert L.ah_diag_combine(1, None, cf, ci, cf) == ahlib.AH_EINVAL
