// ah_common.cuh — shared device-side definitions of the B200 Abelian-Higgs library.
//
// Notation follows the paper (arXiv:2005.14454) and DESIGN.md: phi, Pi on sites,
// th_i = lattice A_i (link angle of Eq. 12), ep_i = lattice E_i (Eq. 10),
// U_i = exp(-i th_i).  This file holds no code shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace ah {

// Per-step scalars, computed on the host in fp64 (ah_api.cu: make_coef) from
// PAPER.md:78-80 and Eqs. 7-8, then rounded once to the kernel's real type.
template <typename real>
struct StepCoef {
    real idx2;      // 1/dx^2
    real c1;        // (1-delta)/(1+delta)            Eq. 7
    real c2;        // dt/(1+delta)
    real w1;        // (1-omega)/(1+omega)            Eq. 8
    real w2;        // dt/(1+omega)
    real half_lam_q;// lambda0 * a^{2s} / 2           Eq. 7
    real sig2;      // sigma^2
    real two_e2_q;  // 2 e0^2 a^{2s}                  Eq. 8
    real dt;        // Delta eta                      Eqs. 9-10
    int compact;    // 1: sin(Phi) force; 0: Phi      reading #10
};

// Diagnostic-step scalars (SURVEY 8(c) diagnostics block).
struct DiagCoef {
    double idx2;        // 1/dx^2
    double q;           // a^{2s} at tau
    double quarter_lam_q;// lambda0 q / 4
    double sig2;
    double inv_2e2q;    // 1/(2 e0^2 q)
    double two_e2_kappa;// 2 e0^2 kappa, kappa = q (1-delta)/(1-omega)   reading #18
    int compact;
    int winding;        // 1: all read-outs; 0: no winding read-out D1 (fused DIAG instantiation only; the
                        // standalone kernel always evaluates everything and the API masks the record)
    // the same scalars rounded once to fp32 on the host, for the fp32 read-out arithmetic
    float f_idx2, f_idx4, f_quarter_lam_q, f_sig2, f_inv_2e2q;
};

template <typename real>
struct Fields {            // 10 SoA arrays, order of ah_b200.h
    real *f[10];
};
template <typename real>
struct ConstFields {
    const real *f[10];
};

enum { PHI_RE = 0, PHI_IM, PI_RE, PI_IM, TH_X, TH_Y, TH_Z, EP_X, EP_Y, EP_Z };

// Planes lo .. hi-1 of the nz allocated ones that a launch updates / reads out.  {0, nz}: the whole periodic lattice.
// A z slab of a multi-GPU run is allocated with one ghost plane below and above its own
// planes and uses {1, nz - 1}: the periodic wrap of the plane index is then never taken.
struct ZRange {
    int lo, hi;
};

// Number of partial-sum slots a diagnostics block writes.
enum {
    DS_NW_XY = 0, DS_NW_XZ, DS_NW_YZ, DS_NEAR, DS_BIG,   // integer counts (stored as double-exact int64)
    DS_NINT = 5,
    DF_SPI = 0, DF_SGR, DF_SL, DF_GSQ, DF_DIVSQ, DF_CHSQ, DF_SPL, DF_SRL, DF_GMAX,   // DF_GMAX (a maximum) stays last
    DS_NFLT = 9
};

struct DiagPartial {
    long long i[DS_NINT];
    double f[DS_NFLT];
};

// ----------------------------------------------------------------------------------- trig
//
// Link variables need cos/sin of an unbounded angle th (Eq. 10 never wraps it); plaquette
// forces need sin of a (normally small) angle Phi.  fp32 path: round-to-nearest multiple of
// pi/2 (resp. pi) by the add-magic-constant trick, two-term Cody-Waite reduction with FMA
// (pi/2 = C1 + C2 to 48 bits, enough for |x| < 2^15), then odd/even polynomials whose coefficients
// are weighted least-squares (near-minimax) fits on Chebyshev nodes of the reduced interval, made
// once with numpy in fp64 and rounded to fp32; the fitting script is not part of the repository,
// the coefficients below are bounded by tests/test_gpu_parity.py::test_trig_against_fp64 and
// ::test_tiled_kernel_trig_against_fp64 (relative error of the polynomials 7.5e-9 / 2.3e-10 / 1.1e-8, i.e.
// below half an fp32 ulp).  Measured against fp64 in tests/test_gpu_parity.py::test_trig.
// Arguments beyond 2^15 take the libm path.  fp64 path: libm.

#define AH_TRIG_LIMIT 32768.0f

__device__ __forceinline__ void sincos_poly_f32(float x, float &s, float &c)
{
    const float magic = 12582912.0f;                          // 1.5 * 2^23
    const float t = fmaf(x, 0.6366197466850281f, magic);      // low mantissa bits = rint(x*2/pi)
    const float k = t - magic;
    float r = fmaf(k, -1.5707963705062866f, x);               // C1 = fl32(pi/2)
    r = fmaf(k, 4.371138828673793e-08f, r);                   // C2 = fl32(pi/2 - C1) (negative)
    const float r2 = r * r;
    // sin(r) = r + r^3 P(r^2) on |r| <= pi/4
    float ps = fmaf(r2, -0.00019482117204461247f, 0.008331847377121449f);
    ps = fmaf(ps, r2, -0.16666647791862488f);
    const float sr = fmaf(ps * r2, r, r);
    // cos(r) = 1 - r^2/2 + r^4 Q(r^2)
    float pc = fmaf(r2, 2.4440761990263127e-05f, -0.0013887434033676982f);
    pc = fmaf(pc, r2, 0.04166664928197861f);
    pc = fmaf(pc, r2, -0.5f);
    const float cr = fmaf(pc, r2, 1.0f);
    const unsigned q = __float_as_uint(t);
    const float s0 = (q & 1u) ? cr : sr;
    const float c0 = (q & 1u) ? sr : cr;
    s = __uint_as_float(__float_as_uint(s0) ^ ((q & 2u) << 30));
    c = __uint_as_float(__float_as_uint(c0) ^ (((q + 1u) & 2u) << 30));
}

__device__ __forceinline__ float sin_poly_f32(float x)
{
    const float magic = 12582912.0f;
    const float t = fmaf(x, 0.31830987334251404f, magic);     // rint(x/pi)
    const float k = t - magic;
    float r = fmaf(k, -3.1415927410125732f, x);               // fl32(pi)
    r = fmaf(k, 8.742277657347586e-08f, r);                   // fl32(pi - fl32(pi)) (negative)
    const float r2 = r * r;
    // sin(r) = r + r^3 P(r^2) on |r| <= pi/2
    float ps = fmaf(r2, 2.5971810373448534e-06f, -0.00019805048941634595f);
    ps = fmaf(ps, r2, 0.008332990109920502f);
    ps = fmaf(ps, r2, -0.16666655242443085f);
    const float sr = fmaf(ps * r2, r, r);
    return __uint_as_float(__float_as_uint(sr) ^ (__float_as_uint(t) << 31));   // (-1)^k
}

// Tiled-kernel variants (fewer instructions, no quadrant logic): reduce by multiples of pi to |r| <= pi/2,
// evaluate sin (degree 9) and cos (degree 10) there and flip both signs for odd multiples.  Absolute error
// <= 1.5e-7 for |x| < 2^18 (two-term Cody-Waite with FMA: pi = C1 + C2 to 48 bits).
__device__ __forceinline__ void sincos_pi_f32(float x, float &s, float &c)
{
    const float magic = 12582912.0f;                          // 1.5 * 2^23
    const float t = fmaf(x, 0.31830987334251404f, magic);     // low mantissa bits = rint(x/pi)
    const float k = t - magic;
    float r = fmaf(k, -3.1415927410125732f, x);               // fl32(pi)
    r = fmaf(k, 8.742277657347586e-08f, r);                   // fl32(pi - fl32(pi)) (negative)
    const float r2 = r * r;
    float ps = fmaf(r2, 2.5971810373448534e-06f, -0.00019805048941634595f);
    ps = fmaf(ps, r2, 0.008332990109920502f);
    ps = fmaf(ps, r2, -0.16666655242443085f);
    const float sr = fmaf(ps * r2, r, r);
    float pc = fmaf(r2, -2.605479494377505e-07f, 2.4762006432865746e-05f);
    pc = fmaf(pc, r2, -0.0013888449175283313f);
    pc = fmaf(pc, r2, 0.04166664928197861f);
    pc = fmaf(pc, r2, -0.5f);
    const float cr = fmaf(pc, r2, 1.0f);
    const unsigned sign = __float_as_uint(t) << 31;           // (-1)^k
    s = __uint_as_float(__float_as_uint(sr) ^ sign);
    c = __uint_as_float(__float_as_uint(cr) ^ sign);
}

// sin(x) for |x| < AH_SMALL_ANGLE = 0.5: x - x^3/6 + x^5/120 - x^7/5040, truncation x^9/9! <= 1.1e-8 |x|
#define AH_SMALL_ANGLE 0.5f
__device__ __forceinline__ float sin_small_f32(float x)
{
    const float x2 = x * x;
    float p = fmaf(x2, -1.9841270e-4f, 8.3333333e-3f);
    p = fmaf(p, x2, -1.6666667e-1f);
    return fmaf(p * x2, x, x);
}

// ---- packed pairs (sm_100a fma.rn.f32x2 -> SASS FFMA2: two fp32 FMAs per issued instruction; each half is the
// IEEE operation of the scalar code above, so results are bit-identical; constants are broadcast operands)
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
#define AH_C2(x) pack2((x), (x))

// sincos_pi_f32 on two angles at once
__device__ __forceinline__ void sincos_pi_f32x2(f32x2 x, f32x2 &s, f32x2 &c)
{
    const f32x2 t = fma2(x, AH_C2(0.31830987334251404f), AH_C2(12582912.0f));
    const f32x2 k = add2(t, AH_C2(-12582912.0f));
    f32x2 r = fma2(k, AH_C2(-3.1415927410125732f), x);
    r = fma2(k, AH_C2(8.742277657347586e-08f), r);
    const f32x2 r2 = mul2(r, r);
    f32x2 ps = fma2(r2, AH_C2(2.5971810373448534e-06f), AH_C2(-0.00019805048941634595f));
    ps = fma2(ps, r2, AH_C2(0.008332990109920502f));
    ps = fma2(ps, r2, AH_C2(-0.16666655242443085f));
    const f32x2 sr = fma2(mul2(ps, r2), r, r);
    f32x2 pc = fma2(r2, AH_C2(-2.605479494377505e-07f), AH_C2(2.4762006432865746e-05f));
    pc = fma2(pc, r2, AH_C2(-0.0013888449175283313f));
    pc = fma2(pc, r2, AH_C2(0.04166664928197861f));
    pc = fma2(pc, r2, AH_C2(-0.5f));
    const f32x2 cr = fma2(pc, r2, AH_C2(1.0f));
    const f32x2 sign = (t << 31) & 0x8000000080000000ull;     // (-1)^k of each half
    s = sr ^ sign;
    c = cr ^ sign;
}
// sin_small_f32 / sin_poly_f32 on two angles at once
__device__ __forceinline__ f32x2 sin_small_f32x2(f32x2 x)
{
    const f32x2 x2 = mul2(x, x);
    f32x2 p = fma2(x2, AH_C2(-1.9841270e-4f), AH_C2(8.3333333e-3f));
    p = fma2(p, x2, AH_C2(-1.6666667e-1f));
    return fma2(mul2(p, x2), x, x);
}
__device__ __forceinline__ f32x2 sin_poly_f32x2(f32x2 x)
{
    const f32x2 t = fma2(x, AH_C2(0.31830987334251404f), AH_C2(12582912.0f));
    const f32x2 k = add2(t, AH_C2(-12582912.0f));
    f32x2 r = fma2(k, AH_C2(-3.1415927410125732f), x);
    r = fma2(k, AH_C2(8.742277657347586e-08f), r);
    const f32x2 r2 = mul2(r, r);
    f32x2 ps = fma2(r2, AH_C2(2.5971810373448534e-06f), AH_C2(-0.00019805048941634595f));
    ps = fma2(ps, r2, AH_C2(0.008332990109920502f));
    ps = fma2(ps, r2, AH_C2(-0.16666655242443085f));
    const f32x2 sr = fma2(mul2(ps, r2), r, r);
    return sr ^ ((t << 31) & 0x8000000080000000ull);
}

// libm slow paths kept out of line: the hot loops stay small enough for the 32 KB instruction cache
static __device__ __noinline__ void sincos_slow_f32(float th, float *s, float *c) { sincosf(th, s, c); }
static __device__ __noinline__ float sin_slow_f32(float x) { return sinf(x); }

__device__ __forceinline__ void link_sincos(float th, float &s, float &c)
{
    sincos_poly_f32(th, s, c);
    if (!(fabsf(th) < AH_TRIG_LIMIT)) sincos_slow_f32(th, &s, &c);
}
__device__ __forceinline__ void link_sincos(double th, double &s, double &c) { sincos(th, &s, &c); }

__device__ __forceinline__ float plaq_sin(float x)
{
    float r = sin_poly_f32(x);
    if (!(fabsf(x) < AH_TRIG_LIMIT)) r = sin_slow_f32(x);
    return r;
}
__device__ __forceinline__ double plaq_sin(double x) { return sin(x); }

// ---- fp32 building blocks with a FIXED rounding sequence (explicit intrinsics, no compiler-chosen FMA
// contraction): the tiled step kernel, its fused read-outs and the standalone diagnostics kernel all evaluate
// these, so a quantity computed in two kernels is the same bit pattern in both.

// forward hop U_i(x) phi(x+i), U = cos th - i sin th (Eq. 12), from c = cos th_i(x), s = sin th_i(x)
__device__ __forceinline__ void hop_fwd_f32(float c, float s, float br, float bi, float &hr, float &hi)
{
    hr = __fmaf_rn(c, br, __fmul_rn(s, bi));
    hi = __fmaf_rn(c, bi, -__fmul_rn(s, br));
}
// hand-over conj(U_i(x)) phi(x) for the site x + i
__device__ __forceinline__ void hop_bwd_f32(float c, float s, float fr, float fi, float &hr, float &hi)
{
    hr = __fmaf_rn(c, fr, -__fmul_rn(s, fi));
    hi = __fmaf_rn(c, fi, __fmul_rn(s, fr));
}
// Phi_ij(x) = th_i(x) + th_j(x+i) - th_i(x+j) - th_j(x)   (Eqs. 14-15, reading #9), summed left to right
__device__ __forceinline__ float plaq_angle_f32(float th_i, float th_j_xi, float th_i_xj, float th_j)
{
    return __fadd_rn(__fadd_rn(__fadd_rn(th_i, th_j_xi), -th_i_xj), -th_j);
}

// ---- programmatic dependent launch (PTX griddepcontrol; sm_90+): the step kernels of consecutive steps are launched
// with cudaLaunchAttributeProgrammaticStreamSerialization, so the launch of kernel k+1 is processed while kernel k
// still runs.  pdl_wait() blocks until the preceding kernel of the stream has completed and its writes are visible;
// it precedes EVERY global access of a kernel launched that way (also on early-exit paths, so that completion of a
// kernel always implies completion of its predecessors).  pdl_launch_dependents() lets the next kernel's CTAs be
// scheduled as soon as there is room for them.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

#ifndef AH_PDL
#define AH_PDL 1   // 0 (measurements only): plain stream serialisation
#endif
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = AH_PDL;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ------------------------------------------------------------------------- block reduction

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ int warp_sum(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ long long warp_sum(long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

}  // namespace ah
