// ah_diag_site.cuh — the network read-outs of ONE site, written once and used by
// both the standalone diagnostics kernel (ah_diag_kernel.cu: neighbours from global memory) and the fused
// DIAG instantiation of the tiled step kernel (ah_tiled_kernel.cu: neighbours from the staged planes).
//
//   D1 winding     W_ij(x) = rint{[d_i(x) + d_j(x+i) - d_i(x+j) - d_j(x) + Phi_ij(x)] / 2 pi},
//                  d_i(x) = Arg(conj(phi(x)) U_i(x) phi(x+i))        (Eq. 16 right)
//   D2 <v^2>_phi   sums of |Pi|^2 L, sum_i |D+_i phi|^2 L, L          (Eqs. 17-18)
//   D3 Gauss       G = div ep / dx^2 - 2 e0^2 kappa Im(conj(phi) Pi)  (Eq. 5)
//
// Link phases.  d_i(x) = Arg(conj(phi(x)) U_i(x) phi(x+i)) is evaluated as the principal value of
// alpha(x+i) - alpha(x) - th_i(x) with alpha = Arg(phi): the same number up to rounding (a few 1e-7 rad in
// fp32, far inside the 1e-5 rad band that flags a plaquette as near-branch), but with ONE atan2 per site,
// shareable between the twelve links that touch it, instead of one sincos + atan2 per link use.  th is first
// reduced modulo 2 pi with a two-term Cody-Waite step so that large link angles lose nothing.  A site with
// phi == 0 exactly has no phase: alpha is NaN there and every link touching it gets d = 0 (the oracle's
// atan2(0,0) := 0 convention).
//
// Per-site terms are evaluated in the state's precision (the winding decision is taken in that precision on
// both sides of a parity test; the Gauss residual, a difference of nearly equal numbers, is evaluated in fp64
// from the stored values) and accumulated in fp64.
//
// The accessor A supplies the snapshot around the site (offsets are 0 or 1 in each direction):
//   a.phi_re(dx,dy,dz), a.phi_im(dx,dy,dz), a.th(i,dx,dy,dz)   old phi, th at x + (dx,dy,dz)
//   a.alpha(dx,dy,dz)                                           site_phase() of phi at x + (dx,dy,dz)
//   a.pi_re(), a.pi_im(), a.ep(i)                               Pi, ep_i at x
//   a.ep_back(i)                                                ep_i at x - i
#pragma once

#include "ah_common.cuh"

namespace ah {

template <typename real> struct DiagConsts;
template <> struct DiagConsts<float> {
    static __device__ __forceinline__ float pi() { return 3.14159265358979323846f; }
    static __device__ __forceinline__ float inv2pi() { return 0.15915494309189533577f; }
    static __device__ __forceinline__ float atan2r(float y, float x) { return atan2f(y, x); }
    static __device__ __forceinline__ float rintr(float x) { return rintf(x); }
};
template <> struct DiagConsts<double> {
    static __device__ __forceinline__ double pi() { return 3.14159265358979323846; }
    static __device__ __forceinline__ double inv2pi() { return 0.15915494309189533577; }
    static __device__ __forceinline__ double atan2r(double y, double x) { return atan2(y, x); }
    static __device__ __forceinline__ double rintr(double x) { return rint(x); }
};

// alpha = Arg(phi) in (-pi, pi], NaN when phi == 0
template <typename real>
__device__ __forceinline__ real site_phase(real re, real im)
{
    if (re == (real)0 && im == (real)0) return (real)NAN;
    return DiagConsts<real>::atan2r(im, re);
}

// y - 2 pi rint(y / 2 pi)
__device__ __forceinline__ float wrap_2pi(float y)
{
    const float magic = 12582912.0f;                          // 1.5 * 2^23
    const float k = fmaf(y, 0.15915494309189535f, magic) - magic;
    float r = fmaf(k, -6.2831854820251465f, y);               // fl32(2 pi)
    return fmaf(k, 1.7484555314695172e-07f, r);               // fl32(2 pi - fl32(2 pi)) (negative)
}
__device__ __forceinline__ double wrap_2pi(double y)
{
    return y - 6.283185307179586476925 * rint(y * 0.15915494309189533577);
}
// link angle modulo 2 pi (two-term Cody-Waite is exact enough for |th| < 2^20; beyond that, in fp64)
__device__ __forceinline__ float reduce_2pi(float th)
{
    if (!(fabsf(th) < 1048576.0f)) return (float)wrap_2pi((double)th);
    return wrap_2pi(th);
}
__device__ __forceinline__ double reduce_2pi(double th) { return wrap_2pi(th); }

// d = principal value of alpha_head - alpha_tail - th; 0 when either end has no phase
template <typename real>
__device__ __forceinline__ real diag_link_phase(real a_tail, real a_head, real th)
{
    const real y = (a_head - a_tail) - reduce_2pi(th);
    return (y == y) ? wrap_2pi(y) : (real)0;
}

// forward hop U_i(a) phi(b) with U = cos th - i sin th
template <typename real>
__device__ __forceinline__ void diag_hop(real th, real br, real bi, real &hr, real &hi)
{
    real s, c;
    link_sincos(th, s, c);
    hr = c * br + s * bi;
    hi = c * bi - s * br;
}

// Adds the site's contributions to cnt[DS_NINT], acc[DS_NFLT]; wi[3], nearf[3] receive the per-plaquette
// winding integers and near-branch flags (xy, xz, yz).
template <typename real, typename A>
__device__ __forceinline__ void diag_site(const A &a, const DiagCoef &k, long long *cnt, double *acc, int *wi,
                                          int *nearf)
{
    const real fr = a.phi_re(0, 0, 0), fi = a.phi_im(0, 0, 0);
    const real t0[3] = {a.th(0, 0, 0, 0), a.th(1, 0, 0, 0), a.th(2, 0, 0, 0)};
    // neighbour phi at x+i
    const real nr[3] = {a.phi_re(1, 0, 0), a.phi_re(0, 1, 0), a.phi_re(0, 0, 1)};
    const real ni[3] = {a.phi_im(1, 0, 0), a.phi_im(0, 1, 0), a.phi_im(0, 0, 1)};

    const real a0 = a.alpha(0, 0, 0);
    const real an[3] = {a.alpha(1, 0, 0), a.alpha(0, 1, 0), a.alpha(0, 0, 1)};

    // own forward hops (for the gradient energy) and link phases d_i(x)
    real hr[3], hi[3], d0[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        diag_hop<real>(t0[i], nr[i], ni[i], hr[i], hi[i]);
        d0[i] = diag_link_phase<real>(a0, an[i], t0[i]);
    }

    // ---- D1: three plaquettes (xy, xz, yz)
    const real lim = DiagConsts<real>::pi() - (real)1e-5;
    real Phi[3];
#pragma unroll
    for (int pq = 0; pq < 3; ++pq) {
        const int i = (pq == 2) ? 1 : 0;
        const int j = (pq == 0) ? 1 : 2;
        const int ix = (i == 0), iy = (i == 1);                 // unit vector of direction i (i is x or y)
        const int jy = (j == 1), jz = (j == 2);                 // unit vector of direction j (j is y or z)
        const real ac = a.alpha(ix, iy + jy, jz);               // alpha(x+i+j)
        const real th_j_i = a.th(j, ix, iy, 0);                 // th_j(x+i)
        const real th_i_j = a.th(i, 0, jy, jz);                 // th_i(x+j)
        const real d2 = diag_link_phase<real>(an[i], ac, th_j_i);   // d_j(x+i): link j from x+i to x+i+j
        const real d3 = diag_link_phase<real>(an[j], ac, th_i_j);   // d_i(x+j): link i from x+j to x+i+j
        const real d1 = d0[i], d4 = d0[j];
        Phi[pq] = t0[i] + th_j_i - th_i_j - t0[j];              // Eqs. 14-15, un-wrapped
        const real w = DiagConsts<real>::rintr((d1 + d2 - d3 - d4 + Phi[pq]) * DiagConsts<real>::inv2pi());
        wi[pq] = (int)w;
        nearf[pq] = (fabs(d1) >= lim) || (fabs(d2) >= lim) || (fabs(d3) >= lim) || (fabs(d4) >= lim);
        cnt[pq] += (wi[pq] < 0) ? -wi[pq] : wi[pq];
        cnt[DS_NEAR] += nearf[pq];
        cnt[DS_BIG] += (fabs(Phi[pq]) > lim) ? 1 : 0;
    }

    // ---- D2: Lagrangian density of the site (reading #15)
    const real idx2 = (real)k.idx2;
    const real pir = a.pi_re(), pii = a.pi_im();
    const real pi2 = pir * pir + pii * pii;
    real grad2 = 0, e2 = 0, b2 = 0;
    real e0v[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const real dr = hr[i] - fr, di = hi[i] - fi;
        grad2 += (dr * dr + di * di) * idx2;
        e0v[i] = a.ep(i);
        e2 += e0v[i] * e0v[i] * idx2;
    }
#pragma unroll
    for (int pq = 0; pq < 3; ++pq) {
        real pe;
        if (k.compact) {
            // 2(1 - cos Phi) = 4 sin^2(Phi/2): same number, no cancellation in fp32
            const real sh = plaq_sin(Phi[pq] * (real)0.5);
            pe = (real)4 * sh * sh;
        } else {
            pe = Phi[pq] * Phi[pq];
        }
        b2 += pe * idx2 * idx2;
    }
    const real m2 = fr * fr + fi * fi - (real)k.sig2;
    const real pot = (real)k.quarter_lam_q * m2 * m2;
    const real L = pi2 - grad2 - pot + (e2 - b2) * (real)k.inv_2e2q;
    acc[DF_SPI] += (double)pi2 * (double)L;
    acc[DF_SGR] += (double)grad2 * (double)L;
    acc[DF_SL] += (double)L;
    // Eq. 17 right, reading #17: energy density and isotropic pressure of the same five pieces
    const real eb = (e2 + b2) * (real)k.inv_2e2q;
    const real rho = pi2 + grad2 + pot + eb;
    const real prs = pi2 - grad2 * (real)(1.0 / 3.0) - pot + eb * (real)(1.0 / 3.0);
    acc[DF_SPL] += (double)prs * (double)L;
    acc[DF_SRL] += (double)rho * (double)L;

    // ---- D3: Gauss residual, fp64 from the stored values
    double div = 0.0;
#pragma unroll
    for (int i = 0; i < 3; ++i) div += (double)e0v[i] - (double)a.ep_back(i);
    div *= k.idx2;
    const double charge = k.two_e2_kappa * ((double)fr * (double)pii - (double)fi * (double)pir);
    const double G = div - charge;
    acc[DF_GSQ] += G * G;
    acc[DF_DIVSQ] += div * div;
    acc[DF_CHSQ] += charge * charge;
    acc[DF_GMAX] = fmax(acc[DF_GMAX], fabs(G));
}


// ======================================================================= fp32 read-outs, fixed rounding sequence
//
// The fused DIAG instantiation of the tiled step kernel evaluates the read-outs of a site from what the step
// already holds in registers for that site (own phi, th; forward hops; plaquette angles; the staged Pi, ep) and
// from a shared-memory table of site phases alpha = Arg(phi).  The routines below are that arithmetic, written
// with explicit rounding intrinsics so that the standalone diagnostics kernel, which gathers the same inputs from
// global memory, produces the SAME bit patterns site by site: integers (winding, flags) and max |G| are then equal
// between the two kernels and the fp64 sums differ only by the order of summation.  Domain: every link angle
// involved has |th| < 2^16 (the tiled kernel's domain); outside it the standalone kernel takes diag_site() above
// and the API replaces a fused record by a standalone one (ah_api.cu).

#define AH_READOUT_TH_LIMIT 65536.0f

// alpha = Arg(phi) in (-pi, pi], NaN when phi == 0: atan(t) = t P(t^2) on t = min/max in [0, 1] (own minimax fit,
// 8 coefficients, |error| <= 1.2e-7 + the 2-ulp division), then the octant / sign fix-ups.  Quadrant and sign come
// from exact comparisons, so the branch (-pi, pi] is that of atan2f; the value may differ from it by ~2.5e-7 rad,
// far inside the 1e-5 rad near-branch band of reading #14.
__device__ __forceinline__ float site_phase_fast(float re, float im)
{
    const float ax = fabsf(re), ay = fabsf(im);
    const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
    const float t = __fdividef(mn, mx);                        // 0/0 -> NaN: a site without a phase
    const float u = __fmul_rn(t, t);
    float p = __fmaf_rn(u, -0.003687542863190174f, 0.020418046042323112f);
    p = __fmaf_rn(p, u, -0.05361030250787735f);
    p = __fmaf_rn(p, u, 0.09452305734157562f);
    p = __fmaf_rn(p, u, -0.13822640478610992f);
    p = __fmaf_rn(p, u, 0.19925765693187714f);
    p = __fmaf_rn(p, u, -0.333274781703949f);
    p = __fmaf_rn(p, u, 0.9999983906745911f);
    p = __fmul_rn(p, t);
    p = (ay > ax) ? __fadd_rn(1.57079637050628662f, -p) : p;
    p = (re < 0.0f) ? __fadd_rn(3.14159274101257324f, -p) : p;
    return (mx == 0.0f) ? NAN : copysignf(p, im);
}

// y - 2 pi rint(y / 2 pi) with the rounding sequence pinned
__device__ __forceinline__ float wrap_2pi_fix(float y)
{
    const float magic = 12582912.0f;                          // 1.5 * 2^23
    const float k = __fadd_rn(__fmaf_rn(y, 0.15915494309189535f, magic), -magic);
    const float r = __fmaf_rn(k, -6.2831854820251465f, y);    // fl32(2 pi)
    return __fmaf_rn(k, 1.7484555314695172e-07f, r);          // fl32(2 pi - fl32(2 pi)) (negative)
}
// d = principal value of alpha_head - alpha_tail - th (|th| < 2^16); NaN when either end has no phase
__device__ __forceinline__ float link_phase_raw(float a_tail, float a_head, float th)
{
    return wrap_2pi_fix(__fadd_rn(__fadd_rn(a_head, -a_tail), -wrap_2pi_fix(th)));
}

struct SiteWinding {
    float absw[3];  // |W_xy|, |W_xz|, |W_yz| as exact small integers in fp32
    int w[3];       // the signed integers (dead code unless the caller uses them)
    int nearf[3];   // any of the four link phases within 1e-5 of +-pi
    int big[3];     // |Phi_ij| > pi - 1e-5
};

// one plaquette: W = rint{[d1 + d2 - d3 - d4 + Phi] / 2 pi} (Eq. 16 right, reading #13).  A link that touches a
// site without a phase (phi == 0 exactly) has d = NaN here and counts as d = 0 (the oracle's atan2(0,0) := 0):
// fmaxf drops NaNs from the near-branch test by itself, and the sum is redone with zeros only when it is NaN.
__device__ __forceinline__ void plaquette_winding(float d1, float d2, float d3, float d4, float Phi, float &absw, int &w,
                                                  int &nearf, int &big)
{
    const float lim = 3.14159274101257324f - 1e-5f;
    const float inv2pi = 0.15915494309189533577f;
    const float magic = 12582912.0f;   // 1.5 * 2^23
    float sum = __fadd_rn(__fadd_rn(__fadd_rn(__fadd_rn(d1, d2), -d3), -d4), Phi);
    if (sum != sum) {
        d1 = (d1 == d1) ? d1 : 0.0f; d2 = (d2 == d2) ? d2 : 0.0f;
        d3 = (d3 == d3) ? d3 : 0.0f; d4 = (d4 == d4) ? d4 : 0.0f;
        sum = __fadd_rn(__fadd_rn(__fadd_rn(__fadd_rn(d1, d2), -d3), -d4), Phi);
    }
    const float wf = __fadd_rn(__fmaf_rn(sum, inv2pi, magic), -magic);   // rint(sum / 2 pi), |.| < 2^22
    absw = fabsf(wf);
    w = (int)wf;
    nearf = fmaxf(fmaxf(fabsf(d1), fabsf(d2)), fmaxf(fabsf(d3), fabsf(d4))) >= lim;
    big = fabsf(Phi) > lim;
}

// D1 of one site.  a0 = alpha(x); ax, ay, az = alpha(x+i); axy, axz, ayz = alpha(x+i+j);
// t0* = th_*(x); t{j}_{i}p = th_j(x+i); P* = Phi_ij(x) (plaq_angle_f32).
__device__ __forceinline__ SiteWinding readout_winding(float a0, float ax, float ay, float az, float axy, float axz,
                                                       float ayz, float t0x, float t0y, float t0z, float ty_xp,
                                                       float tz_xp, float tx_yp, float tz_yp, float tx_zp,
                                                       float ty_zp, float Pxy, float Pxz, float Pyz)
{
    const float dx0 = link_phase_raw(a0, ax, t0x), dy0 = link_phase_raw(a0, ay, t0y), dz0 = link_phase_raw(a0, az, t0z);
    SiteWinding r;
    // xy: d_x(x) + d_y(x+x) - d_x(x+y) - d_y(x)
    plaquette_winding(dx0, link_phase_raw(ax, axy, ty_xp), link_phase_raw(ay, axy, tx_yp), dy0, Pxy, r.absw[0], r.w[0],
                      r.nearf[0], r.big[0]);
    // xz: d_x(x) + d_z(x+x) - d_x(x+z) - d_z(x)
    plaquette_winding(dx0, link_phase_raw(ax, axz, tz_xp), link_phase_raw(az, axz, tx_zp), dz0, Pxz, r.absw[1], r.w[1],
                      r.nearf[1], r.big[1]);
    // yz: d_y(x) + d_z(x+y) - d_y(x+z) - d_z(x)
    plaquette_winding(dy0, link_phase_raw(ay, ayz, tz_yp), link_phase_raw(az, ayz, ty_zp), dz0, Pyz, r.absw[2], r.w[2],
                      r.nearf[2], r.big[2]);
    return r;
}

// sum_{i<j} [2 (1 - cos Phi_ij)] / dx^4 of the three plaquettes owned by the site (compact; Phi^2 otherwise):
// 2(1 - cos Phi) = 4 sin^2(Phi/2), no cancellation in fp32
__device__ __forceinline__ float readout_plaq_energy(float Pxy, float Pxz, float Pyz, int compact, float idx4)
{
    float e0, e1, e2;
    if (compact) {
        const float s0 = sin_poly_f32(__fmul_rn(Pxy, 0.5f)), s1 = sin_poly_f32(__fmul_rn(Pxz, 0.5f));
        const float s2 = sin_poly_f32(__fmul_rn(Pyz, 0.5f));
        e0 = __fmul_rn(__fmul_rn(4.0f, s0), s0);
        e1 = __fmul_rn(__fmul_rn(4.0f, s1), s1);
        e2 = __fmul_rn(__fmul_rn(4.0f, s2), s2);
    } else {
        e0 = __fmul_rn(Pxy, Pxy);
        e1 = __fmul_rn(Pxz, Pxz);
        e2 = __fmul_rn(Pyz, Pyz);
    }
    return __fmul_rn(__fadd_rn(__fadd_rn(e0, e1), e2), idx4);
}

// sum_i |U_i phi(x+i) - phi|^2 / dx^2 from the three forward hops
__device__ __forceinline__ float readout_grad2(float fr, float fi, float hxr, float hxi, float hyr, float hyi,
                                               float hzr, float hzi, float idx2)
{
    const float ar = __fadd_rn(hxr, -fr), ai = __fadd_rn(hxi, -fi);
    const float br = __fadd_rn(hyr, -fr), bi = __fadd_rn(hyi, -fi);
    const float cr = __fadd_rn(hzr, -fr), ci = __fadd_rn(hzi, -fi);
    float g = __fmaf_rn(ar, ar, __fmul_rn(ai, ai));
    g = __fadd_rn(g, __fmaf_rn(br, br, __fmul_rn(bi, bi)));
    g = __fadd_rn(g, __fmaf_rn(cr, cr, __fmul_rn(ci, ci)));
    return __fmul_rn(g, idx2);
}

// D2 of one site (reading #15): L and its weighted companions |Pi|^2 L, grad2 L, and p L, rho L of the
// equation-of-state estimator (Eq. 17 right, reading #17) (fp32 terms, summed in fp64)
__device__ __forceinline__ void readout_lagrangian(float fr, float fi, float grad2, float b2, float pir, float pii,
                                                   float ex, float ey, float ez, const DiagCoef &k, float &pi2L,
                                                   float &gr2L, float &L, float &pL, float &rhoL)
{
    const float pi2 = __fmaf_rn(pir, pir, __fmul_rn(pii, pii));
    const float e2 = __fmul_rn(__fmaf_rn(ez, ez, __fmaf_rn(ey, ey, __fmul_rn(ex, ex))), k.f_idx2);
    const float m2 = __fadd_rn(__fmaf_rn(fr, fr, __fmul_rn(fi, fi)), -k.f_sig2);
    const float pot = __fmul_rn(__fmul_rn(k.f_quarter_lam_q, m2), m2);
    L = __fmaf_rn(__fadd_rn(e2, -b2), k.f_inv_2e2q, __fadd_rn(__fadd_rn(pi2, -grad2), -pot));
    pi2L = __fmul_rn(pi2, L);
    gr2L = __fmul_rn(grad2, L);
    const float eb = __fmul_rn(__fadd_rn(e2, b2), k.f_inv_2e2q);
    const float rho = __fadd_rn(__fadd_rn(__fadd_rn(pi2, grad2), pot), eb);
    const float prs = __fmaf_rn(eb, 0.333333343267440796f, __fadd_rn(__fmaf_rn(grad2, -0.333333343267440796f, pi2), -pot));
    pL = __fmul_rn(prs, L);
    rhoL = __fmul_rn(rho, L);
}

// D3 of one site, in fp64 from the stored fp32 values (a difference of nearly equal numbers)
__device__ __forceinline__ void readout_gauss(float fr, float fi, float pir, float pii, float ex, float ey, float ez,
                                              float exb, float eyb, float ezb, const DiagCoef &k, double &G,
                                              double &div, double &charge)
{
    div = __dmul_rn(__dadd_rn(__dadd_rn(__dadd_rn((double)ex, -(double)exb), __dadd_rn((double)ey, -(double)eyb)),
                              __dadd_rn((double)ez, -(double)ezb)),
                    k.idx2);
    charge = __dmul_rn(k.two_e2_kappa, __fma_rn((double)fr, (double)pii, -__dmul_rn((double)fi, (double)pir)));
    G = __dadd_rn(div, -charge);
}

// adds one site's D2 + D3 terms to the fp64 accumulators
__device__ __forceinline__ void readout_accumulate(double *acc, float pi2L, float gr2L, float L, float pL, float rhoL,
                                                   double G, double div, double charge)
{
    acc[DF_SPI] += (double)pi2L;
    acc[DF_SGR] += (double)gr2L;
    acc[DF_SL] += (double)L;
    acc[DF_SPL] += (double)pL;
    acc[DF_SRL] += (double)rhoL;
    acc[DF_GSQ] = __fma_rn(G, G, acc[DF_GSQ]);
    acc[DF_DIVSQ] = __fma_rn(div, div, acc[DF_DIVSQ]);
    acc[DF_CHSQ] = __fma_rn(charge, charge, acc[DF_CHSQ]);
    acc[DF_GMAX] = fmax(acc[DF_GMAX], fabs(G));
}

}  // namespace ah
