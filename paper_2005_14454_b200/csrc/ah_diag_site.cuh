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

}  // namespace ah
