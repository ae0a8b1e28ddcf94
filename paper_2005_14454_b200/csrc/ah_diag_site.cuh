// ah_diag_site.cuh — the network read-outs of ONE site, written once and used by
// both the standalone diagnostics kernel (ah_diag_kernel.cu: neighbours from global memory) and the fused
// DIAG instantiation of the tiled step kernel (ah_tiled_kernel.cu: neighbours from the staged planes).
//
//   D1 winding     W_ij(x) = rint{[d_i(x) + d_j(x+i) - d_i(x+j) - d_j(x) + Phi_ij(x)] / 2 pi},
//                  d_i(x) = Arg(conj(phi(x)) U_i(x) phi(x+i))        (Eq. 16 right)
//   D2 <v^2>_phi   sums of |Pi|^2 L, sum_i |D+_i phi|^2 L, L          (Eqs. 17-18)
//   D3 Gauss       G = div ep / dx^2 - 2 e0^2 kappa Im(conj(phi) Pi)  (Eq. 5)
//
// Per-site terms are evaluated in the state's precision (the winding decision is taken in that precision on
// both sides of a parity test; the Gauss residual, a difference of nearly equal numbers, is evaluated in fp64
// from the stored values) and accumulated in fp64.
//
// The accessor A supplies the snapshot around the site (offsets are 0 or 1 in each direction):
//   a.phi_re(dx,dy,dz), a.phi_im(dx,dy,dz), a.th(i,dx,dy,dz)   old phi, th at x + (dx,dy,dz)
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

// forward hop U_i(a) phi(b) with U = cos th - i sin th
template <typename real>
__device__ __forceinline__ void diag_hop(real th, real br, real bi, real &hr, real &hi)
{
    real s, c;
    link_sincos(th, s, c);
    hr = c * br + s * bi;
    hi = c * bi - s * br;
}

// d = Arg(conj(phi_a) h)
template <typename real>
__device__ __forceinline__ real diag_link_phase(real ar, real ai, real hr, real hi)
{
    const real re = ar * hr + ai * hi;
    const real im = ar * hi - ai * hr;
    if (re == (real)0 && im == (real)0) return (real)0;
    return DiagConsts<real>::atan2r(im, re);
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

    // own forward hops and link phases d_i(x)
    real hr[3], hi[3], d0[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        diag_hop<real>(t0[i], nr[i], ni[i], hr[i], hi[i]);
        d0[i] = diag_link_phase<real>(fr, fi, hr[i], hi[i]);
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
        const real cr = a.phi_re(ix, iy + jy, jz), ci = a.phi_im(ix, iy + jy, jz);   // phi(x+i+j)
        const real th_j_i = a.th(j, ix, iy, 0);                 // th_j(x+i)
        const real th_i_j = a.th(i, 0, jy, jz);                 // th_i(x+j)
        real gr, gi;
        // d_j(x+i): link j leaving x+i, ending at x+i+j
        diag_hop<real>(th_j_i, cr, ci, gr, gi);
        const real d2 = diag_link_phase<real>(nr[i], ni[i], gr, gi);
        // d_i(x+j): link i leaving x+j, ending at x+i+j
        diag_hop<real>(th_i_j, cr, ci, gr, gi);
        const real d3 = diag_link_phase<real>(nr[j], ni[j], gr, gi);
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
