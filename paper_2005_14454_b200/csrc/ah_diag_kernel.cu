// ah_diag_kernel.cu — network read-outs of one snapshot.
//
//   D1 winding     W_ij(x) = rint{[d_i(x) + d_j(x+i) - d_i(x+j) - d_j(x) + Phi_ij(x)] / 2 pi},
//                  d_i(x) = Arg(conj(phi(x)) U_i(x) phi(x+i))        (Eq. 16 right)
//   D2 <v^2>_phi   sums of |Pi|^2 L, sum_i |D+_i phi|^2 L, L          (Eqs. 17-18)
//   D3 Gauss       G = div ep / dx^2 - 2 e0^2 kappa Im(conj(phi) Pi)  (Eq. 5)
//
// Per-site terms are evaluated in the state's precision (the winding decision is taken in that
// precision on both sides of a parity test; the Gauss residual, a difference of nearly equal
// numbers, is evaluated in fp64 from the stored values), accumulated in fp64, reduced per block
// with warp shuffles, and summed over blocks in a fixed order by a second one-block kernel, so
// results are bit-reproducible run to run.
#include "ah_kernels.h"

namespace ah {

namespace {

constexpr int DBX = 64, DBY = 4;   // block = 64 x 4 sites of a z plane ...
constexpr int DBZ = 8;             // ... marched over 8 consecutive planes

template <typename real> struct Consts;
template <> struct Consts<float> {
    static __device__ __forceinline__ float pi() { return 3.14159265358979323846f; }
    static __device__ __forceinline__ float inv2pi() { return 0.15915494309189533577f; }
    static __device__ __forceinline__ float atan2r(float y, float x) { return atan2f(y, x); }
    static __device__ __forceinline__ float rintr(float x) { return rintf(x); }
};
template <> struct Consts<double> {
    static __device__ __forceinline__ double pi() { return 3.14159265358979323846; }
    static __device__ __forceinline__ double inv2pi() { return 0.15915494309189533577; }
    static __device__ __forceinline__ double atan2r(double y, double x) { return atan2(y, x); }
    static __device__ __forceinline__ double rintr(double x) { return rint(x); }
};

// forward hop U_i(a) phi(b) with U = cos th - i sin th
template <typename real>
__device__ __forceinline__ void hop(real th, real br, real bi, real &hr, real &hi)
{
    real s, c;
    link_sincos(th, s, c);
    hr = c * br + s * bi;
    hi = c * bi - s * br;
}

// d = Arg(conj(phi_a) h)
template <typename real>
__device__ __forceinline__ real link_phase(real ar, real ai, real hr, real hi)
{
    const real re = ar * hr + ai * hi;
    const real im = ar * hi - ai * hr;
    if (re == (real)0 && im == (real)0) return (real)0;
    return Consts<real>::atan2r(im, re);
}

template <typename real>
__global__ void __launch_bounds__(DBX * DBY)
diag_kernel(ConstFields<real> in, DiagCoef k, int nx, int ny, int nz, DiagPartial *partials,
            int8_t *w3, uint8_t *near3)
{
    const int x = blockIdx.x * DBX + threadIdx.x;
    const int y = blockIdx.y * DBY + threadIdx.y;
    const bool active = (x < nx) && (y < ny);

    long long cnt[DS_NINT] = {0, 0, 0, 0, 0};
    double acc[DS_NFLT] = {0, 0, 0, 0, 0, 0, 0};

    const int z_end = min(nz, ((int)blockIdx.z + 1) * DBZ);
    for (int z = blockIdx.z * DBZ; active && z < z_end; ++z) {
        const int xp = (x + 1 == nx) ? 0 : x + 1, xm = (x == 0) ? nx - 1 : x - 1;
        const int yp = (y + 1 == ny) ? 0 : y + 1, ym = (y == 0) ? ny - 1 : y - 1;
        const int zp = (z + 1 == nz) ? 0 : z + 1, zm = (z == 0) ? nz - 1 : z - 1;
        const size_t sxy = (size_t)nx * ny;
        auto at = [&](int xx, int yy, int zz) { return (size_t)xx + (size_t)nx * yy + sxy * zz; };
        const size_t c = at(x, y, z);
        const size_t ip[3] = {at(xp, y, z), at(x, yp, z), at(x, y, zp)};
        const size_t im[3] = {at(xm, y, z), at(x, ym, z), at(x, y, zm)};
        // (+,+) edge neighbours x+i+j for (xy, xz, yz)
        const size_t ipp[3] = {at(xp, yp, z), at(xp, y, zp), at(x, yp, zp)};

        const real *pr = in.f[PHI_RE], *pi = in.f[PHI_IM];
        const real *th[3] = {in.f[TH_X], in.f[TH_Y], in.f[TH_Z]};
        const real *ep[3] = {in.f[EP_X], in.f[EP_Y], in.f[EP_Z]};

        const real fr = pr[c], fi = pi[c];
        const real t0[3] = {th[0][c], th[1][c], th[2][c]};

        // own forward hops and link phases d_i(x)
        real hr[3], hi[3], d0[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            hop<real>(t0[i], pr[ip[i]], pi[ip[i]], hr[i], hi[i]);
            d0[i] = link_phase<real>(fr, fi, hr[i], hi[i]);
        }

        // ---- D1: three plaquettes (xy, xz, yz)
        const real lim = Consts<real>::pi() - (real)1e-5;
        real Phi[3];
#pragma unroll
        for (int pq = 0; pq < 3; ++pq) {
            const int i = (pq == 2) ? 1 : 0;
            const int j = (pq == 0) ? 1 : 2;
            // d_j(x+i): link j leaving x+i, ending at x+i+j
            real ar = pr[ip[i]], ai = pi[ip[i]], gr, gi;
            hop<real>(th[j][ip[i]], pr[ipp[pq]], pi[ipp[pq]], gr, gi);
            const real d2 = link_phase<real>(ar, ai, gr, gi);
            // d_i(x+j): link i leaving x+j, ending at x+i+j
            ar = pr[ip[j]];
            ai = pi[ip[j]];
            hop<real>(th[i][ip[j]], pr[ipp[pq]], pi[ipp[pq]], gr, gi);
            const real d3 = link_phase<real>(ar, ai, gr, gi);
            const real d1 = d0[i], d4 = d0[j];
            Phi[pq] = t0[i] + th[j][ip[i]] - th[i][ip[j]] - t0[j];   // Eqs. 14-15, un-wrapped
            const real w = Consts<real>::rintr((d1 + d2 - d3 - d4 + Phi[pq]) * Consts<real>::inv2pi());
            const int wi = (int)w;
            const int nearf = (fabs(d1) >= lim) || (fabs(d2) >= lim) || (fabs(d3) >= lim) ||
                              (fabs(d4) >= lim);
            cnt[pq] += (wi < 0) ? -wi : wi;
            cnt[DS_NEAR] += nearf;
            cnt[DS_BIG] += (fabs(Phi[pq]) > lim) ? 1 : 0;
            if (w3) w3[(size_t)pq * sxy * nz + c] = (int8_t)wi;
            if (near3) near3[(size_t)pq * sxy * nz + c] = (uint8_t)nearf;
        }

        // ---- D2: Lagrangian density of the site (reading #15)
        const real idx2 = (real)k.idx2;
        const real pir = in.f[PI_RE][c], pii = in.f[PI_IM][c];
        const real pi2 = pir * pir + pii * pii;
        real grad2 = 0, e2 = 0, b2 = 0;
        real e0v[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const real dr = hr[i] - fr, di = hi[i] - fi;
            grad2 += (dr * dr + di * di) * idx2;
            e0v[i] = ep[i][c];
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
        for (int i = 0; i < 3; ++i) div += (double)e0v[i] - (double)ep[i][im[i]];
        div *= k.idx2;
        const double charge = k.two_e2_kappa * ((double)fr * (double)pii - (double)fi * (double)pir);
        const double G = div - charge;
        acc[DF_GSQ] += G * G;
        acc[DF_DIVSQ] += div * div;
        acc[DF_CHSQ] += charge * charge;
        acc[DF_GMAX] = fmax(acc[DF_GMAX], fabs(G));
    }

    // ---- block reduction: warp shuffles, then 8 warps through shared memory
    __shared__ long long s_i[DBX * DBY / 32][DS_NINT];
    __shared__ double s_f[DBX * DBY / 32][DS_NFLT];
    const int tid = threadIdx.y * DBX + threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int a = 0; a < DS_NINT; ++a) cnt[a] = warp_sum(cnt[a]);
#pragma unroll
    for (int a = 0; a < DS_NFLT - 1; ++a) acc[a] = warp_sum(acc[a]);
    acc[DF_GMAX] = warp_max(acc[DF_GMAX]);
    if (lane == 0) {
#pragma unroll
        for (int a = 0; a < DS_NINT; ++a) s_i[warp][a] = cnt[a];
#pragma unroll
        for (int a = 0; a < DS_NFLT; ++a) s_f[warp][a] = acc[a];
    }
    __syncthreads();
    if (tid == 0) {
        DiagPartial p;
#pragma unroll
        for (int a = 0; a < DS_NINT; ++a) {
            long long v = 0;
            for (int w = 0; w < DBX * DBY / 32; ++w) v += s_i[w][a];
            p.i[a] = v;
        }
#pragma unroll
        for (int a = 0; a < DS_NFLT; ++a) {
            double v = 0;
            for (int w = 0; w < DBX * DBY / 32; ++w)
                v = (a == DF_GMAX) ? fmax(v, s_f[w][a]) : v + s_f[w][a];
            p.f[a] = v;
        }
        const size_t b = blockIdx.x + (size_t)gridDim.x * (blockIdx.y + (size_t)gridDim.y * blockIdx.z);
        partials[b] = p;
    }
}

// Fixed-order total of the per-block partials: thread t sums partials t, t+1024, ... ; then a
// shared-memory tree.  One block.
__global__ void __launch_bounds__(1024)
diag_final_kernel(const DiagPartial *partials, int n, DiagPartial *result)
{
    __shared__ long long s_i[1024];
    __shared__ double s_f[1024];
    const int t = threadIdx.x;
    DiagPartial mine;
    for (int a = 0; a < DS_NINT; ++a) mine.i[a] = 0;
    for (int a = 0; a < DS_NFLT; ++a) mine.f[a] = 0;
    for (int b = t; b < n; b += 1024) {
        const DiagPartial p = partials[b];
        for (int a = 0; a < DS_NINT; ++a) mine.i[a] += p.i[a];
        for (int a = 0; a < DS_NFLT; ++a)
            mine.f[a] = (a == DF_GMAX) ? fmax(mine.f[a], p.f[a]) : mine.f[a] + p.f[a];
    }
    for (int a = 0; a < DS_NINT; ++a) {
        s_i[t] = mine.i[a];
        __syncthreads();
        for (int o = 512; o > 0; o >>= 1) {
            if (t < o) s_i[t] += s_i[t + o];
            __syncthreads();
        }
        if (t == 0) result->i[a] = s_i[0];
        __syncthreads();
    }
    for (int a = 0; a < DS_NFLT; ++a) {
        s_f[t] = mine.f[a];
        __syncthreads();
        for (int o = 512; o > 0; o >>= 1) {
            if (t < o) s_f[t] = (a == DF_GMAX) ? fmax(s_f[t], s_f[t + o]) : s_f[t] + s_f[t + o];
            __syncthreads();
        }
        if (t == 0) result->f[a] = s_f[0];
        __syncthreads();
    }
}

}  // namespace

int diag_num_blocks(int nx, int ny, int nz)
{
    return ((nx + DBX - 1) / DBX) * ((ny + DBY - 1) / DBY) * ((nz + DBZ - 1) / DBZ);
}

template <typename real>
cudaError_t launch_diag(const ConstFields<real> &in, const DiagCoef &k, int nx, int ny, int nz,
                        DiagPartial *partials, DiagPartial *result, int8_t *w3, uint8_t *near3,
                        cudaStream_t st)
{
    dim3 block(DBX, DBY, 1);
    dim3 grid((nx + DBX - 1) / DBX, (ny + DBY - 1) / DBY, (nz + DBZ - 1) / DBZ);
    diag_kernel<real><<<grid, block, 0, st>>>(in, k, nx, ny, nz, partials, w3, near3);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    diag_final_kernel<<<1, 1024, 0, st>>>(partials, diag_num_blocks(nx, ny, nz), result);
    return cudaGetLastError();
}

template cudaError_t launch_diag<float>(const ConstFields<float> &, const DiagCoef &, int, int, int,
                                        DiagPartial *, DiagPartial *, int8_t *, uint8_t *, cudaStream_t);
template cudaError_t launch_diag<double>(const ConstFields<double> &, const DiagCoef &, int, int, int,
                                         DiagPartial *, DiagPartial *, int8_t *, uint8_t *, cudaStream_t);

// ------------------------------------------------------------------------- trig test hook

__global__ void test_trig_kernel(const float *x, float *s, float *c, float *ps, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float ss, cc;
    link_sincos(x[i], ss, cc);
    s[i] = ss;
    c[i] = cc;
    ps[i] = plaq_sin(x[i]);
}

cudaError_t launch_test_trig(const float *x, float *s, float *c, float *ps, size_t n, cudaStream_t st)
{
    test_trig_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(x, s, c, ps, n);
    return cudaGetLastError();
}

}  // namespace ah
