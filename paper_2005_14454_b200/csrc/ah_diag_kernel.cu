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
#include <atomic>

#include "ah_kernels.h"
#include "ah_diag_site.cuh"

namespace ah {

namespace {

constexpr int DBX = 64, DBY = 4;   // block = 64 x 4 sites of a z plane ...
constexpr int DBZ = 8;             // ... marched over 8 consecutive planes

// neighbours straight from global memory (periodic wrap on the indices)
template <typename real>
struct GlobalSiteAccessor {
    const ConstFields<real> &in;
    int nx, ny, nz, x, y, z;
    __device__ __forceinline__ size_t at(int dx, int dy, int dz) const
    {
        int xx = x + dx, yy = y + dy, zz = z + dz;
        if (xx >= nx) xx -= nx;
        if (yy >= ny) yy -= ny;
        if (zz >= nz) zz -= nz;
        if (xx < 0) xx += nx;
        if (yy < 0) yy += ny;
        if (zz < 0) zz += nz;
        return (size_t)xx + (size_t)nx * ((size_t)yy + (size_t)ny * (size_t)zz);
    }
    __device__ __forceinline__ real phi_re(int dx, int dy, int dz) const { return in.f[PHI_RE][at(dx, dy, dz)]; }
    __device__ __forceinline__ real phi_im(int dx, int dy, int dz) const { return in.f[PHI_IM][at(dx, dy, dz)]; }
    __device__ __forceinline__ real th(int i, int dx, int dy, int dz) const { return in.f[TH_X + i][at(dx, dy, dz)]; }
    __device__ __forceinline__ real alpha(int dx, int dy, int dz) const
    {
        const size_t c = at(dx, dy, dz);
        return site_phase<real>(in.f[PHI_RE][c], in.f[PHI_IM][c]);
    }
    __device__ __forceinline__ real pi_re() const { return in.f[PI_RE][at(0, 0, 0)]; }
    __device__ __forceinline__ real pi_im() const { return in.f[PI_IM][at(0, 0, 0)]; }
    __device__ __forceinline__ real ep(int i) const { return in.f[EP_X + i][at(0, 0, 0)]; }
    __device__ __forceinline__ real ep_back(int i) const
    {
        return in.f[EP_X + i][at(i == 0 ? -1 : 0, i == 1 ? -1 : 0, i == 2 ? -1 : 0)];
    }
};

// The read-outs of one site into cnt / acc, with the per-plaquette integers in wi / nearf.  fp64 state: diag_site()
// (libm, neighbours through the accessor).  fp32 state inside the tiled kernel's domain (|th| < 2^16): the
// fixed-rounding arithmetic of ah_diag_site.cuh on inputs gathered from global memory — the bit patterns the fused
// DIAG instantiation of the tiled step kernel produces for the same site; outside the domain: diag_site().
__device__ __forceinline__ void site_readouts(const ConstFields<double> &in, const DiagCoef &k, int nx, int ny, int nz,
                                              int x, int y, int z, long long *cnt, double *acc, int *wi, int *nearf)
{
    const GlobalSiteAccessor<double> a{in, nx, ny, nz, x, y, z};
    diag_site<double>(a, k, cnt, acc, wi, nearf);
}

__device__ __forceinline__ void site_readouts(const ConstFields<float> &in, const DiagCoef &k, int nx, int ny, int nz,
                                              int x, int y, int z, long long *cnt, double *acc, int *wi, int *nearf)
{
    const GlobalSiteAccessor<float> a{in, nx, ny, nz, x, y, z};
    const size_t c = a.at(0, 0, 0), cx = a.at(1, 0, 0), cy = a.at(0, 1, 0), cz = a.at(0, 0, 1);
    const size_t cxy = a.at(1, 1, 0), cxz = a.at(1, 0, 1), cyz = a.at(0, 1, 1);
    const float *thx = in.f[TH_X], *thy = in.f[TH_Y], *thz = in.f[TH_Z];
    const float t0x = thx[c], t0y = thy[c], t0z = thz[c];
    const float ty_xp = thy[cx], tz_xp = thz[cx], tx_yp = thx[cy], tz_yp = thz[cy], tx_zp = thx[cz], ty_zp = thy[cz];
    const float tmax = fmaxf(fmaxf(fmaxf(fabsf(t0x), fabsf(t0y)), fmaxf(fabsf(t0z), fabsf(ty_xp))),
                             fmaxf(fmaxf(fabsf(tz_xp), fabsf(tx_yp)),
                                   fmaxf(fabsf(tz_yp), fmaxf(fabsf(tx_zp), fabsf(ty_zp)))));
    if (!(tmax < AH_READOUT_TH_LIMIT)) {
        diag_site<float>(a, k, cnt, acc, wi, nearf);
        return;
    }
    const float *pr = in.f[PHI_RE], *pi = in.f[PHI_IM];
    const float fr = pr[c], fi = pi[c];
    // D1
    const float Pxy = plaq_angle_f32(t0x, ty_xp, tx_yp, t0y), Pxz = plaq_angle_f32(t0x, tz_xp, tx_zp, t0z);
    const float Pyz = plaq_angle_f32(t0y, tz_yp, ty_zp, t0z);
    const SiteWinding sw = readout_winding(
        site_phase_fast(fr, fi), site_phase_fast(pr[cx], pi[cx]), site_phase_fast(pr[cy], pi[cy]),
        site_phase_fast(pr[cz], pi[cz]), site_phase_fast(pr[cxy], pi[cxy]), site_phase_fast(pr[cxz], pi[cxz]),
        site_phase_fast(pr[cyz], pi[cyz]), t0x, t0y, t0z, ty_xp, tz_xp, tx_yp, tz_yp, tx_zp, ty_zp, Pxy, Pxz, Pyz);
#pragma unroll
    for (int pq = 0; pq < 3; ++pq) {
        wi[pq] = sw.w[pq];
        nearf[pq] = sw.nearf[pq];
        cnt[pq] += abs(sw.w[pq]);
        cnt[DS_NEAR] += sw.nearf[pq];
        cnt[DS_BIG] += sw.big[pq];
    }
    // D2: hops with the tiled kernel's link variables
    float sx, cxv, sy, cyv, sz, czv;
    sincos_pi_f32(t0x, sx, cxv);
    sincos_pi_f32(t0y, sy, cyv);
    sincos_pi_f32(t0z, sz, czv);
    float hxr, hxi, hyr, hyi, hzr, hzi;
    hop_fwd_f32(cxv, sx, pr[cx], pi[cx], hxr, hxi);
    hop_fwd_f32(cyv, sy, pr[cy], pi[cy], hyr, hyi);
    hop_fwd_f32(czv, sz, pr[cz], pi[cz], hzr, hzi);
    const float pir = in.f[PI_RE][c], pii = in.f[PI_IM][c];
    const float ex = in.f[EP_X][c], ey = in.f[EP_Y][c], ez = in.f[EP_Z][c];
    float pi2L, gr2L, L, pL, rhoL;
    readout_lagrangian(fr, fi, readout_grad2(fr, fi, hxr, hxi, hyr, hyi, hzr, hzi, k.f_idx2),
                       readout_plaq_energy(Pxy, Pxz, Pyz, k.compact, k.f_idx4), pir, pii, ex, ey, ez, k, pi2L, gr2L, L,
                       pL, rhoL);
    // D3
    double G, div, charge;
    readout_gauss(fr, fi, pir, pii, ex, ey, ez, a.ep_back(0), a.ep_back(1), a.ep_back(2), k, G, div, charge);
    readout_accumulate(acc, pi2L, gr2L, L, pL, rhoL, G, div, charge);
}

// One partial per VIRTUAL block vb = (bx, by, bz) of 64 x 4 x 8 sites; the launched blocks take virtual blocks
// blockIdx.x, blockIdx.x + gridDim.x, ... so that the grid can be smaller than the number of virtual blocks.
// only_if != nullptr: the launch is a conditional re-evaluation (ah_api.cu): nothing happens unless *only_if != 0
// (launched with a small grid, since it normally exits at once).
template <typename real>
__global__ void __launch_bounds__(DBX * DBY)
diag_kernel(ConstFields<real> in, DiagCoef k, int nx, int ny, int nz, int z_lo, int z_hi, int nbx, int nby, int nvb,
            DiagPartial *partials, int8_t *w3, uint8_t *near3, const int *only_if)
{
    if (only_if != nullptr && *only_if == 0) return;
    __shared__ long long s_i[DBX * DBY / 32][DS_NINT];
    __shared__ double s_f[DBX * DBY / 32][DS_NFLT];
    for (int vb = blockIdx.x; vb < nvb; vb += gridDim.x) {
    const int vbx = vb % nbx, vby = (vb / nbx) % nby, vbz = vb / (nbx * nby);
    const int x = vbx * DBX + threadIdx.x;
    const int y = vby * DBY + threadIdx.y;
    const bool active = (x < nx) && (y < ny);

    long long cnt[DS_NINT] = {0, 0, 0, 0, 0};
    double acc[DS_NFLT] = {0, 0, 0, 0, 0, 0, 0, 0, 0};

    const int z_end = min(z_hi, z_lo + (vbz + 1) * DBZ);
    const size_t n = (size_t)nx * ny * nz;
    for (int z = z_lo + vbz * DBZ; active && z < z_end; ++z) {
        int wi[3], nearf[3];
        site_readouts(in, k, nx, ny, nz, x, y, z, cnt, acc, wi, nearf);
        const size_t c = (size_t)x + (size_t)nx * ((size_t)y + (size_t)ny * (size_t)z);
#pragma unroll
        for (int pq = 0; pq < 3; ++pq) {
            if (w3) w3[(size_t)pq * n + c] = (int8_t)wi[pq];
            if (near3) near3[(size_t)pq * n + c] = (uint8_t)nearf[pq];
        }
    }

    // ---- block reduction: warp shuffles, then 8 warps through shared memory
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
        partials[vb] = p;
    }
    __syncthreads();   // s_i, s_f are re-used by the next virtual block
    }
}

// Fixed-order total of the per-block partials: thread t sums partials t, t+1024, ... ; then a
// shared-memory tree.  One block.  The number of partials is n, or n_alt when *use_alt != 0 (the partials then
// come from the conditional re-evaluation by diag_kernel, which has its own grid).
__global__ void __launch_bounds__(1024)
diag_final_kernel(const DiagPartial *partials, int n, int n_alt, const int *use_alt, DiagPartial *result)
{
    if (use_alt != nullptr && *use_alt != 0) n = n_alt;
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

cudaError_t launch_diag_final(const DiagPartial *partials, int n, DiagPartial *result, cudaStream_t st, int n_alt,
                              const int *use_alt)
{
    diag_final_kernel<<<1, 1024, 0, st>>>(partials, n, n_alt, use_alt, result);
    return cudaGetLastError();
}

template <typename real>
cudaError_t launch_diag_partials(const ConstFields<real> &in, const DiagCoef &k, int nx, int ny, int nz, ZRange zr,
                                 DiagPartial *partials, int8_t *w3, uint8_t *near3, const int *only_if,
                                 cudaStream_t st)
{
    dim3 block(DBX, DBY, 1);
    const int nbx = (nx + DBX - 1) / DBX, nby = (ny + DBY - 1) / DBY, nbz = (zr.hi - zr.lo + DBZ - 1) / DBZ;
    const long long nvb = (long long)nbx * nby * nbz;
    if (nvb > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const int grid = (only_if != nullptr && nvb > 148 * 8) ? 148 * 8 : (int)nvb;
    diag_kernel<real><<<grid, block, 0, st>>>(in, k, nx, ny, nz, zr.lo, zr.hi, nbx, nby, (int)nvb, partials, w3, near3,
                                             only_if);
    return cudaGetLastError();
}

template <typename real>
cudaError_t launch_diag(const ConstFields<real> &in, const DiagCoef &k, int nx, int ny, int nz, ZRange zr,
                        DiagPartial *partials, DiagPartial *result, int8_t *w3, uint8_t *near3,
                        cudaStream_t st)
{
    cudaError_t e = launch_diag_partials<real>(in, k, nx, ny, nz, zr, partials, w3, near3, nullptr, st);
    if (e != cudaSuccess) return e;
    return launch_diag_final(partials, diag_num_blocks(nx, ny, zr.hi - zr.lo), result, st);
}

template cudaError_t launch_diag<float>(const ConstFields<float> &, const DiagCoef &, int, int, int, ZRange,
                                        DiagPartial *, DiagPartial *, int8_t *, uint8_t *, cudaStream_t);
template cudaError_t launch_diag<double>(const ConstFields<double> &, const DiagCoef &, int, int, int, ZRange,
                                         DiagPartial *, DiagPartial *, int8_t *, uint8_t *, cudaStream_t);
template cudaError_t launch_diag_partials<float>(const ConstFields<float> &, const DiagCoef &, int, int, int, ZRange,
                                                 DiagPartial *, int8_t *, uint8_t *, const int *, cudaStream_t);

// ------------------------------------------------------------------------- read-outs with no allocation
//
// ah_readout_noalloc (include/ah_b200.h): the two read-out kernels above, with the per-block partials in a fixed
// array that is part of the loaded library image instead of in memory a context obtained from cudaMalloc.  It exists
// for callers that must not allocate device memory when they want a read-out (see the header for who they are).
//
//   * Size: AH_NOALLOC_MAX_PARTIALS DiagPartial of 112 bytes = 7 MiB, resident on every GPU that loads the library
//     until the process exits.  One partial per block of 64 x 4 x 8 sites, so the largest lattice is 512^3
//     (or any other shape with ceil(nx/64) * ceil(ny/4) * ceil(nz/8) <= 65536).
//   * g_noalloc_partials as written in HOST code is only a handle for the runtime, not an address a kernel can use;
//     the device address is looked up once per device with cudaGetSymbolAddress (noalloc_scratch below) and that
//     pointer is what the kernels get.
//   * Nothing in the array has to be zero on entry: the first kernel writes partial vb for EVERY block vb < nvb
//     (thread 0 of a block stores its partial whether or not the block holds active sites) and the second kernel reads
//     exactly those nvb entries, so what an earlier, larger call left behind is never read and nothing is cleared.
//   * All calls on a device share the array: calls whose kernels can be in flight at the same time race on it.

namespace {

constexpr int NOALLOC_MAX_PARTIALS = 65536;
static __device__ __align__(256) DiagPartial g_noalloc_partials[NOALLOC_MAX_PARTIALS];

constexpr int NOALLOC_MAX_DEVICES = 64;
std::atomic<DiagPartial *> g_noalloc_ptr[NOALLOC_MAX_DEVICES];   // zero-initialised: not looked up yet

// Device address of g_noalloc_partials on the CURRENT device.  The first call per device asks the runtime (which may
// load the module on that device then); later calls read the cached pointer.  Two threads that both find the slot
// empty both ask and store the same value.
cudaError_t noalloc_scratch(DiagPartial **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
    DiagPartial *p = g_noalloc_ptr[dev].load(std::memory_order_acquire);
    if (p == nullptr) {
        e = cudaGetSymbolAddress((void **)&p, g_noalloc_partials);
        if (e != cudaSuccess) return e;
        if (p == nullptr) return cudaErrorInvalidSymbol;
        g_noalloc_ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return cudaSuccess;
}

}  // namespace

int diag_noalloc_capacity() { return NOALLOC_MAX_PARTIALS; }

template <typename real>
cudaError_t launch_diag_noalloc(const ConstFields<real> &in, const DiagCoef &k, int nx, int ny, int nz,
                                DiagPartial *result, cudaStream_t st)
{
    if (diag_num_blocks(nx, ny, nz) > NOALLOC_MAX_PARTIALS) return cudaErrorInvalidValue;   // callers check first
    DiagPartial *scratch = nullptr;
    cudaError_t e = noalloc_scratch(&scratch);
    if (e != cudaSuccess) return e;
    return launch_diag<real>(in, k, nx, ny, nz, ZRange{0, nz}, scratch, result, nullptr, nullptr, st);
}

template cudaError_t launch_diag_noalloc<float>(const ConstFields<float> &, const DiagCoef &, int, int, int,
                                                DiagPartial *, cudaStream_t);
template cudaError_t launch_diag_noalloc<double>(const ConstFields<double> &, const DiagCoef &, int, int, int,
                                                 DiagPartial *, cudaStream_t);

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

__global__ void test_trig_fast_kernel(const float *x, float *s, float *c, float *ss, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float sv, cv;
    sincos_pi_f32(x[i], sv, cv);
    s[i] = sv;
    c[i] = cv;
    ss[i] = sin_small_f32(x[i]);
}

cudaError_t launch_test_trig_fast(const float *x, float *s, float *c, float *ss, size_t n, cudaStream_t st)
{
    test_trig_fast_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(x, s, c, ss, n);
    return cudaGetLastError();
}

cudaError_t launch_test_trig(const float *x, float *s, float *c, float *ps, size_t n, cudaStream_t st)
{
    test_trig_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(x, s, c, ps, n);
    return cudaGetLastError();
}

}  // namespace ah
