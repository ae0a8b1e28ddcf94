// ah_site_kernel.cu — one-thread-per-site leapfrog step (any lattice shape, fp32 or fp64) and I0.
//
// This is the general kernel: it evaluates Eqs. 7-10 at one site per thread with
// every neighbour read straight from global memory through L1/L2.  It serves lattices the tiled
// kernel does not cover (nx not a multiple of 64, fp64 state) and is the algebra check of the
// tiled kernel (tests compare the two bit-for-bit-independent paths against the oracle).
#include "ah_kernels.h"

namespace ah {

// Eqs. 7-10 at the single site (x, y, z)
// S: storage type of the state; real: type of the arithmetic (S = real for the fp32 and fp64 builds; S = float,
// real = double is the mixed-precision variant: fp32 storage, every operation of the step in fp64)
template <typename S, typename real>
__device__ __forceinline__ void site_update(const ConstFields<S> &in, const Fields<S> &out,
                                            const StepCoef<real> &k, int nx, int ny, int nz, int x, int y, int z)
{
    const int xp = (x + 1 == nx) ? 0 : x + 1, xm = (x == 0) ? nx - 1 : x - 1;
    const int yp = (y + 1 == ny) ? 0 : y + 1, ym = (y == 0) ? ny - 1 : y - 1;
    const int zp = (z + 1 == nz) ? 0 : z + 1, zm = (z == 0) ? nz - 1 : z - 1;
    const size_t sxy = (size_t)nx * ny;
    auto at = [&](int xx, int yy, int zz) { return (size_t)xx + (size_t)nx * yy + sxy * zz; };
    const size_t c = at(x, y, z);
    const size_t ixp = at(xp, y, z), ixm = at(xm, y, z);
    const size_t iyp = at(x, yp, z), iym = at(x, ym, z);
    const size_t izp = at(x, y, zp), izm = at(x, y, zm);

    // reads convert to the arithmetic type
    struct Rd {
        const S *p;
        __device__ __forceinline__ real operator[](size_t i) const { return (real)p[i]; }
    };
    const Rd pr{in.f[PHI_RE]}, pi{in.f[PHI_IM]}, thx{in.f[TH_X]}, thy{in.f[TH_Y]}, thz{in.f[TH_Z]};

    const real fr = pr[c], fi = pi[c];
    const real tx = thx[c], ty = thy[c], tz = thz[c];

    // Eq. 12: U_i(x) = cos th_i - i sin th_i at x and at the three backward neighbours
    real sx, cx, sy, cy, sz, cz;
    link_sincos(tx, sx, cx);
    link_sincos(ty, sy, cy);
    link_sincos(tz, sz, cz);
    real sxm, cxm, sym, cym, szm, czm;
    link_sincos(thx[ixm], sxm, cxm);
    link_sincos(thy[iym], sym, cym);
    link_sincos(thz[izm], szm, czm);

    // forward hops F_i = U_i(x) phi(x+i); backward hops conj(U_i(x-i)) phi(x-i)   (Eq. 13)
    const real fxr = cx * pr[ixp] + sx * pi[ixp], fxi = cx * pi[ixp] - sx * pr[ixp];
    const real fyr = cy * pr[iyp] + sy * pi[iyp], fyi = cy * pi[iyp] - sy * pr[iyp];
    const real fzr = cz * pr[izp] + sz * pi[izp], fzi = cz * pi[izp] - sz * pr[izp];
    const real bxr = cxm * pr[ixm] - sxm * pi[ixm], bxi = cxm * pi[ixm] + sxm * pr[ixm];
    const real byr = cym * pr[iym] - sym * pi[iym], byi = cym * pi[iym] + sym * pr[iym];
    const real bzr = czm * pr[izm] - szm * pi[izm], bzi = czm * pi[izm] + szm * pr[izm];

    const real six = (real)6;
    const real lap_r = k.idx2 * ((fxr + bxr) + (fyr + byr) + (fzr + bzr) - six * fr);
    const real lap_i = k.idx2 * ((fxi + bxi) + (fyi + byi) + (fzi + bzi) - six * fi);

    // Eq. 7
    const real pot = k.half_lam_q * (fr * fr + fi * fi - k.sig2);
    const real pr_new = k.c1 * (real)in.f[PI_RE][c] + k.c2 * (lap_r - pot * fr);
    const real pi_new = k.c1 * (real)in.f[PI_IM][c] + k.c2 * (lap_i - pot * fi);

    // Eqs. 14-15: plaquette angles Phi_ij at x and at the backward neighbours (reading #9)
    auto F = [&](real phi) { return k.compact ? plaq_sin(phi) : phi; };
    const real thy_xp = thy[ixp], thz_xp = thz[ixp];
    const real thx_yp = thx[iyp], thz_yp = thz[iyp];
    const real thx_zp = thx[izp], thy_zp = thy[izp];
    const real s_xy = F(tx + thy_xp - thx_yp - ty);
    const real s_xz = F(tx + thz_xp - thx_zp - tz);
    const real s_yz = F(ty + thz_yp - thy_zp - tz);
    // Phi_xy(x-y), Phi_xz(x-z): plaquettes below the x link
    const size_t ixpym = at(xp, ym, z), ixpzm = at(xp, y, zm), iypzm = at(x, yp, zm);
    const size_t ixmyp = at(xm, yp, z), ixmzp = at(xm, y, zp), iymzp = at(x, ym, zp);
    const real s_xy_ym = F(thx[iym] + thy[ixpym] - tx - thy[iym]);
    const real s_xz_zm = F(thx[izm] + thz[ixpzm] - tx - thz[izm]);
    // Phi_xy(x-x), Phi_yz(x-z): plaquettes beside / below the y link
    const real s_xy_xm = F(thx[ixm] + ty - thx[ixmyp] - thy[ixm]);
    const real s_yz_zm = F(thy[izm] + thz[iypzm] - ty - thz[izm]);
    // Phi_xz(x-x), Phi_yz(x-y): plaquettes beside the z link
    const real s_xz_xm = F(thx[ixm] + tz - thx[ixmzp] - thz[ixm]);
    const real s_yz_ym = F(thy[iym] + tz - thy[iymzp] - thz[iym]);

    // sum_{j != i} [ sin Phi_ij(x) - sin Phi_ij(x-j) ] with Phi_ji = -Phi_ij
    const real curl_x = (s_xy - s_xy_ym) + (s_xz - s_xz_zm);
    const real curl_y = (s_xy_xm - s_xy) + (s_yz - s_yz_zm);
    const real curl_z = (s_xz_xm - s_xz) + (s_yz_ym - s_yz);

    // current Im[conj(phi) U_i phi(x+i)]
    const real jx = fr * fxi - fi * fxr;
    const real jy = fr * fyi - fi * fyr;
    const real jz = fr * fzi - fi * fzr;

    // Eq. 8
    const real ex_new = k.w1 * (real)in.f[EP_X][c] + k.w2 * (k.two_e2_q * jx - k.idx2 * curl_x);
    const real ey_new = k.w1 * (real)in.f[EP_Y][c] + k.w2 * (k.two_e2_q * jy - k.idx2 * curl_y);
    const real ez_new = k.w1 * (real)in.f[EP_Z][c] + k.w2 * (k.two_e2_q * jz - k.idx2 * curl_z);

    out.f[PI_RE][c] = (S)(pr_new);
    out.f[PI_IM][c] = (S)(pi_new);
    out.f[EP_X][c] = (S)(ex_new);
    out.f[EP_Y][c] = (S)(ey_new);
    out.f[EP_Z][c] = (S)(ez_new);
    // Eqs. 9-10
    out.f[PHI_RE][c] = (S)(fr + k.dt * pr_new);
    out.f[PHI_IM][c] = (S)(fi + k.dt * pi_new);
    out.f[TH_X][c] = (S)(tx + k.dt * ex_new);
    out.f[TH_Y][c] = (S)(ty + k.dt * ey_new);
    out.f[TH_Z][c] = (S)(tz + k.dt * ez_new);
}

template <typename real>
__global__ void __launch_bounds__(256)
site_step_kernel(ConstFields<real> in, Fields<real> out, StepCoef<real> k, int nx, int ny, int nz, int z_lo)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = z_lo + blockIdx.z;
    if (x >= nx || y >= ny) return;
    site_update<real, real>(in, out, k, nx, ny, nz, x, y, z);
}

// mixed precision: fp32 state, the whole step in fp64; results are rounded once, on the store
__global__ void __launch_bounds__(256)
site_step_mixed_kernel(ConstFields<float> in, Fields<float> out, StepCoef<double> k, int nx, int ny, int nz, int z_lo)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = z_lo + blockIdx.z;
    if (x >= nx || y >= ny) return;
    site_update<float, double>(in, out, k, nx, ny, nz, x, y, z);
}

cudaError_t launch_site_step_mixed(const ConstFields<float> &in, const Fields<float> &out,
                                   const StepCoef<double> &k, int nx, int ny, int nz, ZRange zr, cudaStream_t st)
{
    dim3 block(nx >= 64 ? 64 : 32, nx >= 64 ? 4 : 8, 1);
    dim3 grid((nx + block.x - 1) / block.x, (ny + block.y - 1) / block.y, zr.hi - zr.lo);
    site_step_mixed_kernel<<<grid, block, 0, st>>>(in, out, k, nx, ny, nz, zr.lo);
    return cudaGetLastError();
}

// Conditional redo of one step (fixed small grid, grid-stride over sites): does nothing unless the tiled
// kernel raised *flag (a link angle outside its domain); then every site is recomputed with the libm
// paths above.  Thread 0 also clears the flag the NEXT step will use.
__global__ void __launch_bounds__(256)
site_redo_kernel(const int *flag, int *clear, ConstFields<float> in, Fields<float> out, StepCoef<float> k,
                 int nx, int ny, int nz, int z_lo, int z_hi)
{
    pdl_launch_dependents();
    pdl_wait();   // before the flag is read, and before the early exit (ah_common.cuh)
    if (blockIdx.x == 0 && threadIdx.x == 0) *clear = 0;
    if (*flag == 0) return;
    const size_t n = (size_t)nx * ny * (z_hi - z_lo);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % nx), y = (int)((i / nx) % ny), z = z_lo + (int)(i / ((size_t)nx * ny));
        site_update<float, float>(in, out, k, nx, ny, nz, x, y, z);
    }
}

cudaError_t launch_site_redo(const int *flag, int *clear, const ConstFields<float> &in, const Fields<float> &out,
                             const StepCoef<float> &k, int nx, int ny, int nz, ZRange zr, cudaStream_t st)
{
    return launch_pdl(site_redo_kernel, dim3(148 * 4), dim3(256), 0, st, flag, clear, in, out, k, nx, ny, nz, zr.lo, zr.hi);
}

// z slabs: a tiled launch checks the link angles of the planes it OWNS against its polynomial domain, and on a whole
// lattice every plane is owned by some CTA of the same launch.  A slab launch also reads planes it does not own: the
// two ghost planes (another context's), and, when the boundary planes are launched ahead of the interior, the plane
// next to each boundary plane.  This kernel raises the same flag for those planes BEFORE the step's launches, so that
// the conditional redo of every launch that reads them sees it.
__global__ void __launch_bounds__(256)
th_range_check_kernel(int *flag, const float *tx, const float *ty, const float *tz, size_t plane, int z0, int z1, int z2,
                      int z3, int np, float limit)
{
    const int zs[4] = {z0, z1, z2, z3};
    bool bad = false;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < plane * (size_t)np; i += (size_t)gridDim.x * blockDim.x) {
        const size_t at = (size_t)zs[i / plane] * plane + i % plane;
        bad |= !(fmaxf(fabsf(tx[at]), fmaxf(fabsf(ty[at]), fabsf(tz[at]))) < limit);
    }
    if (bad) *flag = 1;
}

cudaError_t launch_th_range_check(int *flag, const ConstFields<float> &in, int nx, int ny, const int *planes, int np,
                                  float limit, cudaStream_t st)
{
    if (np < 1 || np > 4) return cudaErrorInvalidValue;
    int z[4] = {planes[0], planes[0], planes[0], planes[0]};
    for (int a = 0; a < np; ++a) z[a] = planes[a];
    const size_t plane = (size_t)nx * ny;
    const size_t want = (plane * (size_t)np + 255) / 256;
    const unsigned grid = (unsigned)(want < 148 * 8 ? want : 148 * 8);
    th_range_check_kernel<<<grid, 256, 0, st>>>(flag, in.f[TH_X], in.f[TH_Y], in.f[TH_Z], plane, z[0], z[1], z[2], z[3], np,
                                                limit);
    return cudaGetLastError();
}

template <typename real>
cudaError_t launch_site_step(const ConstFields<real> &in, const Fields<real> &out,
                             const StepCoef<real> &k, int nx, int ny, int nz, ZRange zr, cudaStream_t st)
{
    dim3 block(nx >= 64 ? 64 : 32, nx >= 64 ? 4 : 8, 1);
    dim3 grid((nx + block.x - 1) / block.x, (ny + block.y - 1) / block.y, zr.hi - zr.lo);
    site_step_kernel<real><<<grid, block, 0, st>>>(in, out, k, nx, ny, nz, zr.lo);
    return cudaGetLastError();
}

template cudaError_t launch_site_step<float>(const ConstFields<float> &, const Fields<float> &,
                                             const StepCoef<float> &, int, int, int, ZRange, cudaStream_t);
template cudaError_t launch_site_step<double>(const ConstFields<double> &, const Fields<double> &,
                                              const StepCoef<double> &, int, int, int, ZRange, cudaStream_t);

// ------------------------------------------------------------------------------------ I0

// Counter-based uniform of DESIGN.md "I0": splitmix64 finaliser of seed + golden*(idx+1), top 24 bits.
__device__ __forceinline__ uint32_t u24(uint64_t seed, uint64_t idx)
{
    uint64_t z = seed + 0x9E3779B97F4A7C15ull * (idx + 1ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    return (uint32_t)(z >> 40);
}

template <typename real>
__global__ void __launch_bounds__(256)
init_kernel(Fields<real> out, uint64_t seed, double sigma, size_t sxy, size_t n, int nz_global, int z_offset)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    // linear index of the site in the GLOBAL lattice (a z slab's ghost planes get their periodic neighbours' values)
    int zg = (int)(i / sxy) + z_offset;
    zg %= nz_global;
    if (zg < 0) zg += nz_global;
    const uint64_t gi = (uint64_t)zg * sxy + (uint64_t)(i % sxy);
    // vartheta = 2 pi u, u = m / 2^24 exactly; evaluate the phase in fp64 so that fp32 and fp64
    // contexts start from the same point rounded once.
    const double u = (double)u24(seed, gi) * (1.0 / 16777216.0);
    double s, c;
    sincospi(2.0 * u, &s, &c);
    out.f[PHI_RE][i] = (real)(sigma * c);
    out.f[PHI_IM][i] = (real)(sigma * s);
#pragma unroll
    for (int a = 2; a < 10; ++a) out.f[a][i] = (real)0;
}

template <typename real>
cudaError_t launch_init(const Fields<real> &out, uint64_t seed, double sigma, int nx, int ny, int nz_alloc,
                        int nz_global, int z_offset, cudaStream_t st)
{
    const size_t sxy = (size_t)nx * ny, n = sxy * nz_alloc;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    init_kernel<real><<<blocks, 256, 0, st>>>(out, seed, sigma, sxy, n, nz_global, z_offset);
    return cudaGetLastError();
}
template cudaError_t launch_init<float>(const Fields<float> &, uint64_t, double, int, int, int, int, int, cudaStream_t);
template cudaError_t launch_init<double>(const Fields<double> &, uint64_t, double, int, int, int, int, int, cudaStream_t);

}  // namespace ah
