// ah_tiled_kernel.cu — the fused z-marching fp32 leapfrog step (Eqs. 7-10) for sm_100a.
//
// One launch = one whole step: Pi, ep from the old phi, th; then phi, th from the new Pi, ep; state read
// once and written once (80 B per site).  DESIGN.md "Kernels / tiled step" has the derivation.
//
// Decomposition
//   * a thread owns 4 consecutive x sites (128-bit coalesced SoA loads / stores), a warp one 128-site
//     row segment, a CTA a tile of 128 x TY sites; the CTA marches through a chunk of z planes;
//   * every link's U_i = exp(-i th_i) (Eq. 12) is evaluated ONCE (3 sincos per site) and every
//     plaquette sine (Eqs. 14-15) ONCE (3 per site); each is then handed to the other sites that use it:
//       x-1 neighbour : inside the thread, or warp shuffle from the lane to the left;
//       y-1 neighbour : through shared memory (double buffered, ONE __syncthreads per plane);
//       z-1 neighbour : carried in registers from the previous plane of the march;
//   * the raw old values at x+1, y+1, z+1 are plain global loads (the z+1 plane becomes the next
//     iteration's own plane and stays in registers; the y+1 row is an L1/L2 hit);
//   * one extra "helper" warp per CTA evaluates the shared quantities of the halo row y0-1 and, one
//     plane ahead, of the halo column x0-1, so the main warps never branch on tile edges.
//   Periodic wrap is applied to the row / plane / edge-column base offsets only (nx % 128 == 0).
#include "ah_kernels.h"

namespace ah {

namespace {

constexpr int TILE_X = 128;   // sites per warp row segment (32 lanes x 4)
constexpr unsigned FULL = 0xffffffffu;

struct V4 {
    float v[4];
};

__device__ __forceinline__ V4 ld4(const float *__restrict__ p)
{
    const float4 t = __ldg(reinterpret_cast<const float4 *>(p));
    V4 r;
    r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w;
    return r;
}
__device__ __forceinline__ void st4(float *__restrict__ p, const V4 &a)
{
    *reinterpret_cast<float4 *>(p) = make_float4(a.v[0], a.v[1], a.v[2], a.v[3]);
}
__device__ __forceinline__ float4 f4(const V4 &a) { return make_float4(a.v[0], a.v[1], a.v[2], a.v[3]); }

// value of the site to the right of this thread's 4th site: lane+1's first site, or (lane 31) the
// first site of the next row segment, loaded from `edge`
__device__ __forceinline__ float right_of(const V4 &a, const float *__restrict__ edge, int lane)
{
    float r = __shfl_down_sync(FULL, a.v[0], 1);
    if (lane == 31) r = __ldg(edge);
    return r;
}

template <bool COMPACT>
__device__ __forceinline__ float plaq_f(float phi)
{
    return COMPACT ? plaq_sin(phi) : phi;   // reading #10
}

}  // namespace

namespace {

// Shared quantities a site hands to its +x / +y / +z neighbours (all from OLD fields):
//   b_i  = conj(U_i(s)) phi(s)      the backward hop of Eq. 13 as seen from s+i
//   S_ij = sin Phi_ij(s)            Eqs. 14-15 (or Phi_ij itself when !COMPACT)
template <int TY, bool COMPACT>
__global__ void __launch_bounds__((TY + 1) * 32, ((TY + 1) * 32 <= 256) ? 2 : 1)
tiled_step_kernel(ConstFields<float> in, Fields<float> out, StepCoef<float> k, int nx, int ny, int nz, int zc)
{
    // [plane parity][row: 0 = halo row y0-1, r+1 = tile row r][b_y.re, b_y.im, S_xy, S_yz][lane] (4 x-sites each)
    __shared__ float4 s_row[2][TY + 1][4][32];
    // [plane parity][tile row]: (b_x.re, b_x.im, S_xy, S_xz) of the site x0-1 left of the row segment
    __shared__ float4 s_col[2][TY];

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int x0 = blockIdx.x * TILE_X, y0 = blockIdx.y * TY, z0 = blockIdx.z * zc;
    const int z1 = min(nz, z0 + zc);
    const size_t sxy = (size_t)nx * ny;
    const int xe = (x0 + TILE_X == nx) ? 0 : x0 + TILE_X;   // x right of the segment (periodic)
    const int xw = (x0 == 0) ? nx - 1 : x0 - 1;             // x left of the segment

    const float *__restrict__ PR = in.f[PHI_RE], *__restrict__ PI = in.f[PHI_IM];
    const float *__restrict__ TX = in.f[TH_X], *__restrict__ TY_ = in.f[TH_Y], *__restrict__ TZ = in.f[TH_Z];

    const float kA = k.c2 * k.idx2;    // weight of one hop in Pi+          (Eq. 7)
    const float kB = k.w2 * k.idx2;    // weight of one plaquette sine in ep+ (Eq. 8)
    const float kJ = k.w2 * k.two_e2_q;

    const bool is_main = w < TY;
    // ---- main-warp geometry: row y0+w, sites x0+4*lane .. +3
    const int y = y0 + w;
    const bool act = is_main && y < ny;
    const int yc = act ? y : 0;
    const int yp = (yc + 1 == ny) ? 0 : yc + 1;
    const size_t ro = (size_t)yc * nx + x0 + 4 * lane;   // own row
    const size_t ry = (size_t)yp * nx + x0 + 4 * lane;   // row y+1
    const size_t re = (size_t)yc * nx + xe;              // site right of the own segment
    // ---- helper-warp geometry: halo row y0-1 (its y+1 row is y0), and halo column x0-1
    const int yh = (y0 == 0) ? ny - 1 : y0 - 1;
    const size_t hro = (size_t)yh * nx + x0 + 4 * lane;
    const size_t hry = (size_t)y0 * nx + x0 + 4 * lane;
    const size_t hre = (size_t)yh * nx + xe;
    const int ycol = y0 + lane;                           // column site handled by this helper lane
    const bool col_act = !is_main && lane < TY && ycol < ny;
    const int ycolp = (ycol + 1 >= ny) ? 0 : ycol + 1;

    // halo column of plane zz -> s_col[zz & 1]   (helper lanes 0..TY-1)
    auto do_column = [&](int zz) {
        if (!col_act) return;
        const int zzp = (zz + 1 == nz) ? 0 : zz + 1;
        const size_t b = (size_t)zz * sxy + (size_t)ycol * nx;
        const float pr = __ldg(PR + b + xw), pi = __ldg(PI + b + xw);
        const float tx = __ldg(TX + b + xw), ty = __ldg(TY_ + b + xw), tz = __ldg(TZ + b + xw);
        const float ty_r = __ldg(TY_ + b + x0), tz_r = __ldg(TZ + b + x0);
        const float tx_yp = __ldg(TX + (size_t)zz * sxy + (size_t)ycolp * nx + xw);
        const float tx_zp = __ldg(TX + (size_t)zzp * sxy + (size_t)ycol * nx + xw);
        float s, c;
        link_sincos(tx, s, c);
        s_col[zz & 1][lane] = make_float4(c * pr - s * pi, c * pi + s * pr,
                                          plaq_f<COMPACT>(tx + ty_r - tx_yp - ty),
                                          plaq_f<COMPACT>(tx + tz_r - tx_zp - tz));
    };

    // ---- prologue: carry of the plane below the chunk (main), column of the first plane (helper)
    V4 c_pr, c_pi, c_tx, c_ty, c_tz;        // own old phi, th of the current plane
    V4 g_bzr, g_bzi, g_sxz, g_syz;          // b_z, S_xz, S_yz of the site below (z-1)
    if (act) {
        const int zm = (z0 == 0) ? nz - 1 : z0 - 1;
        const size_t oc = (size_t)z0 * sxy, om = (size_t)zm * sxy;
        c_pr = ld4(PR + oc + ro); c_pi = ld4(PI + oc + ro);
        c_tx = ld4(TX + oc + ro); c_ty = ld4(TY_ + oc + ro); c_tz = ld4(TZ + oc + ro);
        const V4 m_pr = ld4(PR + om + ro), m_pi = ld4(PI + om + ro);
        const V4 m_tx = ld4(TX + om + ro), m_ty = ld4(TY_ + om + ro), m_tz = ld4(TZ + om + ro);
        const V4 my_tz = ld4(TZ + om + ry);
        const float me_tz = right_of(m_tz, TZ + om + re, lane);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            float s, c;
            link_sincos(m_tz.v[j], s, c);
            g_bzr.v[j] = c * m_pr.v[j] - s * m_pi.v[j];
            g_bzi.v[j] = c * m_pi.v[j] + s * m_pr.v[j];
            const float tz_xp = (j < 3) ? m_tz.v[j < 3 ? j + 1 : 3] : me_tz;
            g_sxz.v[j] = plaq_f<COMPACT>(m_tx.v[j] + tz_xp - c_tx.v[j] - m_tz.v[j]);
            g_syz.v[j] = plaq_f<COMPACT>(m_ty.v[j] + my_tz.v[j] - c_ty.v[j] - m_tz.v[j]);
        }
    } else if (!is_main) {
        do_column(z0);
    }
    __syncthreads();

    // ---- march
    for (int z = z0; z < z1; ++z) {
        const int buf = z & 1;
        const int zp = (z + 1 == nz) ? 0 : z + 1;
        const size_t oc = (size_t)z * sxy, on = (size_t)zp * sxy;

        V4 n_pr, n_pi, n_tx, n_ty, n_tz;   // own old phi, th of plane z+1
        V4 P_r, P_i, E_x, E_z;             // Pi+, ep+ still lacking the terms that come from row y-1

        if (act) {
            n_pr = ld4(PR + on + ro); n_pi = ld4(PI + on + ro);
            n_tx = ld4(TX + on + ro); n_ty = ld4(TY_ + on + ro); n_tz = ld4(TZ + on + ro);
            const V4 y_pr = ld4(PR + oc + ry), y_pi = ld4(PI + oc + ry);
            const V4 y_tx = ld4(TX + oc + ry), y_tz = ld4(TZ + oc + ry);
            const V4 q_r = ld4(in.f[PI_RE] + oc + ro), q_i = ld4(in.f[PI_IM] + oc + ro);
            const V4 e_x = ld4(in.f[EP_X] + oc + ro), e_y = ld4(in.f[EP_Y] + oc + ro);
            const V4 e_z = ld4(in.f[EP_Z] + oc + ro);
            const float r_pr = right_of(c_pr, PR + oc + re, lane), r_pi = right_of(c_pi, PI + oc + re, lane);
            const float r_ty = right_of(c_ty, TY_ + oc + re, lane), r_tz = right_of(c_tz, TZ + oc + re, lane);

            V4 o_byr, o_byi, o_sxy, o_syz;   // for row y+1, through shared memory
            V4 E_y, h_bzr, h_bzi, h_sxz;     // h_*: this plane's hand-down to z+1 (with S_yz in o_syz)
            float l_bxr = 0.f, l_bxi = 0.f, l_sxy = 0.f, l_sxz = 0.f;   // from the site to the left
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float fr = c_pr.v[j], fi = c_pi.v[j];
                const float tx = c_tx.v[j], ty = c_ty.v[j], tz = c_tz.v[j];
                float sx, cx, sy, cy, sz, cz;
                link_sincos(tx, sx, cx);          // Eq. 12
                link_sincos(ty, sy, cy);
                link_sincos(tz, sz, cz);
                const int jn = (j < 3) ? j + 1 : 3;
                const float xr = (j < 3) ? c_pr.v[jn] : r_pr, xi = (j < 3) ? c_pi.v[jn] : r_pi;
                const float ty_xp = (j < 3) ? c_ty.v[jn] : r_ty, tz_xp = (j < 3) ? c_tz.v[jn] : r_tz;
                // forward hops U_i(s) phi(s+i)                                   (Eq. 13)
                const float fxr = cx * xr + sx * xi, fxi = cx * xi - sx * xr;
                const float fyr = cy * y_pr.v[j] + sy * y_pi.v[j], fyi = cy * y_pi.v[j] - sy * y_pr.v[j];
                const float fzr = cz * n_pr.v[j] + sz * n_pi.v[j], fzi = cz * n_pi.v[j] - sz * n_pr.v[j];
                // hand-overs conj(U_i(s)) phi(s)
                const float bxr = cx * fr - sx * fi, bxi = cx * fi + sx * fr;
                o_byr.v[j] = cy * fr - sy * fi; o_byi.v[j] = cy * fi + sy * fr;
                h_bzr.v[j] = cz * fr - sz * fi; h_bzi.v[j] = cz * fi + sz * fr;
                // plaquettes owned by s                                          (Eqs. 14-15)
                const float Sxy = plaq_f<COMPACT>(tx + ty_xp - y_tx.v[j] - ty);
                const float Sxz = plaq_f<COMPACT>(tx + tz_xp - n_tx.v[j] - tz);
                const float Syz = plaq_f<COMPACT>(ty + y_tz.v[j] - n_ty.v[j] - tz);
                o_sxy.v[j] = Sxy; o_syz.v[j] = Syz; h_sxz.v[j] = Sxz;
                // Eq. 7 without the x-1 (j == 0) and y-1 hops
                float ar = (fxr + fyr) + (fzr + g_bzr.v[j]) - 6.0f * fr;
                float ai = (fxi + fyi) + (fzi + g_bzi.v[j]) - 6.0f * fi;
                // Eq. 8 curls without the x-1 (j == 0) and y-1 plaquettes
                float cux = Sxy + (Sxz - g_sxz.v[j]);
                float cuy = (Syz - g_syz.v[j]) - Sxy;
                float cuz = -Sxz - Syz;
                if (j > 0) {
                    ar += l_bxr; ai += l_bxi; cuy += l_sxy; cuz += l_sxz;
                }
                const float pot = k.half_lam_q * (fr * fr + fi * fi - k.sig2);
                P_r.v[j] = k.c1 * q_r.v[j] + (kA * ar - k.c2 * (pot * fr));
                P_i.v[j] = k.c1 * q_i.v[j] + (kA * ai - k.c2 * (pot * fi));
                E_x.v[j] = k.w1 * e_x.v[j] + (kJ * (fr * fxi - fi * fxr) - kB * cux);
                E_y.v[j] = k.w1 * e_y.v[j] + (kJ * (fr * fyi - fi * fyr) - kB * cuy);
                E_z.v[j] = k.w1 * e_z.v[j] + (kJ * (fr * fzi - fi * fzr) - kB * cuz);
                l_bxr = bxr; l_bxi = bxi; l_sxy = Sxy; l_sxz = Sxz;
            }
            // y-1 hand-over for the row above
            s_row[buf][w + 1][0][lane] = f4(o_byr);
            s_row[buf][w + 1][1][lane] = f4(o_byi);
            s_row[buf][w + 1][2][lane] = f4(o_sxy);
            s_row[buf][w + 1][3][lane] = f4(o_syz);
            // x-1 terms of the first site: lane-1's last site, or (lane 0) the helper's column entry
            l_bxr = __shfl_up_sync(FULL, l_bxr, 1);
            l_bxi = __shfl_up_sync(FULL, l_bxi, 1);
            l_sxy = __shfl_up_sync(FULL, l_sxy, 1);
            l_sxz = __shfl_up_sync(FULL, l_sxz, 1);
            if (lane == 0) {
                const float4 cdat = s_col[buf][w];
                l_bxr = cdat.x; l_bxi = cdat.y; l_sxy = cdat.z; l_sxz = cdat.w;
            }
            P_r.v[0] += kA * l_bxr;
            P_i.v[0] += kA * l_bxi;
            E_y.v[0] -= kB * l_sxy;
            E_z.v[0] -= kB * l_sxz;
            // ep_y+ is complete: store it and th_y+ (Eq. 10)
            V4 t_y;
#pragma unroll
            for (int j = 0; j < 4; ++j) t_y.v[j] = c_ty.v[j] + k.dt * E_y.v[j];
            st4(out.f[EP_Y] + oc + ro, E_y);
            st4(out.f[TH_Y] + oc + ro, t_y);
            // roll the z hand-down
            g_bzr = h_bzr; g_bzi = h_bzi; g_sxz = h_sxz; g_syz = o_syz;
        } else if (!is_main) {
            // helper: shared quantities of the halo row y0-1 at plane z
            const V4 h_pr = ld4(PR + oc + hro), h_pi = ld4(PI + oc + hro);
            const V4 h_tx = ld4(TX + oc + hro), h_ty = ld4(TY_ + oc + hro), h_tz = ld4(TZ + oc + hro);
            const V4 hn_ty = ld4(TY_ + on + hro);
            const V4 hy_tx = ld4(TX + oc + hry), hy_tz = ld4(TZ + oc + hry);
            const float hr_ty = right_of(h_ty, TY_ + oc + hre, lane);
            V4 o_byr, o_byi, o_sxy, o_syz;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float s, c;
                link_sincos(h_ty.v[j], s, c);
                o_byr.v[j] = c * h_pr.v[j] - s * h_pi.v[j];
                o_byi.v[j] = c * h_pi.v[j] + s * h_pr.v[j];
                const float ty_xp = (j < 3) ? h_ty.v[j < 3 ? j + 1 : 3] : hr_ty;
                o_sxy.v[j] = plaq_f<COMPACT>(h_tx.v[j] + ty_xp - hy_tx.v[j] - h_ty.v[j]);
                o_syz.v[j] = plaq_f<COMPACT>(h_ty.v[j] + hy_tz.v[j] - hn_ty.v[j] - h_tz.v[j]);
            }
            s_row[buf][0][0][lane] = f4(o_byr);
            s_row[buf][0][1][lane] = f4(o_byi);
            s_row[buf][0][2][lane] = f4(o_sxy);
            s_row[buf][0][3][lane] = f4(o_syz);
            if (z + 1 < z1) do_column(z + 1);   // one plane ahead: ready before the main warps' next phase 1
        }

        __syncthreads();

        if (act) {
            // add what row y-1 hands over, finish Eqs. 7-10, store
            const float4 a = s_row[buf][w][0][lane], b = s_row[buf][w][1][lane];
            const float4 c = s_row[buf][w][2][lane], d = s_row[buf][w][3][lane];
            const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
            const float cv[4] = {c.x, c.y, c.z, c.w}, dv[4] = {d.x, d.y, d.z, d.w};
            V4 f_r, f_i, t_x, t_z;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                P_r.v[j] += kA * av[j];
                P_i.v[j] += kA * bv[j];
                E_x.v[j] += kB * cv[j];
                E_z.v[j] -= kB * dv[j];
                f_r.v[j] = c_pr.v[j] + k.dt * P_r.v[j];   // Eq. 9
                f_i.v[j] = c_pi.v[j] + k.dt * P_i.v[j];
                t_x.v[j] = c_tx.v[j] + k.dt * E_x.v[j];   // Eq. 10
                t_z.v[j] = c_tz.v[j] + k.dt * E_z.v[j];
            }
            st4(out.f[PI_RE] + oc + ro, P_r);
            st4(out.f[PI_IM] + oc + ro, P_i);
            st4(out.f[EP_X] + oc + ro, E_x);
            st4(out.f[EP_Z] + oc + ro, E_z);
            st4(out.f[PHI_RE] + oc + ro, f_r);
            st4(out.f[PHI_IM] + oc + ro, f_i);
            st4(out.f[TH_X] + oc + ro, t_x);
            st4(out.f[TH_Z] + oc + ro, t_z);
            c_pr = n_pr; c_pi = n_pi; c_tx = n_tx; c_ty = n_ty; c_tz = n_tz;
        }
    }
}

}  // namespace

// --------------------------------------------------------------------------------- launch

constexpr int TILE_Y = 7;    // 7 main warps + 1 helper = 256 threads, 2 CTAs per SM at 128 registers

bool tiled_supported(int nx, int ny, int nz) { return nx >= TILE_X && nx % TILE_X == 0 && ny >= 1 && nz >= 1; }

cudaError_t tiled_setup() { return cudaSuccess; }

// Planes per CTA: long chunks amortise the prologue (one extra plane of loads and a third of a
// plane of arithmetic), but the grid should still be many waves of 148 SMs x 2 resident CTAs.
int tiled_chunk(int nx, int ny, int nz)
{
    const long long cols = (long long)(nx / TILE_X) * ((ny + TILE_Y - 1) / TILE_Y);
    const long long want = 148LL * 2 * 8;            // >= 8 waves when the lattice allows it
    int zc = 64;
    while (zc > 8 && cols * ((nz + zc - 1) / zc) < want) zc >>= 1;
    return zc < nz ? zc : nz;
}

cudaError_t launch_tiled_step(const ConstFields<float> &in, const Fields<float> &out,
                              const StepCoef<float> &k, int nx, int ny, int nz, cudaStream_t st)
{
    if (!tiled_supported(nx, ny, nz)) return cudaErrorInvalidValue;
    const int zc = tiled_chunk(nx, ny, nz);
    dim3 grid(nx / TILE_X, (ny + TILE_Y - 1) / TILE_Y, (nz + zc - 1) / zc);
    dim3 block((TILE_Y + 1) * 32);
    if (grid.y > 65535u || grid.z > 65535u) return cudaErrorInvalidConfiguration;
    if (k.compact)
        tiled_step_kernel<TILE_Y, true><<<grid, block, 0, st>>>(in, out, k, nx, ny, nz, zc);
    else
        tiled_step_kernel<TILE_Y, false><<<grid, block, 0, st>>>(in, out, k, nx, ny, nz, zc);
    return cudaGetLastError();
}

}  // namespace ah
