// ah_tiled_kernel.cu — the fused z-marching fp32 leapfrog step (Eqs. 7-10) for sm_100a.
//
// One launch = one whole step: Pi, ep from the old phi, th; then phi, th from the new Pi, ep; state read
// once and written once (80 B per site).  DESIGN.md "Kernels / tiled step" has the derivation.
//
// Decomposition
//   * a thread owns SPT consecutive x sites, a warp one row segment of 32 SPT sites, a CTA a tile of
//     32 SPT x TY sites; the CTA marches through a chunk of z planes.  SPT = 4 (128-bit accesses, 128-site
//     rows) when nx % 128 == 0, else SPT = 2 (64-bit accesses, 64-site rows; needs nx % 64 == 0).  TY = 6
//     rows for the plain step, 5 for the DIAG instantiations (their read-out ring needs the shared memory);
//     the arithmetic of a site does not depend on the tile it falls in (slabs and the two tilings agree
//     bit for bit).  Numbers below are for SPT = 4;
//   * the OLD phi, th planes (the only fields with a stencil) are staged in shared memory with their
//     halo rows y0-1, y0+TY and halo columns x0-4..x0-1, x0+128..x0+131 by 1-D bulk TMA copies
//     (cp.async.bulk, one per field row, issued by one elected lane of the warp that owns the row) into
//     a 3-slot ring: plane z (own), z+1 (forward) in use, plane z+2 in flight for one whole iteration.
//     Completion is signalled on one mbarrier per slot.  The periodic wrap is applied to the row / plane
//     source addresses; tiles that touch the x boundary copy their two 16-byte halo columns separately;
//   * the OLD Pi, ep (read only at their own site) are staged per warp, one plane ahead, by the same
//     mechanism (one mbarrier per warp); all ten outputs go registers -> global (128-bit stores);
//     nothing the march waits on is a register-destination global load;
//   * every link's U_i = exp(-i th_i) (Eq. 12) is evaluated ONCE (3 sincos per site) and every
//     plaquette sine (Eqs. 14-15) ONCE (3 per site); each is then handed to the other sites that use it:
//       x-1 neighbour : inside the thread, or warp shuffle from the lane to the left;
//       y-1 neighbour : through shared memory (double buffered; ONE __syncthreads per plane);
//       z-1 neighbour : carried in registers from the previous plane of the march;
//   * warp TY (the "helper") copies the two halo rows, arms the plane barriers and evaluates the shared
//     quantities of the halo row y0-1 and of the halo column x0-1, so the main warps never branch on
//     tile edges;
//   * no libm in the march: polynomial sin / cos (ah_common.cuh) valid for |th| < 2^16; a link outside
//     raises a flag and the API redoes the step with the site kernel (ah_api.cu).
#include "ah_kernels.h"
#include "ah_diag_site.cuh"

namespace ah {

namespace {

constexpr int HALO = 4;                // staged halo columns on each side (16 bytes)
constexpr int NST = 3;                 // ring slots
constexpr int NRAW = 5;                // staged fields: phi_re, phi_im, th_x, th_y, th_z
constexpr unsigned FULL = 0xffffffffu;

// SPT consecutive x sites of one thread (4: 128-bit accesses, 128-site warp rows; 2: 64-bit, 64-site rows)
template <int SPT>
struct VN {
    float v[SPT];
};

template <int SPT>
__device__ __forceinline__ VN<SPT> ldsN(const float *p)
{
    VN<SPT> r;
    if constexpr (SPT == 4) {
        const float4 t = *reinterpret_cast<const float4 *>(p);
        r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w;
    } else {
        const float2 t = *reinterpret_cast<const float2 *>(p);
        r.v[0] = t.x; r.v[1] = t.y;
    }
    return r;
}
template <int SPT>
__device__ __forceinline__ VN<SPT> ldgN(const float *p)
{
    VN<SPT> r;
    if constexpr (SPT == 4) {
        const float4 t = __ldg(reinterpret_cast<const float4 *>(p));
        r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w;
    } else {
        const float2 t = __ldg(reinterpret_cast<const float2 *>(p));
        r.v[0] = t.x; r.v[1] = t.y;
    }
    return r;
}
template <int SPT>
__device__ __forceinline__ void stN(float *__restrict__ p, const VN<SPT> &a)
{
    if constexpr (SPT == 4) *reinterpret_cast<float4 *>(p) = make_float4(a.v[0], a.v[1], a.v[2], a.v[3]);
    else *reinterpret_cast<float2 *>(p) = make_float2(a.v[0], a.v[1]);
}
template <int SPT>
__device__ __forceinline__ float vmaxabs(const VN<SPT> &a)
{
    float m = fabsf(a.v[0]);
#pragma unroll
    for (int j = 1; j < SPT; ++j) m = fmaxf(m, fabsf(a.v[j]));
    return m;
}

// ---- mbarrier / bulk-copy primitives (PTX; SASS: SYNCS.*, UBLKCP)
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// L2 policies: the staged phi, th rows are read again by the neighbouring tiles (halo rows / columns) and by
// the next z chunk, so they should outlive the read-once Pi, ep rows and the streamed outputs in L2
__device__ __forceinline__ unsigned long long l2_policy_keep()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long l2_policy_stream()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void bulk_g2s_hint(float *dst, const float *src, unsigned bytes, unsigned long long *bar,
                                              unsigned long long policy)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(float *dst, const float *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// one lane of a converged warp (SASS: ELECT); lets the compiler issue what follows once, with uniform operands
__device__ __forceinline__ bool elect_one()
{
    unsigned p;
    asm volatile(
        "{\n"
        ".reg .pred P;\n"
        "elect.sync _|P, 0xffffffff;\n"
        "selp.u32 %0, 1, 0, P;\n"
        "}\n"
        : "=r"(p));
    return p != 0;
}

template <bool COMPACT>
__device__ __forceinline__ float plaq_f(float phi)
{
    return COMPACT ? sin_poly_f32(phi) : phi;   // reading #10; range check by the caller
}

template <int SPT, int TY, bool DIAG>
struct Smem {
    static constexpr int TX = 32 * SPT;        // sites per warp row segment
    static constexpr int RF = TX + 2 * HALO;   // floats per staged row
    float raw[NST][NRAW][TY + 2][RF];     // staged planes; row r <-> y0 - 1 + r, column c <-> x0 - HALO + c
    float qe[TY][NRAW][TX];               // staged old Pi, ep of the own rows (one plane): pi_re, pi_im, ep_x, ep_y, ep_z
    // y hand-over: (b_y.re, b_y.im, S_xy, S_yz); row 0 = halo row y0-1, row w+1 from warp w.  Double buffered
    // (one barrier per plane).  DIAG: after warp w has consumed row w of a buffer it re-uses the first 128 floats
    // of that row as scratch (the sites' gradient energies, handed from the step to the read-out loop)
    float row[2][TY][4][TX];
    // DIAG: alpha = Arg(phi) (ah_diag_site.cuh) of the staged rows 1 .. TY+1 (columns HALO .. HALO+128) of the
    // plane held by the ring slot of the same index
    float alpha[DIAG ? NST : 1][DIAG ? TY + 1 : 1][DIAG ? RF : 4];
    // DIAG: per-thread partial sums of the main warps, parked here between read-out loops so that they do not
    // occupy registers during the step's arithmetic
    double dacc[DIAG ? DS_NFLT : 1][DIAG ? TY * 32 : 1];
    float dwnd[DIAG ? 3 : 1][DIAG ? TY * 32 : 1];   // |W| sums: exact integers in fp32 (<= 64 planes x 4 sites x |W|)
    int dflg[DIAG ? 2 : 1][DIAG ? TY * 32 : 1];     // near-branch and big-plaquette counts
    float4 col[2][TY];                    // x hand-over of the site x0-1: (b_x.re, b_x.im, S_xy, S_xz)
    unsigned long long full[NST];         // a staged phi, th plane has landed
    unsigned long long qfull[TY];         // a warp's Pi, ep row has landed
};

}  // namespace

namespace {

// Domain of this kernel: every |th_i| < AH_TILED_TH_LIMIT (2^16 rad), so that every plaquette angle is below
// 2^18, where the two-term Cody-Waite reductions of sincos_pi_f32 / sin_poly_f32 still hold their 1.5e-7
// absolute accuracy (ah_common.cuh).  Each thread checks the 12 link angles it owns (every link of the
// input state is owned by exactly one thread) and raises *overflow if one is outside; the API then
// redoes the step with the libm-based site kernel (ah_api.cu: one_step).
#define AH_TILED_TH_LIMIT 65536.0f

// DIAG = true (SURVEY 8(a) row D-fuse): the same step, plus the read-outs D1-D3 of the ENTRY snapshot of every
// site, evaluated in a separate, ROLLED loop at the end of each plane's iteration (after the outputs of the
// plane have been stored, when nothing of the step's arithmetic is live any more):
//   * phase 1 additionally computes the site phases alpha = Arg(phi) (one polynomial atan2 per staged site) of
//     the forward plane into a 3-plane ring in shared memory, and the step's own forward hops give each site's
//     gradient energy, which is handed over through a scratch row;
//   * the read-out loop gives lane l the sites l, l+32, l+64, l+96 of the warp's row (NOT the step's 4l .. 4l+3),
//     so that every scalar it needs — phi, th of the site and its forward neighbours, the seven site phases,
//     the staged Pi, ep, the gradient energy — is a conflict-free shared-memory read; the nine link phases of the
//     site's three plaquettes are wrapped differences of site phases (ah_diag_site.cuh);
//   * both staged planes the read-outs use (own and forward) must therefore survive phase 2: the ring slot of
//     the plane below is refilled after the CTA barrier instead of before it (the longer iteration of a
//     diagnostic step leaves the copy ample time), and the warp's Pi, ep row is refilled after the loop;
//   * the only extra global reads are the backward neighbours ep_y(x-y), ep_z(x-z) (coalesced rows, L2 hits)
//     and one ep_x per row.
// Per-thread partial sums (int32 counts, fp64 sums) live in shared memory between loops, are reduced per CTA
// into partials[linear CTA index]; diag_final_kernel adds them in a fixed order.
// WIND (DIAG only): include the winding read-out D1 (site phases, link phases, |W| and the two plaquette counts);
// without it the DIAG instantiation evaluates the Lagrangian-weighted sums and the Gauss residual only — the set
// the paper's timed runs compute every 5 steps — and needs neither the phase ring nor atan2.
template <int SPT, int TY, bool COMPACT, bool DIAG, bool WIND>
__global__ void __launch_bounds__((TY + 1) * 32, ((TY + 1) * 32 <= 256) ? 2 : 1)
tiled_step_kernel(ConstFields<float> in, Fields<float> out, StepCoef<float> k, int nx, int ny, int nz, int z_lo,
                  int z_hi, int zc, int *overflow, DiagCoef dk, DiagPartial *partials)
{
    extern __shared__ __align__(128) unsigned char smem_bytes[];
    Smem<SPT, TY, DIAG> &sm = *reinterpret_cast<Smem<SPT, TY, DIAG> *>(smem_bytes);
    constexpr int TX = 32 * SPT, RF = TX + 2 * HALO;
    using VS = VN<SPT>;

    const int lane = threadIdx.x & 31;
    const int w = __shfl_sync(FULL, (int)(threadIdx.x >> 5), 0);   // warp-uniform by construction
    // planes z_lo .. z_hi - 1 are updated (the whole periodic lattice: 0 .. nz; a z slab with ghost planes: 1 .. nz - 1,
    // where the wrap of the plane index below never happens)
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = z_lo + blockIdx.z * zc;
    const int z1 = min(z_hi, z0 + zc);
    const int nplanes = z1 - z0;           // planes this CTA updates; loads n = 0 .. nplanes + 1
    const size_t sxy = (size_t)nx * ny;
    const bool is_main = w < TY;

    // ------------------------------------------------------------------ producers
    // load n  <->  plane z0 - 1 + n (periodic), slot n % NST.  Every main warp copies its own staged row (one
    // copy per field), the helper warp the two halo rows 0 and TY+1, and it arms the slot's mbarrier with the
    // byte count of the whole plane.  One elected lane per warp issues them, with warp-uniform operands.
    const bool interior = (x0 > 0) && (x0 + TX < nx);
    auto wrap_y = [&](int yy) {
        yy %= ny;
        return yy < 0 ? yy + ny : yy;
    };
    const size_t p_row0 = (size_t)wrap_y(is_main ? y0 + w : y0 - 1) * nx;   // main: own row; helper: halo row y0-1
    const size_t p_row1 = (size_t)wrap_y(y0 + TY) * nx;                      // helper only: halo row y0+TY
#ifndef AH_L2_HINTS
#define AH_L2_HINTS 1
#endif
    const unsigned long long pol_keep = l2_policy_keep(), pol_stream = l2_policy_stream();
    auto copy1 = [&](float *dst, const float *src, unsigned bytes, unsigned long long *bar) {
        if (AH_L2_HINTS) bulk_g2s_hint(dst, src, bytes, bar, pol_keep);
        else bulk_g2s(dst, src, bytes, bar);
    };
    auto copy_row = [&](int slot, int r, size_t src_off) {
        constexpr int FLD[NRAW] = {PHI_RE, PHI_IM, TH_X, TH_Y, TH_Z};
#pragma unroll
        for (int f = 0; f < NRAW; ++f) {
            const float *srow = in.f[FLD[f]] + src_off;
            float *dst = &sm.raw[slot][f][r][0];
            if (interior) {
                copy1(dst, srow + x0 - HALO, RF * sizeof(float), &sm.full[slot]);
            } else {
                const int xl = (x0 == 0) ? nx - HALO : x0 - HALO;
                const int xr = (x0 + TX == nx) ? 0 : x0 + TX;
                copy1(dst + HALO, srow + x0, TX * sizeof(float), &sm.full[slot]);
                copy1(dst, srow + xl, HALO * sizeof(float), &sm.full[slot]);
                copy1(dst + HALO + TX, srow + xr, HALO * sizeof(float), &sm.full[slot]);
            }
        }
    };
    // running state of the next load (no division in the march): ring slot, plane offset of plane z0 - 1 + n
    //
    // Write-after-read on a ring slot: produce() overwrites (async proxy) the slot whose plane the generic-proxy
    // loads of ALL warps read last in phase 1 of the previous iteration (DIAG: in phase 2 of the iteration before the
    // CTA barrier it follows).  Every call site sits after the __syncthreads that follows those reads, and a read
    // value has gone through dependent arithmetic (or a store) before its thread reaches that barrier, so no read of
    // the old plane can still be in flight when the copy is issued.  A violation would put the next plane's phi, th
    // under a slower warp's loads and change Pi+, ep+ of its row by O(1): test_one_step_fp32 (256,16,11) and
    // test_tiled_step_repeats_bit_identically would fail.
    int ld_slot = 0, ld_z = (z0 == 0) ? nz - 1 : z0 - 1;
    size_t ld_plane = (size_t)ld_z * sxy;
    auto produce = [&]() {
        if (elect_one()) {
            if (is_main) {
                copy_row(ld_slot, w + 1, ld_plane + p_row0);
            } else {
                mbar_expect_tx(&sm.full[ld_slot], (unsigned)(NRAW * (TY + 2) * RF * sizeof(float)));
                copy_row(ld_slot, 0, ld_plane + p_row0);
                copy_row(ld_slot, TY + 1, ld_plane + p_row1);
            }
        }
        ld_slot = (ld_slot == NST - 1) ? 0 : ld_slot + 1;
        ld_plane += sxy;
        if (++ld_z == nz) {
            ld_z = 0;
            ld_plane = 0;
        }
    };

    // Pi, ep of the warp's own row, plane after plane starting at z0 -> sm.qe[w].
    // Write-after-read: only the warp itself reads sm.qe[w]; produce_q() is called after the __syncwarp that follows
    // the last use of the staged values in arithmetic (plain: the final Eq. 7-10 updates; DIAG: the read-out loop), so
    // the refill cannot land under a lane that has not read yet.
    size_t q_off = (size_t)z0 * sxy + (size_t)(y0 + w < ny ? y0 + w : 0) * nx + x0;
    auto produce_q = [&]() {
        if (elect_one()) {
            constexpr int FLD[NRAW] = {PI_RE, PI_IM, EP_X, EP_Y, EP_Z};
            mbar_expect_tx(&sm.qfull[w], (unsigned)(NRAW * TX * sizeof(float)));
#pragma unroll
            for (int f = 0; f < NRAW; ++f)
                if (AH_L2_HINTS) bulk_g2s_hint(&sm.qe[w][f][0], in.f[FLD[f]] + q_off, TX * sizeof(float), &sm.qfull[w], pol_stream);
                else bulk_g2s(&sm.qe[w][f][0], in.f[FLD[f]] + q_off, TX * sizeof(float), &sm.qfull[w]);
        }
        q_off += sxy;
    };

    pdl_launch_dependents();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(&sm.full[s], 1);
#pragma unroll
        for (int s = 0; s < TY; ++s) mbar_init(&sm.qfull[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    pdl_wait();   // the previous step's kernels have completed: its outputs are this step's inputs
    produce();   // loads 0, 1, 2
    produce();
    produce();
    if (is_main && y0 + w < ny) produce_q();

    const float kA = k.c2 * k.idx2;    // weight of one hop in Pi+          (Eq. 7)
    const float kB = k.w2 * k.idx2;    // weight of one plaquette sine in ep+ (Eq. 8)
    const float kJ = k.w2 * k.two_e2_q;

    // ---- main-warp geometry: row y0+w (staged row w+1), sites x0+4*lane .. +3
    const int y = y0 + w;
    const bool act = is_main && y < ny;
    const int r_own = w + 1;
    const int cofs = HALO + SPT * lane;                    // staged column of this thread's first site
    const size_t ro = (size_t)(act ? y : 0) * nx + x0 + SPT * lane;
    // ---- helper-warp geometry: halo row (staged row 0) and halo column x0-1 (staged column HALO-1)
    const bool col_act = !is_main && lane < TY;

    // DIAG: site phases of this warp's staged row (helper: halo row TY+1, and the column x0+128 of every row) of
    // the plane in ring slot `slot` -> sm.alpha[slot].  Lane l takes columns l, l+32, ... (conflict-free).
    auto stage_alpha = [&](int slot) {
        if constexpr (DIAG && WIND) {
            const int r = is_main ? w + 1 : TY + 1;
#pragma unroll
            for (int j = 0; j < SPT; ++j) {
                const int c = HALO + lane + 32 * j;
                sm.alpha[slot][r - 1][c] = site_phase_fast(sm.raw[slot][0][r][c], sm.raw[slot][1][r][c]);
            }
            if (!is_main && lane <= TY)
                sm.alpha[slot][lane][HALO + TX] =
                    site_phase_fast(sm.raw[slot][0][lane + 1][HALO + TX], sm.raw[slot][1][lane + 1][HALO + TX]);
        }
    };

    // ---- prologue: hand-down of the plane below the chunk (needs loads 0 and 1)
    VS c_pr, c_pi, c_tx, c_ty, c_tz;        // own old phi, th of the current plane
    VS g_bzr, g_bzi, g_sxz, g_syz;          // b_z, S_xz, S_yz of the site below (z-1)
    mbar_wait(&sm.full[0], 0);
    mbar_wait(&sm.full[1], 0);
    if (act) {
        c_pr = ldsN<SPT>(&sm.raw[1][0][r_own][cofs]); c_pi = ldsN<SPT>(&sm.raw[1][1][r_own][cofs]);
        c_tx = ldsN<SPT>(&sm.raw[1][2][r_own][cofs]); c_ty = ldsN<SPT>(&sm.raw[1][3][r_own][cofs]);
        c_tz = ldsN<SPT>(&sm.raw[1][4][r_own][cofs]);
        if (!(fmaxf(vmaxabs<SPT>(c_tx), fmaxf(vmaxabs<SPT>(c_ty), vmaxabs<SPT>(c_tz))) < AH_TILED_TH_LIMIT))
            *overflow = 1;
        const VS m_pr = ldsN<SPT>(&sm.raw[0][0][r_own][cofs]), m_pi = ldsN<SPT>(&sm.raw[0][1][r_own][cofs]);
        const VS m_tx = ldsN<SPT>(&sm.raw[0][2][r_own][cofs]), m_ty = ldsN<SPT>(&sm.raw[0][3][r_own][cofs]);
        const VS m_tz = ldsN<SPT>(&sm.raw[0][4][r_own][cofs]);
        const VS my_tz = ldsN<SPT>(&sm.raw[0][4][r_own + 1][cofs]), my_tx = ldsN<SPT>(&sm.raw[0][2][r_own + 1][cofs]);
        float me_tz = __shfl_down_sync(FULL, m_tz.v[0], 1), me_ty = __shfl_down_sync(FULL, m_ty.v[0], 1);
        if (lane == 31) {
            me_tz = sm.raw[0][4][r_own][cofs + SPT];
            me_ty = sm.raw[0][3][r_own][cofs + SPT];
        }
        // The hand-down of the plane below is what that plane's own iteration (in the CTA of the chunk below)
        // computes and carries in registers: the same expressions in the same rounding sequence, including the
        // warp-wide choice between the two plaquette-sine polynomials, so that a site's result does not depend on
        // where the z chunks (or the z slabs of a multi-GPU run) are cut.
        VS a_xz, a_yz;
        float amax = 0.f;
#pragma unroll
        for (int j = 0; j < SPT; ++j) {
            const int jn = (j < SPT - 1) ? j + 1 : SPT - 1;
            const float ty_xp = (j < SPT - 1) ? m_ty.v[jn] : me_ty, tz_xp = (j < SPT - 1) ? m_tz.v[jn] : me_tz;
            const float a_xy = plaq_angle_f32(m_tx.v[j], ty_xp, my_tx.v[j], m_ty.v[j]);
            a_xz.v[j] = plaq_angle_f32(m_tx.v[j], tz_xp, c_tx.v[j], m_tz.v[j]);
            a_yz.v[j] = plaq_angle_f32(m_ty.v[j], my_tz.v[j], c_ty.v[j], m_tz.v[j]);
            amax = fmaxf(amax, fmaxf(fmaxf(fabsf(a_xy), fabsf(a_xz.v[j])), fabsf(a_yz.v[j])));
        }
        const bool small = __all_sync(FULL, amax < AH_SMALL_ANGLE);
#pragma unroll
        for (int j = 0; j < SPT; ++j) {
            float s, c;
            sincos_pi_f32(m_tz.v[j], s, c);
            hop_bwd_f32(c, s, m_pr.v[j], m_pi.v[j], g_bzr.v[j], g_bzi.v[j]);
            if (COMPACT) {
                g_sxz.v[j] = small ? sin_small_f32(a_xz.v[j]) : sin_poly_f32(a_xz.v[j]);
                g_syz.v[j] = small ? sin_small_f32(a_yz.v[j]) : sin_poly_f32(a_yz.v[j]);
            } else {
                g_sxz.v[j] = a_xz.v[j];
                g_syz.v[j] = a_yz.v[j];
            }
        }
    }
    stage_alpha(1);
    __syncthreads();   // slot 0 (load 0) is free from here on

    int sf = 1, sf_par = 0;                           // slot and mbarrier parity of the forward plane (load n + 1)
    size_t oc = (size_t)z0 * sxy + ro - sxy;          // this thread's element offset in plane z0 + n - 1
    if constexpr (DIAG) {
        if (is_main) {
#pragma unroll
            for (int a = 0; a < DS_NFLT; ++a) sm.dacc[a][threadIdx.x] = 0.0;
#pragma unroll
            for (int a = 0; a < 3; ++a) sm.dwnd[a][threadIdx.x] = 0.0f;
            sm.dflg[0][threadIdx.x] = sm.dflg[1][threadIdx.x] = 0;
        }
    }

    // ---- march: iteration n updates plane z0 + n - 1 (slot n % 3), forward plane in slot (n + 1) % 3.
    // One __syncthreads per plane separates phase 1 (hand-overs written, staged planes read) from phase 2 (hand-overs
    // consumed, outputs stored); the three roles run separate loops with the same barrier count.
    // Re-use of a ring slot: the slot of load n+2 held plane n-1, last read in phase 1 of iteration n-1, i.e. before
    // the barrier that every warp has passed when it issues its copies at the top of iteration n.  DIAG reads the
    // planes n and n+1 in phase 2 as well (read-out loop), so there the copies of load n+2 are issued right after
    // the barrier of iteration n instead.
    // (A warp-to-warp mbarrier protocol without the CTA barrier was measured 15 % slower and removed.)
    if (!is_main) {
#pragma unroll 1
        for (int n = 1; n <= nplanes; ++n) {
            const int buf = n & 1;
            const int so = sf;
            if (++sf == NST) { sf = 0; sf_par ^= 1; }
            if (!DIAG && n + 2 <= nplanes + 1) produce();
            mbar_wait(&sm.full[sf], sf_par);
            stage_alpha(sf);
            // helper: shared quantities of the halo row y0-1 (staged row 0) at this plane
            const VS h_pr = ldsN<SPT>(&sm.raw[so][0][0][cofs]), h_pi = ldsN<SPT>(&sm.raw[so][1][0][cofs]);
            const VS h_tx = ldsN<SPT>(&sm.raw[so][2][0][cofs]), h_ty = ldsN<SPT>(&sm.raw[so][3][0][cofs]);
            const VS h_tz = ldsN<SPT>(&sm.raw[so][4][0][cofs]);
            const VS hn_ty = ldsN<SPT>(&sm.raw[sf][3][0][cofs]), hn_tx = ldsN<SPT>(&sm.raw[sf][2][0][cofs]);
            const VS hy_tx = ldsN<SPT>(&sm.raw[so][2][1][cofs]), hy_tz = ldsN<SPT>(&sm.raw[so][4][1][cofs]);
            float hr_ty = __shfl_down_sync(FULL, h_ty.v[0], 1), hr_tz = __shfl_down_sync(FULL, h_tz.v[0], 1);
            if (lane == 31) {
                hr_ty = sm.raw[so][3][0][cofs + SPT];
                hr_tz = sm.raw[so][4][0][cofs + SPT];
            }
            // the same expressions, rounding sequence and warp-wide choice of the sine polynomial as the main warp
            // that owns this row in the tile below: a site's result must not depend on where the y tiles are cut
            // (the plain and the DIAG instantiation cut them differently)
            VS o_byr, o_byi, o_sxy, o_syz;
            float amax = 0.f;
#pragma unroll
            for (int j = 0; j < SPT; ++j) {
                const int jn = (j < SPT - 1) ? j + 1 : SPT - 1;
                const float ty_xp = (j < SPT - 1) ? h_ty.v[jn] : hr_ty, tz_xp = (j < SPT - 1) ? h_tz.v[jn] : hr_tz;
                o_sxy.v[j] = plaq_angle_f32(h_tx.v[j], ty_xp, hy_tx.v[j], h_ty.v[j]);
                const float a_xz = plaq_angle_f32(h_tx.v[j], tz_xp, hn_tx.v[j], h_tz.v[j]);
                o_syz.v[j] = plaq_angle_f32(h_ty.v[j], hy_tz.v[j], hn_ty.v[j], h_tz.v[j]);
                amax = fmaxf(amax, fmaxf(fmaxf(fabsf(o_sxy.v[j]), fabsf(a_xz)), fabsf(o_syz.v[j])));
            }
            const bool small = __all_sync(FULL, amax < AH_SMALL_ANGLE);
#pragma unroll
            for (int j = 0; j < SPT; ++j) {
                float s, c;
                sincos_pi_f32(h_ty.v[j], s, c);
                hop_bwd_f32(c, s, h_pr.v[j], h_pi.v[j], o_byr.v[j], o_byi.v[j]);
                if (COMPACT) {
                    o_sxy.v[j] = small ? sin_small_f32(o_sxy.v[j]) : sin_poly_f32(o_sxy.v[j]);
                    o_syz.v[j] = small ? sin_small_f32(o_syz.v[j]) : sin_poly_f32(o_syz.v[j]);
                }
            }
            stN<SPT>(&sm.row[buf][0][0][SPT * lane], o_byr);
            stN<SPT>(&sm.row[buf][0][1][SPT * lane], o_byi);
            stN<SPT>(&sm.row[buf][0][2][SPT * lane], o_sxy);
            stN<SPT>(&sm.row[buf][0][3][SPT * lane], o_syz);
            // halo column x0-1 (staged column HALO-1) of tile row `lane`
            if (col_act) {
                const int r = lane + 1, cw = HALO - 1;
                const float pr = sm.raw[so][0][r][cw], pi = sm.raw[so][1][r][cw];
                const float tx = sm.raw[so][2][r][cw], ty = sm.raw[so][3][r][cw], tz = sm.raw[so][4][r][cw];
                const float ty_r = sm.raw[so][3][r][cw + 1], tz_r = sm.raw[so][4][r][cw + 1];
                const float tx_yp = sm.raw[so][2][r + 1][cw], tx_zp = sm.raw[sf][2][r][cw];
                float s, c;
                sincos_pi_f32(tx, s, c);
                const float a_xy = tx + ty_r - tx_yp - ty, a_xz = tx + tz_r - tx_zp - tz;
                const float sxy_ = plaq_f<COMPACT>(a_xy), sxz_ = plaq_f<COMPACT>(a_xz);
                sm.col[buf][lane] = make_float4(c * pr - s * pi, c * pi + s * pr, sxy_, sxz_);
            }
            __syncthreads();
            if (DIAG && n + 2 <= nplanes + 1) produce();
        }
    } else if (!act) {
        // a row beyond ny (ragged last tile): keeps the protocol going, computes nothing
#pragma unroll 1
        for (int n = 1; n <= nplanes; ++n) {
            if (!DIAG && n + 2 <= nplanes + 1) produce();
            if constexpr (DIAG) {   // the row above the last active one is this warp's (periodic wrap): its phases are needed
                if (++sf == NST) { sf = 0; sf_par ^= 1; }
                mbar_wait(&sm.full[sf], sf_par);
                stage_alpha(sf);
            }
            __syncthreads();
            if (DIAG && n + 2 <= nplanes + 1) produce();
        }
    } else {
#pragma unroll 1
        for (int n = 1; n <= nplanes; ++n) {
            const int buf = n & 1;
            const int so = sf;
            if (++sf == NST) { sf = 0; sf_par ^= 1; }
            oc += sxy;
            VS P_r, P_i, E_x, E_y, E_z;   // Pi+, ep+ still lacking the old Pi, ep and the terms from row y-1 / site x0-1
            if (!DIAG && n + 2 <= nplanes + 1) produce();
            // DIAG: the backward ep neighbours that are not on chip (row y-1 of this plane, this row of the plane
            // below, and - lane 0 - the site x0-1), requested a whole phase before the read-out loop needs them
            VS d_eby, d_ebz;
            float d_exl = 0.f;
            if constexpr (DIAG) {
                const int z = z0 + n - 1, zm = (z == 0) ? nz - 1 : z - 1, ym = (y == 0) ? ny - 1 : y - 1;
                d_eby = ldgN<SPT>(in.f[EP_Y] + (size_t)z * sxy + (size_t)ym * nx + x0 + SPT * lane);
                d_ebz = ldgN<SPT>(in.f[EP_Z] + (size_t)zm * sxy + ro);
                if (lane == 0) d_exl = __ldg(in.f[EP_X] + (size_t)z * sxy + (size_t)y * nx + ((x0 == 0) ? nx - 1 : x0 - 1));
            }
            mbar_wait(&sm.full[sf], sf_par);
            stage_alpha(sf);   // DIAG: site phases of the forward plane
            VS o_byr, o_byi, o_sxy, o_syz;   // for row y+1, through shared memory
            VS h_bzr, h_bzi, h_sxz;          // this plane's hand-down to z+1 (with S_yz in o_syz)
            float l_bxr = 0.f, l_bxi = 0.f, l_sxy = 0.f, l_sxz = 0.f;   // from the site to the left
            const VS y_pr = ldsN<SPT>(&sm.raw[so][0][r_own + 1][cofs]), y_pi = ldsN<SPT>(&sm.raw[so][1][r_own + 1][cofs]);
            const VS y_tx = ldsN<SPT>(&sm.raw[so][2][r_own + 1][cofs]), y_tz = ldsN<SPT>(&sm.raw[so][4][r_own + 1][cofs]);
            const VS n_pr = ldsN<SPT>(&sm.raw[sf][0][r_own][cofs]), n_pi = ldsN<SPT>(&sm.raw[sf][1][r_own][cofs]);
            const VS n_tx = ldsN<SPT>(&sm.raw[sf][2][r_own][cofs]), n_ty = ldsN<SPT>(&sm.raw[sf][3][r_own][cofs]);
            // right neighbours of the 4th site: lane+1's first site, or (lane 31) the staged halo column
            float r_pr = __shfl_down_sync(FULL, c_pr.v[0], 1), r_pi = __shfl_down_sync(FULL, c_pi.v[0], 1);
            float r_ty = __shfl_down_sync(FULL, c_ty.v[0], 1), r_tz = __shfl_down_sync(FULL, c_tz.v[0], 1);
            if (lane == 31) {
                r_pr = sm.raw[so][0][r_own][cofs + SPT]; r_pi = sm.raw[so][1][r_own][cofs + SPT];
                r_ty = sm.raw[so][3][r_own][cofs + SPT]; r_tz = sm.raw[so][4][r_own][cofs + SPT];
            }

            // plaquette angles owned by the 4 sites (Eqs. 14-15), then their sines: when every angle of the
            // warp is small (the physical regime) a Taylor polynomial without range reduction is exact to fp32
            VS S_xy, S_xz, S_yz;
            float amax = 0.f;
#pragma unroll
            for (int j = 0; j < SPT; ++j) {
                const int jn = (j < SPT - 1) ? j + 1 : SPT - 1;
                const float ty_xp = (j < SPT - 1) ? c_ty.v[jn] : r_ty, tz_xp = (j < SPT - 1) ? c_tz.v[jn] : r_tz;
                S_xy.v[j] = plaq_angle_f32(c_tx.v[j], ty_xp, y_tx.v[j], c_ty.v[j]);
                S_xz.v[j] = plaq_angle_f32(c_tx.v[j], tz_xp, n_tx.v[j], c_tz.v[j]);
                S_yz.v[j] = plaq_angle_f32(c_ty.v[j], y_tz.v[j], n_ty.v[j], c_tz.v[j]);
                amax = fmaxf(amax, fmaxf(fmaxf(fabsf(S_xy.v[j]), fabsf(S_xz.v[j])), fabsf(S_yz.v[j])));
            }
            if (COMPACT) {
                // two angles per issued instruction (FFMA2); bit-identical to the scalar polynomials
                auto sines = [&](VS &a, bool small) {
#pragma unroll
                    for (int h = 0; h < SPT; h += 2) {
                        const f32x2 x = pack2(a.v[h], a.v[h + 1]);
                        unpack2(small ? sin_small_f32x2(x) : sin_poly_f32x2(x), a.v[h], a.v[h + 1]);
                    }
                };
                if (__all_sync(FULL, amax < AH_SMALL_ANGLE)) {
                    sines(S_xy, true); sines(S_xz, true); sines(S_yz, true);
                } else {
                    sines(S_xy, false); sines(S_xz, false); sines(S_yz, false);
                }
            }

            // link variables of the 4 sites (Eq. 12), two angles per issued instruction
            VS s_x, c_x, s_y, c_y, s_z, c_z;
            {
                auto sincos4 = [&](const VS &t, VS &sn, VS &cs) {
#pragma unroll
                    for (int h = 0; h < SPT; h += 2) {
                        f32x2 s2, c2;
                        sincos_pi_f32x2(pack2(t.v[h], t.v[h + 1]), s2, c2);
                        unpack2(s2, sn.v[h], sn.v[h + 1]);
                        unpack2(c2, cs.v[h], cs.v[h + 1]);
                    }
                };
                sincos4(c_tx, s_x, c_x);
                sincos4(c_ty, s_y, c_y);
                sincos4(c_tz, s_z, c_z);
            }
            VS d_g2;   // DIAG: gradient energy of the 4 sites, for the read-out loop
#pragma unroll
            for (int j = 0; j < SPT; ++j) {
                const float fr = c_pr.v[j], fi = c_pi.v[j];
                const float tx = c_tx.v[j], ty = c_ty.v[j], tz = c_tz.v[j];
                const int jn = (j < SPT - 1) ? j + 1 : SPT - 1;
                const float xr = (j < SPT - 1) ? c_pr.v[jn] : r_pr, xi = (j < SPT - 1) ? c_pi.v[jn] : r_pi;
                const float Sxy = S_xy.v[j], Sxz = S_xz.v[j], Syz = S_yz.v[j];
                const float sx = s_x.v[j], cx = c_x.v[j], sy = s_y.v[j], cy = c_y.v[j], sz = s_z.v[j], cz = c_z.v[j];
                // forward hops U_i(s) phi(s+i)                                   (Eq. 13)
                float fxr, fxi, fyr, fyi, fzr, fzi;
                hop_fwd_f32(cx, sx, xr, xi, fxr, fxi);
                hop_fwd_f32(cy, sy, y_pr.v[j], y_pi.v[j], fyr, fyi);
                hop_fwd_f32(cz, sz, n_pr.v[j], n_pi.v[j], fzr, fzi);
                // hand-overs conj(U_i(s)) phi(s)
                float bxr, bxi;
                hop_bwd_f32(cx, sx, fr, fi, bxr, bxi);
                hop_bwd_f32(cy, sy, fr, fi, o_byr.v[j], o_byi.v[j]);
                hop_bwd_f32(cz, sz, fr, fi, h_bzr.v[j], h_bzi.v[j]);
                if constexpr (DIAG) d_g2.v[j] = readout_grad2(fr, fi, fxr, fxi, fyr, fyi, fzr, fzi, dk.f_idx2);
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
                // (the old Pi, ep terms are added after the barrier: their copies have the whole phase to land)
                P_r.v[j] = kA * ar - k.c2 * (pot * fr);
                P_i.v[j] = kA * ai - k.c2 * (pot * fi);
                E_x.v[j] = kJ * (fr * fxi - fi * fxr) - kB * cux;
                E_y.v[j] = kJ * (fr * fyi - fi * fyr) - kB * cuy;
                E_z.v[j] = kJ * (fr * fzi - fi * fzr) - kB * cuz;
                l_bxr = bxr; l_bxi = bxi; l_sxy = Sxy; l_sxz = Sxz;
            }
            // y-1 hand-over for the row above
            if (w + 1 < TY) {
                stN<SPT>(&sm.row[buf][w + 1][0][SPT * lane], o_byr);
                stN<SPT>(&sm.row[buf][w + 1][1][SPT * lane], o_byi);
                stN<SPT>(&sm.row[buf][w + 1][2][SPT * lane], o_sxy);
                stN<SPT>(&sm.row[buf][w + 1][3][SPT * lane], o_syz);
            }
            // x-1 terms of the first site: lane-1's last site (lane 0: the helper's column entry, after the barrier)
            l_bxr = __shfl_up_sync(FULL, l_bxr, 1);
            l_bxi = __shfl_up_sync(FULL, l_bxi, 1);
            l_sxy = __shfl_up_sync(FULL, l_sxy, 1);
            l_sxz = __shfl_up_sync(FULL, l_sxz, 1);
            if (lane > 0) {
                P_r.v[0] += kA * l_bxr;
                P_i.v[0] += kA * l_bxi;
                E_y.v[0] -= kB * l_sxy;
                E_z.v[0] -= kB * l_sxz;
            }
            // roll the z hand-down
            g_bzr = h_bzr; g_bzi = h_bzi; g_sxz = h_sxz; g_syz = o_syz;
            __syncthreads();
            if (DIAG && n + 2 <= nplanes + 1) produce();
            // add what row y-1 (and, lane 0, site x0-1) hands over, finish Eqs. 7-10, store
            const VS av = ldsN<SPT>(&sm.row[buf][w][0][SPT * lane]), bv = ldsN<SPT>(&sm.row[buf][w][1][SPT * lane]);
            const VS cv = ldsN<SPT>(&sm.row[buf][w][2][SPT * lane]), dv = ldsN<SPT>(&sm.row[buf][w][3][SPT * lane]);
            if (lane == 0) {
                const float4 cdat = sm.col[buf][w];
                P_r.v[0] += kA * cdat.x;
                P_i.v[0] += kA * cdat.y;
                E_y.v[0] -= kB * cdat.z;
                E_z.v[0] -= kB * cdat.w;
            }
            // old Pi, ep of the own sites: staged one plane ahead by this warp
            mbar_wait(&sm.qfull[w], (n - 1) & 1);
            const VS q_r = ldsN<SPT>(&sm.qe[w][0][SPT * lane]), q_i = ldsN<SPT>(&sm.qe[w][1][SPT * lane]);
            const VS e_x = ldsN<SPT>(&sm.qe[w][2][SPT * lane]), e_y = ldsN<SPT>(&sm.qe[w][3][SPT * lane]);
            const VS e_z = ldsN<SPT>(&sm.qe[w][4][SPT * lane]);
            VS f_r, f_i, t_x, t_y, t_z;
#pragma unroll
            for (int j = 0; j < SPT; ++j) {
                P_r.v[j] = k.c1 * q_r.v[j] + (P_r.v[j] + kA * av.v[j]);
                P_i.v[j] = k.c1 * q_i.v[j] + (P_i.v[j] + kA * bv.v[j]);
                E_x.v[j] = k.w1 * e_x.v[j] + (E_x.v[j] + kB * cv.v[j]);
                E_y.v[j] = k.w1 * e_y.v[j] + E_y.v[j];
                E_z.v[j] = k.w1 * e_z.v[j] + (E_z.v[j] - kB * dv.v[j]);
                f_r.v[j] = c_pr.v[j] + k.dt * P_r.v[j];   // Eq. 9
                f_i.v[j] = c_pi.v[j] + k.dt * P_i.v[j];
                t_x.v[j] = c_tx.v[j] + k.dt * E_x.v[j];   // Eq. 10
                t_y.v[j] = c_ty.v[j] + k.dt * E_y.v[j];
                t_z.v[j] = c_tz.v[j] + k.dt * E_z.v[j];
            }
            // the staged Pi, ep row has been consumed (its values went through the arithmetic above): refill it
            // with the next plane's row, which then has almost a whole iteration to land (DIAG: after the read-outs)
            __syncwarp();
            if (!DIAG && n + 1 <= nplanes) produce_q();
            stN<SPT>(out.f[PI_RE] + oc, P_r);
            stN<SPT>(out.f[PI_IM] + oc, P_i);
            stN<SPT>(out.f[EP_X] + oc, E_x);
            stN<SPT>(out.f[EP_Y] + oc, E_y);
            stN<SPT>(out.f[EP_Z] + oc, E_z);
            stN<SPT>(out.f[PHI_RE] + oc, f_r);
            stN<SPT>(out.f[PHI_IM] + oc, f_i);
            stN<SPT>(out.f[TH_X] + oc, t_x);
            stN<SPT>(out.f[TH_Y] + oc, t_y);
            stN<SPT>(out.f[TH_Z] + oc, t_z);
            if constexpr (DIAG) {
                // ---- read-outs D1-D3 of the entry snapshot of this plane: lane l takes the sites l + 32 j of the row
                // scratch: this warp's hand-over row, consumed above and free until iteration n + 2: 4 x 128 floats
                float *scr = reinterpret_cast<float *>(&sm.row[buf][w][0][0]);
                stN<SPT>(scr + SPT * lane, d_g2);
                stN<SPT>(scr + TX + SPT * lane, d_eby);
                stN<SPT>(scr + 2 * TX + SPT * lane, d_ebz);
                const float ex_left = d_exl;
                __syncwarp();
                float wnd[3];
                int n_near = sm.dflg[0][threadIdx.x], n_big = sm.dflg[1][threadIdx.x];
                double acc[DS_NFLT];
#pragma unroll
                for (int a = 0; a < 3; ++a) wnd[a] = sm.dwnd[a][threadIdx.x];
#pragma unroll
                for (int a = 0; a < DS_NFLT; ++a) acc[a] = sm.dacc[a][threadIdx.x];
#pragma unroll 1
                for (int j = 0; j < SPT; ++j) {
                    const int cq = lane + 32 * j, c = HALO + cq;
                    const float eby = scr[TX + cq], ebz = scr[2 * TX + cq];
                    // D1: winding of the three plaquettes the site owns (Eq. 16 right)
                    const float t0x = sm.raw[so][2][r_own][c], t0y = sm.raw[so][3][r_own][c], t0z = sm.raw[so][4][r_own][c];
                    const float ty_xp = sm.raw[so][3][r_own][c + 1], tz_xp = sm.raw[so][4][r_own][c + 1];
                    const float tx_yp = sm.raw[so][2][r_own + 1][c], tz_yp = sm.raw[so][4][r_own + 1][c];
                    const float tx_zp = sm.raw[sf][2][r_own][c], ty_zp = sm.raw[sf][3][r_own][c];
                    const float Pxy = plaq_angle_f32(t0x, ty_xp, tx_yp, t0y), Pxz = plaq_angle_f32(t0x, tz_xp, tx_zp, t0z);
                    const float Pyz = plaq_angle_f32(t0y, tz_yp, ty_zp, t0z);
                    if constexpr (WIND) {
                        const SiteWinding sw = readout_winding(
                            sm.alpha[so][w][c], sm.alpha[so][w][c + 1], sm.alpha[so][w + 1][c], sm.alpha[sf][w][c],
                            sm.alpha[so][w + 1][c + 1], sm.alpha[sf][w][c + 1], sm.alpha[sf][w + 1][c], t0x, t0y, t0z, ty_xp,
                            tz_xp, tx_yp, tz_yp, tx_zp, ty_zp, Pxy, Pxz, Pyz);
#pragma unroll
                        for (int pq = 0; pq < 3; ++pq) {
                            wnd[pq] += sw.absw[pq];
                            n_near += sw.nearf[pq];
                            n_big += sw.big[pq];
                        }
                    }
                    // D2, D3 (Eqs. 17-18, Eq. 5) from the staged phi, Pi, ep and the step's gradient energy
                    const float fr = sm.raw[so][0][r_own][c], fi = sm.raw[so][1][r_own][c];
                    const float pir = sm.qe[w][0][cq], pii = sm.qe[w][1][cq];
                    const float ex = sm.qe[w][2][cq], ey = sm.qe[w][3][cq], ez = sm.qe[w][4][cq];
                    const float exl = sm.qe[w][2][cq > 0 ? cq - 1 : 0];
                    const float exb = (cq == 0) ? ex_left : exl;
                    float pi2L, gr2L, L, pL, rhoL;
                    readout_lagrangian(fr, fi, scr[cq], readout_plaq_energy(Pxy, Pxz, Pyz, COMPACT ? 1 : 0, dk.f_idx4), pir,
                                       pii, ex, ey, ez, dk, pi2L, gr2L, L, pL, rhoL);
                    double G, div, charge;
                    readout_gauss(fr, fi, pir, pii, ex, ey, ez, exb, eby, ebz, dk, G, div, charge);
                    readout_accumulate(acc, pi2L, gr2L, L, pL, rhoL, G, div, charge);
                }
#pragma unroll
                for (int a = 0; a < 3; ++a) sm.dwnd[a][threadIdx.x] = wnd[a];
                sm.dflg[0][threadIdx.x] = n_near;
                sm.dflg[1][threadIdx.x] = n_big;
#pragma unroll
                for (int a = 0; a < DS_NFLT; ++a) sm.dacc[a][threadIdx.x] = acc[a];
                __syncwarp();   // every lane is done with the staged Pi, ep row
                if (n + 1 <= nplanes) produce_q();
            }
            // the forward plane becomes the own plane
            c_pr = ldsN<SPT>(&sm.raw[sf][0][r_own][cofs]); c_pi = ldsN<SPT>(&sm.raw[sf][1][r_own][cofs]);
            c_tx = ldsN<SPT>(&sm.raw[sf][2][r_own][cofs]); c_ty = ldsN<SPT>(&sm.raw[sf][3][r_own][cofs]);
            c_tz = ldsN<SPT>(&sm.raw[sf][4][r_own][cofs]);
            if (n < nplanes) {
                if (!(fmaxf(vmaxabs<SPT>(c_tx), fmaxf(vmaxabs<SPT>(c_ty), vmaxabs<SPT>(c_tz))) < AH_TILED_TH_LIMIT))
                    *overflow = 1;
            }
        }
    }

    if constexpr (DIAG) {
        // CTA reduction: warp shuffles, then the warps through shared memory (the hand-over rows are free now)
        int d_cnt[DS_NINT] = {0, 0, 0, 0, 0};
        double d_acc[DS_NFLT] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        if (is_main) {
#pragma unroll
            for (int a = 0; a < 3; ++a) d_cnt[a] = (int)sm.dwnd[a][threadIdx.x];
            d_cnt[DS_NEAR] = sm.dflg[0][threadIdx.x];
            d_cnt[DS_BIG] = sm.dflg[1][threadIdx.x];
#pragma unroll
            for (int a = 0; a < DS_NFLT; ++a) d_acc[a] = sm.dacc[a][threadIdx.x];
        }
        __syncthreads();
        double *s_f = reinterpret_cast<double *>(&sm.row[0][0][0][0]);       // [TY + 1][DS_NFLT]
        long long *s_i = reinterpret_cast<long long *>(s_f + (TY + 1) * DS_NFLT);   // [TY + 1][DS_NINT]
#pragma unroll
        for (int a = 0; a < DS_NINT; ++a) d_cnt[a] = warp_sum(d_cnt[a]);   // <= 32 x 64 x 12: fits int32
#pragma unroll
        for (int a = 0; a < DS_NFLT - 1; ++a) d_acc[a] = warp_sum(d_acc[a]);
        d_acc[DF_GMAX] = warp_max(d_acc[DF_GMAX]);
        if (lane == 0) {
#pragma unroll
            for (int a = 0; a < DS_NINT; ++a) s_i[w * DS_NINT + a] = (long long)d_cnt[a];
#pragma unroll
            for (int a = 0; a < DS_NFLT; ++a) s_f[w * DS_NFLT + a] = d_acc[a];
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            DiagPartial p;
            for (int a = 0; a < DS_NINT; ++a) {
                long long v = 0;
                for (int ww = 0; ww <= TY; ++ww) v += s_i[ww * DS_NINT + a];
                p.i[a] = v;
            }
            for (int a = 0; a < DS_NFLT; ++a) {
                double v = 0;
                for (int ww = 0; ww <= TY; ++ww)
                    v = (a == DF_GMAX) ? fmax(v, s_f[ww * DS_NFLT + a]) : v + s_f[ww * DS_NFLT + a];
                p.f[a] = v;
            }
            partials[blockIdx.x + (size_t)gridDim.x * (blockIdx.y + (size_t)gridDim.y * blockIdx.z)] = p;
        }
    }
}

}  // namespace

// --------------------------------------------------------------------------------- launch

constexpr int TILE_Y = 6;        // plain step: 6 main warps + 1 helper = 224 threads, 2 CTAs per SM (106 KB shared memory each)
constexpr int TILE_Y_DIAG = 5;   // fused read-outs: the site-phase ring and the parked partial sums take the room of one row

// sites per thread: 4 (128-site warp rows, 128-bit accesses) when nx allows it, else 2 (64-site rows, 64-bit accesses)
static int spt_for(int nx) { return nx % 128 == 0 ? 4 : 2; }

bool tiled_supported(int nx, int ny, int nz) { return nx >= 64 && nx % 64 == 0 && ny >= 1 && nz >= 1; }

template <int SPT, int TY, bool COMPACT, bool DIAG, bool WIND>
static cudaError_t setup_one()
{
    cudaError_t e = cudaFuncSetAttribute(tiled_step_kernel<SPT, TY, COMPACT, DIAG, WIND>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<SPT, TY, DIAG>));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(tiled_step_kernel<SPT, TY, COMPACT, DIAG, WIND>,
                                cudaFuncAttributePreferredSharedMemoryCarveout, 100);
}

template <int SPT>
static cudaError_t setup_spt()
{
    cudaError_t e = setup_one<SPT, TILE_Y, true, false, false>();
    if (e == cudaSuccess) e = setup_one<SPT, TILE_Y, false, false, false>();
    if (e == cudaSuccess) e = setup_one<SPT, TILE_Y_DIAG, true, true, true>();
    if (e == cudaSuccess) e = setup_one<SPT, TILE_Y_DIAG, false, true, true>();
    if (e == cudaSuccess) e = setup_one<SPT, TILE_Y_DIAG, true, true, false>();
    if (e == cudaSuccess) e = setup_one<SPT, TILE_Y_DIAG, false, true, false>();
    return e;
}

cudaError_t tiled_setup()
{
    cudaError_t e = setup_spt<4>();
    if (e == cudaSuccess) e = setup_spt<2>();
    return e;
}

// Planes per CTA: long chunks amortise the prologue (two extra planes of staging and a third of a
// plane of arithmetic), but the grid should still be many waves of 148 SMs x 2 resident CTAs.
// Measured at 1024^3: 64 and 128 planes tie, 256 loses 4 % to the partial last wave.
// Choice: minimise (number of waves of 148 SMs x 2 resident CTAs) x (planes per CTA + prologue), i.e. the
// time of the slowest SM, over chunk lengths up to AH_ZC_MAX; for small lattices this picks a chunk count that
// fills one wave (or a whole number of them) instead of leaving a mostly empty last wave (128^3: +40 %,
// 256^3: +9 %).  With six or more waves the last partial wave is not modelled as a whole one (measured: it costs
// little, the CTAs left share the freed bandwidth).
#ifndef AH_ZC_MAX
#define AH_ZC_MAX 64
#endif
static int chunk_for(int nx, int ny, int nz, int ty)
{
    const long long cols = (long long)(nx / (32 * spt_for(nx))) * ((ny + ty - 1) / ty);
    const long long resident = 148LL * 2;
    int best = nz < 8 ? nz : 8;
    double best_cost = 1e300;
    for (int nchunk = 1; nchunk <= nz; ++nchunk) {
        const int zc = (nz + nchunk - 1) / nchunk;
        if (zc > AH_ZC_MAX) continue;
        if (zc < 4 && nz >= 4) break;
        const long long ctas = cols * ((nz + zc - 1) / zc);
        const double waves = ctas >= 6 * resident ? (double)ctas / (double)resident
                                                  : (double)((ctas + resident - 1) / resident);
        const double cost = waves * (zc + 2.5);     // 2.5 planes ~ ring fill + hand-down of the plane below
        if (cost < best_cost * (1.0 - 1e-9)) {
            best_cost = cost;
            best = zc;
        }
    }
    return best;
}

int tiled_chunk(int nx, int ny, int nz, bool diag) { return chunk_for(nx, ny, nz, diag ? TILE_Y_DIAG : TILE_Y); }

float tiled_th_limit() { return AH_TILED_TH_LIMIT; }

// nz: number of planes the launch updates
int tiled_num_blocks(int nx, int ny, int nz, bool diag)
{
    if (!tiled_supported(nx, ny, nz)) return 0;
    const int ty = diag ? TILE_Y_DIAG : TILE_Y;
    const int zc = chunk_for(nx, ny, nz, ty);
    return (nx / (32 * spt_for(nx))) * ((ny + ty - 1) / ty) * ((nz + zc - 1) / zc);
}

template <int SPT, int TY, bool COMPACT, bool DIAG, bool WIND>
static cudaError_t launch_one(const ConstFields<float> &in, const Fields<float> &out, const StepCoef<float> &k, int nx,
                              int ny, int nz, ZRange zr, int *overflow, cudaStream_t st, const DiagCoef &d,
                              DiagPartial *partials)
{
    const int zc = chunk_for(nx, ny, zr.hi - zr.lo, TY);
    dim3 grid(nx / (32 * SPT), (ny + TY - 1) / TY, (zr.hi - zr.lo + zc - 1) / zc);
    dim3 block((TY + 1) * 32);
    if (grid.y > 65535u || grid.z > 65535u) return cudaErrorInvalidConfiguration;
    return launch_pdl(tiled_step_kernel<SPT, TY, COMPACT, DIAG, WIND>, grid, block, sizeof(Smem<SPT, TY, DIAG>), st, in, out, k, nx,
                      ny, nz, zr.lo, zr.hi, zc, overflow, d, partials);
}

template <int SPT>
static cudaError_t launch_spt(const ConstFields<float> &in, const Fields<float> &out, const StepCoef<float> &k, int nx,
                              int ny, int nz, ZRange zr, int *overflow, cudaStream_t st, bool diag, const DiagCoef &d,
                              DiagPartial *partials)
{
    if (!diag)
        return k.compact ? launch_one<SPT, TILE_Y, true, false, false>(in, out, k, nx, ny, nz, zr, overflow, st, d, nullptr)
                         : launch_one<SPT, TILE_Y, false, false, false>(in, out, k, nx, ny, nz, zr, overflow, st, d, nullptr);
    if (d.winding)
        return k.compact ? launch_one<SPT, TILE_Y_DIAG, true, true, true>(in, out, k, nx, ny, nz, zr, overflow, st, d, partials)
                         : launch_one<SPT, TILE_Y_DIAG, false, true, true>(in, out, k, nx, ny, nz, zr, overflow, st, d, partials);
    return k.compact ? launch_one<SPT, TILE_Y_DIAG, true, true, false>(in, out, k, nx, ny, nz, zr, overflow, st, d, partials)
                     : launch_one<SPT, TILE_Y_DIAG, false, true, false>(in, out, k, nx, ny, nz, zr, overflow, st, d, partials);
}

// partials == nullptr: plain step.  Otherwise the DIAG instantiation, which also writes one DiagPartial per
// CTA (tiled_num_blocks(.., planes updated, true) of them) holding the read-outs of the entry snapshot.
// zr: the planes to update; {0, nz} is the whole periodic lattice.
cudaError_t launch_tiled_step(const ConstFields<float> &in, const Fields<float> &out,
                              const StepCoef<float> &k, int nx, int ny, int nz, ZRange zr, int *overflow, cudaStream_t st,
                              const DiagCoef *dk, DiagPartial *partials)
{
    if (!tiled_supported(nx, ny, nz) || zr.lo < 0 || zr.hi > nz || zr.lo >= zr.hi) return cudaErrorInvalidValue;
    const bool diag = partials != nullptr && dk != nullptr;
    const DiagCoef d = diag ? *dk : DiagCoef{};
    return spt_for(nx) == 4 ? launch_spt<4>(in, out, k, nx, ny, nz, zr, overflow, st, diag, d, partials)
                            : launch_spt<2>(in, out, k, nx, ny, nz, zr, overflow, st, diag, d, partials);
}

}  // namespace ah
