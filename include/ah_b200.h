/*
 * ah_b200.h — C ABI of the B200 (sm_100a) Abelian-Higgs leapfrog library.
 *
 * Hot path of Correia & Martins, "Abelian-Higgs cosmic string evolution with
 * multiple GPUs" (arXiv:2005.14454): the damped leapfrog step of the lattice
 * U(1) gauge-Higgs model in an FRW background (Eqs. 7-11, with
 * the stencils of Eqs. 12-15) and the network read-outs
 * (winding, Eq. 16; Lagrangian-weighted <v^2>, PAPER.md:107-111
 * Eqs. 17-18; Gauss law, Eq. 5 and :83).  Readings of the garbled
 * or silent passages are listed in DESIGN.md ("Readings").
 *
 * Conventions
 *   - One periodic nx*ny*nz lattice in ONE GPU's memory; site x=(x,y,z) has
 *     linear index x + nx*(y + ny*z) (x fastest).
 *   - State = 10 real scalars per site, structure-of-arrays, in this order:
 *       0 phi_re 1 phi_im 2 pi_re 3 pi_im 4 th_x 5 th_y 6 th_z 7 ep_x 8 ep_y 9 ep_z
 *     th_i(x) is the paper's lattice link angle A_i(x) of Eq. 12 (U_i = exp(-i th_i)),
 *     ep_i(x) the paper's lattice E_i(x) of Eq. 10 (= d th_i / d tau).
 *   - phi, th live at tau_k; Pi, ep at tau_k - dt/2.
 *   - All pointers named dev_* are DEVICE pointers, host_* are HOST pointers.
 *   - Every function returns 0 on success or a negative AH_E* code; no C++
 *     exception crosses this boundary; ah_last_error() gives a message for the
 *     calling thread's most recent failure.
 *   - Nothing here falls back to the CPU: without a CUDA device every compute
 *     entry point returns AH_ECUDA.
 *   - Test and measurement hooks (kernel selection, launch counters, launch geometry, the device trig
 *     evaluators) are NOT part of this interface: they live in ah_b200_test.h.
 */
#ifndef AH_B200_H
#define AH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define AH_OK 0
#define AH_EINVAL (-1) /* bad parameter, null pointer, tau <= 0 with p != 0, cap too small */
#define AH_ECUDA (-2)  /* CUDA runtime failure (message in ah_last_error)                 */
#define AH_ESTATE (-3) /* call made in the wrong state (e.g. stepping before any fields)  */

#define AH_NFIELDS 10

/* ah_params.fp64 */
#define AH_PRECISION_FP32 0
#define AH_PRECISION_FP64 1
#define AH_PRECISION_MIXED 2 /* fp32 storage, fp64 arithmetic; results rounded once, on the store */

/* z slabs (below): fields whose boundary planes neighbours exchange, and the raw partial sums of a slab's read-outs */
#define AH_NHALO 6      /* phi_re, phi_im, th_x, th_y, th_z, ep_z */
#define AH_NDIAG_INT 5  /* |W| sums xy, xz, yz; near-branch count; big-plaquette count            */
#define AH_NDIAG_FLT 9  /* sums of |Pi|^2 L, grad2 L, L, G^2, div^2, charge^2, p L, rho L; then max |G| (last) */

typedef struct ah_ctx ah_ctx; /* opaque */

/* Model and lattice parameters.  Plain data, host side. */
typedef struct {
    int32_t nx, ny, nz; /* periodic extents, each >= 1                                             */
    double dx;          /* lattice spacing (0.5 in the paper)                          */
    double lambda0, e0, sigma; /* couplings (2, 1, 1: critical coupling)              */
    double s;           /* core-growth exponent of Eq. 6: 0 constant comoving width, 1 physical     */
    double p;           /* dln a/dln tau = m/(1-m) (Eq. 11): 0 Minkowski, 1 radiation, 2 matter      */
    double tau_ref;     /* a(tau) = (tau/tau_ref)^p (reading #6); ignored when p == 0 or s == 0      */
    double alpha;       /* damping constant of PAPER.md:78; 2 = physical Hubble damping              */
    int32_t compact;    /* 1: sin(plaquette) force, 2(1-cos) energy (reading #10); 0: non-compact     */
    int32_t fp64;       /* AH_PRECISION_*: 0 fp32 state and arithmetic (the product); 1 fp64 state and arithmetic
                           (site kernel); 2 fp32 state, every operation of the step in fp64 (site kernel)   */
} ah_params;

/* Diagnostics of one snapshot. */
typedef struct {
    double tau;
    int64_t n_wind, n_wind_xy, n_wind_xz, n_wind_yz; /* sum |W_ij| (Eq. 16 right)                   */
    int64_t n_near_branch; /* plaquettes with a link phase within 1e-5 of +-pi (reading #14)        */
    int64_t n_big_plaq;    /* plaquettes with |Phi_ij| > pi - 1e-5 (reading #13)                    */
    double string_length, xi_w; /* dx*n_wind ; sqrt(V/L_W), +inf when n_wind == 0                   */
    double sum_pi2_L, sum_grad2_L, sum_L, v2_phi; /* Eqs. 17-18                                      */
    double gauss_max, gauss_l2, gauss_rel;        /* Eq. 5 residual                                  */
    double gauss_div_l2, gauss_charge_l2;
    double xi_l; /* Lagrangian estimator sqrt(-mu V / sum_x L_x dx^3), mu = 2 pi sigma^2 (Eq. 16 left,
                    PAPER.md:102; reading #16); +inf when the sum is not negative                        */
    double sum_p_L, sum_rho_L; /* sum_x p_x L_x, sum_x rho_x L_x: isotropic pressure and energy density of the five
                    pieces of L_x, weighted with L_x (reading #17)                               */
    double v2_omega; /* equation-of-state estimator (1 + 3 sum p L / sum rho L) / 2 (Eq. 17 right)  */
    double xi_w_corr; /* xi_w above is the RAW estimator: string_length counts every pierced plaquette as one lattice
                    spacing (a Manhattan length), which over-counts a smooth string; the values the paper prints for
                    xi_W (Table 1) carry the usual correction L -> (pi/6) L of that over-count
                    (reading #13).  xi_w_corr = sqrt(V / ((pi/6) string_length)) = xi_w sqrt(6/pi) is the
                    number to compare with the paper; +inf when n_wind == 0, NaN without the winding read-out      */
} ah_diag;

/*
 * ah_create — make a context on the current CUDA device.
 *   dev_bufs : 2*AH_NFIELDS caller-owned device arrays (e.g. PyTorch tensors), each of
 *              nx*ny*nz elements (float, or double when params->fp64), 16-byte aligned.
 *              Buffers [0,10) hold the current state (order above); [10,20) are the
 *              ping-pong partners.  The context only borrows them: it never frees them,
 *              and they must outlive it.  After an odd number of steps the current state
 *              lives in [10,20); use ah_current_bufs / ah_get_fields, never assume.
 *   nbufs    : must be 20.   bytes_each: must equal nx*ny*nz*sizeof(element).
 *   cuda_stream : a cudaStream_t (0 = legacy default stream); all work is enqueued on it.
 * Allocates only small context-owned scratch (reduction partials, a few hundred KB).
 */
int ah_create(ah_ctx **out, const ah_params *params, void *const dev_bufs[], int nbufs,
              size_t bytes_each, void *cuda_stream);

/* Frees context-owned scratch only, never the field buffers.  NULL is a no-op. */
int ah_destroy(ah_ctx *ctx);

/* I0: phi = sigma*exp(2 pi i u(seed, linear index)), Pi = th = ep = 0, with the
 * counter-based u of DESIGN.md "I0".  Asynchronous on the stream.  Resets the ping-pong parity. */
int ah_init_fields(ah_ctx *ctx, uint64_t seed);

/* Upload / download a snapshot: host_soa10 holds 10 contiguous arrays of nx*ny*nz elements
 * (float or double as the context) in the field order above.  Both synchronise the stream. */
int ah_set_fields(ah_ctx *ctx, const void *host_soa10);
int ah_get_fields(ah_ctx *ctx, void *host_soa10);

/* Which 10 device pointers hold the current state (ping-pong parity resolved). */
int ah_current_bufs(ah_ctx *ctx, void *dev_ptrs_out[AH_NFIELDS]);

/*
 * ah_step — advance n leapfrog steps (Eqs. 7-10) starting from conformal time tau, with phi, th
 * at tau and Pi, ep at tau - dt/2.  Step j uses the coefficients (a, delta, omega of
 * PAPER.md:78-80) at tau_j = tau + j*dt, the product evaluated in fp64.  Asynchronous on the
 * stream; allocates nothing.  n == 0 is a no-op.  AH_EINVAL if n < 0, dt <= 0 or (p != 0 and
 * tau <= 0); AH_ESTATE if no fields were ever set.
 */
int ah_step(ah_ctx *ctx, int n, double tau, double dt);

/*
 * ah_step_cooling — n leapfrog steps with a CONSTANT artificial damping delta on both Pi and ep and the couplings at
 * their a = 1 values (the "artificial damping (cooling) period" of PAPER.md:63; used to relax initial conditions,
 * e.g. onto a static string).  Identical to ah_step on a context with p = 1, s = 0, alpha = 2 called n times at the
 * fixed time tau = dt / delta; the context's own parameters are not modified (re-entrant with respect to
 * them).  AH_EINVAL if n < 0, dt <= 0 or delta <= 0 or delta >= 1.
 */
int ah_step_cooling(ah_ctx *ctx, int n, double delta, double dt);

/* Diagnostics D1-D3 of the current snapshot (fields at tau, momenta at tau - dt/2).
 * Synchronous: returns after the result is in *host_out.  AH_EINVAL when omega = (1-s) delta = 1 at tau
 * (the Gauss coefficient kappa = q (1-delta)/(1-omega) of DESIGN.md reading #18 does not exist there). */
int ah_diagnostics(ah_ctx *ctx, double tau, double dt, ah_diag *host_out);

/*
 * ah_step_diag — n steps with diagnostics of the ENTRY snapshot of every step j with
 * j % every == 0 (SURVEY 8(a) row D-fuse): identical to calling ah_diagnostics(tau_j) before
 * step j.  Records are written to host_out[0..*n_written).  AH_EINVAL, without stepping, when
 * cap < ceil(n/every) or every < 1.  Synchronous at return.
 */
int ah_step_diag(ah_ctx *ctx, int n, double tau, double dt, int every, ah_diag *host_out, int cap,
                 int *n_written);

/*
 * ah_step_diag_sums — as ah_step_diag, but the records carry the Lagrangian-weighted estimators (xi_L, <v^2>_phi,
 * <v^2>_omega and their sums) and the Gauss residual only: the set the paper's timed runs evaluate every 5 steps
 * (PAPER.md:181).  The winding read-out is skipped (on the tiled kernel neither site phases nor link phases are
 * computed): n_wind* = n_near_branch = n_big_plaq = -1, string_length = xi_w = xi_w_corr = NaN.  All other fields are bit-identical
 * to ah_step_diag's, and so are the fields the steps leave.
 */
int ah_step_diag_sums(ah_ctx *ctx, int n, double tau, double dt, int every, ah_diag *host_out, int cap,
                      int *n_written);

/* Per-plaquette winding integers of the current snapshot: host_w3 receives 3 arrays (xy, xz, yz)
 * of nx*ny*nz int8; host_near3 (may be NULL) the near-branch flags as uint8.  Synchronous. */
int ah_winding_field(ah_ctx *ctx, int8_t *host_w3, uint8_t *host_near3);

/*
 * ---- z slabs: one periodic lattice cut along z over several GPUs (the paper's domain decomposition, PAPER.md:122-142,
 * in its natural single-node form: 1-D slabs, one exchange of boundary planes per step, overlapped with the update of
 * the interior).  BASELINE's north_star keeps the measured build on ONE GPU.  What has been executed: a lattice cut
 * into slab contexts on ONE GPU (device-to-device copies stand in for the exchange), bit-identical to the single
 * lattice.  What has NOT: the exchange between ranks over NCCL on more than one GPU (no multi-GPU node on this pool;
 * tests/test_gpu_slabs.py holds a two-rank test that is skipped below two GPUs).
 * Bit identity with the single lattice holds while every link angle stays inside the tiled kernel's domain
 * (|th| < 2^16 rad): outside it the step is redone with the libm-based site kernel by the slab that READS the angle
 * (its own planes, its ghost planes, the planes next to its boundary planes), not by the whole lattice, so the other
 * slabs keep the tiled kernel's bits; every slab's result stays within the one-step tolerance either way.
 *
 * A slab context owns nz_own consecutive planes z_first .. z_first+nz_own-1 of the global lattice params->nz and
 * stores nz_own + 2 planes per array: plane 0 is the ghost copy of global plane z_first-1, planes 1 .. nz_own the
 * own planes, plane nz_own+1 the ghost copy of global plane z_first+nz_own (indices modulo nz).  dev_bufs are 20
 * caller-owned arrays of nx*ny*(nz_own+2) elements.  ah_init_fields fills own AND ghost planes (the generator is
 * counter-based on the global site index); ah_set_fields / ah_get_fields move all nz_own+2 planes.
 *
 * Per step:   ah_slab_step(ctx, tau, dt, want_diag, comm_stream)
 *             copy the planes ah_slab_halo_ptrs names, on comm_stream (NCCL send/recv between ranks, or plain
 *               device copies between slabs of one process):  my send_lo -> lower neighbour's recv_hi,
 *                                                              my send_hi -> upper neighbour's recv_lo
 *             ah_slab_exchange_done(ctx, comm_stream)
 * ah_slab_step updates the two boundary planes first, makes comm_stream wait for exactly those launches, then
 * updates the interior on the context's stream, so the copies overlap the interior.  ah_slab_exchange_done makes the
 * context's stream wait for what has been enqueued on comm_stream.  comm_stream may be the context's own stream
 * (no overlap, no events).  ah_step / ah_step_diag / ah_diagnostics return AH_ESTATE on a slab context.
 */
int ah_create_slab(ah_ctx **out, const ah_params *global_params, int nz_own, int z_first, void *const dev_bufs[],
                   int nbufs, size_t bytes_each, void *cuda_stream);

/* One step of the slab's own planes.  want_diag != 0: also the read-outs D1-D3 of the ENTRY snapshot of the own
 * planes (fused on the tiled kernel, boundary planes first there too, so the exchange overlaps the interior on read-out
 * steps as well), left on the device for ah_slab_diag_partial. */
int ah_slab_step(ah_ctx *ctx, double tau, double dt, int want_diag, void *comm_stream);

/* Device pointers of the boundary / ghost planes of the CURRENT state, per exchanged field (AH_NHALO of them, order
 * above), each plane_bytes = nx*ny*sizeof(element) long. */
int ah_slab_halo_ptrs(ah_ctx *ctx, void *dev_send_lo[AH_NHALO], void *dev_send_hi[AH_NHALO], void *dev_recv_lo[AH_NHALO],
                      void *dev_recv_hi[AH_NHALO], size_t *plane_bytes);

int ah_slab_exchange_done(ah_ctx *ctx, void *comm_stream);

/* Read-outs of the own planes of the current snapshot (standalone kernel), left on the device. */
int ah_slab_diagnostics(ah_ctx *ctx, double tau, double dt);

/* The slab's raw partial sums of the last requested read-out (synchronises the stream).  Slabs combine them by
 * adding counts and sums[0..7] and taking the maximum of sums[8] (an all-reduce of 14 numbers), then ah_diag_finish. */
int ah_slab_diag_partial(ah_ctx *ctx, int64_t host_counts[AH_NDIAG_INT], double host_sums[AH_NDIAG_FLT]);

/* Totals of a whole lattice from the raw partial sums of its n_parts slabs (host arithmetic only): part r's counts are
 * host_counts[r*AH_NDIAG_INT ..], its sums host_sums[r*AH_NDIAG_FLT ..]; counts and sums[0..7] add in the order
 * given (fixed order: reproducible), sums[8] (max |G|) takes the maximum.  AH_EINVAL for null pointers or n_parts < 1. */
int ah_diag_combine(int n_parts, const int64_t *host_counts, const double *host_sums,
                    int64_t host_counts_out[AH_NDIAG_INT], double host_sums_out[AH_NDIAG_FLT]);

/* Totals of a whole lattice -> the ah_diag record; host arithmetic only: xi_W, xi_L, <v^2>_phi, Gauss norms. */
int ah_diag_finish(const ah_params *global_params, const int64_t host_counts[AH_NDIAG_INT],
                   const double host_sums[AH_NDIAG_FLT], double tau, ah_diag *host_out);

/*
 * ah_readout_noalloc — the read-outs D1-D3 of one whole-lattice snapshot (what ah_diagnostics computes: winding
 * counts, Eq. 16 right; Lagrangian-weighted sums, Eqs. 17-18; Gauss residual,
 * Eq. 5) WITHOUT a context and without allocating anything, on the device or on the host.
 *
 * Who needs it.  Every other read-out call goes through an ah_ctx, and ah_create obtains the context's scratch with
 * cudaMalloc / cudaMallocHost.  Some callers cannot do that at the moment they want a read-out:
 *   - a host program that handed (nearly) all of the GPU's memory to its own pool up front (a 1024^3 run already
 *     holds 86 GB of fields; a framework's caching allocator typically owns the rest), so a driver allocation
 *     may fail, or may succeed only after the pool is trimmed;
 *   - a monitoring or steering loop that must not stall the GPU: cudaMalloc and cudaFree synchronise the whole
 *     device, so a read-out that allocates would drain every stream of the process each time it is asked for;
 *   - code that runs inside somebody else's no-allocation region (a plugin or callback contract that forbids
 *     changes to the memory map, a fixed-footprint service that is audited for a constant memory use).
 * Such callers own the field arrays already (they are the inputs) and can set 112 bytes aside for the result; the
 * only other memory the read-out needs is the per-block partial sums, and for this call those live in a fixed array
 * inside the library image.
 *
 *   params     : the model and the extents of the lattice (host pointer); fp64 = 0 or 2 reads float arrays, 1 double.
 *   dev_fields : AH_NFIELDS DEVICE arrays of nx*ny*nz elements in the field order above (e.g. what ah_current_bufs
 *                returned, or the caller's own buffers); read only.
 *   tau, dt    : as for ah_diagnostics (fields at tau, momenta at tau - dt/2).
 *   dev_totals : DEVICE buffer of AH_NOALLOC_TOTALS_BYTES, 8-byte aligned, caller-owned: receives int64
 *                counts[AH_NDIAG_INT] followed by double sums[AH_NDIAG_FLT], the raw totals that ah_slab_diag_partial
 *                also returns.  Copy them to the host when convenient and pass them to ah_diag_finish (host
 *                arithmetic only) for xi_W, xi_L, <v^2>, the Gauss norms.
 *   cuda_stream: the two kernels are enqueued on it; the call returns without synchronising.
 *
 * Limit.  The fixed array holds AH_NOALLOC_MAX_PARTIALS partial sums, one per block of 64 x 4 x 8 sites:
 * ceil(nx/64) * ceil(ny/4) * ceil(nz/8) must not exceed it, so 512^3 is the largest cube.  Larger lattices get
 * AH_EINVAL with a message naming the limit; nothing is launched.  The array costs 7 MiB of device memory on every GPU
 * on which the library's code is loaded, from then until the process ends, whether or not this call is ever made.
 *
 * First call.  The first call on each device asks the CUDA runtime for the array's device address
 * (cudaGetSymbolAddress, once per device, with that device current) and keeps it; later calls only launch.  Make that
 * first call at start-up, with the device you will use current and before any stream capture begins.
 *
 * Sharing.  There is ONE array per device, shared by every call from every thread, and it keeps whatever the last call
 * left in it.  Nothing in it needs clearing (each call overwrites every entry it later reads), but two calls whose
 * kernels can run at the same time on one GPU — different streams with no ordering between them — race on it and both
 * results are then garbage.  Keep the calls of one device on one stream, or order them with events.
 *
 * Results are bit-identical to ah_diagnostics on the same snapshot (same kernels, same summation order).
 * Errors: AH_EINVAL (null or misaligned pointer, bad params, dt <= 0, tau <= 0 with p != 0, omega = 1, lattice beyond
 * the limit), AH_ECUDA (no device, address look-up or launch failed).
 */
#define AH_NOALLOC_MAX_PARTIALS 65536
#define AH_NOALLOC_TOTALS_BYTES (8 * (AH_NDIAG_INT + AH_NDIAG_FLT))
int ah_readout_noalloc(const ah_params *params, const void *const dev_fields[AH_NFIELDS], double tau, double dt,
                       void *dev_totals, void *cuda_stream);

/* Host-side coefficients as the kernels receive them (for tests): a, q = a^{2s}, delta, omega. */
int ah_coeffs(const ah_params *params, double tau, double dt, double *a, double *q, double *delta,
              double *omega);

/* Message for the calling thread's most recent error ("" if none).  Never NULL. */
const char *ah_last_error(void);

/* Library version string. */
const char *ah_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AH_B200_H */
