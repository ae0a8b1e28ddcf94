// ah_api.cu — the C ABI of include/ah_b200.h: argument checking, per-step coefficients on the
// host in fp64, kernel launches on the caller's stream.  No field arithmetic happens here.
#include "../../include/ah_b200.h"
#include "../../include/ah_b200_test.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <limits>
#include <new>

#include "ah_kernels.h"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int cuda_fail(cudaError_t e, const char *what)
{
    return fail(AH_ECUDA, "%s: %s (%s)", what, cudaGetErrorString(e), cudaGetErrorName(e));
}

#define AH_CUDA(call)                                       \
    do {                                                    \
        cudaError_t e__ = (call);                           \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)

// PAPER.md:78-80 with readings #4-#6: a = (tau/tau_ref)^p, q = a^{2s},
// delta = (alpha/2) p dt / tau, omega = (1-s) delta.
void coeffs(const ah_params &P, double tau, double dt, double &a, double &q, double &delta,
            double &omega)
{
    a = (P.p == 0.0) ? 1.0 : std::pow(tau / P.tau_ref, P.p);
    q = (P.s == 0.0) ? 1.0 : std::pow(a, 2.0 * P.s);
    delta = (P.p == 0.0) ? 0.0 : 0.5 * P.alpha * P.p * dt / tau;
    omega = delta * (1.0 - P.s);
}

template <typename real>
ah::StepCoef<real> make_coef(const ah_params &P, double tau, double dt)
{
    double a, q, d, w;
    coeffs(P, tau, dt, a, q, d, w);
    ah::StepCoef<real> k;
    k.idx2 = (real)(1.0 / (P.dx * P.dx));
    k.c1 = (real)((1.0 - d) / (1.0 + d));
    k.c2 = (real)(dt / (1.0 + d));
    k.w1 = (real)((1.0 - w) / (1.0 + w));
    k.w2 = (real)(dt / (1.0 + w));
    k.half_lam_q = (real)(0.5 * P.lambda0 * q);
    k.sig2 = (real)(P.sigma * P.sigma);
    k.two_e2_q = (real)(2.0 * P.e0 * P.e0 * q);
    k.dt = (real)dt;
    k.compact = P.compact;
    return k;
}

ah::DiagCoef make_diag_coef(const ah_params &P, double tau, double dt)
{
    double a, q, d, w;
    coeffs(P, tau, dt, a, q, d, w);
    ah::DiagCoef k;
    k.idx2 = 1.0 / (P.dx * P.dx);
    k.q = q;
    k.quarter_lam_q = 0.25 * P.lambda0 * q;
    k.sig2 = P.sigma * P.sigma;
    k.inv_2e2q = 1.0 / (2.0 * P.e0 * P.e0 * q);
    // reading #18; omega == 1 (the momentum half step would sit on the damping pole) has no Gauss coefficient:
    // callers check it (ah_diagnostics returns AH_EINVAL); 0 keeps the kernel's sums finite
    k.two_e2_kappa = (w == 1.0) ? 0.0 : 2.0 * P.e0 * P.e0 * q * (1.0 - d) / (1.0 - w);
    k.compact = P.compact;
    k.winding = 1;
    k.f_idx2 = (float)k.idx2;
    k.f_idx4 = (float)(k.idx2 * k.idx2);
    k.f_quarter_lam_q = (float)k.quarter_lam_q;
    k.f_sig2 = (float)k.sig2;
    k.f_inv_2e2q = (float)k.inv_2e2q;
    return k;
}

}  // namespace

struct ah_ctx {
    ah_params P;       // the model; nx, ny, nz are the extents of the GLOBAL periodic lattice
    void *bufs[2 * AH_NFIELDS];
    int cur;           // 0: state in bufs[0..10), 1: in bufs[10..20)
    bool have_fields;
    cudaStream_t st;
    // storage: nza planes of nx*ny sites per array.  Whole lattice: nza = nz, zr = {0, nz}.  z slab (ah_create_slab):
    // nza = own planes + 2 ghost planes, zr = {1, nza - 1}, plane zl is global plane z_offset + zl.
    int nza;
    ah::ZRange zr;
    int z_offset;
    bool slab;
    cudaEvent_t ev_boundary, ev_exchange;   // slab: boundary planes of the new state are final / ghost planes have landed
    size_t n;          // sites stored per array (nx*ny*nza)
    size_t elem;       // bytes per element
    int kernel;        // resolved AH_KERNEL_SITE / AH_KERNEL_TILED
    int64_t launches;
    ah::DiagPartial *d_partials;
    int n_partials;
    ah::DiagPartial *d_results;
    ah::DiagPartial *h_results;  // pinned
    int cap_results;
    int *d_overflow;   // two flags (step parity): tiled kernel met a link angle outside its domain
    int step_parity;
};

namespace {

template <typename real>
ah::ConstFields<real> cur_fields(const ah_ctx *c)
{
    ah::ConstFields<real> f;
    for (int a = 0; a < AH_NFIELDS; ++a) f.f[a] = (const real *)c->bufs[c->cur * AH_NFIELDS + a];
    return f;
}
template <typename real>
ah::Fields<real> next_fields(const ah_ctx *c)
{
    ah::Fields<real> f;
    for (int a = 0; a < AH_NFIELDS; ++a) f.f[a] = (real *)c->bufs[(1 - c->cur) * AH_NFIELDS + a];
    return f;
}
template <typename real>
ah::Fields<real> cur_fields_mut(const ah_ctx *c)
{
    ah::Fields<real> f;
    for (int a = 0; a < AH_NFIELDS; ++a) f.f[a] = (real *)c->bufs[c->cur * AH_NFIELDS + a];
    return f;
}

bool is_fp64(const ah_params &P) { return P.fp64 == AH_PRECISION_FP64; }
bool is_mixed(const ah_params &P) { return P.fp64 == AH_PRECISION_MIXED; }

int check_time(const ah_ctx *c, double tau, double dt)
{
    if (!(dt > 0.0) || !std::isfinite(dt) || !std::isfinite(tau))
        return fail(AH_EINVAL, "dt must be positive and finite (dt=%g, tau=%g)", dt, tau);
    if (c->P.p != 0.0 && !(tau > 0.0))
        return fail(AH_EINVAL, "tau must be > 0 in an expanding background (tau=%g, p=%g)", tau, c->P.p);
    return AH_OK;
}

// Launches of one step over the planes zr of the current state into the other buffer set; no context state changes
// here except the launch counter.  Tiled kernel: the fast path, then a conditional redo of the same planes with the
// libm-based site kernel (runs only if the fast path flagged a link angle beyond its polynomial range).
// diag_slot >= 0 (tiled fp32 kernel only): the fused DIAG instantiation also leaves the read-outs of the entry
// snapshot of those planes in d_results[diag_slot] (SURVEY 8(a) row D-fuse).
cudaError_t enqueue_step(ah_ctx *c, const ah_params &P, double tau, double dt, ah::ZRange zr, int diag_slot, int *flag,
                         int *next_flag, bool winding = true)
{
    cudaError_t e;
    const int nx = P.nx, ny = P.ny, nza = c->nza;
    if (is_fp64(P)) {
        e = ah::launch_site_step<double>(cur_fields<double>(c), next_fields<double>(c), make_coef<double>(P, tau, dt), nx,
                                         ny, nza, zr, c->st);
        if (e == cudaSuccess) c->launches += 1;
    } else if (is_mixed(P)) {
        e = ah::launch_site_step_mixed(cur_fields<float>(c), next_fields<float>(c), make_coef<double>(P, tau, dt), nx, ny,
                                       nza, zr, c->st);
        if (e == cudaSuccess) c->launches += 1;
    } else if (c->kernel == AH_KERNEL_TILED) {
        const ah::StepCoef<float> k = make_coef<float>(P, tau, dt);
        if (diag_slot >= 0) {
            ah::DiagCoef dk = make_diag_coef(P, tau, dt);
            dk.winding = winding ? 1 : 0;
            e = ah::launch_tiled_step(cur_fields<float>(c), next_fields<float>(c), k, nx, ny, nza, zr, flag, c->st, &dk,
                                      c->d_partials);
            // a link angle outside the tiled kernel's domain spoils its read-outs as well: the standalone kernel
            // then re-evaluates the entry snapshot (conditional launch, exits at once when the flag is clear)
            if (e == cudaSuccess) {
                c->launches += 1;
                e = ah::launch_diag_partials<float>(cur_fields<float>(c), dk, nx, ny, nza, zr, c->d_partials, nullptr,
                                                    nullptr, flag, c->st);
            }
            if (e == cudaSuccess) {
                c->launches += 1;
                e = ah::launch_diag_final(c->d_partials, ah::tiled_num_blocks(nx, ny, zr.hi - zr.lo, true),
                                          c->d_results + diag_slot, c->st, ah::diag_num_blocks(nx, ny, zr.hi - zr.lo), flag);
            }
        } else {
            e = ah::launch_tiled_step(cur_fields<float>(c), next_fields<float>(c), k, nx, ny, nza, zr, flag, c->st);
        }
        if (e == cudaSuccess) {
            c->launches += 1;
            e = ah::launch_site_redo(flag, next_flag, cur_fields<float>(c), next_fields<float>(c), k, nx, ny, nza, zr, c->st);
        }
        if (e == cudaSuccess) c->launches += 1;
    } else {
        e = ah::launch_site_step<float>(cur_fields<float>(c), next_fields<float>(c), make_coef<float>(P, tau, dt), nx, ny,
                                        nza, zr, c->st);
        if (e == cudaSuccess) c->launches += 1;
    }
    return e;
}

// One whole step.  Context state (ping-pong parity, flag parity) changes only after EVERY launch of the step was
// accepted; a failed launch leaves the context on the entry snapshot with both overflow flags cleared.
// P: the model the step uses (the context's own, or ah_step_cooling's constant-damping copy of it)
int one_step(ah_ctx *c, const ah_params &P, double tau, double dt, int diag_slot = -1, bool winding = true)
{
    int *flag = c->d_overflow + c->step_parity, *next_flag = c->d_overflow + (1 - c->step_parity);
    const cudaError_t e = enqueue_step(c, P, tau, dt, c->zr, diag_slot, flag, next_flag, winding);
    if (e != cudaSuccess) {
        cudaMemsetAsync(c->d_overflow, 0, 2 * sizeof(int), c->st);   // a half-issued step must not leave a stale flag
        return cuda_fail(e, "step kernel launch");
    }
    c->step_parity = 1 - c->step_parity;
    c->cur = 1 - c->cur;
    return AH_OK;
}

int ensure_diag_scratch(ah_ctx *c, int records)
{
    const int own = c->zr.hi - c->zr.lo;
    int nb = ah::diag_num_blocks(c->P.nx, c->P.ny, own);
    int nbt = ah::tiled_num_blocks(c->P.nx, c->P.ny, own, true);
    if (c->slab && own > 2)   // boundary planes and interior read out by three launches (ah_slab_step)
        nbt = 2 * ah::tiled_num_blocks(c->P.nx, c->P.ny, 1, true) + ah::tiled_num_blocks(c->P.nx, c->P.ny, own - 2, true);
    if (nbt > nb) nb = nbt;
    if (c->n_partials < nb) {
        if (c->d_partials) cudaFree(c->d_partials);
        c->d_partials = nullptr;
        c->n_partials = 0;
        AH_CUDA(cudaMalloc(&c->d_partials, sizeof(ah::DiagPartial) * (size_t)nb));
        c->n_partials = nb;
    }
    if (c->cap_results < records) {
        if (c->d_results) cudaFree(c->d_results);
        if (c->h_results) cudaFreeHost(c->h_results);
        c->d_results = nullptr;
        c->h_results = nullptr;
        c->cap_results = 0;
        int cap = records < 256 ? 256 : records;
        AH_CUDA(cudaMalloc(&c->d_results, sizeof(ah::DiagPartial) * (size_t)cap));
        AH_CUDA(cudaMallocHost(&c->h_results, sizeof(ah::DiagPartial) * (size_t)cap));
        c->cap_results = cap;
    }
    return AH_OK;
}

// the Gauss coefficient kappa = q (1 - delta) / (1 - omega) of reading #18 needs omega != 1
int check_diag_time(const ah_ctx *c, double tau, double dt)
{
    int rc = check_time(c, tau, dt);
    if (rc != AH_OK) return rc;
    double a, q, d, w;
    coeffs(c->P, tau, dt, a, q, d, w);
    if (w == 1.0)
        return fail(AH_EINVAL, "diagnostics: omega = (1-s) delta = 1 at tau=%g, dt=%g: no Gauss coefficient", tau, dt);
    return AH_OK;
}

// standalone read-outs of the own planes of the current snapshot into d_results[slot]
// winding_only: coefficients of the static a = 1 model (the winding integers depend on none of them)
int enqueue_diag(ah_ctx *c, double tau, double dt, int slot, int8_t *w3, uint8_t *near3, bool winding_only = false)
{
    ah_params P = c->P;
    if (winding_only) P.p = 0.0, P.s = 0.0;
    const ah::DiagCoef k = make_diag_coef(P, tau, dt);
    cudaError_t e;
    if (is_fp64(P))
        e = ah::launch_diag<double>(cur_fields<double>(c), k, P.nx, P.ny, c->nza, c->zr, c->d_partials,
                                    c->d_results + slot, w3, near3, c->st);
    else
        e = ah::launch_diag<float>(cur_fields<float>(c), k, P.nx, P.ny, c->nza, c->zr, c->d_partials,
                                   c->d_results + slot, w3, near3, c->st);
    if (e != cudaSuccess) return cuda_fail(e, "diagnostics kernel launch");
    c->launches += 2;
    return AH_OK;
}

// totals -> the derived numbers of ah_diag (P: the GLOBAL lattice the totals belong to).
// winding == false: the record carries no winding read-out (counts -1, lengths NaN), whatever the kernel summed.
void finish_diag(const ah_params &P, const ah::DiagPartial &r, double tau, ah_diag *out, bool winding = true)
{
    out->tau = tau;
    if (winding) {
        out->n_wind_xy = r.i[ah::DS_NW_XY];
        out->n_wind_xz = r.i[ah::DS_NW_XZ];
        out->n_wind_yz = r.i[ah::DS_NW_YZ];
        out->n_wind = out->n_wind_xy + out->n_wind_xz + out->n_wind_yz;
        out->n_near_branch = r.i[ah::DS_NEAR];
        out->n_big_plaq = r.i[ah::DS_BIG];
        out->string_length = P.dx * (double)out->n_wind;   // L_W = dx * n_W (reading #13)
        const double V = (double)P.nx * P.ny * P.nz * P.dx * P.dx * P.dx;
        out->xi_w = out->n_wind > 0 ? std::sqrt(V / out->string_length)
                                    : std::numeric_limits<double>::infinity();
        // the paper's xi_W: Manhattan length reduced by pi/6 (reading #13)
        out->xi_w_corr = out->xi_w * std::sqrt(6.0 / 3.14159265358979323846);
    } else {
        out->n_wind = out->n_wind_xy = out->n_wind_xz = out->n_wind_yz = out->n_near_branch = out->n_big_plaq = -1;
        out->string_length = out->xi_w = out->xi_w_corr = std::numeric_limits<double>::quiet_NaN();
    }
    out->sum_pi2_L = r.f[ah::DF_SPI];
    out->sum_grad2_L = r.f[ah::DF_SGR];
    out->sum_L = r.f[ah::DF_SL];
    {   // Eq. 16 left: xi_L = sqrt(-mu V / int L), int L = sum_x L_x dx^3, V = N dx^3, mu = 2 pi sigma^2
        const double mu = 2.0 * 3.14159265358979323846 * P.sigma * P.sigma;
        const double nsites = (double)P.nx * P.ny * P.nz;
        out->xi_l = out->sum_L < 0.0 ? std::sqrt(-mu * nsites / out->sum_L) : std::numeric_limits<double>::infinity();
    }
    if (out->sum_grad2_L != 0.0) {
        const double R = out->sum_pi2_L / out->sum_grad2_L;   // Eq. 18
        out->v2_phi = 2.0 * R / (1.0 + R);                    // Eq. 17 left
    } else {
        out->v2_phi = 0.0;
    }
    out->sum_p_L = r.f[ah::DF_SPL];
    out->sum_rho_L = r.f[ah::DF_SRL];
    // Eq. 17 right with reading #17
    out->v2_omega = out->sum_rho_L != 0.0 ? 0.5 * (1.0 + 3.0 * out->sum_p_L / out->sum_rho_L) : 0.0;
    out->gauss_max = r.f[ah::DF_GMAX];
    out->gauss_l2 = std::sqrt(r.f[ah::DF_GSQ]);
    out->gauss_div_l2 = std::sqrt(r.f[ah::DF_DIVSQ]);
    out->gauss_charge_l2 = std::sqrt(r.f[ah::DF_CHSQ]);
    const double den = out->gauss_div_l2 + out->gauss_charge_l2;
    out->gauss_rel = den > 0.0 ? out->gauss_l2 / den : 0.0;
}

int check_params(const ah_params *P, const char *who)
{
    if (P->nx < 1 || P->ny < 1 || P->nz < 1)
        return fail(AH_EINVAL, "%s: extents must be >= 1 (%d,%d,%d)", who, P->nx, P->ny, P->nz);
    if (!(P->dx > 0.0) || !(P->e0 != 0.0) || !(P->alpha >= 0.0) || !std::isfinite(P->lambda0) ||
        !std::isfinite(P->sigma) || !std::isfinite(P->s) || !std::isfinite(P->p))
        return fail(AH_EINVAL, "%s: bad model parameters", who);
    if (P->p != 0.0 && P->s != 0.0 && !(P->tau_ref > 0.0))
        return fail(AH_EINVAL, "%s: tau_ref must be > 0 when p != 0 and s != 0", who);
    if (P->fp64 != AH_PRECISION_FP32 && P->fp64 != AH_PRECISION_FP64 && P->fp64 != AH_PRECISION_MIXED)
        return fail(AH_EINVAL, "%s: fp64 must be 0 (fp32), 1 (fp64) or 2 (fp32 storage, fp64 arithmetic)", who);
    return AH_OK;
}

// nz_own planes starting at global plane z_first; slab: with one ghost plane on each side
int create_ctx(ah_ctx **out, const ah_params *P, bool slab, int nz_own, int z_first, void *const dev_bufs[], int nbufs,
               size_t bytes_each, void *cuda_stream, const char *who)
{
    if (!out || !P || !dev_bufs) return fail(AH_EINVAL, "%s: null pointer", who);
    *out = nullptr;
    int rc = check_params(P, who);
    if (rc != AH_OK) return rc;
    if (slab && (nz_own < 1 || z_first < 0 || z_first + nz_own > P->nz))
        return fail(AH_EINVAL, "%s: slab planes [%d, %d) do not lie inside [0, %d)", who, z_first, z_first + nz_own, P->nz);
    if (nbufs != 2 * AH_NFIELDS) return fail(AH_EINVAL, "%s: nbufs must be 20 (got %d)", who, nbufs);
    const int nza = slab ? nz_own + 2 : P->nz;
    const size_t n = (size_t)P->nx * P->ny * nza;
    const size_t elem = is_fp64(*P) ? sizeof(double) : sizeof(float);
    if (bytes_each != n * elem)
        return fail(AH_EINVAL, "%s: bytes_each=%zu but nx*ny*planes*sizeof(elem)=%zu", who, bytes_each, n * elem);
    for (int i = 0; i < nbufs; ++i) {
        if (!dev_bufs[i]) return fail(AH_EINVAL, "%s: dev_bufs[%d] is null", who, i);
        if (((uintptr_t)dev_bufs[i]) & 15u)
            return fail(AH_EINVAL, "%s: dev_bufs[%d] is not 16-byte aligned", who, i);
        for (int j = 0; j < i; ++j)
            if (dev_bufs[i] == dev_bufs[j]) return fail(AH_EINVAL, "%s: dev_bufs[%d] == dev_bufs[%d]", who, i, j);
    }
    int ndev = 0;
    AH_CUDA(cudaGetDeviceCount(&ndev));
    if (ndev < 1) return fail(AH_ECUDA, "%s: no CUDA device", who);

    ah_ctx *c = new (std::nothrow) ah_ctx;
    if (!c) return fail(AH_ECUDA, "%s: out of host memory", who);
    std::memset(c, 0, sizeof(*c));
    c->P = *P;
    for (int i = 0; i < nbufs; ++i) c->bufs[i] = dev_bufs[i];
    c->st = (cudaStream_t)cuda_stream;
    c->nza = nza;
    c->zr = slab ? ah::ZRange{1, nza - 1} : ah::ZRange{0, nza};
    c->z_offset = slab ? z_first - 1 : 0;
    c->slab = slab;
    c->n = n;
    c->elem = elem;
    const bool can_tile = P->fp64 == AH_PRECISION_FP32 && ah::tiled_supported(P->nx, P->ny, nza);
    c->kernel = can_tile ? AH_KERNEL_TILED : AH_KERNEL_SITE;
    if (c->kernel == AH_KERNEL_TILED) {
        cudaError_t e = ah::tiled_setup();
        if (e != cudaSuccess) {
            delete c;
            return cuda_fail(e, "tiled kernel setup");
        }
    }
    rc = ensure_diag_scratch(c, 256);
    if (rc != AH_OK) {
        ah_destroy(c);
        return rc;
    }
    {
        cudaError_t e = cudaMalloc(&c->d_overflow, 2 * sizeof(int));
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d_overflow, 0, 2 * sizeof(int), c->st);
        if (e == cudaSuccess && slab) e = cudaEventCreateWithFlags(&c->ev_boundary, cudaEventDisableTiming);
        if (e == cudaSuccess && slab) e = cudaEventCreateWithFlags(&c->ev_exchange, cudaEventDisableTiming);
        if (e != cudaSuccess) {
            ah_destroy(c);
            return cuda_fail(e, "context scratch");
        }
    }
    *out = c;
    return AH_OK;
}

const int HALO_FIELDS[AH_NHALO] = {ah::PHI_RE, ah::PHI_IM, ah::TH_X, ah::TH_Y, ah::TH_Z, ah::EP_Z};

}  // namespace

extern "C" {

const char *ah_last_error(void) { return g_err; }
const char *ah_version(void) { return "ah_b200 0.2 (sm_100a)"; }

int ah_coeffs(const ah_params *P, double tau, double dt, double *a, double *q, double *delta,
              double *omega)
{
    if (!P || !a || !q || !delta || !omega) return fail(AH_EINVAL, "ah_coeffs: null pointer");
    if (P->p != 0.0 && !(tau > 0.0)) return fail(AH_EINVAL, "ah_coeffs: tau must be > 0 when p != 0");
    coeffs(*P, tau, dt, *a, *q, *delta, *omega);
    return AH_OK;
}

int ah_create(ah_ctx **out, const ah_params *P, void *const dev_bufs[], int nbufs, size_t bytes_each,
              void *cuda_stream)
{
    return create_ctx(out, P, false, P ? P->nz : 0, 0, dev_bufs, nbufs, bytes_each, cuda_stream, "ah_create");
}

int ah_create_slab(ah_ctx **out, const ah_params *global_params, int nz_own, int z_first, void *const dev_bufs[],
                   int nbufs, size_t bytes_each, void *cuda_stream)
{
    return create_ctx(out, global_params, true, nz_own, z_first, dev_bufs, nbufs, bytes_each, cuda_stream,
                      "ah_create_slab");
}

int ah_destroy(ah_ctx *c)
{
    if (!c) return AH_OK;
    if (c->d_partials) cudaFree(c->d_partials);
    if (c->d_results) cudaFree(c->d_results);
    if (c->h_results) cudaFreeHost(c->h_results);
    if (c->d_overflow) cudaFree(c->d_overflow);
    if (c->ev_boundary) cudaEventDestroy(c->ev_boundary);
    if (c->ev_exchange) cudaEventDestroy(c->ev_exchange);
    delete c;
    return AH_OK;
}

int ah_set_kernel(ah_ctx *c, int kernel)
{
    if (!c) return fail(AH_EINVAL, "ah_set_kernel: null context");
    const bool can_tile = c->P.fp64 == AH_PRECISION_FP32 && ah::tiled_supported(c->P.nx, c->P.ny, c->nza);
    if (kernel == AH_KERNEL_AUTO) kernel = can_tile ? AH_KERNEL_TILED : AH_KERNEL_SITE;
    if (kernel == AH_KERNEL_TILED) {
        if (!can_tile) return fail(AH_EINVAL, "ah_set_kernel: tiled kernel needs fp32 and nx %% 64 == 0");
        AH_CUDA(ah::tiled_setup());
    } else if (kernel != AH_KERNEL_SITE) {
        return fail(AH_EINVAL, "ah_set_kernel: unknown kernel %d", kernel);
    }
    c->kernel = kernel;
    return AH_OK;
}

int ah_get_kernel(const ah_ctx *c)
{
    if (!c) return fail(AH_EINVAL, "ah_get_kernel: null context");
    return c->P.fp64 != AH_PRECISION_FP32 ? AH_KERNEL_SITE : c->kernel;
}

int ah_tiled_launch_info(int nx, int ny, int nz, int *planes_per_cta, int *n_ctas)
{
    if (!planes_per_cta || !n_ctas) return fail(AH_EINVAL, "ah_tiled_launch_info: null pointer");
    if (!ah::tiled_supported(nx, ny, nz)) return fail(AH_EINVAL, "ah_tiled_launch_info: tiled kernel needs nx %% 64 == 0");
    *planes_per_cta = ah::tiled_chunk(nx, ny, nz);
    *n_ctas = ah::tiled_num_blocks(nx, ny, nz);
    return AH_OK;
}

int64_t ah_launch_count(const ah_ctx *c) { return c ? c->launches : 0; }

int ah_init_fields(ah_ctx *c, uint64_t seed)
{
    if (!c) return fail(AH_EINVAL, "ah_init_fields: null context");
    c->cur = 0;
    const ah_params &P = c->P;
    cudaError_t e = is_fp64(P) ? ah::launch_init<double>(cur_fields_mut<double>(c), seed, P.sigma, P.nx, P.ny, c->nza, P.nz,
                                                         c->z_offset, c->st)
                               : ah::launch_init<float>(cur_fields_mut<float>(c), seed, P.sigma, P.nx, P.ny, c->nza, P.nz,
                                                        c->z_offset, c->st);
    if (e != cudaSuccess) return cuda_fail(e, "init kernel launch");
    c->launches += 1;
    c->have_fields = true;
    return AH_OK;
}

int ah_set_fields(ah_ctx *c, const void *host)
{
    if (!c || !host) return fail(AH_EINVAL, "ah_set_fields: null pointer");
    c->cur = 0;
    const size_t bytes = c->n * c->elem;
    for (int a = 0; a < AH_NFIELDS; ++a)
        AH_CUDA(cudaMemcpyAsync(c->bufs[a], (const char *)host + bytes * a, bytes, cudaMemcpyHostToDevice, c->st));
    AH_CUDA(cudaStreamSynchronize(c->st));
    c->have_fields = true;
    return AH_OK;
}

int ah_get_fields(ah_ctx *c, void *host)
{
    if (!c || !host) return fail(AH_EINVAL, "ah_get_fields: null pointer");
    if (!c->have_fields) return fail(AH_ESTATE, "ah_get_fields: no fields were set");
    const size_t bytes = c->n * c->elem;
    for (int a = 0; a < AH_NFIELDS; ++a)
        AH_CUDA(cudaMemcpyAsync((char *)host + bytes * a, c->bufs[c->cur * AH_NFIELDS + a], bytes,
                                cudaMemcpyDeviceToHost, c->st));
    AH_CUDA(cudaStreamSynchronize(c->st));
    return AH_OK;
}

int ah_current_bufs(ah_ctx *c, void *out[AH_NFIELDS])
{
    if (!c || !out) return fail(AH_EINVAL, "ah_current_bufs: null pointer");
    for (int a = 0; a < AH_NFIELDS; ++a) out[a] = c->bufs[c->cur * AH_NFIELDS + a];
    return AH_OK;
}

int ah_step(ah_ctx *c, int n, double tau, double dt)
{
    if (!c) return fail(AH_EINVAL, "ah_step: null context");
    if (n < 0) return fail(AH_EINVAL, "ah_step: n must be >= 0 (got %d)", n);
    if (!c->have_fields) return fail(AH_ESTATE, "ah_step: no fields were set");
    if (c->slab) return fail(AH_ESTATE, "ah_step: a z-slab context steps with ah_slab_step (ghost planes need an exchange)");
    int rc = check_time(c, tau, dt);
    if (rc != AH_OK) return rc;
    for (int j = 0; j < n; ++j) {
        rc = one_step(c, c->P, tau + (double)j * dt, dt);
        if (rc != AH_OK) return rc;
    }
    return AH_OK;
}

int ah_step_cooling(ah_ctx *c, int n, double delta, double dt)
{
    if (!c) return fail(AH_EINVAL, "ah_step_cooling: null context");
    if (n < 0) return fail(AH_EINVAL, "ah_step_cooling: n must be >= 0 (got %d)", n);
    if (!c->have_fields) return fail(AH_ESTATE, "ah_step_cooling: no fields were set");
    if (c->slab) return fail(AH_ESTATE, "ah_step_cooling: not available on a z-slab context");
    if (!(dt > 0.0) || !std::isfinite(dt) || !(delta > 0.0) || !(delta < 1.0))
        return fail(AH_EINVAL, "ah_step_cooling: need dt > 0 and 0 < delta < 1 (dt=%g, delta=%g)", dt, delta);
    // constant damping = the Hubble term frozen at tau = dt/delta with p = 1, alpha = 2; s = 0 keeps q = 1
    ah_params P = c->P;   // a copy: the context's own model is never touched
    P.p = 1.0;
    P.s = 0.0;
    P.alpha = 2.0;
    int rc = AH_OK;
    for (int j = 0; j < n && rc == AH_OK; ++j) rc = one_step(c, P, dt / delta, dt);
    return rc;
}

int ah_diagnostics(ah_ctx *c, double tau, double dt, ah_diag *out)
{
    if (!c || !out) return fail(AH_EINVAL, "ah_diagnostics: null pointer");
    if (!c->have_fields) return fail(AH_ESTATE, "ah_diagnostics: no fields were set");
    if (c->slab) return fail(AH_ESTATE, "ah_diagnostics: a z-slab context reads out with ah_slab_diag_partial");
    int rc = check_diag_time(c, tau, dt);
    if (rc != AH_OK) return rc;
    rc = ensure_diag_scratch(c, 1);
    if (rc != AH_OK) return rc;
    rc = enqueue_diag(c, tau, dt, 0, nullptr, nullptr);
    if (rc != AH_OK) return rc;
    AH_CUDA(cudaMemcpyAsync(c->h_results, c->d_results, sizeof(ah::DiagPartial), cudaMemcpyDeviceToHost, c->st));
    AH_CUDA(cudaStreamSynchronize(c->st));
    finish_diag(c->P, c->h_results[0], tau, out);
    return AH_OK;
}

static int step_diag_impl(ah_ctx *c, int n, double tau, double dt, int every, ah_diag *out, int cap, int *n_written,
                          bool winding);

int ah_step_diag(ah_ctx *c, int n, double tau, double dt, int every, ah_diag *out, int cap, int *n_written)
{
    return step_diag_impl(c, n, tau, dt, every, out, cap, n_written, true);
}

int ah_step_diag_sums(ah_ctx *c, int n, double tau, double dt, int every, ah_diag *out, int cap, int *n_written)
{
    return step_diag_impl(c, n, tau, dt, every, out, cap, n_written, false);
}

static int step_diag_impl(ah_ctx *c, int n, double tau, double dt, int every, ah_diag *out, int cap, int *n_written,
                          bool winding)
{
    if (!c || !out || !n_written) return fail(AH_EINVAL, "ah_step_diag: null pointer");
    *n_written = 0;
    if (n < 0 || every < 1) return fail(AH_EINVAL, "ah_step_diag: need n >= 0 and every >= 1");
    if (!c->have_fields) return fail(AH_ESTATE, "ah_step_diag: no fields were set");
    if (c->slab) return fail(AH_ESTATE, "ah_step_diag: a z-slab context steps with ah_slab_step");
    int rc = check_time(c, tau, dt);
    for (int j = 0; j < n && rc == AH_OK; j += every) rc = check_diag_time(c, tau + (double)j * dt, dt);
    if (rc != AH_OK) return rc;
    const int records = (n + every - 1) / every;
    if (cap < records) return fail(AH_EINVAL, "ah_step_diag: cap=%d < %d records", cap, records);
    rc = ensure_diag_scratch(c, records);
    if (rc != AH_OK) return rc;
    int r = 0;
    for (int j = 0; j < n; ++j) {
        const double tj = tau + (double)j * dt;
        const bool diag = (j % every == 0);
        const bool fused = diag && c->P.fp64 == AH_PRECISION_FP32 && c->kernel == AH_KERNEL_TILED;
        if (diag && !fused) {   // site / fp64 kernels: read-outs by the standalone kernel, then the step
            rc = enqueue_diag(c, tj, dt, r, nullptr, nullptr);
            if (rc != AH_OK) return rc;
        }
        rc = one_step(c, c->P, tj, dt, fused ? r : -1, winding);
        if (rc != AH_OK) return rc;
        if (diag) ++r;
    }
    if (r > 0)
        AH_CUDA(cudaMemcpyAsync(c->h_results, c->d_results, sizeof(ah::DiagPartial) * (size_t)r,
                                cudaMemcpyDeviceToHost, c->st));
    AH_CUDA(cudaStreamSynchronize(c->st));
    for (int i = 0; i < r; ++i) finish_diag(c->P, c->h_results[i], tau + (double)(i * every) * dt, out + i, winding);
    *n_written = r;
    return AH_OK;
}

int ah_winding_field(ah_ctx *c, int8_t *host_w3, uint8_t *host_near3)
{
    if (!c || !host_w3) return fail(AH_EINVAL, "ah_winding_field: null pointer");
    if (!c->have_fields) return fail(AH_ESTATE, "ah_winding_field: no fields were set");
    int rc = ensure_diag_scratch(c, 1);
    if (rc != AH_OK) return rc;
    int8_t *d_w = nullptr;
    uint8_t *d_near = nullptr;
    AH_CUDA(cudaMalloc(&d_w, 3 * c->n));
    cudaError_t e = cudaMemsetAsync(d_w, 0, 3 * c->n, c->st);   // ghost planes of a slab stay 0
    if (e == cudaSuccess && host_near3) {
        e = cudaMalloc(&d_near, 3 * c->n);
        if (e == cudaSuccess) e = cudaMemsetAsync(d_near, 0, 3 * c->n, c->st);
    }
    if (e != cudaSuccess) {
        cudaFree(d_w);
        if (d_near) cudaFree(d_near);
        return cuda_fail(e, "winding field scratch");
    }
    // winding does not depend on tau or on the couplings
    rc = enqueue_diag(c, 1.0, 1.0, 0, d_w, d_near, /*winding_only=*/true);
    if (rc == AH_OK) e = cudaMemcpyAsync(host_w3, d_w, 3 * c->n, cudaMemcpyDeviceToHost, c->st);
    if (rc == AH_OK && e == cudaSuccess && host_near3)
        e = cudaMemcpyAsync(host_near3, d_near, 3 * c->n, cudaMemcpyDeviceToHost, c->st);
    cudaError_t e2 = cudaStreamSynchronize(c->st);
    cudaFree(d_w);
    if (d_near) cudaFree(d_near);
    if (rc != AH_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "winding field download");
    if (e2 != cudaSuccess) return cuda_fail(e2, "cudaStreamSynchronize");
    return AH_OK;
}

// ------------------------------------------------------------------------------------------------ z slabs

int ah_slab_step(ah_ctx *c, double tau, double dt, int want_diag, void *comm_stream)
{
    if (!c) return fail(AH_EINVAL, "ah_slab_step: null context");
    if (!c->slab) return fail(AH_ESTATE, "ah_slab_step: not a z-slab context");
    if (!c->have_fields) return fail(AH_ESTATE, "ah_slab_step: no fields were set");
    int rc = want_diag ? check_diag_time(c, tau, dt) : check_time(c, tau, dt);
    if (rc != AH_OK) return rc;
    int *flag = c->d_overflow + c->step_parity, *next_flag = c->d_overflow + (1 - c->step_parity);
    const ah::ZRange own = c->zr;
    const bool tiled = c->P.fp64 == AH_PRECISION_FP32 && c->kernel == AH_KERNEL_TILED;
    cudaError_t e = cudaSuccess;
    if (want_diag) {
        rc = ensure_diag_scratch(c, 1);
        if (rc != AH_OK) return rc;
        if (!tiled) {
            rc = enqueue_diag(c, tau, dt, 0, nullptr, nullptr);
            if (rc != AH_OK) return rc;
        }
    }
    const bool split = own.hi - own.lo > 2;
    if (tiled) {
        // the planes the launches below read without owning them: the ghost planes and, when the boundary planes go
        // first, their inner neighbours (ah_site_kernel.cu: th_range_check_kernel)
        const int planes[4] = {own.lo - 1, own.hi, own.lo + 1, own.hi - 2};
        e = ah::launch_th_range_check(flag, cur_fields<float>(c), c->P.nx, c->P.ny, planes, split ? 4 : 2,
                                      ah::tiled_th_limit(), c->st);
        if (e == cudaSuccess) c->launches += 1;
    }
    if (e != cudaSuccess) {
        // nothing of the step has been enqueued yet
    } else if (want_diag && tiled && split) {
        // fused read-outs with the paper's order kept: the two boundary planes go through the DIAG
        // instantiation first, each leaving its per-CTA partials behind the previous launch's, then the exchange may
        // start; the interior follows, and ONE fixed-order total covers the partials of all three launches.  A link
        // angle outside the tiled domain (flag, cumulative over the launches) makes the standalone kernel re-evaluate
        // the whole own range into the same array, which the total then reads instead.
        const int nx = c->P.nx, ny = c->P.ny, nza = c->nza;
        const ah::StepCoef<float> k = make_coef<float>(c->P, tau, dt);
        const ah::DiagCoef dk = make_diag_coef(c->P, tau, dt);
        const ah::ConstFields<float> in = cur_fields<float>(c);
        const ah::Fields<float> out = next_fields<float>(c);
        const ah::ZRange parts[3] = {{own.lo, own.lo + 1}, {own.hi - 1, own.hi}, {own.lo + 1, own.hi - 1}};
        int at = 0;
        for (int r = 0; r < 3 && e == cudaSuccess; ++r) {
            e = ah::launch_tiled_step(in, out, k, nx, ny, nza, parts[r], flag, c->st, &dk, c->d_partials + at);
            if (e != cudaSuccess) break;
            c->launches += 1;
            at += ah::tiled_num_blocks(nx, ny, parts[r].hi - parts[r].lo, true);
            if (r == 2) {
                e = ah::launch_diag_partials<float>(in, dk, nx, ny, nza, own, c->d_partials, nullptr, nullptr, flag, c->st);
                if (e == cudaSuccess)
                    e = ah::launch_diag_final(c->d_partials, at, c->d_results, c->st,
                                              ah::diag_num_blocks(nx, ny, own.hi - own.lo), flag);
                if (e != cudaSuccess) break;
                c->launches += 2;
            }
            e = ah::launch_site_redo(flag, next_flag, in, out, k, nx, ny, nza, parts[r], c->st);
            if (e == cudaSuccess) c->launches += 1;
            if (e == cudaSuccess && r == 1) e = cudaEventRecord(c->ev_boundary, c->st);
        }
    } else if (want_diag && tiled) {
        // at most two own planes: one fused launch
        e = enqueue_step(c, c->P, tau, dt, own, 0, flag, next_flag);
        if (e == cudaSuccess) e = cudaEventRecord(c->ev_boundary, c->st);
    } else if (!split) {
        e = enqueue_step(c, c->P, tau, dt, own, -1, flag, next_flag);
        if (e == cudaSuccess) e = cudaEventRecord(c->ev_boundary, c->st);
    } else {
        // the paper's order: the planes the neighbours need first, then their exchange can run
        // while the interior is updated
        e = enqueue_step(c, c->P, tau, dt, ah::ZRange{own.lo, own.lo + 1}, -1, flag, next_flag);
        if (e == cudaSuccess) e = enqueue_step(c, c->P, tau, dt, ah::ZRange{own.hi - 1, own.hi}, -1, flag, next_flag);
        if (e == cudaSuccess) e = cudaEventRecord(c->ev_boundary, c->st);
        if (e == cudaSuccess) e = enqueue_step(c, c->P, tau, dt, ah::ZRange{own.lo + 1, own.hi - 1}, -1, flag, next_flag);
    }
    if (e == cudaSuccess && comm_stream != (void *)c->st)
        e = cudaStreamWaitEvent((cudaStream_t)comm_stream, c->ev_boundary, 0);
    if (e != cudaSuccess) {
        cudaMemsetAsync(c->d_overflow, 0, 2 * sizeof(int), c->st);
        return cuda_fail(e, "slab step launch");
    }
    c->step_parity = 1 - c->step_parity;
    c->cur = 1 - c->cur;
    return AH_OK;
}

int ah_slab_halo_ptrs(ah_ctx *c, void *send_lo[AH_NHALO], void *send_hi[AH_NHALO], void *recv_lo[AH_NHALO],
                      void *recv_hi[AH_NHALO], size_t *plane_bytes)
{
    if (!c || !send_lo || !send_hi || !recv_lo || !recv_hi || !plane_bytes)
        return fail(AH_EINVAL, "ah_slab_halo_ptrs: null pointer");
    if (!c->slab) return fail(AH_ESTATE, "ah_slab_halo_ptrs: not a z-slab context");
    const size_t pb = (size_t)c->P.nx * c->P.ny * c->elem;
    for (int a = 0; a < AH_NHALO; ++a) {
        char *base = (char *)c->bufs[c->cur * AH_NFIELDS + HALO_FIELDS[a]];
        recv_lo[a] = base;                                   // ghost plane below the own planes
        send_lo[a] = base + pb;                              // first own plane  -> the lower neighbour's recv_hi
        send_hi[a] = base + pb * (size_t)(c->nza - 2);       // last own plane   -> the upper neighbour's recv_lo
        recv_hi[a] = base + pb * (size_t)(c->nza - 1);       // ghost plane above
    }
    *plane_bytes = pb;
    return AH_OK;
}

int ah_slab_exchange_done(ah_ctx *c, void *comm_stream)
{
    if (!c) return fail(AH_EINVAL, "ah_slab_exchange_done: null context");
    if (!c->slab) return fail(AH_ESTATE, "ah_slab_exchange_done: not a z-slab context");
    if (comm_stream == (void *)c->st) return AH_OK;
    AH_CUDA(cudaEventRecord(c->ev_exchange, (cudaStream_t)comm_stream));
    AH_CUDA(cudaStreamWaitEvent(c->st, c->ev_exchange, 0));
    return AH_OK;
}

int ah_slab_diagnostics(ah_ctx *c, double tau, double dt)
{
    if (!c) return fail(AH_EINVAL, "ah_slab_diagnostics: null context");
    if (!c->slab) return fail(AH_ESTATE, "ah_slab_diagnostics: not a z-slab context");
    if (!c->have_fields) return fail(AH_ESTATE, "ah_slab_diagnostics: no fields were set");
    int rc = check_diag_time(c, tau, dt);
    if (rc != AH_OK) return rc;
    rc = ensure_diag_scratch(c, 1);
    if (rc != AH_OK) return rc;
    return enqueue_diag(c, tau, dt, 0, nullptr, nullptr);
}

int ah_slab_diag_partial(ah_ctx *c, int64_t counts[AH_NDIAG_INT], double sums[AH_NDIAG_FLT])
{
    if (!c || !counts || !sums) return fail(AH_EINVAL, "ah_slab_diag_partial: null pointer");
    if (!c->slab) return fail(AH_ESTATE, "ah_slab_diag_partial: not a z-slab context");
    if (!c->d_results) return fail(AH_ESTATE, "ah_slab_diag_partial: no read-out was requested");
    AH_CUDA(cudaMemcpyAsync(c->h_results, c->d_results, sizeof(ah::DiagPartial), cudaMemcpyDeviceToHost, c->st));
    AH_CUDA(cudaStreamSynchronize(c->st));
    for (int a = 0; a < AH_NDIAG_INT; ++a) counts[a] = c->h_results[0].i[a];
    for (int a = 0; a < AH_NDIAG_FLT; ++a) sums[a] = c->h_results[0].f[a];
    return AH_OK;
}

int ah_diag_combine(int n_parts, const int64_t *counts, const double *sums, int64_t counts_out[AH_NDIAG_INT],
                    double sums_out[AH_NDIAG_FLT])
{
    if (!counts || !sums || !counts_out || !sums_out) return fail(AH_EINVAL, "ah_diag_combine: null pointer");
    if (n_parts < 1) return fail(AH_EINVAL, "ah_diag_combine: n_parts must be >= 1 (got %d)", n_parts);
    for (int a = 0; a < AH_NDIAG_INT; ++a) counts_out[a] = 0;
    for (int a = 0; a < AH_NDIAG_FLT; ++a) sums_out[a] = 0.0;
    for (int r = 0; r < n_parts; ++r) {
        for (int a = 0; a < AH_NDIAG_INT; ++a) counts_out[a] += counts[r * AH_NDIAG_INT + a];
        for (int a = 0; a < AH_NDIAG_FLT; ++a) {
            const double v = sums[r * AH_NDIAG_FLT + a];
            sums_out[a] = (a == ah::DF_GMAX) ? std::fmax(sums_out[a], v) : sums_out[a] + v;
        }
    }
    return AH_OK;
}

int ah_diag_finish(const ah_params *global_params, const int64_t counts[AH_NDIAG_INT], const double sums[AH_NDIAG_FLT],
                   double tau, ah_diag *out)
{
    if (!global_params || !counts || !sums || !out) return fail(AH_EINVAL, "ah_diag_finish: null pointer");
    ah::DiagPartial r;
    for (int a = 0; a < AH_NDIAG_INT; ++a) r.i[a] = counts[a];
    for (int a = 0; a < AH_NDIAG_FLT; ++a) r.f[a] = sums[a];
    finish_diag(*global_params, r, tau, out);
    return AH_OK;
}

// ------------------------------------------------------------------------------------------------ no allocation

// Read-outs D1-D3 for callers that may not allocate (see ah_b200.h).  Everything is checked before the first CUDA call;
// no cudaMalloc / cudaFree / cudaMallocHost / event or stream creation happens here or below (the per-block partials
// live in the fixed device array of ah_diag_kernel.cu, the totals go to the caller's dev_totals).
static_assert(sizeof(ah::DiagPartial) == AH_NOALLOC_TOTALS_BYTES && ah::DS_NINT == AH_NDIAG_INT &&
                  ah::DS_NFLT == AH_NDIAG_FLT,
              "dev_totals layout of ah_b200.h: int64 counts, then double sums");

int ah_readout_noalloc(const ah_params *P, const void *const dev_fields[AH_NFIELDS], double tau, double dt,
                       void *dev_totals, void *cuda_stream)
{
    if (!P || !dev_fields || !dev_totals) return fail(AH_EINVAL, "ah_readout_noalloc: null pointer");
    int rc = check_params(P, "ah_readout_noalloc");
    if (rc != AH_OK) return rc;
    const size_t elem = is_fp64(*P) ? sizeof(double) : sizeof(float);
    for (int a = 0; a < AH_NFIELDS; ++a) {
        if (!dev_fields[a]) return fail(AH_EINVAL, "ah_readout_noalloc: dev_fields[%d] is null", a);
        if (((uintptr_t)dev_fields[a]) & (elem - 1))
            return fail(AH_EINVAL, "ah_readout_noalloc: dev_fields[%d] is not aligned to its element size", a);
    }
    if (((uintptr_t)dev_totals) & 7u) return fail(AH_EINVAL, "ah_readout_noalloc: dev_totals is not 8-byte aligned");
    if (!(dt > 0.0) || !std::isfinite(dt) || !std::isfinite(tau))
        return fail(AH_EINVAL, "ah_readout_noalloc: dt must be positive and finite (dt=%g, tau=%g)", dt, tau);
    if (P->p != 0.0 && !(tau > 0.0))
        return fail(AH_EINVAL, "ah_readout_noalloc: tau must be > 0 in an expanding background (tau=%g, p=%g)", tau, P->p);
    {
        double a, q, d, w;
        coeffs(*P, tau, dt, a, q, d, w);
        if (w == 1.0)
            return fail(AH_EINVAL, "ah_readout_noalloc: omega = (1-s) delta = 1 at tau=%g, dt=%g: no Gauss coefficient",
                        tau, dt);
    }
    const long long need = (long long)((P->nx + 63) / 64) * ((P->ny + 3) / 4) * ((P->nz + 7) / 8);
    if (need > (long long)ah::diag_noalloc_capacity())
        return fail(AH_EINVAL,
                    "ah_readout_noalloc: a %d x %d x %d lattice needs %lld partial sums (one per 64 x 4 x 8 sites), the "
                    "library's fixed scratch array holds %d (AH_NOALLOC_MAX_PARTIALS; 512^3 is the largest cube): use "
                    "ah_diagnostics on a context for larger lattices",
                    P->nx, P->ny, P->nz, need, ah::diag_noalloc_capacity());
    const ah::DiagCoef k = make_diag_coef(*P, tau, dt);
    cudaError_t e;
    if (is_fp64(*P)) {
        ah::ConstFields<double> f;
        for (int a = 0; a < AH_NFIELDS; ++a) f.f[a] = (const double *)dev_fields[a];
        e = ah::launch_diag_noalloc<double>(f, k, P->nx, P->ny, P->nz, (ah::DiagPartial *)dev_totals,
                                            (cudaStream_t)cuda_stream);
    } else {
        ah::ConstFields<float> f;
        for (int a = 0; a < AH_NFIELDS; ++a) f.f[a] = (const float *)dev_fields[a];
        e = ah::launch_diag_noalloc<float>(f, k, P->nx, P->ny, P->nz, (ah::DiagPartial *)dev_totals,
                                           (cudaStream_t)cuda_stream);
    }
    if (e != cudaSuccess) return cuda_fail(e, "ah_readout_noalloc: scratch look-up or kernel launch");
    return AH_OK;
}

// ------------------------------------------------------------------------------------------------ test hooks

int ah_test_trig(const float *dev_x, float *dev_sin, float *dev_cos, float *dev_plaq_sin, size_t n,
                 void *cuda_stream)
{
    if (!dev_x || !dev_sin || !dev_cos || !dev_plaq_sin) return fail(AH_EINVAL, "ah_test_trig: null pointer");
    if (n == 0) return AH_OK;
    cudaError_t e = ah::launch_test_trig(dev_x, dev_sin, dev_cos, dev_plaq_sin, n, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "trig test kernel launch");
    return AH_OK;
}

int ah_test_trig_fast(const float *dev_x, float *dev_sin, float *dev_cos, float *dev_small_sin, size_t n,
                      void *cuda_stream)
{
    if (!dev_x || !dev_sin || !dev_cos || !dev_small_sin) return fail(AH_EINVAL, "ah_test_trig_fast: null pointer");
    if (n == 0) return AH_OK;
    cudaError_t e = ah::launch_test_trig_fast(dev_x, dev_sin, dev_cos, dev_small_sin, n, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "fast trig test kernel launch");
    return AH_OK;
}

}  // extern "C"
