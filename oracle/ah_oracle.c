/*
 * ah_oracle.c — ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, fp64 CPU statement of the lattice Abelian-Higgs leapfrog step
 * and its network read-outs, written from the paper's equations
 * (/root/reference/PAPER.md, arXiv:2005.14454, Sect. 2) with the readings of
 * its garbled / silent passages listed in DESIGN.md ("Readings").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, link or call this file.  It shares no
 * code, header, constant table or helper with the CUDA path under
 * paper_2005_14454_b200/csrc/ and neither includes the other.
 *
 * Pins (tests/test_oracle_*.py): Gauss law to round-off, gauge covariance,
 * plane-wave dispersion (closed form), Minkowski energy conservation with an
 * energy written independently in numpy, vortex-antivortex pair (static,
 * mu = 2 pi sigma^2), brute-force winding (including |Phi_ij| > pi, where the
 * un-wrapped plaquette angle decides the integer), closed forms of L_x and
 * <v^2>_phi on uniform states (kinetic, electric, potential, gradient and
 * magnetic terms each fixed by arithmetic) besides the naive numpy <v^2> sums,
 * splitmix known answers; <v^2>_omega (Eq. 17 right; the paper leaves its
 * weight, rho and p undefined: DESIGN.md reading #17) by the same uniform-state
 * closed forms, by p = -rho/3 on the relaxed (critical-coupling) string pair,
 * by p = rho/3 for pure gauge radiation.  Those pins fix rho and p for ANY weight.
 * Parity unpinned (stated in DESIGN.md): the normalisation a(tau_ref) = 1 and the tau grid (the paper fixes neither:
 * readings #6, #7), and the WEIGHT W_x = L_x of <v^2>_omega (reading #17): no CPU-side pin discriminates it; the only
 * check that sees it is the GPU-side regression against the paper's printed Table 1 (1024^3 rows, 3 printed sigma).
 *
 * Conventions:
 *   site x = (x,y,z), linear index x + nx*(y + ny*z), periodic in all three;
 *   stored link angle  th_i(x) = paper's lattice A_i(x) of Eq. 12,
 *   stored link field  ep_i(x) = paper's lattice E_i(x) of Eq. 10 (= d th_i/d tau);
 *   U_i(x) = exp(-i th_i(x))                                   (Eq. 12)
 *   fields phi, th live at tau_k; momenta Pi, ep at tau_k - dt/2.
 * Field block f10: 10 contiguous arrays of n = nx*ny*nz doubles in the order
 *   phi_re, phi_im, pi_re, pi_im, th_x, th_y, th_z, ep_x, ep_y, ep_z.
 *
 * The only concession to run time is "#pragma omp parallel for" on the
 * outermost z loop (each site's arithmetic is untouched by it).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t nx, ny, nz;
    double dx;
    double lambda0, e0, sigma;
    double s;        /* core-growth exponent: 0 constant comoving width, 1 physical */
    double p;        /* dln a / dln tau = m/(1-m): 0 Minkowski, 1 radiation, 2 matter (Eq. 11) */
    double tau_ref;  /* a(tau) = (tau/tau_ref)^p   (reading #6) */
    double alpha;    /* 2 = physical Hubble damping (reading #4) */
    int32_t compact; /* 1: sin(plaquette) force / 2(1-cos) energy; 0: non-compact (reading #10) */
} ahref_params;

typedef struct {
    double tau;
    int64_t n_wind, n_wind_xy, n_wind_xz, n_wind_yz, n_near_branch, n_big_plaq;
    double string_length, xi_w;
    double sum_pi2_L, sum_grad2_L, sum_L, v2_phi;
    double gauss_max, gauss_l2, gauss_rel;
    double gauss_div_l2, gauss_charge_l2;
    double xi_l;
    double sum_p_L, sum_rho_L, v2_omega; /* Eq. 17 right, reading #17 */
} ahref_diag;

#define AHREF_PI 3.14159265358979323846264338327950288

int ahref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------- indexing */

static size_t site(const ahref_params *P, const int c[3])
{
    return (size_t)c[0] + (size_t)P->nx * ((size_t)c[1] + (size_t)P->ny * (size_t)c[2]);
}

static int extent(const ahref_params *P, int dir)
{
    return dir == 0 ? P->nx : (dir == 1 ? P->ny : P->nz);
}

/* coordinates of x + sgn * k_dir with periodic wrap */
static void shifted(const ahref_params *P, const int c[3], int dir, int sgn, int out[3])
{
    int n = extent(P, dir);
    out[0] = c[0];
    out[1] = c[1];
    out[2] = c[2];
    out[dir] = (c[dir] + sgn + n) % n;
}

static size_t nb(const ahref_params *P, const int c[3], int dir, int sgn)
{
    int t[3];
    shifted(P, c, dir, sgn, t);
    return site(P, t);
}

/* ------------------------------------------------------------ coefficients */

/* a, q = a^{2s}, delta, omega at conformal time tau (Eq. 11 :80;
 * readings #4, #5, #6): a = (tau/tau_ref)^p, delta = (alpha/2) p dt / tau,
 * omega = delta (1 - s). */
void ahref_coeffs(const ahref_params *P, double tau, double dt,
                  double *a, double *q, double *delta, double *omega)
{
    double aa = (P->p == 0.0) ? 1.0 : pow(tau / P->tau_ref, P->p);
    double qq = (P->s == 0.0) ? 1.0 : pow(aa, 2.0 * P->s);
    double d = 0.5 * P->alpha * P->p * dt / tau;
    if (P->p == 0.0)
        d = 0.0;
    *a = aa;
    *q = qq;
    *delta = d;
    *omega = d * (1.0 - P->s);
}

/* ---------------------------------------------------------- lattice pieces */

/* Phi_ij(x) = th_i(x) + th_j(x+i) - th_i(x+j) - th_j(x)   (Eqs. 14-15, reading #9) */
static double plaq(const ahref_params *P, const double *const th[3], const int c[3], int i, int j)
{
    size_t x0 = site(P, c), xi = nb(P, c, i, +1), xj = nb(P, c, j, +1);
    return th[i][x0] + th[j][xi] - th[i][xj] - th[j][x0];
}

/* derivative of the plaquette energy w.r.t. the angle: sin Phi (compact) or Phi */
static double plaq_force(const ahref_params *P, double Phi)
{
    return P->compact ? sin(Phi) : Phi;
}

/* plaquette energy density numerator: 2(1-cos Phi) (compact) or Phi^2 */
static double plaq_energy(const ahref_params *P, double Phi)
{
    return P->compact ? 2.0 * (1.0 - cos(Phi)) : Phi * Phi;
}

/* U_i(x) phi(x+i) as (re, im); U = cos th - i sin th  (Eq. 12) */
static void hop_fwd(const ahref_params *P, const double *pr, const double *pim,
                    const double *const th[3], const int c[3], int i, double out[2])
{
    size_t x0 = site(P, c), xi = nb(P, c, i, +1);
    double cu = cos(th[i][x0]), su = -sin(th[i][x0]); /* U = cu + i su */
    out[0] = cu * pr[xi] - su * pim[xi];
    out[1] = cu * pim[xi] + su * pr[xi];
}

/* conj(U_i(x-i)) phi(x-i) */
static void hop_bwd(const ahref_params *P, const double *pr, const double *pim,
                    const double *const th[3], const int c[3], int i, double out[2])
{
    size_t xm = nb(P, c, i, -1);
    double cu = cos(th[i][xm]), su = sin(th[i][xm]); /* conj(U) = cu + i su, su = +sin th */
    out[0] = cu * pr[xm] - su * pim[xm];
    out[1] = cu * pim[xm] + su * pr[xm];
}

/* ------------------------------------------------------------------- init */

/* Counter-based uniform u in [0,1): splitmix64 finaliser of
 * seed + 0x9E3779B97F4A7C15*(idx+1); top 24 bits / 2^24. */
double ahref_uniform(uint64_t seed, uint64_t idx)
{
    uint64_t z = seed + 0x9E3779B97F4A7C15ULL * (idx + 1ULL);
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return (double)(z >> 40) / 16777216.0;
}

/* I0: random phase for phi with |phi| = sigma, all else zero. */
int ahref_init_fields(const ahref_params *P, uint64_t seed, double *f10)
{
    size_t n = (size_t)P->nx * P->ny * P->nz;
    memset(f10, 0, 10 * n * sizeof(double));
    for (size_t k = 0; k < n; ++k) {
        double vartheta = 2.0 * AHREF_PI * ahref_uniform(seed, (uint64_t)k);
        f10[0 * n + k] = P->sigma * cos(vartheta);
        f10[1 * n + k] = P->sigma * sin(vartheta);
    }
    return 0;
}

/* ------------------------------------------------------------------- step */

/* One leapfrog step at time level tau (Eqs. 7-10).
 * Loop 1 updates Pi and ep everywhere from the OLD phi, th (each only reads its
 * own Pi / ep, so in place); loop 2 then updates phi and th — the paper's order
 * ("At such a point, we can simply update phi and A"). */
static void one_step(const ahref_params *P, double *f10, double tau, double dt)
{
    const int nx = P->nx, ny = P->ny, nz = P->nz;
    const size_t n = (size_t)nx * ny * nz;
    double *pr = f10, *pim = f10 + n, *pir = f10 + 2 * n, *pii = f10 + 3 * n;
    double *thm[3] = {f10 + 4 * n, f10 + 5 * n, f10 + 6 * n};
    const double *const th[3] = {thm[0], thm[1], thm[2]};
    double *ep[3] = {f10 + 7 * n, f10 + 8 * n, f10 + 9 * n};
    double a, q, delta, omega;
    ahref_coeffs(P, tau, dt, &a, &q, &delta, &omega);
    const double idx2 = 1.0 / (P->dx * P->dx);
    const double sig2 = P->sigma * P->sigma;

#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const int c[3] = {x, y, z};
                const size_t x0 = site(P, c);
                /* Eq. 13: covariant Laplacian */
                double lap_re = 0.0, lap_im = 0.0;
                double fwd[3][2];
                for (int i = 0; i < 3; ++i) {
                    double b[2];
                    hop_fwd(P, pr, pim, th, c, i, fwd[i]);
                    hop_bwd(P, pr, pim, th, c, i, b);
                    lap_re += fwd[i][0] - 2.0 * pr[x0] + b[0];
                    lap_im += fwd[i][1] - 2.0 * pim[x0] + b[1];
                }
                lap_re *= idx2;
                lap_im *= idx2;
                /* Eq. 7 */
                const double mod2 = pr[x0] * pr[x0] + pim[x0] * pim[x0];
                const double pot = 0.5 * P->lambda0 * q * (mod2 - sig2);
                const double f_re = lap_re - pot * pr[x0];
                const double f_im = lap_im - pot * pim[x0];
                pir[x0] = ((1.0 - delta) * pir[x0] + dt * f_re) / (1.0 + delta);
                pii[x0] = ((1.0 - delta) * pii[x0] + dt * f_im) / (1.0 + delta);
                /* Eq. 8 */
                for (int i = 0; i < 3; ++i) {
                    double curl = 0.0;
                    for (int j = 0; j < 3; ++j) {
                        if (j == i)
                            continue;
                        int cm[3];
                        shifted(P, c, j, -1, cm);
                        curl += plaq_force(P, plaq(P, th, c, i, j)) -
                                plaq_force(P, plaq(P, th, cm, i, j));
                    }
                    /* Im[conj(phi(x)) U_i(x) phi(x+i)] */
                    const double cur = pr[x0] * fwd[i][1] - pim[x0] * fwd[i][0];
                    const double force = -idx2 * curl + 2.0 * P->e0 * P->e0 * q * cur;
                    ep[i][x0] = ((1.0 - omega) * ep[i][x0] + dt * force) / (1.0 + omega);
                }
            }

    /* Eqs. 9-10 */
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const int c[3] = {x, y, z};
                const size_t x0 = site(P, c);
                pr[x0] += dt * pir[x0];
                pim[x0] += dt * pii[x0];
                for (int i = 0; i < 3; ++i)
                    thm[i][x0] += dt * ep[i][x0];
            }
}

/* n steps from tau; step j uses tau_j = tau + j*dt (a product, not an accumulation). */
int ahref_step(const ahref_params *P, double *f10, int n, double tau, double dt)
{
    if (!P || !f10 || n < 0 || P->nx < 1 || P->ny < 1 || P->nz < 1 || !(P->dx > 0.0))
        return -1;
    if (P->p != 0.0 && !(tau > 0.0))
        return -1;
    for (int j = 0; j < n; ++j)
        one_step(P, f10, tau + (double)j * dt, dt);
    return 0;
}

/* ------------------------------------------------------------ diagnostics */

static double link_phase(const ahref_params *P, const double *pr, const double *pim,
                         const double *const th[3], const int c[3], int i)
{
    /* d_i(x) = Arg( conj(phi(x)) U_i(x) phi(x+i) ) in (-pi, pi]; atan2(0,0) = 0 */
    double h[2];
    size_t x0 = site(P, c);
    hop_fwd(P, pr, pim, th, c, i, h);
    double re = pr[x0] * h[0] + pim[x0] * h[1];
    double im = pr[x0] * h[1] - pim[x0] * h[0];
    if (re == 0.0 && im == 0.0)
        return 0.0;
    return atan2(im, re);
}

static const int PAIRS[3][2] = {{0, 1}, {0, 2}, {1, 2}}; /* xy, xz, yz */

/* Winding of plaquette (i,j) at x (Eq. 16 right; Kajantie et al. form,
 * reading #13).  *near is set when any of the four link phases lies within 1e-5 of +-pi,
 * *big when |Phi_ij| > pi - 1e-5. */
static int winding_at(const ahref_params *P, const double *pr, const double *pim,
                      const double *const th[3], const int c[3], int i, int j,
                      int *near, int *big)
{
    int ci[3], cj[3];
    shifted(P, c, i, +1, ci);
    shifted(P, c, j, +1, cj);
    const double d1 = link_phase(P, pr, pim, th, c, i);  /* d_i(x)   */
    const double d2 = link_phase(P, pr, pim, th, ci, j); /* d_j(x+i) */
    const double d3 = link_phase(P, pr, pim, th, cj, i); /* d_i(x+j) */
    const double d4 = link_phase(P, pr, pim, th, c, j);  /* d_j(x)   */
    const double Phi = plaq(P, th, c, i, j);
    const double lim = AHREF_PI - 1e-5;
    *near = (fabs(d1) >= lim) || (fabs(d2) >= lim) || (fabs(d3) >= lim) || (fabs(d4) >= lim);
    *big = fabs(Phi) > lim;
    return (int)rint((d1 + d2 - d3 - d4 + Phi) / (2.0 * AHREF_PI));
}

/* Per-plaquette winding field: w3 = 3 arrays (xy, xz, yz) of n int8; near3 same shape or NULL. */
int ahref_winding(const ahref_params *P, const double *f10, int8_t *w3, uint8_t *near3)
{
    const size_t n = (size_t)P->nx * P->ny * P->nz;
    const double *pr = f10, *pim = f10 + n;
    const double *const th[3] = {f10 + 4 * n, f10 + 5 * n, f10 + 6 * n};
#pragma omp parallel for schedule(static)
    for (int z = 0; z < P->nz; ++z)
        for (int y = 0; y < P->ny; ++y)
            for (int x = 0; x < P->nx; ++x) {
                const int c[3] = {x, y, z};
                const size_t x0 = site(P, c);
                for (int k = 0; k < 3; ++k) {
                    int near, big;
                    int w = winding_at(P, pr, pim, th, c, PAIRS[k][0], PAIRS[k][1], &near, &big);
                    w3[(size_t)k * n + x0] = (int8_t)w;
                    if (near3)
                        near3[(size_t)k * n + x0] = (uint8_t)near;
                }
            }
    return 0;
}

/* Lagrangian density of site x (reading #15):
 *  L = |Pi|^2 - sum_i |U_i phi(x+i) - phi|^2/dx^2 - (lambda0 q/4)(|phi|^2-sigma^2)^2
 *      + (1/(2 e0^2 q)) [ sum_i ep_i^2/dx^2 - sum_{i<j} 2(1-cos Phi_ij)/dx^4 ]
 * also returns |Pi|^2, the gradient sum, and the energy density and isotropic pressure of the same five pieces
 * (reading #17, for the equation-of-state estimator of Eq. 17 right):
 *  rho = |Pi|^2 + grad2 + V + (E2 + B2),   p = |Pi|^2 - grad2/3 - V + (E2 + B2)/3,
 * with E2 = sum_i ep_i^2/(2 e0^2 q dx^2), B2 = sum_{i<j} 2(1-cos Phi_ij)/(2 e0^2 q dx^4), V the potential term. */
static double lagrangian_at(const ahref_params *P, const double *f10, const int c[3], double q,
                            double *pi2_out, double *grad2_out, double *rho_out, double *p_out)
{
    const size_t n = (size_t)P->nx * P->ny * P->nz;
    const double *pr = f10, *pim = f10 + n, *pir = f10 + 2 * n, *pii = f10 + 3 * n;
    const double *const th[3] = {f10 + 4 * n, f10 + 5 * n, f10 + 6 * n};
    const double *const ep[3] = {f10 + 7 * n, f10 + 8 * n, f10 + 9 * n};
    const size_t x0 = site(P, c);
    const double idx2 = 1.0 / (P->dx * P->dx);
    const double pi2 = pir[x0] * pir[x0] + pii[x0] * pii[x0];
    double grad2 = 0.0, e2 = 0.0, b2 = 0.0;
    for (int i = 0; i < 3; ++i) {
        double h[2];
        hop_fwd(P, pr, pim, th, c, i, h);
        const double dr = h[0] - pr[x0], di = h[1] - pim[x0];
        grad2 += (dr * dr + di * di) * idx2;
        e2 += ep[i][x0] * ep[i][x0] * idx2;
    }
    for (int k = 0; k < 3; ++k)
        b2 += plaq_energy(P, plaq(P, th, c, PAIRS[k][0], PAIRS[k][1])) * idx2 * idx2;
    const double mod2 = pr[x0] * pr[x0] + pim[x0] * pim[x0];
    const double sig2 = P->sigma * P->sigma;
    const double pot = 0.25 * P->lambda0 * q * (mod2 - sig2) * (mod2 - sig2);
    *pi2_out = pi2;
    *grad2_out = grad2;
    {
        const double E2 = e2 / (2.0 * P->e0 * P->e0 * q), B2 = b2 / (2.0 * P->e0 * P->e0 * q);
        *rho_out = pi2 + grad2 + pot + (E2 + B2);
        *p_out = pi2 - grad2 / 3.0 - pot + (E2 + B2) / 3.0;
    }
    return pi2 - grad2 - pot + (e2 - b2) / (2.0 * P->e0 * P->e0 * q);
}

/* Diagnostics of the snapshot (phi,th at tau; Pi,ep at tau - dt/2). */
int ahref_diagnostics(const ahref_params *P, const double *f10, double tau, double dt, ahref_diag *out)
{
    if (!P || !f10 || !out)
        return -1;
    const int nx = P->nx, ny = P->ny, nz = P->nz;
    const size_t n = (size_t)nx * ny * nz;
    const double *pr = f10, *pim = f10 + n, *pir = f10 + 2 * n, *pii = f10 + 3 * n;
    const double *const th[3] = {f10 + 4 * n, f10 + 5 * n, f10 + 6 * n};
    const double *const ep[3] = {f10 + 7 * n, f10 + 8 * n, f10 + 9 * n};
    double a, q, delta, omega;
    ahref_coeffs(P, tau, dt, &a, &q, &delta, &omega);
    const double idx2 = 1.0 / (P->dx * P->dx);
    /* Gauss coefficient at the momenta's half step (reading #18) */
    const double kappa = q * (1.0 - delta) / (1.0 - omega);

    int64_t nw[3] = {0, 0, 0}, n_near = 0, n_big = 0;
    double s_pi = 0.0, s_gr = 0.0, s_L = 0.0, s_pL = 0.0, s_rL = 0.0;
    double g_max = 0.0, g_sq = 0.0, div_sq = 0.0, ch_sq = 0.0;

    /* serial accumulation in site order: the definition, nothing else */
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const int c[3] = {x, y, z};
                const size_t x0 = site(P, c);
                /* D1 winding */
                for (int k = 0; k < 3; ++k) {
                    int near, big;
                    int w = winding_at(P, pr, pim, th, c, PAIRS[k][0], PAIRS[k][1], &near, &big);
                    nw[k] += (w < 0) ? -w : w;
                    n_near += near;
                    n_big += big;
                }
                /* D2 Lagrangian-weighted sums (Eqs. 17-18) */
                double pi2, grad2, rho, prs;
                const double L = lagrangian_at(P, f10, c, q, &pi2, &grad2, &rho, &prs);
                s_pi += pi2 * L;
                s_gr += grad2 * L;
                s_L += L;
                /* Eq. 17 right with the weight W_x = L_x (reading #17) */
                s_pL += prs * L;
                s_rL += rho * L;
                /* D3 Gauss residual (Eq. 5) */
                double div = 0.0;
                for (int i = 0; i < 3; ++i)
                    div += ep[i][x0] - ep[i][nb(P, c, i, -1)];
                div *= idx2;
                const double charge = 2.0 * P->e0 * P->e0 * kappa * (pr[x0] * pii[x0] - pim[x0] * pir[x0]);
                const double G = div - charge;
                if (fabs(G) > g_max)
                    g_max = fabs(G);
                g_sq += G * G;
                div_sq += div * div;
                ch_sq += charge * charge;
            }

    out->tau = tau;
    out->n_wind_xy = nw[0];
    out->n_wind_xz = nw[1];
    out->n_wind_yz = nw[2];
    out->n_wind = nw[0] + nw[1] + nw[2];
    out->n_near_branch = n_near;
    out->n_big_plaq = n_big;
    out->string_length = P->dx * (double)out->n_wind;
    {
        const double V = (double)nx * ny * nz * P->dx * P->dx * P->dx;
        out->xi_w = out->n_wind > 0 ? sqrt(V / out->string_length) : INFINITY;
    }
    out->sum_pi2_L = s_pi;
    out->sum_grad2_L = s_gr;
    out->sum_L = s_L;
    /* Eq. 16 left: xi_L = sqrt(-mu V / integral of L), mu = 2 pi sigma^2 (beta = 1);
     * V = N dx^3 and the integral is sum_x L_x dx^3, so the dx^3 cancel. */
    out->xi_l = (s_L < 0.0) ? sqrt(-(2.0 * AHREF_PI * P->sigma * P->sigma) * ((double)nx * ny * nz) / s_L) : INFINITY;
    {
        const double R = s_pi / s_gr;
        out->v2_phi = (s_gr != 0.0) ? 2.0 * R / (1.0 + R) : 0.0;
    }
    out->sum_p_L = s_pL;
    out->sum_rho_L = s_rL;
    out->v2_omega = (s_rL != 0.0) ? 0.5 * (1.0 + 3.0 * s_pL / s_rL) : 0.0;
    out->gauss_max = g_max;
    out->gauss_l2 = sqrt(g_sq);
    out->gauss_div_l2 = sqrt(div_sq);
    out->gauss_charge_l2 = sqrt(ch_sq);
    {
        const double den = out->gauss_div_l2 + out->gauss_charge_l2;
        out->gauss_rel = den > 0.0 ? out->gauss_l2 / den : 0.0;
    }
    return 0;
}
