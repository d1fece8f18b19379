/*
 * sph_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, FP64 CPU statement of what the SPH interaction sweep of
 * arxiv/paper_2511_11425 ("SPH in pkdgrav3 ... I. Hydrodynamics") computes:
 * neighbour sets within the kernel support 2h, the density / smoothing-length
 * solve, the hydro force pass with Monaghan artificial viscosity and the
 * ideal-gas EOS, and the per-particle / global time step.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code
 * with the CUDA path (paper_2511_11425_b200/csrc) and neither includes the
 * other.  Every function cites the passage of /root/reference/PAPER.md it
 * follows; where the paper is silent the reading Rn of DESIGN.md section 3 is
 * named.
 *
 * Two families of entry points:
 *   orc_*_brute : the definition. For each requested target i an O(N) loop
 *                 over ALL particles j.  Used for parity (all targets at small
 *                 N, a seeded sample of targets at the full sizes).
 *   orc_*_cells : the same sums with the j-loop restricted by a uniform cell
 *                 list (27-cell stencil, cell side >= the largest support in
 *                 use) and OpenMP over targets.  Pinned against the brute
 *                 force (tests/test_oracle_pins.py::test_cells_equals_brute);
 *                 it is what bench.py times as the CPU baseline.
 *
 * Parity pins: kernel normalisation and derivatives, root residual and
 * monotonicity, infinite-lattice density, momentum / energy / angular-momentum
 * conservation, Galilean / translation / permutation invariance, two-particle
 * and homologous-flow closed forms, static-gas dt, the entropy-conserving
 * variant (viscous heating alone conserves energy; P / rho^gamma invariant),
 * the block-step bookkeeping (ruler sequence, exact leap-frog under constant
 * acceleration for any rung history) --
 * see tests/test_oracle_pins.py.  No function here is "parity unpinned".
 *
 * All arithmetic is double precision.  Inputs arrive as double arrays holding
 * the exact values of the caller's FP32 inputs.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288

typedef struct {
    double lo[3];       /* lower corner of the box                          */
    double len[3];      /* side lengths                                     */
    int32_t periodic[3];/* 1: periodic in that dimension     */
} orc_box;

typedef struct {
    int32_t kernel;     /* 0 cubic spline, 1 Wendland C2, 2 C4, 3 C6 */
    double n_ngb;       /* kernel mass in units of m_i (Eq. 6, reading R4)  */
    double gamma;       /* ideal gas                         */
    double av_alpha, av_beta, av_eps; /* Eqs. 15-16; eps reading R8         */
    double eta_cfl, eta_acc;          /* Eq. 26 / PAPER.md:263              */
    int32_t entropy;    /* 1: Eq. (14) is discarded, du/dt is the
                           viscous heating of Eq. (18) alone; reading R31     */
} orc_params;

/* ------------------------------------------------------------------------- *
 * Kernel functions, PAPER.md:105 (names only; reading R3: Dehnen & Aly 2012
 * forms, rescaled to support radius 2h, reading R2).  W(r,h) = w(q)/h^3,
 * q = r/h, w(q) = 0 for q >= 2.  x = q/2 below.
 * ------------------------------------------------------------------------- */
double orc_w(int kernel, double q)
{
    if (q >= 2.0 || q < 0.0) return 0.0;
    double x = 0.5 * q, y = 1.0 - x;
    switch (kernel) {
    case 0: /* cubic spline (Monaghan 1992), support 2h */
        if (q < 1.0) return (1.0 / ORC_PI) * (1.0 - 1.5 * q * q + 0.75 * q * q * q);
        return (1.0 / ORC_PI) * 0.25 * (2.0 - q) * (2.0 - q) * (2.0 - q);
    case 1: /* Wendland C2 */
        return (21.0 / (16.0 * ORC_PI)) * y * y * y * y * (1.0 + 4.0 * x);
    case 2: /* Wendland C4 */
        return (495.0 / (256.0 * ORC_PI)) * pow(y, 6) * (1.0 + 6.0 * x + (35.0 / 3.0) * x * x);
    case 3: /* Wendland C6 */
        return (1365.0 / (512.0 * ORC_PI)) * pow(y, 8) *
               (1.0 + 8.0 * x + 25.0 * x * x + 32.0 * x * x * x);
    }
    return NAN;
}

/* dw/dq, same conventions. */
double orc_dw(int kernel, double q)
{
    if (q >= 2.0 || q < 0.0) return 0.0;
    double x = 0.5 * q, y = 1.0 - x;
    switch (kernel) {
    case 0:
        if (q < 1.0) return (1.0 / ORC_PI) * (-3.0 * q + 2.25 * q * q);
        return -(1.0 / ORC_PI) * 0.75 * (2.0 - q) * (2.0 - q);
    case 1: /* d/dx[(1-x)^4(1+4x)] = -20 x (1-x)^3 ; dx/dq = 1/2 */
        return (21.0 / (16.0 * ORC_PI)) * 0.5 * (-20.0 * x * y * y * y);
    case 2: /* d/dx[(1-x)^6(1+6x+35x^2/3)] = -(56/3) x (1-x)^5 (1+5x) */
        return (495.0 / (256.0 * ORC_PI)) * 0.5 * (-(56.0 / 3.0) * x * pow(y, 5) * (1.0 + 5.0 * x));
    case 3: /* d/dx[(1-x)^8(1+8x+25x^2+32x^3)] = -22 x (1-x)^7 (1+7x+16x^2) */
        return (1365.0 / (512.0 * ORC_PI)) * 0.5 *
               (-22.0 * x * pow(y, 7) * (1.0 + 7.0 * x + 16.0 * x * x));
    }
    return NAN;
}

/* O1: displacement component with the minimum-image convention in periodic
 * dimensions (periodic replicas; no replica of a particle
 * lies in its own kernel, so the nearest image is the only one that counts). */
static inline double orc_disp(double xi, double xj, double L, int periodic)
{
    double d = xi - xj;
    if (periodic) d -= L * nearbyint(d / L);
    return d;
}

static inline double orc_r2(const double *x, const double *y, const double *z, int64_t i,
                            int64_t j, const orc_box *b, double d[3])
{
    d[0] = orc_disp(x[i], x[j], b->len[0], b->periodic[0]);
    d[1] = orc_disp(y[i], y[j], b->len[1], b->periodic[1]);
    d[2] = orc_disp(z[i], z[j], b->len[2], b->periodic[2]);
    return d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
}

/* Squared distance only (exported for tests). */
double orc_dist2(const double *x, const double *y, const double *z, int64_t i, int64_t j,
                 const orc_box *b)
{
    double d[3];
    return orc_r2(x, y, z, i, j, b, d);
}

/* ------------------------------------------------------------------------- *
 * Density pass, PAPER.md:137-154 (Section 2.3.3).
 *
 *   Eq. (5)  rho_i = sum_j m_j W_ij(h_i)             (gather, self included, R1/R6)
 *   Eq. (6)  (4/3) pi R_kernel(h_i)^3 rho_i = M_tot^i, R_kernel = 2h (R2),
 *            M_tot^i = N_ngb m_i (R4)
 *   Eq. (7)  Omega_i = 1 + h_i/(3 rho_i) sum_j m_j dW_ij(h_i)/dh_i
 *
 * With S(h) = sum_j m_j w(r_ij/h):  rho = S/h^3 and Eq. (6) reads
 *   G_i(h) = (32 pi/3) S(h) - N_ngb m_i = 0.
 * w is non-increasing in q, so G_i is non-decreasing in h: the root is unique
 * and the paper's Newton-Raphson iteration is only a fast way
 * to reach it.  The oracle brackets the root and bisects (O3).
 * dW/dh = -(3 w + q w')/h^4  ==>  Omega = 1 - D/(3S), D = sum_j m_j (3w + q w').
 * ------------------------------------------------------------------------- */

/* S and D over an explicit list of (r^2, m) pairs. */
static void orc_sums(int kernel, int64_t cnt, const double *r2, const double *mm, double h,
                     double *S, double *D, int64_t *nn)
{
    double s = 0.0, dd = 0.0;
    int64_t c = 0;
    for (int64_t k = 0; k < cnt; k++) {
        double q = sqrt(r2[k]) / h;
        if (r2[k] < 4.0 * h * h) c++;         /* neighbour: r^2 < (2h)^2 (R7) */
        if (q >= 2.0) continue;
        double w = orc_w(kernel, q), dw = orc_dw(kernel, q);
        s += mm[k] * w;
        dd += mm[k] * (3.0 * w + q * dw);
    }
    *S = s; *D = dd; *nn = c;
}

/* Solve particle i given the squared distances to a list of candidate particles that
 * contains every particle within 2*hcap of i.  Returns 0, or -1 if the
 * bracket would have to exceed hcap (then the candidate list is not enough). */
static int orc_solve_h(const orc_params *p, int64_t cnt, const double *r, const double *mm,
                       double mi, double hint, double hcap, double *h_out, double *rho,
                       double *omega, int32_t *nngb)
{
    const double c43 = 32.0 * ORC_PI / 3.0;
    double S, D; int64_t nn;
    double lo = hint, hi = hint;
    for (;;) {                       /* lower end: G(lo) < 0 */
        orc_sums(p->kernel, cnt, r, mm, lo, &S, &D, &nn);
        if (c43 * S - p->n_ngb * mi < 0.0) break;
        hi = lo; lo *= 0.5;
        if (lo < 1e-300) return -2;
    }
    for (;;) {                       /* upper end: G(hi) >= 0 */
        orc_sums(p->kernel, cnt, r, mm, hi, &S, &D, &nn);
        if (c43 * S - p->n_ngb * mi >= 0.0) break;
        lo = hi; hi *= 2.0;
        if (hi > hcap) { hi = hcap;
            orc_sums(p->kernel, cnt, r, mm, hi, &S, &D, &nn);
            if (c43 * S - p->n_ngb * mi >= 0.0) break;
            return -1; }
    }
    for (int it = 0; it < 200 && (hi - lo) > 1e-15 * hi; it++) {   /* bisection */
        double mid = 0.5 * (lo + hi);
        orc_sums(p->kernel, cnt, r, mm, mid, &S, &D, &nn);
        if (c43 * S - p->n_ngb * mi < 0.0) lo = mid; else hi = mid;
    }
    double h = 0.5 * (lo + hi);
    orc_sums(p->kernel, cnt, r, mm, h, &S, &D, &nn);
    *h_out = h;
    *rho = S / (h * h * h);          /* Eq. (5) */
    *omega = 1.0 - D / (3.0 * S);    /* Eq. (7) */
    *nngb = (int32_t)nn;
    return 0;
}

/* The largest h for which the minimum image is the only image inside the
 * kernel: 2h < L/2 in every periodic dimension. */
static double orc_hcap(const orc_box *b)
{
    double cap = 1e300;
    for (int d = 0; d < 3; d++)
        if (b->periodic[d] && 0.25 * b->len[d] < cap) cap = 0.25 * b->len[d];
    return cap;
}

/* Brute force: for each target an O(N) loop over all particles.
 * targets == NULL means all particles 0..nt-1.  Outputs are indexed by the
 * position in the target list.  Returns 0 or a negative error. */
int orc_density_brute(int64_t n, const double *x, const double *y, const double *z,
                      const double *m, const double *h_hint, const orc_box *box,
                      const orc_params *p, int64_t nt, const int64_t *targets, double *h,
                      double *rho, double *omega, int32_t *nngb)
{
    int err = 0;
    double hcap = orc_hcap(box);
#pragma omp parallel
    {
        double *r = (double *)malloc(sizeof(double) * (size_t)n);
#pragma omp for schedule(dynamic, 8)
        for (int64_t t = 0; t < nt; t++) {
            int64_t i = targets ? targets[t] : t;
            double d[3];
            for (int64_t j = 0; j < n; j++) r[j] = orc_r2(x, y, z, i, j, box, d);
            int rc = orc_solve_h(p, n, r, m, m[i], h_hint[i], hcap, &h[t], &rho[t], &omega[t],
                                 &nngb[t]);
            if (rc) {
#pragma omp critical
                err = rc;
            }
        }
        free(r);
    }
    return err;
}

/* Density sums at a PRESCRIBED h (no solve): S/h^3, Omega and the neighbour
 * count n_i = #{j : r_ij^2 < 4 h_i^2} (self included).  Used to compare the
 * device's rho/Omega/n at the device's own converged h (reading R7). */
int orc_density_at_h_brute(int64_t n, const double *x, const double *y, const double *z,
                           const double *m, const double *h_in, const orc_box *box,
                           const orc_params *p, int64_t nt, const int64_t *targets,
                           double *rho, double *omega, int32_t *nngb, double *resid)
{
    const double c43 = 32.0 * ORC_PI / 3.0;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t t = 0; t < nt; t++) {
        int64_t i = targets ? targets[t] : t;
        double hi = h_in[i], S = 0.0, D = 0.0, d[3];
        int32_t c = 0;
        for (int64_t j = 0; j < n; j++) {
            double r2 = orc_r2(x, y, z, i, j, box, d);
            if (r2 < 4.0 * hi * hi) {
                c++;
                double q = sqrt(r2) / hi;
                double w = orc_w(p->kernel, q), dw = orc_dw(p->kernel, q);
                S += m[j] * w;
                D += m[j] * (3.0 * w + q * dw);
            }
        }
        rho[t] = S / (hi * hi * hi);
        omega[t] = 1.0 - D / (3.0 * S);
        nngb[t] = c;
        if (resid) resid[t] = (c43 * S - p->n_ngb * m[i]) / (p->n_ngb * m[i]);
    }
    return 0;
}

/* Neighbour lists at a prescribed h.
 * mode 0: gather  j in N_i  <=>  r_ij^2 < 4 h_i^2            (self included)
 * mode 1: gather-or-scatter, j != i, 0 < r_ij^2 < 4 max(h_i,h_j)^2 (R14, R15)
 * Two calls: indices == NULL fills offsets[0..nt]; then with indices. */
int orc_neighbors_brute(int64_t n, const double *x, const double *y, const double *z,
                        const double *h, const orc_box *box, int mode, int64_t nt,
                        const int64_t *targets, int64_t *offsets, int64_t *indices)
{
    if (!indices) {
        offsets[0] = 0;
#pragma omp parallel for schedule(dynamic, 8)
        for (int64_t t = 0; t < nt; t++) {
            int64_t i = targets ? targets[t] : t, c = 0;
            double d[3];
            for (int64_t j = 0; j < n; j++) {
                double r2 = orc_r2(x, y, z, i, j, box, d);
                double hh = (mode == 1 && h[j] > h[i]) ? h[j] : h[i];
                if (mode == 0 ? (r2 < 4.0 * hh * hh) : (j != i && r2 > 0.0 && r2 < 4.0 * hh * hh)) c++;
            }
            offsets[t + 1] = c;
        }
        for (int64_t t = 0; t < nt; t++) offsets[t + 1] += offsets[t];
        return 0;
    }
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t t = 0; t < nt; t++) {
        int64_t i = targets ? targets[t] : t, c = offsets[t];
        double d[3];
        for (int64_t j = 0; j < n; j++) {
            double r2 = orc_r2(x, y, z, i, j, box, d);
            double hh = (mode == 1 && h[j] > h[i]) ? h[j] : h[i];
            if (mode == 0 ? (r2 < 4.0 * hh * hh) : (j != i && r2 > 0.0 && r2 < 4.0 * hh * hh))
                indices[c++] = j;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- *
 * EOS, PAPER.md:111 (built-in ideal gas; the paper prints no formula, O5):
 *   P = (gamma-1) rho u,  c = sqrt(gamma P / rho).
 * ------------------------------------------------------------------------- */
void orc_eos(int64_t n, const double *rho, const double *u, double gamma, double *P, double *c)
{
    for (int64_t i = 0; i < n; i++) {
        P[i] = (gamma - 1.0) * rho[i] * u[i];
        c[i] = sqrt(gamma * P[i] / rho[i]);
    }
}

/* ------------------------------------------------------------------------- *
 * One ordered pair (i,j) of the force pass, PAPER.md:186-219 (Section 2.3.5).
 *
 *  Eq. (13) dv_i/dt|H  = - sum_j m_j [ P_i/(Om_i rho_i^2) dW_ij(h_i)/dr_i
 *                                    + P_j/(Om_j rho_j^2) dW_ij(h_j)/dr_i ]
 *  Eq. (14) du_i/dt|H  = P_i/(Om_i rho_i^2) sum_j m_j (v_i-v_j).dW_ij(h_i)/dr_i
 *  Eq. (15) Pi_ij = (-alpha cbar mu + beta mu^2)/rhobar  if v_ij.r_ij < 0, else 0
 *  Eq. (16) mu_ij = hbar (v_ij.r_ij) / (r_ij^2 + eps hbar^2)        (R9, R10)
 *  Eq. (17) dv_i/dt|Pi = - sum_j m_j Pi_ij dWbar_ij/dr_i
 *  Eq. (18) du_i/dt|Pi = 1/2 sum_j m_j Pi_ij (v_i-v_j).dWbar_ij/dr_i
 *  Wbar_ij = 0.5 (W_ij(h_i) + W_ij(h_j)).
 *
 * dW_ij(h)/dr_i = (w'(r/h)/h^4) d_ij/r, zero outside that kernel's own
 * support and at r = 0 (R14, R15).  Returns 0 if the pair is not in the
 * gather-or-scatter set.
 * ------------------------------------------------------------------------- */
typedef struct { double a[3], dudt, mu, absC, absU; } orc_pair;

static int orc_pair_force(const orc_params *p, const double d[3], double r2, double hi, double hj,
                          double mj, const double vij[3], double Ai, double Aj, double ci,
                          double cj, double rhoi, double rhoj, orc_pair *out)
{
    double hm = hi > hj ? hi : hj;
    if (!(r2 > 0.0 && r2 < 4.0 * hm * hm)) return 0;
    double r = sqrt(r2);
    double Fi = orc_dw(p->kernel, r / hi) / (hi * hi * hi * hi);   /* dW/dr at h_i */
    double Fj = orc_dw(p->kernel, r / hj) / (hj * hj * hj * hj);   /* dW/dr at h_j */
    double Fbar = 0.5 * (Fi + Fj);
    double vr = vij[0] * d[0] + vij[1] * d[1] + vij[2] * d[2];     /* v_ij . r_ij */
    double hbar = 0.5 * (hi + hj), cbar = 0.5 * (ci + cj), rhobar = 0.5 * (rhoi + rhoj);
    double mu = hbar * vr / (r2 + p->av_eps * hbar * hbar);        /* Eq. (16) */
    double Pi = 0.0;
    if (vr < 0.0) Pi = (-p->av_alpha * cbar * mu + p->av_beta * mu * mu) / rhobar; /* Eq. (15) */
    double C = Ai * Fi + Aj * Fj + Pi * Fbar;                      /* Eqs. (13)+(17) */
    for (int k = 0; k < 3; k++) out->a[k] = -mj * C * d[k] / r;
    double vrhat = vr / r;
    double E = 0.5 * Pi * Fbar * vrhat;                            /* Eq. (18) */
    if (!p->entropy) E += Ai * Fi * vrhat;                         /* Eq. (14) */
    out->dudt = mj * E;
    out->mu = mu;
    out->absC = mj * fabs(C);
    out->absU = mj * fabs(E);
    return 1;
}

/* Brute-force force pass over a list of targets.  rho, h, omega, u are given
 * for ALL particles (the caller decides whose they are: the oracle's own or
 * the device's, for stage-isolated parity).  Outputs, indexed by position in
 * the target list: a (3), du/dt, mu_min = min(0, min_j mu_ij) (for Eq. 26),
 * and the normalisers Sa = sum_j m_j |C_ij|, Su = sum_j m_j |E_ij| the parity
 * tolerance is stated against (BASELINE.json north_star). n_pairs counts the
 * pairs in the gather-or-scatter set. */
int orc_forces_brute(int64_t n, const double *x, const double *y, const double *z,
                     const double *m, const double *vx, const double *vy, const double *vz,
                     const double *u, const double *rho, const double *h, const double *omega,
                     const orc_box *box, const orc_params *p, int64_t nt, const int64_t *targets,
                     double *ax, double *ay, double *az, double *dudt, double *mumin,
                     double *Sa, double *Su, int32_t *n_pairs)
{
    double *P = (double *)malloc(sizeof(double) * (size_t)n);
    double *c = (double *)malloc(sizeof(double) * (size_t)n);
    double *A = (double *)malloc(sizeof(double) * (size_t)n);
    orc_eos(n, rho, u, p->gamma, P, c);
    for (int64_t i = 0; i < n; i++) A[i] = P[i] / (omega[i] * rho[i] * rho[i]);
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t t = 0; t < nt; t++) {
        int64_t i = targets ? targets[t] : t;
        double a[3] = {0, 0, 0}, du = 0, mm = 0, sa = 0, su = 0, d[3];
        int32_t cnt = 0;
        for (int64_t j = 0; j < n; j++) {
            if (j == i) continue;
            double r2 = orc_r2(x, y, z, i, j, box, d);
            double vij[3] = {vx[i] - vx[j], vy[i] - vy[j], vz[i] - vz[j]};
            orc_pair pr;
            if (!orc_pair_force(p, d, r2, h[i], h[j], m[j], vij, A[i], A[j], c[i], c[j], rho[i],
                                rho[j], &pr))
                continue;
            cnt++;
            a[0] += pr.a[0]; a[1] += pr.a[1]; a[2] += pr.a[2];
            du += pr.dudt; sa += pr.absC; su += pr.absU;
            if (pr.mu < mm) mm = pr.mu;
        }
        ax[t] = a[0]; ay[t] = a[1]; az[t] = a[2];
        dudt[t] = du; mumin[t] = mm; Sa[t] = sa; Su[t] = su;
        if (n_pairs) n_pairs[t] = cnt;
    }
    free(P); free(c); free(A);
    return 0;
}

/* ------------------------------------------------------------------------- *
 * Time step, PAPER.md:263-268 (Section 2.3.6) and the global step of
 * PAPER.md:325 (Sedov: "a dynamic global time step ... smaller than the
 * smallest needed by any particle").
 *   dt_a   = eta_a sqrt(eps/|a_i|), eps = the SPH kernel size 2 h_i (R18);
 *            no constraint when |a_i| = 0
 *   dt_CFL = eta_C h_i / ((1+0.6 alpha) c_i + 0.6 beta |min_j min(0,mu_ij)|)   Eq. (26), R17
 *   dt_i   = min(dt_a, dt_CFL);  dt = min_i dt_i.
 * ------------------------------------------------------------------------- */
int orc_timestep(int64_t n, const double *h, const double *c, const double *ax,
                 const double *ay, const double *az, const double *mumin, const orc_params *p,
                 double *dt_i, double *dt_min)
{
    double best = INFINITY;
    for (int64_t i = 0; i < n; i++) {
        double an = sqrt(ax[i] * ax[i] + ay[i] * ay[i] + az[i] * az[i]);
        double dta = an > 0.0 ? p->eta_acc * sqrt(2.0 * h[i] / an) : INFINITY;
        double dtc = p->eta_cfl * h[i] /
                     ((1.0 + 0.6 * p->av_alpha) * c[i] + 0.6 * p->av_beta * fabs(mumin[i]));
        double dt = dta < dtc ? dta : dtc;
        dt_i[i] = dt;
        if (dt < best) best = dt;
    }
    *dt_min = best;
    return 0;
}

/* ------------------------------------------------------------------------- *
 * Cell-list variants: identical sums, with the j-loop restricted to the 27
 * cells around the target's cell.  A uniform grid with cell side >= s covers
 * every particle within distance s of the target, so the restriction is exact
 * whenever the support in use is <= s.  Not part of the definition: pinned
 * against the brute force above.
 * ------------------------------------------------------------------------- */
typedef struct {
    int64_t nc[3];
    int64_t *start;   /* nc0*nc1*nc2 + 1 */
    int64_t *order;   /* particle indices grouped by cell */
} orc_grid;

static int64_t orc_cell_of(double v, double lo, double len, int64_t nc)
{
    int64_t c = (int64_t)floor((v - lo) / len * (double)nc);
    if (c < 0) c = 0;
    if (c >= nc) c = nc - 1;
    return c;
}

static void orc_grid_build(orc_grid *g, int64_t n, const double *x, const double *y,
                           const double *z, const orc_box *b, double s)
{
    for (int d = 0; d < 3; d++) {
        g->nc[d] = (int64_t)floor(b->len[d] / s);
        if (g->nc[d] < 1) g->nc[d] = 1;
        if (g->nc[d] > 1024) g->nc[d] = 1024;
    }
    int64_t ncell = g->nc[0] * g->nc[1] * g->nc[2];
    g->start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
    g->order = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    int64_t *cid = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    for (int64_t i = 0; i < n; i++) {
        int64_t cx = orc_cell_of(x[i], b->lo[0], b->len[0], g->nc[0]);
        int64_t cy = orc_cell_of(y[i], b->lo[1], b->len[1], g->nc[1]);
        int64_t cz = orc_cell_of(z[i], b->lo[2], b->len[2], g->nc[2]);
        cid[i] = (cz * g->nc[1] + cy) * g->nc[0] + cx;
        g->start[cid[i] + 1]++;
    }
    for (int64_t c = 0; c < ncell; c++) g->start[c + 1] += g->start[c];
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)ncell);
    memcpy(fill, g->start, sizeof(int64_t) * (size_t)ncell);
    for (int64_t i = 0; i < n; i++) g->order[fill[cid[i]]++] = i;
    free(fill); free(cid);
}

static void orc_grid_free(orc_grid *g) { free(g->start); free(g->order); }

/* Upper bound on the number of particles in any 27-cell stencil. */
static int64_t orc_grid_max_stencil(const orc_grid *g)
{
    int64_t ncell = g->nc[0] * g->nc[1] * g->nc[2], mx = 0;
    for (int64_t c = 0; c < ncell; c++)
        if (g->start[c + 1] - g->start[c] > mx) mx = g->start[c + 1] - g->start[c];
    return 27 * mx + 1;
}

/* The distinct cells of the 3-cell stencil around cell c in one dimension. */
static int orc_stencil_1d(int64_t c, int64_t nc, int periodic, int64_t out[3])
{
    int k = 0;
    for (int64_t o = -1; o <= 1; o++) {
        int64_t cc = c + o;
        if (periodic) cc = ((cc % nc) + nc) % nc;
        else if (cc < 0 || cc >= nc) continue;
        int dup = 0;
        for (int q = 0; q < k; q++) if (out[q] == cc) dup = 1;
        if (!dup) out[k++] = cc;
    }
    return k;
}

/* Gather the particle indices of the stencil around particle i into cand[]. */
static int64_t orc_candidates(const orc_grid *g, const orc_box *b, double xi, double yi,
                              double zi, int64_t *cand)
{
    int64_t sx[3], sy[3], sz[3], cnt = 0;
    int kx = orc_stencil_1d(orc_cell_of(xi, b->lo[0], b->len[0], g->nc[0]), g->nc[0], b->periodic[0], sx);
    int ky = orc_stencil_1d(orc_cell_of(yi, b->lo[1], b->len[1], g->nc[1]), g->nc[1], b->periodic[1], sy);
    int kz = orc_stencil_1d(orc_cell_of(zi, b->lo[2], b->len[2], g->nc[2]), g->nc[2], b->periodic[2], sz);
    for (int c = 0; c < kz; c++)
        for (int bq = 0; bq < ky; bq++)
            for (int a = 0; a < kx; a++) {
                int64_t cell = (sz[c] * g->nc[1] + sy[bq]) * g->nc[0] + sx[a];
                for (int64_t q = g->start[cell]; q < g->start[cell + 1]; q++) cand[cnt++] = g->order[q];
            }
    return cnt;
}

/* Density / h solve for ALL particles with a cell list of side >= cell_side.
 * A particle whose root bracket would leave the covered radius (h > cell_side/2)
 * falls back to the brute-force loop, so the result never depends on cell_side. */
int orc_density_cells(int64_t n, const double *x, const double *y, const double *z,
                      const double *m, const double *h_hint, const orc_box *box,
                      const orc_params *p, double cell_side, double *h, double *rho,
                      double *omega, int32_t *nngb, int64_t *n_fallback)
{
    orc_grid g;
    orc_grid_build(&g, n, x, y, z, box, cell_side);
    /* actual cell sides are >= cell_side unless a dimension had to be clamped */
    double cover = 1e300;
    for (int d = 0; d < 3; d++) {
        double side = box->len[d] / (double)g.nc[d];
        if (g.nc[d] > 1 && side < cover) cover = side;
        if (g.nc[d] == 1 && !box->periodic[d]) { /* whole dimension in the stencil */ }
    }
    double hcap_box = orc_hcap(box);
    double hcap = 0.5 * cover < hcap_box ? 0.5 * cover : hcap_box;
    int err = 0;
    int64_t nfb = 0, cap = orc_grid_max_stencil(&g);
#pragma omp parallel
    {
        int64_t *cand = (int64_t *)malloc(sizeof(int64_t) * (size_t)cap);
        double *r2 = (double *)malloc(sizeof(double) * (size_t)cap);
        double *mm = (double *)malloc(sizeof(double) * (size_t)cap);
#pragma omp for schedule(dynamic, 64) reduction(+ : nfb)
        for (int64_t i = 0; i < n; i++) {
            double d[3];
            int64_t cnt = orc_candidates(&g, box, x[i], y[i], z[i], cand);
            for (int64_t k = 0; k < cnt; k++) {
                r2[k] = orc_r2(x, y, z, i, cand[k], box, d);
                mm[k] = m[cand[k]];
            }
            int rc = orc_solve_h(p, cnt, r2, mm, m[i], h_hint[i], hcap, &h[i], &rho[i], &omega[i],
                                 &nngb[i]);
            if (rc == -1) {            /* bracket left the covered radius: brute force */
                nfb++;
                double *r2all = (double *)malloc(sizeof(double) * (size_t)n);
                for (int64_t j = 0; j < n; j++) r2all[j] = orc_r2(x, y, z, i, j, box, d);
                rc = orc_solve_h(p, n, r2all, m, m[i], h_hint[i], hcap_box, &h[i], &rho[i],
                                 &omega[i], &nngb[i]);
                free(r2all);
            }
            if (rc) {
#pragma omp critical
                err = rc;
            }
        }
        free(cand); free(r2); free(mm);
    }
    if (n_fallback) *n_fallback = nfb;
    orc_grid_free(&g);
    return err;
}

/* Force pass for ALL particles with a cell list; cell_side must be
 * >= 2 max_i h_i (checked; returns -3 otherwise). */
int orc_forces_cells(int64_t n, const double *x, const double *y, const double *z,
                     const double *m, const double *vx, const double *vy, const double *vz,
                     const double *u, const double *rho, const double *h, const double *omega,
                     const orc_box *box, const orc_params *p, double cell_side, double *ax,
                     double *ay, double *az, double *dudt, double *mumin, double *Sa,
                     double *Su, int32_t *n_pairs)
{
    orc_grid g;
    orc_grid_build(&g, n, x, y, z, box, cell_side);
    double hmax = 0.0;
    for (int64_t i = 0; i < n; i++) if (h[i] > hmax) hmax = h[i];
    for (int d = 0; d < 3; d++)
        if (g.nc[d] > 1 && box->len[d] / (double)g.nc[d] < 2.0 * hmax) { orc_grid_free(&g); return -3; }
    double *P = (double *)malloc(sizeof(double) * (size_t)n);
    double *c = (double *)malloc(sizeof(double) * (size_t)n);
    double *A = (double *)malloc(sizeof(double) * (size_t)n);
    orc_eos(n, rho, u, p->gamma, P, c);
    for (int64_t i = 0; i < n; i++) A[i] = P[i] / (omega[i] * rho[i] * rho[i]);
    int64_t cap = orc_grid_max_stencil(&g);
#pragma omp parallel
    {
        int64_t *cand = (int64_t *)malloc(sizeof(int64_t) * (size_t)cap);
#pragma omp for schedule(dynamic, 64)
        for (int64_t i = 0; i < n; i++) {
            double a[3] = {0, 0, 0}, du = 0, mm = 0, sa = 0, su = 0, d[3];
            int32_t cnt = 0;
            int64_t nc = orc_candidates(&g, box, x[i], y[i], z[i], cand);
            for (int64_t k = 0; k < nc; k++) {
                int64_t j = cand[k];
                if (j == i) continue;
                double r2 = orc_r2(x, y, z, i, j, box, d);
                double vij[3] = {vx[i] - vx[j], vy[i] - vy[j], vz[i] - vz[j]};
                orc_pair pr;
                if (!orc_pair_force(p, d, r2, h[i], h[j], m[j], vij, A[i], A[j], c[i], c[j],
                                    rho[i], rho[j], &pr))
                    continue;
                cnt++;
                a[0] += pr.a[0]; a[1] += pr.a[1]; a[2] += pr.a[2];
                du += pr.dudt; sa += pr.absC; su += pr.absU;
                if (pr.mu < mm) mm = pr.mu;
            }
            ax[i] = a[0]; ay[i] = a[1]; az[i] = a[2];
            dudt[i] = du; mumin[i] = mm; Sa[i] = sa; Su[i] = su;
            if (n_pairs) n_pairs[i] = cnt;
        }
        free(cand);
    }
    free(P); free(c); free(A);
    orc_grid_free(&g);
    return 0;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- *
 * Time integration with a global step, PAPER.md:227-261 (Section 2.3.6),
 * Eqs. (19)-(25): kick-drift-kick with predicted v, u for the force pass.
 *   Eqs. (19)-(20)  predict:  q_pred = q_{i-1/2} + (dt/2) qdot_{i-1}   (q = v, u)
 *   Eqs. (21)-(24)  kick:     q     += (dt/2) qdot_i   (closing and opening kick)
 *   Eq.  (25)       drift:    x_{i+1} = x_i + dt v_{i+1/2}, wrapped into the
 *                   periodic box [lo, lo+len) (PAPER.md:297 periodic tests)
 * Plain statements of the update formulas; one array at a time.
 * ------------------------------------------------------------------------- */
void orc_axpy(int64_t n, double a, const double *x, const double *y, double *out)
{   /* out = y + a x : the form shared by Eqs. (19)-(24) with a = dt/2 */
    for (int64_t i = 0; i < n; i++) out[i] = y[i] + a * x[i];
}

/* Entropy-conserving update of the ideal gas: "uses the old
 * density and internal energy to calculate the isentropic evolution to the new
 * density, by having the EOS solve u_new = u(rho_new, s(rho_old, u_old))".  For
 * P = (gamma-1) rho u an isentrope is P / rho^gamma = const
 * (the entropic function of Springel & Hernquist 2002, cited there), hence
 *   u_new = u_old (rho_new / rho_old)^(gamma-1).           (reading R31) */
void orc_isentropic_u(int64_t n, double gamma, const double *rho_old, const double *rho_new,
                      const double *u_old, double *u_new)
{
    for (int64_t i = 0; i < n; i++) u_new[i] = u_old[i] * pow(rho_new[i] / rho_old[i], gamma - 1.0);
}

void orc_drift(int64_t n, double dt, const double *v, double lo, double len, int periodic,
               double *x)
{
    for (int64_t i = 0; i < n; i++) {
        double xn = x[i] + dt * v[i];                       /* Eq. (25) */
        if (periodic) {
            xn -= len * floor((xn - lo) / len);
            if (xn >= lo + len) xn = lo;                    /* rounding at the upper face */
        }
        x[i] = xn;
    }
}

/* ------------------------------------------------------------------------- *
 * Block time steps, PAPER.md:229 ("each particle is integrated with a time
 * step size that is a power-of-two fraction of the global timestep"), the
 * substep of PAPER.md:231-261 per particle, rung changes of PAPER.md:270.
 * Reading R32: time is counted in substeps of delta = dt0 / 2^R,
 * R the deepest rung; a step of rung r spans L(r) = 2^(R-r) substeps.  Per
 * particle: rung, tnext (the substep at which its running step ends, i.e. at
 * which it is active next) and hk (the half-step length of its last opening
 * kick; 0 before the first one), so that its v, u are those of the time
 * tnext delta - hk.
 * ------------------------------------------------------------------------- */

/* the lowest rung whose steps begin at substep s ("moving to a lower rung is only
 * possible on substeps that correspond to the rung it wants to move to") */
int32_t orc_block_floor_rung(int64_t s, int32_t R)
{
    for (int32_t r = 0; r < R; r++)
        if (s % ((int64_t)1 << (R - r)) == 0) return r;
    return R;
}

/* Eqs. (19)-(20) for every particle, active or not (the sources of the force pass need
 * predicted values too): from the time of its v, u to the time s delta of the substep */
void orc_block_predict(int64_t n, int64_t s, double delta, const int32_t *tnext, const double *hk,
                       const double *base, const double *rate, double *out)
{
    for (int64_t i = 0; i < n; i++) {
        double tau = (double)(s - (int64_t)tnext[i]) * delta + hk[i];
        out[i] = base[i] + tau * rate[i];
    }
}

/* Step 4 of PAPER.md:245-259 for the particles whose step ends at substep s: closing kick
 * over the old half step (Eqs. 21-22), rung change (up at once, down only as far as the
 * substep allows, capped at R), opening kick over the new half step (Eqs. 23-24).
 * q, rate: nq arrays of n values each, one after the other.  open = 0: the closing kick
 * alone (to bring v, u to the current time, e.g. for an output); hk becomes 0 and tnext
 * stays s, the state in which a run starts.                                              */
void orc_block_kick(int64_t n, int64_t s, int32_t R, double delta, const int32_t *rung_des,
                    int32_t *rung, int32_t *tnext, double *hk, int32_t nq, double *q,
                    const double *rate, int32_t open)
{
    int32_t fl = orc_block_floor_rung(s, R);
    for (int64_t i = 0; i < n; i++) {
        if ((int64_t)tnext[i] != s) continue;
        for (int32_t k = 0; k < nq; k++) q[k * n + i] += hk[i] * rate[k * n + i];
        if (!open) { hk[i] = 0.0; continue; }   /* v, u now at the time s delta, as at the start */
        int32_t r = rung_des[i] > fl ? rung_des[i] : fl;
        if (r > R) r = R;
        int64_t L = (int64_t)1 << (R - r);
        hk[i] = 0.5 * (double)L * delta;
        for (int32_t k = 0; k < nq; k++) q[k * n + i] += hk[i] * rate[k * n + i];
        tnext[i] = (int32_t)(s + L);
        rung[i] = r;
    }
}

/* ------------------------------------------------------------------------- *
 * Interface correction, PAPER.md:158-182 (Section 2.3.4), Eqs. (8)-(12), for
 * the built-in ideal gas.  Brute force: every target against all particles.
 *
 *   Eq. (8)   I_i = alpha |sum_j kappa_ij (r_j - r_i) m_j W_ij(h_i)|
 *                   / (h_i sum_j m_j W_ij(h_i)),
 *             kappa_ij = +1 same material, -1 different material; the sums run
 *             over the gather neighbours r_ij < 2 h_i, self included (reading
 *             R25; the self term adds nothing to the numerator).  alpha is "a
 *             normalization parameter" (no value in the paper, reading R24).
 *   Eq. (9)   Tbar_i = sum_j T_j e^{-I_j^2} W_ij(h_i) / sum_j e^{-I_j^2} W_ij(h_i),
 *             Pbar_i likewise (no m_j in the weights, as printed: reading R27)
 *   Eq. (10)  P~_i = e^{-I_i^2} P_i + (1 - e^{-I_i^2}) Pbar_i
 *   Eq. (11)  T~_i likewise
 *   Eq. (12)  rho~_i = rho_EOS(T~_i, P~_i); ideal gas with T = u / c_v:
 *             rho~ = P~ / ((gamma-1) u~), c_v cancels (reading R26), so the
 *             "temperature" handled here is u itself.
 * mat == NULL means one material.
 * ------------------------------------------------------------------------- */
int orc_imbalance_brute(int64_t n, const double *x, const double *y, const double *z,
                        const double *m, const double *h, const int32_t *mat, const orc_box *box,
                        const orc_params *p, double alpha, int64_t nt, const int64_t *targets,
                        double *imb)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t t = 0; t < nt; t++) {
        int64_t i = targets ? targets[t] : t;
        double s[3] = {0.0, 0.0, 0.0}, den = 0.0, d[3];
        for (int64_t j = 0; j < n; j++) {
            double r2 = orc_r2(x, y, z, i, j, box, d);   /* d = x_i - x_j */
            if (r2 >= 4.0 * h[i] * h[i]) continue;
            double w = orc_w(p->kernel, sqrt(r2) / h[i]);      /* W up to the common h^-3 */
            double kappa = (mat && mat[i] != mat[j]) ? -1.0 : 1.0;
            for (int k = 0; k < 3; k++) s[k] += kappa * (-d[k]) * m[j] * w;   /* r_j - r_i */
            den += m[j] * w;
        }
        imb[t] = alpha * sqrt(s[0] * s[0] + s[1] * s[1] + s[2] * s[2]) / (h[i] * den);
    }
    return 0;
}

int orc_interface_brute(int64_t n, const double *x, const double *y, const double *z,
                        const double *h, const double *u, const double *rho, const double *imb,
                        const orc_box *box, const orc_params *p, int64_t nt,
                        const int64_t *targets, double *rho_corr, double *P_corr, double *u_corr)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t t = 0; t < nt; t++) {
        int64_t i = targets ? targets[t] : t;
        double nT = 0.0, nP = 0.0, den = 0.0, d[3];
        for (int64_t j = 0; j < n; j++) {
            double r2 = orc_r2(x, y, z, i, j, box, d);
            if (r2 >= 4.0 * h[i] * h[i]) continue;
            double w = orc_w(p->kernel, sqrt(r2) / h[i]) * exp(-imb[j] * imb[j]);
            double Pj = (p->gamma - 1.0) * rho[j] * u[j];
            nT += u[j] * w; nP += Pj * w; den += w;                       /* Eq. (9) */
        }
        double e = exp(-imb[i] * imb[i]);
        double Pi = (p->gamma - 1.0) * rho[i] * u[i];
        double Pt = e * Pi + (1.0 - e) * nP / den;                        /* Eq. (10) */
        double Tt = e * u[i] + (1.0 - e) * nT / den;                      /* Eq. (11) */
        rho_corr[t] = Pt / ((p->gamma - 1.0) * Tt);                       /* Eq. (12) */
        if (P_corr) P_corr[t] = Pt;
        if (u_corr) u_corr[t] = Tt;
    }
    return 0;
}

/* ------------------------------------------------------------------------- *
 * Time-step rungs.
 *   Eq. (27)  the desired rung r_i: min(dt_a, dt_CFL) >= 2^-r_i dt0; taken as
 *             the SMALLEST such r_i >= 0 (the largest admissible step), capped
 *             at max_rung.
 *   Limiter   (Saitoh & Makino 2009): no particle may have a step
 *             larger than four times that of any particle it interacts with:
 *             r_i >= r_j - 2 for all neighbours j.  One pass over the rungs of
 *             Eq. (27) (reading R28); "interacts with" = the force pair set
 *             0 < r_ij < 2 max(h_i, h_j) (reading R14).
 * ------------------------------------------------------------------------- */
void orc_rungs(int64_t n, const double *dt_i, double dt0, int32_t max_rung, int32_t *rung)
{
    for (int64_t i = 0; i < n; i++) {
        int32_t r = 0;
        double t = dt0;
        while (r < max_rung && t > dt_i[i]) { t *= 0.5; r++; }
        rung[i] = r;
    }
}

void orc_rung_limiter_brute(int64_t n, const double *x, const double *y, const double *z,
                            const double *h, const orc_box *box, const int32_t *rung_in,
                            int64_t nt, const int64_t *targets, int32_t *rung_out)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t t = 0; t < nt; t++) {
        int64_t i = targets ? targets[t] : t;
        int32_t r = rung_in[i];
        double d[3];
        for (int64_t j = 0; j < n; j++) {
            if (j == i) continue;
            double r2 = orc_r2(x, y, z, i, j, box, d);
            double hh = h[j] > h[i] ? h[j] : h[i];
            if (r2 > 0.0 && r2 < 4.0 * hh * hh && rung_in[j] - 2 > r) r = rung_in[j] - 2;
        }
        rung_out[t] = r;
    }
}

/* The FastGas marking pass: "we mark all particles that would end up on
 * interaction lists of active particles".  mark_i = 1 if src_i, or if a particle j with
 * src_j interacts with i: 0 < r_ij < 2 max(h_i, h_j) (the pair set of PAPER.md:191;
 * DESIGN.md reading R29).  Brute force over all pairs. */
void orc_mark_brute(int64_t n, const double *x, const double *y, const double *z,
                    const double *h, const orc_box *box, const uint8_t *src, uint8_t *mark)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = 0; i < n; i++) {
        uint8_t mk = src[i] ? 1 : 0;
        double d[3];
        for (int64_t j = 0; j < n && !mk; j++) {
            if (j == i || !src[j]) continue;
            double r2 = orc_r2(x, y, z, i, j, box, d);
            double hh = h[j] > h[i] ? h[j] : h[i];
            if (r2 > 0.0 && r2 < 4.0 * hh * hh) mk = 1;
        }
        mark[i] = mk;
    }
}
