/*
 * stag_oracle.c -- CPU ORACLE for the staggered-fermion CG hot path of
 * arXiv:1111.0125 (Jang, Kim, Lee, Lattice 2011).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is the plain, slow,
 * obviously-correct fp64 statement of what the CUDA path must compute.  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference leg may call it.  It shares no code with the CUDA library.
 *
 * Each function cites the passage of /root/reference/PAPER.md ("P:Lnn") it
 * follows.  Conventions ("Conventions"):
 *   site idx = x0 + X0*(x1 + X1*(x2 + X2*x3)); parity p = sum(x)&1; cb = idx>>1
 *   links    W[mu][p][cb][i][j][re,im]  -- eta_mu(x)*bc_mu(x)*U_mu(x), the
 *            phases already folded in by the caller
 *   spinor   chi[cb][i][re,im] on one parity
 *
 * Pins: tests/test_oracle_*.py (anti-hermiticity, positivity identity,
 * free-field closed form, gauge covariance, dense brute force from an
 * independent numpy construction, flop/byte counters, degenerate cases, CG
 * invariants).  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* threads the loops below run on (reported beside the timed CPU baseline; no arithmetic) */
int so_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

typedef struct { int X[4]; long V, Vh; } geom_t;

typedef struct { uint64_t flops, bytes; } so_counters_t;

static int geom_init(geom_t *g, const int dims[4])
{
    g->V = 1;
    for (int m = 0; m < 4; ++m) {
        if (dims[m] < 2 || (dims[m] & 1)) return -1;
        g->X[m] = dims[m];
        g->V *= dims[m];
    }
    g->Vh = g->V / 2;
    return 0;
}

static inline long lex_index(const geom_t *g, const int x[4])
{
    return x[0] + (long)g->X[0] * (x[1] + (long)g->X[1] * (x[2] + (long)g->X[2] * x[3]));
}

/* coordinates of the site with parity p and checkerboard index cb */
static inline void cb_coords(const geom_t *g, int p, long cb, int x[4])
{
    long idx = 2 * cb;                 /* the even member of the pair (2cb, 2cb+1) */
    long r = idx / g->X[0];
    x[1] = (int)(r % g->X[1]); r /= g->X[1];
    x[2] = (int)(r % g->X[2]); r /= g->X[2];
    x[3] = (int)r;
    x[0] = (int)(idx % g->X[0]);       /* even; the pair differs only in x0 */
    if (((x[0] + x[1] + x[2] + x[3]) & 1) != p) x[0] += 1;
}

/* ---- counted complex arithmetic: 6 flop per multiply, 2 per add ---------- */

typedef struct { double re, im; } cplx;

static inline cplx c_mul(cplx a, cplx b, so_counters_t *c)
{
    if (c) c->flops += 6;
    cplx r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re };
    return r;
}
static inline cplx c_add(cplx a, cplx b, so_counters_t *c)
{
    if (c) c->flops += 2;
    cplx r = { a.re + b.re, a.im + b.im };
    return r;
}
static inline cplx c_sub(cplx a, cplx b, so_counters_t *c)
{
    if (c) c->flops += 2;
    cplx r = { a.re - b.re, a.im - b.im };
    return r;
}
static inline cplx c_conj(cplx a) { cplx r = { a.re, -a.im }; return r; }

static inline const cplx *load_link(const double *W, const geom_t *g, int mu, int p, long cb,
                                    so_counters_t *c)
{
    if (c) c->bytes += 18 * sizeof(double);
    return (const cplx *)(W + (((size_t)mu * 2 + (size_t)p) * (size_t)g->Vh + (size_t)cb) * 18);
}
static inline const cplx *load_vec(const double *chi, long cb, so_counters_t *c)
{
    if (c) c->bytes += 6 * sizeof(double);
    return (const cplx *)(chi + (size_t)cb * 6);
}

/*
 * One output site of eq. 2.5:
 *   D chi(x) = sum_mu [ U_mu(x) chi(x+mu) - U_mu^dag(x-mu) chi(x-mu) ]
 * with (U chi)_i = sum_j U_ij chi_j and (U^dag chi)_i = sum_j conj(U_ji) chi_j.
 * No factor 1/2 (reading Q1).  Coordinates wrap mod X_mu; the
 * boundary sign lives in the link (reading Q3).
 */
static void dslash_site(cplx out[3], const double *in, const double *W, const geom_t *g,
                        int p, long cb, so_counters_t *c)
{
    int x[4];
    cb_coords(g, p, cb, x);
    cplx acc[3] = { {0, 0}, {0, 0}, {0, 0} };
    for (int mu = 0; mu < 4; ++mu) {
        int xf[4] = { x[0], x[1], x[2], x[3] };
        int xb[4] = { x[0], x[1], x[2], x[3] };
        xf[mu] = (x[mu] + 1) % g->X[mu];
        xb[mu] = (x[mu] + g->X[mu] - 1) % g->X[mu];
        long cbf = lex_index(g, xf) >> 1;
        long cbb = lex_index(g, xb) >> 1;

        /* + U_mu(x) chi(x+mu) */
        const cplx *U = load_link(W, g, mu, p, cb, c);
        const cplx *vf = load_vec(in, cbf, c);
        for (int i = 0; i < 3; ++i) {
            cplx t = c_mul(U[3*i+0], vf[0], c);
            t = c_add(t, c_mul(U[3*i+1], vf[1], c), c);
            t = c_add(t, c_mul(U[3*i+2], vf[2], c), c);
            acc[i] = c_add(acc[i], t, c);
        }
        /* - U_mu(x-mu)^dag chi(x-mu); the link lives on the other parity */
        const cplx *Ub = load_link(W, g, mu, 1 - p, cbb, c);
        const cplx *vb = load_vec(in, cbb, c);
        for (int i = 0; i < 3; ++i) {
            cplx t = c_mul(c_conj(Ub[3*0+i]), vb[0], c);
            t = c_add(t, c_mul(c_conj(Ub[3*1+i]), vb[1], c), c);
            t = c_add(t, c_mul(c_conj(Ub[3*2+i]), vb[2], c), c);
            acc[i] = c_sub(acc[i], t, c);
        }
    }
    out[0] = acc[0]; out[1] = acc[1]; out[2] = acc[2];
}

/*
 * out (parity_out sites) = D in (the other parity's sites): one "parity hop"
 * of eq. 2.5.  parity_out = 1 is D_oe, parity_out = 0 is D_eo.
 */
int so_dslash(double *out, const double *in, const double *W, const int dims[4], int parity_out)
{
    geom_t g;
    if (!out || !in || !W || geom_init(&g, dims) || (parity_out & ~1)) return -1;
#pragma omp parallel for schedule(static)
    for (long cb = 0; cb < g.Vh; ++cb) {
        cplx o[3];
        dslash_site(o, in, W, &g, parity_out, cb, NULL);
        memcpy(out + (size_t)cb * 6, o, sizeof(o));
    }
    return 0;
}

/*
 * The same hop, serial, with every flop and every byte of eq. 2.5 tallied.
 * The paper states 576 flop and 1584 bytes per site: 8 links x 18
 * reals + 8 neighbour vectors x 6 reals + 1 store x 6 reals, 8 bytes each.
 */
int so_dslash_counted(double *out, const double *in, const double *W, const int dims[4],
                      int parity_out, uint64_t *flops, uint64_t *bytes)
{
    geom_t g;
    if (!out || !in || !W || geom_init(&g, dims) || (parity_out & ~1)) return -1;
    so_counters_t c = { 0, 0 };
    for (long cb = 0; cb < g.Vh; ++cb) {
        cplx o[3];
        dslash_site(o, in, W, &g, parity_out, cb, &c);
        memcpy(out + (size_t)cb * 6, o, sizeof(o));
        c.bytes += 6 * sizeof(double);
    }
    *flops = c.flops;
    *bytes = c.bytes;
    return 0;
}

/*
 * A = -D^2 + m^2 (eq. 2.3) restricted to even sites:
 *   out_e = m^2 in_e - D_eo ( D_oe in_e ).
 * tmp_o is caller scratch of one odd-parity spinor.
 */
int so_apply_A(double *out_e, const double *in_e, const double *W, const int dims[4],
               double mass, double *tmp_o)
{
    geom_t g;
    if (!out_e || !in_e || !W || !tmp_o || geom_init(&g, dims)) return -1;
    so_dslash(tmp_o, in_e, W, dims, 1);
    so_dslash(out_e, tmp_o, W, dims, 0);
    const double m2 = mass * mass;
    const long n = g.Vh * 6;
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) out_e[k] = m2 * in_e[k] - out_e[k];
    return 0;
}

/* ---- vector algebra of Fig. 1, fp64 ---------------------------- */

/* Re <a,b> = sum_k a_k b_k over the 6*Vh reals.  Summed in fixed blocks so the
 * value does not depend on the OpenMP thread count. */
#define SO_BLK 4096
double so_redot(const double *a, const double *b, long n)
{
    long nb = (n + SO_BLK - 1) / SO_BLK;
    double *part = (double *)malloc((size_t)nb * sizeof(double));
#pragma omp parallel for schedule(static)
    for (long ib = 0; ib < nb; ++ib) {
        long lo = ib * SO_BLK, hi = lo + SO_BLK < n ? lo + SO_BLK : n;
        double s = 0;
        for (long k = lo; k < hi; ++k) s += a[k] * b[k];
        part[ib] = s;
    }
    double s = 0;
    for (long ib = 0; ib < nb; ++ib) s += part[ib];
    free(part);
    return s;
}

static void axpy(double *y, double a, const double *x, long n)
{
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) y[k] += a * x[k];
}

static void xpay(double *y, const double *x, double b, long n) /* y = x + b*y */
{
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) y[k] = x[k] + b * y[k];
}

/* r = b - A x ; returns |r|^2 */
static double residual(double *r, const double *x, const double *b, const double *W,
                       const int dims[4], double mass, double *tmp_o, long n)
{
    so_apply_A(r, x, W, dims, mass, tmp_o);
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) r[k] = b[k] - r[k];
    return so_redot(r, r, n);
}

/*
 * Conjugate gradient, Fig. 1, line by line:
 *   r = b - A x ; d = r ; delta_new = r^dag r
 *   for (i = 0; i < maxiter && delta_new > tol^2 delta_ref; ++i) {
 *       alpha = delta_new / d^dag A d
 *       x += alpha d ;  r -= alpha A d
 *       delta_old = delta_new ; delta_new = r^dag r
 *       beta = delta_new / delta_old ;  d = r + beta d
 *   }
 * Readings: delta_ref = |b|^2 (Q6; equals Fig. 1's delta_0 for
 * x0 = 0); N_dim is maxiter (Q7); on loop exit the TRUE residual
 * rho = |b - A x| / |b| is recomputed and, if rho > tol with iterations left,
 * CG restarts from r = b - A x, d = r (Q6b).  x holds x0 on entry.
 * Returns 0 = converged, 1 = maxiter reached, 2 = breakdown (d^dag A d <= 0
 * or NaN), -1 = bad argument.
 */
int so_cg(double *x, const double *b, const double *W, const int dims[4], double mass,
          double tol, int maxiter, int *iters_out, double *resid_out, int *restarts_out)
{
    geom_t g;
    if (!x || !b || !W || geom_init(&g, dims) || !(tol > 0) || maxiter < 0) return -1;
    const long n = g.Vh * 6;
    double *r = (double *)malloc((size_t)n * sizeof(double));
    double *d = (double *)malloc((size_t)n * sizeof(double));
    double *q = (double *)malloc((size_t)n * sizeof(double));
    double *tmp = (double *)malloc((size_t)n * sizeof(double));
    int rc = 0, i = 0, restarts = 0;
    const double delta_ref = so_redot(b, b, n);
    double rho = 0.0;

    if (delta_ref == 0.0) {            /* b = 0  =>  x = 0 exactly, no 0/0 */
        memset(x, 0, (size_t)n * sizeof(double));
        goto done;
    }
    for (;;) {
        double delta_new = residual(r, x, b, W, dims, mass, tmp, n);   /* r = b - A x */
        memcpy(d, r, (size_t)n * sizeof(double));                      /* d = r       */
        for (; i < maxiter && delta_new > tol * tol * delta_ref; ++i) {
            so_apply_A(q, d, W, dims, mass, tmp);                      /* q = A d     */
            double dAd = so_redot(d, q, n);
            if (!(dAd > 0.0)) { rc = 2; break; }
            double alpha = delta_new / dAd;
            axpy(x, alpha, d, n);                                      /* x += alpha d */
            axpy(r, -alpha, q, n);                                     /* r -= alpha q */
            double delta_old = delta_new;
            delta_new = so_redot(r, r, n);
            double beta = delta_new / delta_old;
            xpay(d, r, beta, n);                                       /* d = r + beta d */
        }
        rho = sqrt(residual(r, x, b, W, dims, mass, tmp, n) / delta_ref);
        if (rc == 2) break;
        if (rho <= tol) break;
        if (i >= maxiter) { rc = 1; break; }
        ++restarts;
    }
done:
    if (iters_out) *iters_out = i;
    if (resid_out) *resid_out = rho;
    if (restarts_out) *restarts_out = restarts;
    free(r); free(d); free(q); free(tmp);
    return rc;
}

/* ---- the full-lattice operator M = D + m and its solve ------------------------
 *
 * The paper solves h = A chi with A = -D^2 + m^2 (eq. 2.2-2.3) where
 * "h is given as a source vector and chi is a staggered fermion field which
 * corresponds to the CG solution", on the even sites.  The
 * production use of that solve is the staggered propagator
 * (D + m) psi = h on the whole lattice.  Because D^dag = -D (eq. 2.4),
 *   (D + m)^dag (D + m) = (-D + m)(D + m) = -D^2 + m^2 = A,
 * and A does not mix parities, so psi follows from one even-site solve
 * (reading Q23).  Full-lattice fields are [parity][cb][3][re,im].
 */

/* out = (D + m) in on the whole lattice: out_p = m in_p + D_{p,1-p} in_{1-p}  (eq. 2.5) */
int so_apply_M(double *out_full, const double *in_full, const double *W, const int dims[4],
               double mass)
{
    geom_t g;
    if (!out_full || !in_full || !W || geom_init(&g, dims)) return -1;
    const long n = g.Vh * 6;
    for (int p = 0; p < 2; ++p) {
        so_dslash(out_full + (size_t)p * n, in_full + (size_t)(1 - p) * n, W, dims, p);
#pragma omp parallel for schedule(static)
        for (long k = 0; k < n; ++k) out_full[(size_t)p * n + k] += mass * in_full[(size_t)p * n + k];
    }
    return 0;
}

/*
 * Solve (D + m) psi = h, step by step (Q23):
 *   1. b_e   = m h_e - D_eo h_o            the even part of (D+m)^dag h
 *   2. psi_e : A psi_e = b_e               Fig. 1 CG (so_cg above), tolerance tol on |b_e|
 *   3. psi_o = (h_o - D_oe psi_e) / m      the odd rows of (D+m) psi = h
 * resid_out = |h - (D+m) psi| / |h| on the whole lattice, recomputed with so_apply_M.
 * Returns so_cg's status (0 converged, 1 maxiter, 2 breakdown), -1 on a bad argument
 * (mass == 0 is one: step 3 divides by it).
 */
int so_solve_M(double *psi_full, const double *h_full, const double *W, const int dims[4],
               double mass, double tol, int maxiter, int *iters_out, double *resid_out)
{
    geom_t g;
    if (!psi_full || !h_full || !W || geom_init(&g, dims) || !(tol > 0) || maxiter < 0 ||
        mass == 0.0)
        return -1;
    const long n = g.Vh * 6;
    const double *h_e = h_full, *h_o = h_full + n;
    double *psi_e = psi_full, *psi_o = psi_full + n;
    double *b_e = (double *)malloc((size_t)n * sizeof(double));
    double *t = (double *)malloc((size_t)2 * n * sizeof(double));

    so_dslash(b_e, h_o, W, dims, 0);                                   /* D_eo h_o */
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) b_e[k] = mass * h_e[k] - b_e[k];      /* step 1 */

    memset(psi_e, 0, (size_t)n * sizeof(double));
    int rc = so_cg(psi_e, b_e, W, dims, mass, tol, maxiter, iters_out, NULL, NULL);   /* step 2 */

    so_dslash(psi_o, psi_e, W, dims, 1);                               /* D_oe psi_e */
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) psi_o[k] = (h_o[k] - psi_o[k]) / mass;   /* step 3 */

    so_apply_M(t, psi_full, W, dims, mass);
#pragma omp parallel for schedule(static)
    for (long k = 0; k < 2 * n; ++k) t[k] = h_full[k] - t[k];
    const double hh = so_redot(h_full, h_full, 2 * n);
    if (resid_out) *resid_out = hh > 0.0 ? sqrt(so_redot(t, t, 2 * n) / hh) : 0.0;
    free(b_e); free(t);
    return rc;
}
