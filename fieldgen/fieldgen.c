/*
 * fieldgen.c -- seeded synthetic lattice inputs (gauge links, sources, gauge
 * transforms) for the staggered-CG build.
 *
 * This module only MAKES INPUTS.  It holds none of the method's arithmetic
 * (no Dslash, no A, no CG) and is the one piece of code that both the CPU
 * oracle's tests and the CUDA path's tests/bench may call.
 *
 * Recipe (BASELINE.json configs[0..4]):
 *   - counter-based RNG: every value is a pure function of
 *     (seed, field tag, lexicographic site index, mu, component), so the
 *     fields do not depend on thread count or traversal order;
 *   - random SU(3): complex Gaussian 3x3, rows Gram-Schmidt'ed, third row
 *     conj(r0 x r1) (det = +1 exactly);
 *   - smooth links: U = exp(i eps H), H = (G+G^dag)/2 - tr/3, re-projected
 *     the same way;
 *   - staggered phases eta_mu(x) = (-1)^(x_0+..+x_{mu-1}) and the
 *     antiperiodic time boundary (a -1 on mu=3 links leaving x3 = X3-1) are
 *     folded into the links here, as the paper says the CPS library does
 *     before the solver is called.
 *
 * Canonical layouts (all fp64, C order), shared by oracle and C-ABI boundary:
 *   site    : idx = x0 + X0*(x1 + X1*(x2 + X2*x3)), parity p = (x0+x1+x2+x3)&1,
 *             checkerboard index cb = idx >> 1  (all X_mu even)
 *   links   : W[mu][p][cb][i][j][re,im]        4*2*Vh*18 doubles
 *   spinor  : chi[cb][i][re,im] for one parity Vh*6 doubles
 *   gauge G : G[p][cb][i][j][re,im]            2*Vh*18 doubles
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#include <string.h>

#define FG_TAG_LINK   0x4C494E4Bull
#define FG_TAG_SOURCE 0x53524345ull
#define FG_TAG_GAUGE  0x47415547ull

static inline uint64_t splitmix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

/* one 64-bit draw addressed by (seed, tag, idx, k) */
static inline uint64_t fg_u64(uint64_t seed, uint64_t tag, uint64_t idx, uint64_t k)
{
    uint64_t h = splitmix64(seed ^ (tag * 0xD6E8FEB86659FD93ull));
    h = splitmix64(h ^ (idx * 0xA24BAED4963EE407ull));
    return splitmix64(h + k);
}

static inline double fg_uniform(uint64_t seed, uint64_t tag, uint64_t idx, uint64_t k)
{
    return ((double)(fg_u64(seed, tag, idx, k) >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

/* N(0,1) number k at (seed, tag, idx): Box-Muller on uniforms (2j, 2j+1), j = k>>1 */
static inline double fg_normal(uint64_t seed, uint64_t tag, uint64_t idx, uint64_t k)
{
    uint64_t j = k >> 1;
    double u1 = fg_uniform(seed, tag, idx, 2 * j);
    double u2 = fg_uniform(seed, tag, idx, 2 * j + 1);
    double r = sqrt(-2.0 * log(u1));
    double a = 6.283185307179586476925286766559 * u2;
    return (k & 1) ? r * sin(a) : r * cos(a);
}

/* exported so tests can pin the generator's statistics and reproducibility */
double fg_normal_at(uint64_t seed, uint64_t tag, uint64_t idx, uint64_t k)
{
    return fg_normal(seed, tag, idx, k);
}

typedef struct { int X[4]; long V, Vh; } geom_t;

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

static inline void site_coords(const geom_t *g, long idx, int x[4])
{
    x[0] = (int)(idx % g->X[0]); idx /= g->X[0];
    x[1] = (int)(idx % g->X[1]); idx /= g->X[1];
    x[2] = (int)(idx % g->X[2]); idx /= g->X[2];
    x[3] = (int)idx;
}

/* ---- 3x3 complex helpers; m[i][j][re/im] flattened as m[(3*i+j)*2 + c] ---- */

static void row_cross_conj(const double *a, const double *b, double *c)
{
    /* c = conj(a x b) for 3-vectors of complex numbers */
    for (int i = 0; i < 3; ++i) {
        int j = (i + 1) % 3, k = (i + 2) % 3;
        double re = (a[2*j] * b[2*k] - a[2*j+1] * b[2*k+1]) - (a[2*k] * b[2*j] - a[2*k+1] * b[2*j+1]);
        double im = (a[2*j] * b[2*k+1] + a[2*j+1] * b[2*k]) - (a[2*k] * b[2*j+1] + a[2*k+1] * b[2*j]);
        c[2*i] = re;
        c[2*i+1] = -im;
    }
}

/* rows: r0 normalised, r1 orthonormalised against r0, r2 = conj(r0 x r1) */
static void project_su3(double *m)
{
    double *r0 = m, *r1 = m + 6, *r2 = m + 12;
    double n = 0;
    for (int i = 0; i < 6; ++i) n += r0[i] * r0[i];
    n = 1.0 / sqrt(n);
    for (int i = 0; i < 6; ++i) r0[i] *= n;
    /* <r0, r1> = sum conj(r0_i) r1_i */
    double dre = 0, dim = 0;
    for (int i = 0; i < 3; ++i) {
        dre += r0[2*i] * r1[2*i] + r0[2*i+1] * r1[2*i+1];
        dim += r0[2*i] * r1[2*i+1] - r0[2*i+1] * r1[2*i];
    }
    for (int i = 0; i < 3; ++i) {
        r1[2*i]   -= dre * r0[2*i] - dim * r0[2*i+1];
        r1[2*i+1] -= dre * r0[2*i+1] + dim * r0[2*i];
    }
    n = 0;
    for (int i = 0; i < 6; ++i) n += r1[i] * r1[i];
    n = 1.0 / sqrt(n);
    for (int i = 0; i < 6; ++i) r1[i] *= n;
    row_cross_conj(r0, r1, r2);
}

static void mat_mul(const double *a, const double *b, double *c)
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double re = 0, im = 0;
            for (int k = 0; k < 3; ++k) {
                const double *p = a + (3*i+k)*2, *q = b + (3*k+j)*2;
                re += p[0]*q[0] - p[1]*q[1];
                im += p[0]*q[1] + p[1]*q[0];
            }
            c[(3*i+j)*2] = re;
            c[(3*i+j)*2+1] = im;
        }
}

/* e = exp(a) for a 3x3 complex matrix: scale by 2^-s, 14-term Taylor, square s times */
static void mat_exp(const double *a, double *e)
{
    double nrm = 0;
    for (int i = 0; i < 18; ++i) nrm += a[i] * a[i];
    nrm = sqrt(nrm);
    int s = 0;
    while (nrm > 0.25 && s < 40) { nrm *= 0.5; ++s; }
    double as[18], term[18], tmp[18];
    double sc = ldexp(1.0, -s);
    for (int i = 0; i < 18; ++i) as[i] = a[i] * sc;
    memset(e, 0, 18 * sizeof(double));
    memset(term, 0, 18 * sizeof(double));
    for (int i = 0; i < 3; ++i) { e[(3*i+i)*2] = 1.0; term[(3*i+i)*2] = 1.0; }
    for (int n = 1; n <= 14; ++n) {
        mat_mul(term, as, tmp);
        for (int i = 0; i < 18; ++i) { term[i] = tmp[i] / n; e[i] += term[i]; }
    }
    for (int k = 0; k < s; ++k) {
        mat_mul(e, e, tmp);
        memcpy(e, tmp, sizeof(tmp));
    }
}

/* eta_mu(x) * bc_mu(x): the sign folded into W_mu(x) */
static inline double phase_sign(const geom_t *g, const int x[4], int mu, int antiperiodic_t)
{
    int s = 0;
    for (int nu = 0; nu < mu; ++nu) s += x[nu];
    double sg = (s & 1) ? -1.0 : 1.0;
    if (antiperiodic_t && mu == 3 && x[3] == g->X[3] - 1) sg = -sg;
    return sg;
}

/* The link W_mu(x) of the site with lexicographic index idx: a pure function of (seed, idx, mu).
 * kind: 0 = unit links, 1 = random SU(3), 2 = smooth exp(i eps H).
 * fold: multiply by eta*bc (antiperiodic_t selects the time boundary sign). */
static void link_at(const geom_t *g, long idx, const int x[4], int mu, int kind, uint64_t seed,
                    double eps, int fold, int antiperiodic_t, double m[18])
{
    uint64_t ctr = (uint64_t)idx * 4 + (uint64_t)mu;
    if (kind == 0) {
        memset(m, 0, 18 * sizeof(double));
        m[0] = m[8] = m[16] = 1.0;
    } else if (kind == 1) {
        for (int k = 0; k < 18; ++k) m[k] = fg_normal(seed, FG_TAG_LINK, ctr, k);
        project_su3(m);
    } else {
        double gm[18], ih[18];
        for (int k = 0; k < 18; ++k) gm[k] = fg_normal(seed, FG_TAG_LINK, ctr, k);
        /* H = (G + G^dag)/2 - tr/3 ; ih = i*eps*H */
        double h[18];
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) {
                h[(3*i+j)*2]   = 0.5 * (gm[(3*i+j)*2]   + gm[(3*j+i)*2]);
                h[(3*i+j)*2+1] = 0.5 * (gm[(3*i+j)*2+1] - gm[(3*j+i)*2+1]);
            }
        double tr = (h[0] + h[8] + h[16]) / 3.0;
        h[0] -= tr; h[8] -= tr; h[16] -= tr;
        for (int k = 0; k < 9; ++k) {
            ih[2*k]   = -eps * h[2*k+1];
            ih[2*k+1] =  eps * h[2*k];
        }
        mat_exp(ih, m);
        project_su3(m);
    }
    if (fold) {
        double sg = phase_sign(g, x, mu, antiperiodic_t);
        for (int k = 0; k < 18; ++k) m[k] *= sg;
    }
}

/* The whole field W[mu][p][cb][3][3]. */
int fg_links(double *W, const int dims[4], int kind, uint64_t seed, double eps,
             int fold, int antiperiodic_t)
{
    geom_t g;
    if (!W || geom_init(&g, dims) || kind < 0 || kind > 2) return -1;
#pragma omp parallel for schedule(static)
    for (long idx = 0; idx < g.V; ++idx) {
        int x[4];
        site_coords(&g, idx, x);
        int p = (x[0] + x[1] + x[2] + x[3]) & 1;
        long cb = idx >> 1;
        for (int mu = 0; mu < 4; ++mu) {
            double m[18];
            link_at(&g, idx, x, mu, kind, seed, eps, fold, antiperiodic_t, m);
            double *dst = W + (((size_t)mu * 2 + (size_t)p) * (size_t)g.Vh + (size_t)cb) * 18;
            memcpy(dst, m, sizeof(m));
        }
    }
    return 0;
}

/* Time slices t0, t0+1, ..., t0+nt-1 (mod X3) of the same field, W[mu][p][cb'][3][3] with
 * cb' = (slice number j)*s3 + (index inside the slice): what one rank of a T-slab decomposition
 * needs, generated without the rest of the lattice.  Every value equals the one fg_links writes
 * for that site (the generator is counter-based). */
int fg_links_slices(double *W, const int dims[4], int kind, uint64_t seed, double eps,
                    int fold, int antiperiodic_t, int t0, int nt)
{
    geom_t g;
    if (!W || geom_init(&g, dims) || kind < 0 || kind > 2 || nt < 1 || nt > dims[3]) return -1;
    const long vslice = g.V / g.X[3];          /* sites per time slice, both parities */
    const long s3 = vslice / 2;
#pragma omp parallel for schedule(static)
    for (long k = 0; k < (long)nt * vslice; ++k) {
        const int j = (int)(k / vslice);
        const int t = ((t0 + j) % g.X[3] + g.X[3]) % g.X[3];
        const long idx = (long)t * vslice + k % vslice;
        int x[4];
        site_coords(&g, idx, x);
        int p = (x[0] + x[1] + x[2] + x[3]) & 1;
        long cbl = (long)j * s3 + ((idx >> 1) - (long)t * s3);
        for (int mu = 0; mu < 4; ++mu) {
            double m[18];
            link_at(&g, idx, x, mu, kind, seed, eps, fold, antiperiodic_t, m);
            double *dst = W + (((size_t)mu * 2 + (size_t)p) * (size_t)(nt * s3) + (size_t)cbl) * 18;
            memcpy(dst, m, sizeof(m));
        }
    }
    return 0;
}

/* complex Gaussian (re, im ~ N(0,1)) on the sites of one parity */
int fg_spinor_gaussian(double *chi, const int dims[4], int parity, uint64_t seed)
{
    geom_t g;
    if (!chi || geom_init(&g, dims) || (parity & ~1)) return -1;
#pragma omp parallel for schedule(static)
    for (long idx = 0; idx < g.V; ++idx) {
        int x[4];
        site_coords(&g, idx, x);
        if (((x[0] + x[1] + x[2] + x[3]) & 1) != parity) continue;
        double *dst = chi + (size_t)(idx >> 1) * 6;
        for (int k = 0; k < 6; ++k) dst[k] = fg_normal(seed, FG_TAG_SOURCE, (uint64_t)idx, k);
    }
    return 0;
}

/* chi(x) = exp(i p.x) v on one parity; p_mu = 2 pi n_mu / X_mu, and
 * p_3 = 2 pi (n_3 + 1/2) / X_3 when antiperiodic_t (SURVEY.md 8c pin 3) */
int fg_spinor_planewave(double *chi, const int dims[4], int parity, const int n[4],
                        const double v[6], int antiperiodic_t)
{
    geom_t g;
    if (!chi || !n || !v || geom_init(&g, dims) || (parity & ~1)) return -1;
    double pm[4];
    for (int mu = 0; mu < 4; ++mu) {
        double nn = n[mu] + ((mu == 3 && antiperiodic_t) ? 0.5 : 0.0);
        pm[mu] = 6.283185307179586476925286766559 * nn / g.X[mu];
    }
#pragma omp parallel for schedule(static)
    for (long idx = 0; idx < g.V; ++idx) {
        int x[4];
        site_coords(&g, idx, x);
        if (((x[0] + x[1] + x[2] + x[3]) & 1) != parity) continue;
        double ph = pm[0]*x[0] + pm[1]*x[1] + pm[2]*x[2] + pm[3]*x[3];
        double c = cos(ph), s = sin(ph);
        double *dst = chi + (size_t)(idx >> 1) * 6;
        for (int i = 0; i < 3; ++i) {
            dst[2*i]   = c * v[2*i] - s * v[2*i+1];
            dst[2*i+1] = c * v[2*i+1] + s * v[2*i];
        }
    }
    return 0;
}

/* random SU(3) matrix per site, for gauge-covariance tests */
int fg_gauge(double *G, const int dims[4], uint64_t seed)
{
    geom_t g;
    if (!G || geom_init(&g, dims)) return -1;
#pragma omp parallel for schedule(static)
    for (long idx = 0; idx < g.V; ++idx) {
        int x[4];
        site_coords(&g, idx, x);
        int p = (x[0] + x[1] + x[2] + x[3]) & 1;
        double m[18];
        for (int k = 0; k < 18; ++k) m[k] = fg_normal(seed, FG_TAG_GAUGE, (uint64_t)idx, k);
        project_su3(m);
        memcpy(G + ((size_t)p * (size_t)g.Vh + (size_t)(idx >> 1)) * 18, m, sizeof(m));
    }
    return 0;
}
