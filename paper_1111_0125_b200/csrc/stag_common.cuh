// stag_common.cuh -- geometry, complex arithmetic and reduction helpers shared by the
// CUDA translation units of libstag.  (Nothing here is shared with oracle/ or fieldgen/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/stag.h"

namespace stag {

constexpr int TILE = 32;   // sites per link tile = one warp of output sites

// Lattice geometry in the form the kernels want it (passed by value: lives in the
// constant bank).  Conventions: include/stag.h "Geometry".
struct Geom {
    int X0h, X1, X2, X3;   // X0h = X0/2 sites of one parity per x0-row
    int Vh, Vh_pad;        // sites per parity, rounded up to TILE
    int s1, s2, s3;        // checkerboard strides of mu = 1,2,3
    int antiperiodic;      // caller folded bc = -1 into W_3 at x3 = X3-1 (only 12-real needs it)
    int t0, X3g;           // T-slab of a larger lattice (stag_slab_*): this lattice is time slices
                           // [t0, t0+X3) of a global extent X3g; a whole lattice has t0 = 0, X3g = X3
};

inline bool make_geom(Geom &g, const int dims[4], int antiperiodic)
{
    if (!dims) return false;
    long v = 1;
    for (int m = 0; m < 4; ++m) {
        if (dims[m] < 2 || (dims[m] & 1)) return false;
        v *= dims[m];
    }
    if (v / 2 > (1L << 30)) return false;   // 32-bit site indices
    g.X0h = dims[0] / 2; g.X1 = dims[1]; g.X2 = dims[2]; g.X3 = dims[3];
    g.Vh = (int)(v / 2);
    g.Vh_pad = (g.Vh + TILE - 1) / TILE * TILE;
    g.s1 = g.X0h; g.s2 = g.X0h * g.X1; g.s3 = g.X0h * g.X1 * g.X2;
    g.antiperiodic = antiperiodic ? 1 : 0;
    g.t0 = 0; g.X3g = g.X3;
    return true;
}

// ---- per-precision vector types ---------------------------------------------------
template <typename T> struct Cplx;
template <> struct Cplx<float>  { using type = float2; };
template <> struct Cplx<double> { using type = double2; };
template <typename T> using cplx_t = typename Cplx<T>::type;

template <typename T> __device__ __forceinline__ cplx_t<T> mk(T re, T im)
{
    cplx_t<T> r; r.x = re; r.y = im; return r;
}

// acc += a * b
template <typename C> __device__ __forceinline__ void cfma(C &acc, const C a, const C b)
{
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}
// a * b
template <typename C> __device__ __forceinline__ C cmul(const C a, const C b)
{
    C r;
    r.x = a.x * b.x - a.y * b.y;
    r.y = a.x * b.y + a.y * b.x;
    return r;
}

// ---- site decoding and the eight neighbours -------------------------------------
// Output site of parity p with checkerboard index cb.  nbr[d], d = 0..3: checkerboard index
// (on the other parity) of x + d^; d = 4..7: of x - (d-4)^.  Coordinates wrap mod X_mu.
struct Site {
    int x0, x1, x2, x3;
    int nbr[8];
};

__device__ __forceinline__ void decode_site(const Geom &g, int p, int cb, Site &s)
{
    unsigned r = (unsigned)cb;
    const unsigned xh = r % (unsigned)g.X0h; r /= (unsigned)g.X0h;
    const unsigned x1 = r % (unsigned)g.X1;  r /= (unsigned)g.X1;
    const unsigned x2 = r % (unsigned)g.X2;
    const unsigned x3 = r / (unsigned)g.X2;
    const int q = (int)((x1 + x2 + x3 + (unsigned)p) & 1u);   // x0 = 2 xh + q
    s.x0 = 2 * (int)xh + q; s.x1 = (int)x1; s.x2 = (int)x2; s.x3 = (int)x3;
    // mu = 0: the neighbour's parity bit is 1-q, so it shares xh or sits one pair over
    s.nbr[0] = q ? (((int)xh + 1 == g.X0h) ? cb - (g.X0h - 1) : cb + 1) : cb;
    s.nbr[4] = q ? cb : ((xh == 0) ? cb + (g.X0h - 1) : cb - 1);
    s.nbr[1] = ((int)x1 + 1 == g.X1) ? cb - (g.X1 - 1) * g.s1 : cb + g.s1;
    s.nbr[5] = (x1 == 0) ? cb + (g.X1 - 1) * g.s1 : cb - g.s1;
    s.nbr[2] = ((int)x2 + 1 == g.X2) ? cb - (g.X2 - 1) * g.s2 : cb + g.s2;
    s.nbr[6] = (x2 == 0) ? cb + (g.X2 - 1) * g.s2 : cb - g.s2;
    s.nbr[3] = ((int)x3 + 1 == g.X3) ? cb - (g.X3 - 1) * g.s3 : cb + g.s3;
    s.nbr[7] = (x3 == 0) ? cb + (g.X3 - 1) * g.s3 : cb - g.s3;
}

// det M_d(x) = +-1 for the gathered matrices (include/stag.h): forward d = mu has
// det = eta_mu(x) bc_mu(x); backward d = 4+mu has det(-W_mu(x-mu)^dag) = -eta_mu(x) bc_mu(x-mu)
// (eta_mu does not depend on x_mu).  eta_mu(x) = (-1)^(x0+..+x_{mu-1}); bc = -1 only on the
// mu = 3 link that leaves x3 = X3-1 (Q12).  Returned as a bit mask: bit d set
// means the sign is -1.
__device__ __forceinline__ unsigned det_sign_mask(const Geom &g, const Site &s)
{
    const unsigned e1 = (unsigned)s.x0 & 1u;
    const unsigned e2 = (unsigned)(s.x0 + s.x1) & 1u;
    const unsigned e3 = (unsigned)(s.x0 + s.x1 + s.x2) & 1u;
    const unsigned bf = (g.antiperiodic && s.x3 + g.t0 == g.X3g - 1) ? 1u : 0u;   // global time
    const unsigned bb = (g.antiperiodic && s.x3 + g.t0 == 0) ? 1u : 0u;
    unsigned m = 0;
    m |= 0u << 0;                 // eta_0 = +1
    m |= e1 << 1;
    m |= e2 << 2;
    m |= (e3 ^ bf) << 3;
    m |= 1u << 4;                 // -eta_0
    m |= (e1 ^ 1u) << 5;
    m |= (e2 ^ 1u) << 6;
    m |= (e3 ^ bb ^ 1u) << 7;
    return m;
}

// ---- reductions ---------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block; the result is valid in thread 0.  red must hold >= 32 doubles.
__device__ __forceinline__ double block_sum(double v, double *red)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    v = warp_sum(v);
    if (lane == 0) red[w] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    double t = (threadIdx.x < nw) ? red[threadIdx.x] : 0.0;
    if (w == 0) t = warp_sum(t);
    __syncthreads();
    return t;
}

// Device-resident solver scalars and control.  One per solve.  A solve
// carries nrhs <= MAX_RHS right-hand sides in lockstep: one Fig. 1 recurrence each (its own
// alpha, beta, delta), one shared iteration counter and one shared state, so that every hop
// reads the gauge field once for all of them.
constexpr int MAX_RHS = STAG_MAX_RHS;

struct CgCtrl {
    double delta[MAX_RHS];   // |r|^2 entering the iteration (delta_new of Fig. 1)
    double dAd[MAX_RHS];     // <d, A d>
    double alpha[MAX_RHS], beta[MAX_RHS];
    double maxr[MAX_RHS];    // max |r| since the last update (Q9) / |r| at the last update (mode 2)
    double tol2b[MAX_RHS];   // tol^2 |b|^2 : the stopping threshold on delta (Q6)
    double inner2[MAX_RHS];  // mode 2: inner stopping threshold on delta
    double bnorm2[MAX_RHS];
    double sum0[MAX_RHS];    // |b - A x|^2 of the last fp64 residual evaluation
    double sum1[MAX_RHS];    // the iterated |r|^2 of the last iteration
    double eps_in;
    int active[MAX_RHS];     // 1: this right-hand side is still iterating; 0: frozen (done)
    int iters[MAX_RHS];      // loop passes during which it was active (Q7)
    int state;               // CG_RUN ...
    int iter, maxiter;       // shared loop counter
    int mode;
    int n_updates;
    int nrhs;
    unsigned ticket[4];      // last-block tickets, one per reducing kernel role
    // written by the persistent iteration kernel (stag_persist.cuh) when it returns:
    int have_true;           // 1: the launch ended with a reliable update done IN the kernel, so sum0 is
                             //    |b - A x|^2 of the current x; 0: passes followed it (or none was done)
    int n_inkernel;          // reliable updates done in the kernel so far (each one fp64 application of A)
};
constexpr int CTRL_SLOT = 2048;   // bytes reserved for CgCtrl in the workspace
static_assert(sizeof(CgCtrl) <= CTRL_SLOT, "CgCtrl must fit its workspace slot");

// ---- T-slab exchange region header (stag_slab.cuh describes the protocol) ----------------------
constexpr size_t XCH_HDR = 1024;    // bytes of header in front of the halo buffers
constexpr size_t XCH_RED = 256;     // offset of the reduction slots inside the header area
struct XchHeader {
    unsigned long long flag_back;   // PEER-written: number of the last exchange pushed into my "back" halo
    unsigned long long flag_fwd;    // PEER-written: ... into my "fwd" halo
    // local only (never peer-written).  Kept in device memory, not in kernel arguments, so that a
    // captured CUDA graph of iterations can be replayed: every kernel reads the current number.
    unsigned long long epoch;       // exchanges I have started (face_push_kernel increments it)
    unsigned long long red_seq;     // global sums I have published
    unsigned ticket;                // last-block ticket of my face_push_kernel
    // watchdog of the acquire-waits: a wait that polls wait_limit times without seeing its flag gives
    // up, sets timed_out and lets the kernel finish on stale data, so a missing or mis-ordered peer
    // shows up as an error from the next host call instead of a GPU that spins for ever
    unsigned timed_out;
    unsigned long long wait_limit;  // polls (~1 us each); 0 = the default below
    // diagnostics (stag_slab_wait_stats): acquire-waits that did not find their flag set at once, and
    // the polls they spent; proof that a test really ran ranks concurrently
    unsigned long long waits_spun, polls_spent;
};
constexpr unsigned long long XCH_DEFAULT_WAIT_POLLS = 1ull << 23;     // roughly ten seconds
static_assert(sizeof(XchHeader) <= XCH_RED, "exchange header must fit its slot");
__host__ __device__ inline size_t xch_halo_offset(int s3, unsigned long long epoch, int dir)
{
    return XCH_HDR + ((size_t)((epoch & 1ull) * 2 + dir) * 3 * s3) * 16;
}

enum { CG_RUN = 0, CG_CONVERGED = 1, CG_UPDATE = 2, CG_MAXITER = 3, CG_BREAKDOWN = 4 };

}  // namespace stag
