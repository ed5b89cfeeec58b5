// stag_persist.cuh -- a chunk of CG iterations (Fig. 1's loop body) as ONE persistent kernel.
//
// The kernel-per-step iteration (stag_host_cg.cuh: xpay -> hop -> hop + dot -> update, a CUDA graph of
// 32 passes) pays four kernel boundaries per pass, about 12 us that do not shrink with the lattice;
// the T-slab iteration (stag_host_slab.cuh) pays six, about 34 us.  On 28^3 x 96 that is 7 % of the
// pass, on 16^3 x 32 or on one rank of an eight-way split it is most of it (DESIGN.md sections 14, 16).
// Here the blocks of one launch stay resident (cooperative launch, 148 SMs x BPS blocks) and walk
// through the four phases of every pass themselves, separated by a barrier among the blocks of the
// RANK GROUP instead of a kernel boundary:
//
//   P0  d = r + beta d                      [slab: the faces of d stored into the neighbours' halos]
//   --- barrier ---                         [slab: block 0 fences at system scope, sets the neighbours' flags]
//   P1  tmp = D_oe d                        [slab: boundary slices last, halo after an acquire-wait;
//   --- barrier ---                          the faces of tmp pushed, flags as above]
//   P2  q = m^2 d - D_eo tmp, <d,q> partials
//   --- barrier ---   every block adds the partials in index order   [slab: publish, gather over ranks]
//   P3  alpha; y += alpha d; r -= alpha q; |r|^2 partials
//   --- barrier ---   every block adds them, runs the scalar step on its own copy of the scalars
//   [mode 3, on the trigger of P:L97: x += y, y = 0 | barrier | tmp = D_oe x (fp64) | barrier |
//    r = b - (m^2 x - D_eo tmp), fp32 copy, |r|^2 | barrier | sum, beta from the corrected residual]
//
// Scalars are REPLICATED: every block carries delta, beta, maxr, the counters and the state in shared
// memory and evolves them from the same sums in the same order, so no block ever reads a scalar
// another block wrote inside the loop; block 0 stores them back to CgCtrl when the launch ends.
// Sites are dealt to warps (one 32-site link tile per warp per trip, warp w of the group takes tiles
// w, w + W, ...), vector packets to threads, both grid-stride over the group.  Per site the hop is
// hop_site (stag_dslash.cuh): the same arithmetic in the same order as dslash_kernel.  Vectors written
// in one phase and read in the next go through coherent loads (the barrier's acquire invalidates L1);
// only the links, constant for the launch, use the non-coherent path.
//
// A launch carries one rank group per rank in IterArgs: a real run has one (the whole grid); the
// single-GPU emulation of a multi-GPU run puts ALL ranks into one cooperative launch, each rank its
// own slice of the grid with its own barrier, so the ranks run concurrently by construction -- every
// block is resident -- and wait for each other only through the exchange regions, exactly as processes
// on different GPUs do (B200_PROFILING.md: ranks that wait on one another must not be separate launches).
#pragma once
#include "stag_blas.cuh"
#include "stag_dslash.cuh"
#include "stag_slab.cuh"

namespace stag {

#ifndef STAG_PERSIST_THREADS
#define STAG_PERSIST_THREADS 256
#endif
constexpr int PERSIST_THREADS = STAG_PERSIST_THREADS;

// -DSTAG_PERSIST_TIMING: block 0 of rank group 0 stamps %globaltimer after every phase and barrier of
// pass 20; the host prints the differences after the launch (profiles/README.md, round 2).  Off in
// the product build.
#ifdef STAG_PERSIST_TIMING
__device__ unsigned long long g_persist_stamps[16];
__device__ __forceinline__ unsigned long long persist_now()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define PSTAMP(k) do { if (blockIdx.x == 0 && threadIdx.x == 0 && pass == 20) g_persist_stamps[k] = persist_now(); } while (0)
#else
#define PSTAMP(k) do { } while (0)
#endif

// How many blocks per SM the launch bounds promise ptxas (registers per thread = 65536 / (256 * BPS)).
template <typename T, int NR> struct PersistTune { static constexpr int BPS = 512 / PERSIST_THREADS; };

// What the reliable + group-wise update of section 3.2 (step S6) needs when it is done
// INSIDE the kernel (fp32 iteration, mode 3): links_even == null leaves it to the host as before.
struct IterUpdate {
    double *x;                               // the fp64 solution x += y goes into
    const double *b;                         // the right-hand side (pad lanes read as zero)
    double *tmp;                             // odd-site scratch of A x in fp64
    const double2 *links_even, *links_odd;   // fp64, 18-real gathered fields
    double m2;
};

template <typename T> struct IterRank {
    T *y, *r, *d, *q, *tmp;                  // flat spinors, 6*Vh_pad reals; y = x itself in mode 0
    const pkt_t<T> *links_even, *links_odd;  // gathered fields of the even / odd OUTPUT sites
    Geom g;
    CgCtrl *ctrl;
    double *partials;                        // 2 * nblocks doubles
    unsigned *bar;                           // arrival counter of the group's barrier; 0 at launch (the host zeroes it)
    T m2;
    int block0, nblocks;                     // this rank's slice of the grid
    // T-slab only (xch == null: a whole lattice, periodic wrap inside decode_site)
    char *xch, *peer_fwd, *peer_bwd;
    char *const *peers;
    int nranks, myrank;
    IterUpdate up;
};
template <typename T> struct IterArgs {
    IterRank<T> rk[MAX_RANKS];
    int nlocal;                              // rank groups in this launch
    int max_iters;                           // passes of the loop at most (fewer when the state leaves CG_RUN)
};

struct IterScalars {
    double delta, beta, maxr, tol2b, inner2, eps_in, dAd, alpha, sum1, sum0;
    int state, iter, maxiter, mode, iters, active, n_updates, have_true, n_inkernel;
};

// Barrier among the nb blocks of one rank group: a monotonic arrival counter, zeroed by the host
// before the launch.  Barrier number k (k = 1, 2, ...) is passed once the counter shows k*nb: one
// fire-and-forget release-add per block, then acquire-polls -- no returning atomic, no reset, no
// generation word, so the critical path is one L2 write plus one L2 read after the last arrival.
// hdr != null (slab): the spin is bounded by the slab's watchdog like every other wait; a timeout
// marks the slab dead and returns false.
__device__ __forceinline__ bool group_barrier(unsigned *bar, unsigned target, XchHeader *hdr)
{
    __shared__ bool ok;
    __syncthreads();
    if (threadIdx.x == 0) {
        ok = true;
        // release at gpu scope: cumulative over the block's writes (ordered before it by the block barrier)
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" :: "l"(bar) : "memory");
        unsigned v;
        unsigned long long polls = 0, limit = 0;
        if (hdr) { limit = __ldcg(&hdr->wait_limit); if (limit == 0) limit = XCH_DEFAULT_WAIT_POLLS; limit *= 8; }
        for (;;) {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
            if (v >= target) break;
            if (hdr && ++polls >= limit) { *(volatile unsigned *)&hdr->timed_out = 1u; ok = false; break; }
        }
    }
    __syncthreads();
    return ok;
}

// The scalar step of one pass for one right-hand side on a block's own copy: cg_iteration_epilogue
// (stag_blas.cuh) restated on IterScalars.  dn = the new |r|^2.
__device__ __forceinline__ void iter_epilogue_local(IterScalars &S, const double dn)
{
    const int it = S.iter + 1;
    S.iter = it;
    S.iters += 1;
    S.sum1 = dn;
    S.have_true = 0;
    bool breakdown = false, trigger = false, conv = false;
    if (!(S.dAd > 0.0) || !(dn == dn)) breakdown = true;
    else if (S.mode == STAG_CG_RELIABLE) {
        const double rn = sqrt(dn);
        if (dn <= S.tol2b || rn < S.eps_in * S.maxr) trigger = true;       // P:L97, Q11
        else S.maxr = fmax(S.maxr, rn);                                    // Q9
    } else if (S.mode == STAG_CG_DEFECT) {
        conv = dn <= S.inner2;                                             // Fig. 2 inner
    } else {
        conv = dn <= S.tol2b;                                              // Fig. 1
    }
    int st = CG_RUN;
    if (breakdown) st = CG_BREAKDOWN;
    else if (trigger) st = CG_UPDATE;
    else {
        S.beta = dn / S.delta;
        S.delta = dn;
        if (conv) { S.active = 0; st = CG_CONVERGED; }
    }
    if (st == CG_RUN && it >= S.maxiter) st = CG_MAXITER;
    S.state = st;
}

// Tiles are dealt to the group's warps statically (warp w takes tiles w, w + W, ...).  A dynamic deal
// from one atomic counter was tried to trim the 4-8 us of stragglers at the barrier after each hop on
// 28^3 x 96 (14 trips for some warps, 13 for others; SMs of unequal speed): 33 k same-address atomics
// per phase serialise in L2 and the hop went from 62 to 96 us; chunks of 1-4 tiles per ticket, drawn one
// chunk ahead (8 k atomics per phase), left the hop at 66-71 us against 62-67 and cost 28^3 x 12 six
// microseconds per pass (profiles/README.md, round 2).  The stragglers are not the deal's.
// LRES: the links of both parities and the five vectors fit L2 together (the host decides): the link
// packets are then loaded with the keep policy and every pass after the first reads them from L2.
// The scalar step after a reliable update done in the kernel: residual_epilogue<RES_UPDATE>
// (stag_blas.cuh) restated on IterScalars.  dn = |b - A x|^2 in fp64 (Q9, Q10, Q11).
__device__ __forceinline__ void update_epilogue_local(IterScalars &S, const double dn)
{
    S.sum0 = dn;
    S.have_true = 1;
    S.n_updates += 1;
    S.n_inkernel += 1;
    const bool bad = !(dn == dn);
    if (!bad && S.active) {
        S.maxr = sqrt(dn);                                                 // Q9
        if (dn <= S.tol2b) S.active = 0;
        else { S.beta = dn / S.delta; S.delta = dn; }                      // Q10
    }
    int st = S.active ? CG_RUN : CG_CONVERGED;
    if (bad) st = CG_BREAKDOWN;
    else if (S.active && S.iter >= S.maxiter) st = CG_MAXITER;
    S.state = st;
}

// The scalar step after an outer step of Fig. 2 (mode 2) done in the kernel: residual_epilogue<RES_INIT>
// restated on IterScalars -- a fresh inner CG from the fp64 residual (beta = 0 makes the next P0 d = r).
__device__ __forceinline__ void outer_epilogue_local(IterScalars &S, const double dn)
{
    S.sum0 = dn;
    S.have_true = 1;
    S.n_inkernel += 1;
    const bool bad = !(dn == dn);
    if (!bad) {
        S.delta = dn;
        S.beta = 0.0;
        S.maxr = sqrt(dn);
        S.inner2 = fmax(S.eps_in * S.eps_in * dn, S.tol2b);               // Fig. 2, Q8
        S.active = dn > S.tol2b;
    }
    int st = S.active ? CG_RUN : CG_CONVERGED;
    if (bad) st = CG_BREAKDOWN;
    else if (S.active && S.iter >= S.maxiter) st = CG_MAXITER;
    S.state = st;
}

template <typename T, int NR, bool SLAB, bool LRES>
__global__ void __launch_bounds__(PERSIST_THREADS, PersistTune<T, NR>::BPS)
cg_iter_persistent_kernel(const __grid_constant__ IterArgs<T> A)
{
    using C = cplx_t<T>;
    using V = typename Vec4<T>::type;
    constexpr int N = Vec4<T>::N;
    constexpr int CPK = N / 2;                      // complex numbers per 16-byte packet
    constexpr int PT = PERSIST_THREADS;

    int rk = 0;
    while (rk + 1 < A.nlocal && (int)blockIdx.x >= A.rk[rk + 1].block0) ++rk;
    const IterRank<T> &R = A.rk[rk];
    const Geom &g = R.g;
    const int lb = (int)blockIdx.x - R.block0, nb = R.nblocks;
    XchHeader *hdr = SLAB ? (XchHeader *)R.xch : nullptr;
    if (SLAB && slab_dead(R.xch)) return;           // uniform over the group: the mark predates the launch

    __shared__ IterScalars S;
    __shared__ double red[32];
    __shared__ double s_sum;
    __shared__ bool s_ok;
    unsigned long long epoch = 0, seq = 0;
    unsigned bar_target = 0;                        // arrivals that complete the next barrier
    if constexpr (SLAB) { epoch = __ldcg(&hdr->epoch); seq = __ldcg(&hdr->red_seq); }
    if (threadIdx.x == 0) {
        const CgCtrl *c = R.ctrl;
        S.delta = __ldcg(&c->delta[0]); S.beta = __ldcg(&c->beta[0]); S.maxr = __ldcg(&c->maxr[0]);
        S.tol2b = __ldcg(&c->tol2b[0]); S.inner2 = __ldcg(&c->inner2[0]); S.eps_in = __ldcg(&c->eps_in);
        S.dAd = __ldcg(&c->dAd[0]); S.alpha = __ldcg(&c->alpha[0]); S.sum1 = __ldcg(&c->sum1[0]);
        S.state = __ldcg(&c->state); S.iter = __ldcg(&c->iter); S.maxiter = __ldcg(&c->maxiter);
        S.mode = __ldcg(&c->mode); S.iters = __ldcg(&c->iters[0]); S.active = __ldcg(&c->active[0]);
        S.sum0 = __ldcg(&c->sum0[0]); S.n_updates = __ldcg(&c->n_updates);
        S.have_true = 0; S.n_inkernel = __ldcg(&c->n_inkernel);
        if (!S.active && S.state == CG_RUN) S.state = CG_CONVERGED;
    }
    __syncthreads();

    const long n = 6L * g.Vh_pad, nv = n / N;
    const long tid = (long)lb * PT + threadIdx.x, nthreads = (long)nb * PT;
    const int lane = threadIdx.x & 31;
    const int warp_g = (int)(tid >> 5), nwarps = (int)(nthreads >> 5);
    const int ntiles = g.Vh_pad / TILE;
    V *dv = reinterpret_cast<V *>(R.d);
    const V *rv = reinterpret_cast<const V *>(R.r);
    double *partA = R.partials, *partB = R.partials + nb;
    C *d_c = reinterpret_cast<C *>(R.d), *tmp_c = reinterpret_cast<C *>(R.tmp), *q_c = reinterpret_cast<C *>(R.q);

    // release the neighbours' flags for the exchange whose stores the last barrier ordered (block 0, one thread)
    auto raise_flags = [&](unsigned long long e) {
        if (lb == 0 && threadIdx.x == 0) {
            raise_halo_flags(R.peer_fwd, R.peer_bwd, e);   // cumulative over every block's peer stores (they precede the barrier)
        }
    };
    // local fixed-order total of this group's partials -> (slab) sum over ranks, the same bits everywhere
    auto total_over_ranks = [&](const double *part, double *out) -> bool {
        double t = block_total_fixed(part, nb, red);
        if constexpr (SLAB) {
            ++seq;
            if (threadIdx.x < 32) {               // warp 0: lane r talks to rank r
                if (lb == 0) publish_total(R.peers, R.nranks, R.myrank, seq, t);
                bool ok;
                const double tot = gather_total(R.xch, R.nranks, seq, &ok);
                if (threadIdx.x == 0) { s_sum = tot; s_ok = ok; }
            }
            __syncthreads();
            if (!s_ok) return false;
            t = s_sum;
            __syncthreads();
        }
        *out = t;
        return true;
    };

    for (int pass = 0; pass < A.max_iters && S.state == CG_RUN; ++pass) {
        // ---- P0: d = r + beta d (eq. 3.1 after an update) ------------------------------
        PSTAMP(0);
        {
            const T beta = (T)S.beta;
            V *fwd_back = nullptr, *bwd_fwd = nullptr;
            if constexpr (SLAB) {
                fwd_back = (V *)(R.peer_fwd + xch_halo_offset(g.s3, epoch + 1, 0));
                bwd_fwd = (V *)(R.peer_bwd + xch_halo_offset(g.s3, epoch + 1, 1));
            }
            for (long i = tid; i < nv; i += nthreads) {
                T a[N], b[N];
                unpack<T>(ld_keep(rv + i), a);
                if (beta == (T)0) {
#pragma unroll
                    for (int j = 0; j < N; ++j) b[j] = a[j];
                } else {
                    unpack<T>(ld_keep(dv + i), b);
#pragma unroll
                    for (int j = 0; j < N; ++j) b[j] = fma(beta, b[j], a[j]);
                }
                const V pk = pack(b);
                st_keep(dv + i, pk);
                if constexpr (SLAB) {
                    const long ci = i * CPK;
                    const int c = (ci >= 2L * g.Vh_pad) ? 2 : (ci >= g.Vh_pad ? 1 : 0);
                    const int cb = (int)(ci - (long)c * g.Vh_pad);
                    if (cb < g.s3) bwd_fwd[((long)c * g.s3 + cb) / CPK] = pk;
                    else if (cb >= g.Vh - g.s3 && cb < g.Vh) fwd_back[((long)c * g.s3 + (cb - (g.Vh - g.s3))) / CPK] = pk;
                }
            }
        }
        PSTAMP(1);
        if (!group_barrier(R.bar, bar_target += (unsigned)nb, hdr)) return;
        if constexpr (SLAB) { if (slab_dead(R.xch)) return; ++epoch; raise_flags(epoch); }
        PSTAMP(2);

        // ---- P1: tmp = D_oe d (eq. 2.5 on the odd sites) ------------------------------------
        for (int t = warp_g; t < ntiles; t += nwarps) {
            int cb = t * TILE + lane;
            if constexpr (SLAB) { cb += g.s3; if (cb >= g.Vh_pad) cb -= g.Vh_pad; }     // boundary slices last
            Site s;
            decode_site(g, 1, cb < g.Vh ? cb : 0, s);
            unsigned neg = 0;
            if (NR != 3) neg = det_sign_mask(g, s);
            C acc[3];
            const bool fresh = hop_site<T, NR, SLAB, false, LRES>(acc, d_c, R.links_odd, g, cb, s, neg, R.xch, [=]() { return epoch; });
#pragma unroll
            for (int c = 0; c < 3; ++c) st_keep(tmp_c + (size_t)c * g.Vh_pad + cb, acc[c]);
            if constexpr (SLAB) {
                if (fresh && cb < g.Vh && (s.x3 == 0 || s.x3 == g.X3 - 1)) {      // a timed-out wait publishes nothing
                    C *dst = (s.x3 == 0)
                        ? (C *)(R.peer_bwd + xch_halo_offset(g.s3, epoch + 1, 1)) + cb
                        : (C *)(R.peer_fwd + xch_halo_offset(g.s3, epoch + 1, 0)) + (cb - (g.Vh - g.s3));
#pragma unroll
                    for (int c = 0; c < 3; ++c) dst[(size_t)c * g.s3] = acc[c];
                }
            }
        }
        PSTAMP(3);
        if (!group_barrier(R.bar, bar_target += (unsigned)nb, hdr)) return;
        if constexpr (SLAB) { if (slab_dead(R.xch)) return; ++epoch; raise_flags(epoch); }
        PSTAMP(4);

        // ---- P2: q = m^2 d - D_eo tmp (eq. 2.3), <d,q> in fp64 -------------------------
        double dot = 0.0;
        for (int t = warp_g; t < ntiles; t += nwarps) {
            int cb = t * TILE + lane;
            if constexpr (SLAB) { cb += g.s3; if (cb >= g.Vh_pad) cb -= g.Vh_pad; }
            Site s;
            decode_site(g, 0, cb < g.Vh ? cb : 0, s);
            unsigned neg = 0;
            if (NR != 3) neg = det_sign_mask(g, s);
            C acc[3];
            hop_site<T, NR, SLAB, false, LRES>(acc, tmp_c, R.links_even, g, cb, s, neg, R.xch, [=]() { return epoch; });
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const C o = ld_keep(d_c + (size_t)c * g.Vh_pad + cb);
                C v;
                v.x = fma(R.m2, o.x, -acc[c].x);
                v.y = fma(R.m2, o.y, -acc[c].y);
                st_keep(q_c + (size_t)c * g.Vh_pad + cb, v);
                dot += (double)o.x * (double)v.x + (double)o.y * (double)v.y;
            }
        }
        {
            const double bs = block_sum(dot, red);
            if (threadIdx.x == 0) partA[lb] = bs;
        }
        PSTAMP(5);
        if (!group_barrier(R.bar, bar_target += (unsigned)nb, hdr)) return;
        if constexpr (SLAB) { if (slab_dead(R.xch)) return; }
        PSTAMP(6);
        double dAd;
        if (!total_over_ranks(partA, &dAd)) return;
        PSTAMP(7);

        // ---- P3: alpha = delta / <d,Ad>; y += alpha d; r -= alpha q; |r|^2 ----
        const double alpha_d = (dAd > 0.0) ? S.delta / dAd : 0.0;
        double s2 = 0.0;
        {
            const T alpha = (T)alpha_d;
            V *yv = reinterpret_cast<V *>(R.y);
            V *rw = reinterpret_cast<V *>(R.r);
            const V *qv = reinterpret_cast<const V *>(R.q);
            for (long i = tid; i < nv; i += nthreads) {
                T yy[N], rr[N], dd[N], qq[N];
                unpack<T>(ld_pass(yv + i), yy);
                unpack<T>(ld_keep(rw + i), rr);
                unpack<T>(ld_keep(dv + i), dd);
                unpack<T>(ld_keep(qv + i), qq);
#pragma unroll
                for (int j = 0; j < N; ++j) {
                    yy[j] = fma(alpha, dd[j], yy[j]);
                    rr[j] = fma(-alpha, qq[j], rr[j]);
                    s2 += (double)rr[j] * (double)rr[j];
                }
                st_pass(yv + i, pack(yy));
                st_keep(rw + i, pack(rr));
            }
        }
        {
            const double bs = block_sum(s2, red);
            if (threadIdx.x == 0) partB[lb] = bs;
        }
        PSTAMP(8);
        if (!group_barrier(R.bar, bar_target += (unsigned)nb, hdr)) return;
        if constexpr (SLAB) { if (slab_dead(R.xch)) return; }
        PSTAMP(9);
        double dn;
        if (!total_over_ranks(partB, &dn)) return;
        PSTAMP(10);
        if (threadIdx.x == 0) {
            S.dAd = dAd;
            S.alpha = alpha_d;
            iter_epilogue_local(S, dn);
        }
        __syncthreads();

        // ---- S6 in the kernel: x += y, y = 0 (group-wise); r = b - A x in fp64, its fp32 copy and
        // |r|^2 (reliable); beta from the corrected residual with d kept (eq. 3.1, Q10).  The same
        // three phases serve the outer step of Fig. 2 (mode 2), which restarts from d = r ---------
        if constexpr (sizeof(T) == 4) {
            const bool outer = S.mode == STAG_CG_DEFECT && S.state == CG_CONVERGED;      // Fig. 2: the inner CG met its target
            if ((S.state == CG_UPDATE || outer) && R.up.links_even != nullptr) {
                const IterUpdate &U = R.up;
                using D2 = double2;
                D2 *x_c = reinterpret_cast<D2 *>(U.x), *t_c = reinterpret_cast<D2 *>(U.tmp);
                {   // U0: x += y ; y = 0 -- one float4 of y = two complex numbers of x   [slab: the faces of x pushed]
                    float4 *yv = reinterpret_cast<float4 *>(R.y);
                    for (long i = tid; i < nv; i += nthreads) {
                        const float4 yy = ld_pass(yv + i);
                        D2 a = x_c[2 * i], b2 = x_c[2 * i + 1];
                        a.x += (double)yy.x; a.y += (double)yy.y; b2.x += (double)yy.z; b2.y += (double)yy.w;
                        x_c[2 * i] = a; x_c[2 * i + 1] = b2;
                        st_pass(yv + i, make_float4(0.f, 0.f, 0.f, 0.f));
                        if constexpr (SLAB) {
                            const long ci = 2 * i;
                            const int c = (ci >= 2L * g.Vh_pad) ? 2 : (ci >= g.Vh_pad ? 1 : 0);
                            const int cb = (int)(ci - (long)c * g.Vh_pad);
                            if (cb < g.s3) {
                                D2 *dst = (D2 *)(R.peer_bwd + xch_halo_offset(g.s3, epoch + 1, 1)) + (long)c * g.s3 + cb;
                                dst[0] = a; dst[1] = b2;
                            } else if (cb >= g.Vh - g.s3 && cb < g.Vh) {
                                D2 *dst = (D2 *)(R.peer_fwd + xch_halo_offset(g.s3, epoch + 1, 0)) + (long)c * g.s3 + (cb - (g.Vh - g.s3));
                                dst[0] = a; dst[1] = b2;
                            }
                        }
                    }
                }
                if (!group_barrier(R.bar, bar_target += (unsigned)nb, hdr)) return;
                if constexpr (SLAB) { if (slab_dead(R.xch)) return; ++epoch; raise_flags(epoch); }
                // U1: tmp = D_oe x in fp64 on the 18-real links
                for (int t = warp_g; t < ntiles; t += nwarps) {
                    int cb = t * TILE + lane;
                    if constexpr (SLAB) { cb += g.s3; if (cb >= g.Vh_pad) cb -= g.Vh_pad; }
                    Site s;
                    decode_site(g, 1, cb < g.Vh ? cb : 0, s);
                    D2 acc[3];
                    const bool fresh = hop_site<double, 3, SLAB, false, false>(acc, x_c, U.links_odd, g, cb, s, 0u, R.xch, [=]() { return epoch; });
#pragma unroll
                    for (int c = 0; c < 3; ++c) t_c[(size_t)c * g.Vh_pad + cb] = acc[c];
                    if constexpr (SLAB) {
                        if (fresh && cb < g.Vh && (s.x3 == 0 || s.x3 == g.X3 - 1)) {
                            D2 *dst = (s.x3 == 0)
                                ? (D2 *)(R.peer_bwd + xch_halo_offset(g.s3, epoch + 1, 1)) + cb
                                : (D2 *)(R.peer_fwd + xch_halo_offset(g.s3, epoch + 1, 0)) + (cb - (g.Vh - g.s3));
#pragma unroll
                            for (int c = 0; c < 3; ++c) dst[(size_t)c * g.s3] = acc[c];
                        }
                    }
                }
                if (!group_barrier(R.bar, bar_target += (unsigned)nb, hdr)) return;
                if constexpr (SLAB) { if (slab_dead(R.xch)) return; ++epoch; raise_flags(epoch); }
                // U2: r = b - (m^2 x - D_eo tmp), its fp32 copy, |r|^2
                double s3sum = 0.0;
                const D2 *b_c = reinterpret_cast<const D2 *>(U.b);
                float2 *r_c = reinterpret_cast<float2 *>(R.r);
                for (int t = warp_g; t < ntiles; t += nwarps) {
                    int cb = t * TILE + lane;
                    if constexpr (SLAB) { cb += g.s3; if (cb >= g.Vh_pad) cb -= g.Vh_pad; }
                    Site s;
                    decode_site(g, 0, cb < g.Vh ? cb : 0, s);
                    D2 acc[3];
                    hop_site<double, 3, SLAB, false, false>(acc, t_c, U.links_even, g, cb, s, 0u, R.xch, [=]() { return epoch; });
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const D2 o = x_c[(size_t)c * g.Vh_pad + cb];
                        D2 bb = make_double2(0.0, 0.0);
                        if (cb < g.Vh) bb = b_c[(size_t)c * g.Vh_pad + cb];       // b's pad lanes count as zero
                        const double vx = bb.x - fma(U.m2, o.x, -acc[c].x), vy = bb.y - fma(U.m2, o.y, -acc[c].y);
                        r_c[(size_t)c * g.Vh_pad + cb] = make_float2((float)vx, (float)vy);
                        s3sum += vx * vx + vy * vy;
                    }
                }
                {
                    const double bs = block_sum(s3sum, red);
                    if (threadIdx.x == 0) partA[lb] = bs;
                }
                if (!group_barrier(R.bar, bar_target += (unsigned)nb, hdr)) return;
                if constexpr (SLAB) { if (slab_dead(R.xch)) return; }
                double rn2;
                if (!total_over_ranks(partA, &rn2)) return;
                if (threadIdx.x == 0) {
                    if (outer) outer_epilogue_local(S, rn2);
                    else update_epilogue_local(S, rn2);
                }
                __syncthreads();
            }
        }
    }

    if (lb == 0 && threadIdx.x == 0) {
        CgCtrl *c = R.ctrl;
        c->delta[0] = S.delta; c->beta[0] = S.beta; c->maxr[0] = S.maxr; c->inner2[0] = S.inner2;
        c->dAd[0] = S.dAd; c->alpha[0] = S.alpha; c->sum1[0] = S.sum1;
        c->iter = S.iter; c->iters[0] = S.iters; c->active[0] = S.active;
        c->sum0[0] = S.sum0; c->n_updates = S.n_updates; c->have_true = S.have_true; c->n_inkernel = S.n_inkernel;
        c->state = S.state;
        if constexpr (SLAB) { hdr->epoch = epoch; hdr->red_seq = seq; }
    }
}

}  // namespace stag
