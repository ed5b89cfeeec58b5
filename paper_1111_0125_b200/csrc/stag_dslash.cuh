// stag_dslash.cuh -- the staggered Dslash parity hop (eq. 2.5) on sm_100a.
//
// One thread per output site, one warp per 32-site link tile.  Per site the kernel
// streams eight link matrices from the gathered, tiled field (include/stag.h,
// stag_links_create) with evict-first loads -- the gauge field is read exactly once per hop
// and must not push the spinors out of L2 -- gathers the eight neighbour colour vectors
// through L1/L2 (each is needed by eight output sites, the farthest reuse one time slice
// away), and accumulates eight 3x3 complex matrix-vector products: 8*(66+6) = 576 flop
// (P:L62).  HBM-bound: 8*18 + 6 + 6 reals per site compulsory.
#pragma once
#include "stag_common.cuh"

namespace stag {

constexpr int DSLASH_BLOCK = 128;

enum { HOP_PLAIN = 0,   // out = D in
       HOP_XPAY = 1,    // out = m2*own - D in                       (second hop of A, eq. 2.3)
       HOP_XPAY_DOT = 2 // same, plus <own,out> -> ctrl->dAd, alpha  (Fig. 1)
};

// streaming (read-once) and cached loads of one complex number
template <typename C> __device__ __forceinline__ C ld_stream(const C *p) { return __ldcs(p); }
template <typename C> __device__ __forceinline__ C ld_cached(const C *p) { return __ldg(p); }

// Row 2 of a matrix whose rows 0,1 are m[0..5] and whose determinant is +-1:
// row2 = s * conj(row0 x row1)  (Q12).
template <typename T>
__device__ __forceinline__ void rebuild_row2(cplx_t<T> *m, bool neg)
{
    const T s = neg ? (T)-1 : (T)1;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int a = (j + 1) % 3, b = (j + 2) % 3;
        // c = r0[a]*r1[b] - r0[b]*r1[a]
        T re = m[a].x * m[3 + b].x - m[a].y * m[3 + b].y - (m[b].x * m[3 + a].x - m[b].y * m[3 + a].y);
        T im = m[a].x * m[3 + b].y + m[a].y * m[3 + b].x - (m[b].x * m[3 + a].y + m[b].y * m[3 + a].x);
        m[6 + j].x = s * re;
        m[6 + j].y = -s * im;
    }
}

// T: float or double.  NR: rows of each link held in memory (3 = 18-real, 2 = 12-real).
// links: the gathered field of the OUTPUT parity, L[tile][d][k][lane].
// in:  the other parity's spinor planes; out / own: this parity's.
template <typename T, int NR, int MODE>
__global__ void __launch_bounds__(DSLASH_BLOCK)
dslash_kernel(cplx_t<T> *__restrict__ out, const cplx_t<T> *__restrict__ in,
              const cplx_t<T> *__restrict__ links, const Geom g, const int p, const T m2,
              const cplx_t<T> *__restrict__ own, double *__restrict__ partials,
              CgCtrl *__restrict__ ctrl)
{
    using C = cplx_t<T>;
    constexpr int K = 3 * NR;
    if (ctrl != nullptr && ctrl->state != CG_RUN) return;

    const int cb = blockIdx.x * DSLASH_BLOCK + threadIdx.x;
    double dot = 0.0;
    if (cb < g.Vh_pad) {
        // pad lanes (cb >= Vh) read zero links, so they produce zeros without a branch
        Site s;
        decode_site(g, p, cb < g.Vh ? cb : 0, s);
        const C *L = links + (size_t)(cb >> 5) * (size_t)(8 * K * TILE) + (cb & 31);

        C v[8][3];
#pragma unroll
        for (int d = 0; d < 8; ++d)
#pragma unroll
            for (int c = 0; c < 3; ++c) v[d][c] = ld_cached(in + (size_t)c * g.Vh_pad + s.nbr[d]);

        unsigned neg = 0;
        if (NR == 2) neg = det_sign_mask(g, s);

        C acc[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) acc[i] = mk<T>(0, 0);

#pragma unroll
        for (int d = 0; d < 8; ++d) {
            C m[9];
#pragma unroll
            for (int k = 0; k < K; ++k) m[k] = ld_stream(L + (d * K + k) * TILE);
            if (NR == 2) rebuild_row2<T>(m, (neg >> d) & 1u);
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = 0; j < 3; ++j) cfma(acc[i], m[3 * i + j], v[d][j]);
        }

        if (MODE == HOP_PLAIN) {
#pragma unroll
            for (int c = 0; c < 3; ++c) out[(size_t)c * g.Vh_pad + cb] = acc[c];
        } else {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const C o = own[(size_t)c * g.Vh_pad + cb];
                C r;
                r.x = fma(m2, o.x, -acc[c].x);
                r.y = fma(m2, o.y, -acc[c].y);
                out[(size_t)c * g.Vh_pad + cb] = r;
                if (MODE == HOP_XPAY_DOT)
                    dot += (double)o.x * (double)r.x + (double)o.y * (double)r.y;
            }
        }
    }

    if (MODE == HOP_XPAY_DOT) {
        __shared__ double red[32];
        __shared__ bool last;
        double bs = block_sum(dot, red);
        if (threadIdx.x == 0) {
            partials[blockIdx.x] = bs;
            __threadfence();
            last = (atomicAdd(&ctrl->ticket[0], 1u) == gridDim.x - 1);
        }
        __syncthreads();
        if (last) {
            // fixed-order second stage: the value does not depend on block scheduling
            double t = 0.0;
            for (unsigned i = threadIdx.x; i < gridDim.x; i += DSLASH_BLOCK) t += __ldcg(partials + i);
            t = block_sum(t, red);
            if (threadIdx.x == 0) {
                ctrl->dAd = t;
                if (t > 0.0) ctrl->alpha = ctrl->delta / t;        // alpha = delta_new / d^dag A d
                else ctrl->state = CG_BREAKDOWN;                   // also catches NaN
                ctrl->ticket[0] = 0;
            }
        }
    }
}

}  // namespace stag
