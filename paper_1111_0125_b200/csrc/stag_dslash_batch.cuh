// stag_dslash_batch.cuh -- the fp32 hop for N = 2..4 right-hand sides sharing one pass over the links.
//
// Same mathematics, same per-right-hand-side arithmetic order as dslash_kernel (stag_dslash.cuh):
// out_k(x) = sum_d M_d(x) in_k(nbr_d(x)), eq. 2.5, 576 flop per site and right-hand side.
// What differs is how the loads are put in flight.  With N accumulators the generic kernel leaves
// ptxas too few registers to hoist the loads of the next group of directions above the arithmetic
// of the current one: ncu on 28^3 x 96, N = 4 shows issue slots 52 % busy, DRAM at 5.5 TB/s, and
// half of all warp samples stalled at five instructions, each the first use of a value loaded
// 2 - 25 instructions earlier (profiles/).  Here the pipeline is explicit and sized to fit 128
// registers:
//   * links: the packets of direction d+LD are loaded before direction d is multiplied (one
//     direction = K/2 packets rounded up: 3 for 12-real, 5 for 18-real where directions share a
//     packet, 2 for the 8-parameter form; LD = 2 directions ahead, 1 for 18-real);
//   * neighbour vectors: in UNITS of one pair of right-hand sides (three 16-byte gathers) or one
//     single right-hand side (three 8-byte gathers); the unit after the one being multiplied is
//     already in flight (double buffer of 12 registers, not of N x 6).
// Tried first and dropped: the whole link record copied global -> shared with per-thread cp.async
// (no register held in flight).  126 us against 108 us for N = 4 on 12-real links: the copies
// double the traffic through the L1 / shared-memory pipe that the 4 x 24 gathers already load, and
// queue in front of them; with an L2 cache hint the cp.async faulted ("illegal instruction").
#pragma once
#include "stag_dslash.cuh"

namespace stag {

// MINB: resident blocks per SM promised to ptxas; LD: how many directions ahead the links are loaded.
// Sweep on 28^3 x 96, 12-real links, us per hop for N = 2 / 3 / 4 (profiles/README.md, round 2):
//   LD 1: 80.0 / 94.5 / 103.6    LD 2: 80.2 / 94.3 / 102.7    LD 3: 80.4 / 90.4 / 104.3
//   3 blocks per SM (LD 2): 80.2 / 98.7 / 110.9               5 blocks per SM (LD 1): 78.1 / 94.4 / 112.8
// Measured slower and no longer in the tree (numbers in profiles/README.md, round 2): prefetching link
// tiles towards L2 ahead of the demand loads (prefetch.global.L2 or cp.async.bulk.prefetch.L2), the
// packed fp32 FMA (fma.rn.f32x2) for the two right-hand sides of a pair, and a shared-memory ring of
// link half-tiles filled by cp.async.bulk.
template <int NR, int N> struct BatchTune {
    static constexpr int MINB = 4;
    static constexpr int LD = (NR == 3) ? 1 : (N == 3 ? 3 : 2);
};

// NR, MODE, N, PAIRED as in dslash_kernel; float only; no halo.
template <int NR, int MODE, int N, bool PAIRED>
__global__ void __launch_bounds__(DSLASH_BLOCK, BatchTune<NR, N>::MINB)
dslash_batch_kernel(float2 *__restrict__ out, const float2 *__restrict__ in,
                    const float4 *__restrict__ links, const Geom g, const int p, const float a, const float cD,
                    const float2 *__restrict__ own, double *__restrict__ partials,
                    const CgCtrl *__restrict__ ctrl)
{
    static_assert(N >= 2 && N <= 4, "batch hop: 2..4 right-hand sides per pass");
    using C = float2;
    constexpr int K = link_slots(NR);          // complex numbers per direction
    constexpr int PPS = 8 * K / 2;             // 16-byte packets per site
    constexpr int PPD = (K + 2) / 2;           // packets that cover one direction (an odd K shares one with the next)
    constexpr int NU = PAIRED ? (N + 1) / 2 : N;   // gather units per direction
    constexpr int LD = BatchTune<NR, N>::LD;       // link prefetch depth in directions
    constexpr int NLB = LD + 1;                    // link buffers
    if (ctrl != nullptr && ctrl->state != CG_RUN) return;

    const int cb = blockIdx.x * DSLASH_BLOCK + threadIdx.x;
    const size_t rs = (size_t)3 * g.Vh_pad;
    double dot[N];
#pragma unroll
    for (int k = 0; k < N; ++k) dot[k] = 0.0;

    if (cb < g.Vh_pad) {
        const float4 *L = links + (size_t)(cb >> 5) * (size_t)(PPS * TILE) + (cb & 31);
        // packets first_d .. first_d + PPD - 1 hold direction d's numbers K*d .. K*d + K - 1
        auto load_links = [&](float4 (&pk)[PPD], const int d) {
            const int first = (K * d) >> 1, last = (K * d + K - 1) >> 1;
#pragma unroll
            for (int i = 0; i < PPD; ++i)
                if (first + i <= last) pk[i] = ld_stream(L + (first + i) * TILE);
        };
        float4 lk[NLB][PPD];
#pragma unroll
        for (int d = 0; d < LD; ++d) load_links(lk[d], d);

        // pad lanes (cb >= Vh) read zero links, so they produce zeros without a branch
        Site s;
        decode_site(g, p, cb < g.Vh ? cb : 0, s);
        unsigned neg = 0;
        if (NR != 3) neg = det_sign_mask(g, s);

        // unit u of direction nb: right-hand sides (2u, 2u+1) as one float4 per colour, or one single
        struct Unit { float4 q[3]; };
        auto gather_from = [&](const float2 *base, Unit &v, const int u, int nb) {
            if (PAIRED && 2 * u + 1 < N) {
#pragma unroll
                for (int c = 0; c < 3; ++c) v.q[c] = ld_keep_nc((const float4 *)(base + 2 * u * rs) + (size_t)c * g.Vh_pad + nb);
            } else {
                const int k = PAIRED ? N - 1 : u;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const float2 t = ld_keep_nc(base + k * rs + (size_t)c * g.Vh_pad + nb);
                    v.q[c] = make_float4(t.x, t.y, 0.f, 0.f);
                }
            }
        };
        auto gather = [&](Unit &v, const int u, int nb) { gather_from(in, v, u, nb); };

        C acc[N][3];
#pragma unroll
        for (int k = 0; k < N; ++k)
#pragma unroll
            for (int i = 0; i < 3; ++i) acc[k][i] = make_float2(0.f, 0.f);

        Unit vb[2];
        Unit ow[NU];       // the own-site vectors of the epilogue (MODE != HOP_PLAIN)
        gather(vb[0], 0, s.nbr[0]);
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            if (d + LD < 8) load_links(lk[(d + LD) % NLB], d + LD);
            // once no link is left to prefetch its registers carry the own-site vectors instead: loaded
            // after the last direction they cost every thread one exposed memory latency at its end
            if (MODE != HOP_PLAIN && d + LD == 8) {
#pragma unroll
                for (int u = 0; u < NU; ++u) gather_from(own, ow[u], u, cb);
            }
            C m[9];
            {
                const int first = (K * d) >> 1;
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    const int idx = K * d + k, i = (idx >> 1) - first;
                    const float4 q = lk[d % NLB][i];
                    m[k] = (idx & 1) ? make_float2(q.z, q.w) : make_float2(q.x, q.y);
                }
            }
            if (NR == 2) rebuild_row2<float>(m, (neg >> d) & 1u);
            if (NR == 1) rebuild_from8<float>(m, (neg >> d) & 1u);
#pragma unroll
            for (int u = 0; u < NU; ++u) {
                const int step = d * NU + u;                 // this unit sits in vb[step & 1]
                if (step + 1 < 8 * NU) gather(vb[(step + 1) & 1], (u + 1) % NU, s.nbr[(step + 1) / NU]);
                const Unit &v = vb[step & 1];
                if (PAIRED && 2 * u + 1 < N) {
#pragma unroll
                    for (int i = 0; i < 3; ++i)
#pragma unroll
                        for (int j = 0; j < 3; ++j) {
                            cfma(acc[2 * u][i], m[3 * i + j], make_float2(v.q[j].x, v.q[j].y));
                            cfma(acc[2 * u + 1][i], m[3 * i + j], make_float2(v.q[j].z, v.q[j].w));
                        }
                } else {
                    const int k = PAIRED ? N - 1 : u;
#pragma unroll
                    for (int i = 0; i < 3; ++i)
#pragma unroll
                        for (int j = 0; j < 3; ++j) cfma(acc[k][i], m[3 * i + j], make_float2(v.q[j].x, v.q[j].y));
                }
            }
        }

        if (NR == 1 && cb >= g.Vh) {
            // a rebuilt 8-parameter matrix is unitary, never zero: pad lanes are zeroed here
#pragma unroll
            for (int k = 0; k < N; ++k)
#pragma unroll
                for (int i = 0; i < 3; ++i) acc[k][i] = make_float2(0.f, 0.f);
        }

        // ---- epilogue: out = D in, or a*own - [cD] D in, with the <own,out> partial sums --------
        if constexpr (PAIRED) {
#pragma unroll
            for (int j = 0; j < N / 2; ++j)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    float4 *po = (float4 *)(out + 2 * j * rs) + (size_t)c * g.Vh_pad + cb;
                    if (MODE == HOP_PLAIN) {
                        st_keep(po, make_float4(acc[2 * j][c].x, acc[2 * j][c].y, acc[2 * j + 1][c].x, acc[2 * j + 1][c].y));
                    } else {
                        const float4 o = ow[j].q[c];
                        const float sc = (MODE == HOP_AXPBY) ? cD : 1.f;
                        float4 r;
                        r.x = fma(a, o.x, -sc * acc[2 * j][c].x);     r.y = fma(a, o.y, -sc * acc[2 * j][c].y);
                        r.z = fma(a, o.z, -sc * acc[2 * j + 1][c].x); r.w = fma(a, o.w, -sc * acc[2 * j + 1][c].y);
                        st_keep(po, r);
                        if (MODE == HOP_XPAY_DOT) {
                            dot[2 * j] += (double)o.x * (double)r.x + (double)o.y * (double)r.y;
                            dot[2 * j + 1] += (double)o.z * (double)r.z + (double)o.w * (double)r.w;
                        }
                    }
                }
        }
#pragma unroll
        for (int k = PAIRED ? (N / 2) * 2 : 0; k < N; ++k)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                C *po = out + k * rs + (size_t)c * g.Vh_pad + cb;
                if (MODE == HOP_PLAIN) {
                    st_keep(po, acc[k][c]);
                } else {
                    const float4 oq = ow[PAIRED ? NU - 1 : k].q[c];
                    const C o = make_float2(oq.x, oq.y);
                    const float sc = (MODE == HOP_AXPBY) ? cD : 1.f;
                    C r;
                    r.x = fma(a, o.x, -sc * acc[k][c].x);
                    r.y = fma(a, o.y, -sc * acc[k][c].y);
                    st_keep(po, r);
                    if (MODE == HOP_XPAY_DOT) dot[k] += (double)o.x * (double)r.x + (double)o.y * (double)r.y;
                }
            }
    }

    if (MODE == HOP_XPAY_DOT) {
        // one block barrier for all N sums (N calls of block_sum cost 2N barriers at the tail of a block
        // that lives ~6 us: the x3 hop with the dot took 114 us under ncu against 88 without).  The four
        // warp totals are added as block_sum's shuffle tree adds them: (w0 + w2) + (w1 + w3).
        constexpr int NW = DSLASH_BLOCK / 32;
        static_assert(NW == 4, "the partial-sum order below is written for four warps");
        __shared__ double red[N][NW];
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
        for (int k = 0; k < N; ++k) {
            const double t = warp_sum(dot[k]);
            if (lane == 0) red[k][w] = t;
        }
        __syncthreads();
        if (threadIdx.x < N) {
            const int k = threadIdx.x;
            partials[(size_t)k * gridDim.x + blockIdx.x] = (red[k][0] + red[k][2]) + (red[k][1] + red[k][3]);
        }
    }
}

}  // namespace stag
