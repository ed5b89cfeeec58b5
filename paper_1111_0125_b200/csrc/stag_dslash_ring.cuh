// stag_dslash_ring.cuh -- the paired fp32 batch hop on 12-real links with the link tiles staged in shared
// memory by an asynchronous ring (cp.async.bulk + mbarrier), EXPERIMENT (STAG_BATCH_RING=1 in the environment).
//
// Why: dslash_batch_kernel (stag_dslash_batch.cuh) spends half of its warp samples waiting for loads with
// every register in use (profiles/r2_batch_fp32r12x4_ncu_full.md).  Here the link bytes in flight hold
// no register: a warp's link tile (8 directions x 6 complex x 32 sites = 12 KB, contiguous in the
// gathered field) is brought in as two halves of 6 KB (directions 0-3, 4-7) by one bulk copy each, issued
// by lane 0 and completed on an mbarrier; the blocks are persistent (148 x 4 of them, warp w of the grid
// walks tiles w, w + W, ...), so while a warp multiplies one half the other half -- and then the next
// tile's first half -- is already on its way.  Per site and right-hand side the arithmetic and its order
// are those of dslash_batch_kernel: the outputs are bit-identical (tests/test_gpu_mrhs.py passes with
// STAG_BATCH_RING=1).
//
// MEASURED (28^3 x 96, A/B in one call, us per hop): x2 82.2 against 80.4, x3 104.5 against 89.8, x4 121.5
// against 101.8 -- SLOWER, like the per-thread cp.async staging and the L2 prefetches before it.  The links
// now cross the L1 / shared-memory data pipe twice (the bulk copy's fill, then the LDS), a pipe the
// 4 x 24 gathers already keep 43 % busy, and persistent blocks with a static deal of tiles lose the
// hardware's block-by-block load balancing (the same few per cent the persistent CG kernel loses on
// this lattice).  Kept as the reproducer of that result, not as a path.
#pragma once
#include "stag_dslash_batch.cuh"

namespace stag {

constexpr int RING_HALF_PACKETS = 12;                                   // 4 directions x 3 packets
constexpr int RING_HALF_BYTES = RING_HALF_PACKETS * TILE * 16;          // 6144
constexpr int RING_WARPS = DSLASH_BLOCK / 32;
constexpr int RING_SMEM = RING_WARPS * 2 * RING_HALF_BYTES + 128;       // stages + barriers

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void ring_issue(void *stage, unsigned long long *bar, const void *src)
{
    // one lane: expect RING_HALF_BYTES on the barrier, then the bulk copy that completes them (evict-first in L2)
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(RING_HALF_BYTES) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 :: "r"(smem_u32(stage)), "l"(src), "r"(RING_HALF_BYTES), "r"(smem_u32(bar)), "l"(policy_evict_first()) : "memory");
}
__device__ __forceinline__ void ring_wait(unsigned long long *bar, unsigned parity)
{
    unsigned done = 0;
    while (!done) {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    }
}

// HOP_PLAIN only for now (the stand-alone hop): out_k = D in_k for the N right-hand sides of a paired batch.
template <int N>
__global__ void __launch_bounds__(DSLASH_BLOCK, 4)
dslash_batch_ring_kernel(float2 *__restrict__ out, const float2 *__restrict__ in,
                         const float4 *__restrict__ links, const Geom g, const int p)
{
    static_assert(N >= 2 && N <= 4, "batch hop: 2..4 right-hand sides per pass");
    using C = float2;
    constexpr int K = 6, PPS = 24;
    constexpr int NU = (N + 1) / 2;
    extern __shared__ __align__(128) unsigned char ring_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float4 *stage0 = reinterpret_cast<float4 *>(ring_smem + (size_t)(warp * 2) * RING_HALF_BYTES);
    float4 *stage1 = reinterpret_cast<float4 *>(ring_smem + (size_t)(warp * 2 + 1) * RING_HALF_BYTES);
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(ring_smem + (size_t)RING_WARPS * 2 * RING_HALF_BYTES);
    unsigned long long *bar0 = bars + warp * 2, *bar1 = bars + warp * 2 + 1;
    if (lane == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(bar0)) : "memory");
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(bar1)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    const size_t rs = (size_t)3 * g.Vh_pad;
    const int ntiles = g.Vh_pad / TILE;
    const int W = gridDim.x * RING_WARPS;
    int t = blockIdx.x * RING_WARPS + warp;
    unsigned ph0 = 0, ph1 = 0;
    if (t < ntiles && lane == 0) {
        const float4 *src = links + (size_t)t * (size_t)(PPS * TILE);
        ring_issue(stage0, bar0, src);
        ring_issue(stage1, bar1, src + RING_HALF_PACKETS * TILE);
    }
    struct Unit { float4 q[3]; };
    for (; t < ntiles; t += W) {
        const int cb = t * TILE + lane;
        Site s;
        decode_site(g, p, cb < g.Vh ? cb : 0, s);
        const unsigned neg = det_sign_mask(g, s);
        auto gather = [&](Unit &v, const int u, const int nb) {
            if (2 * u + 1 < N) {
#pragma unroll
                for (int c = 0; c < 3; ++c) v.q[c] = ld_keep_nc((const float4 *)(in + 2 * u * rs) + (size_t)c * g.Vh_pad + nb);
            } else {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const float2 tt = ld_keep_nc(in + (N - 1) * rs + (size_t)c * g.Vh_pad + nb);
                    v.q[c] = make_float4(tt.x, tt.y, 0.f, 0.f);
                }
            }
        };
        C acc[N][3];
#pragma unroll
        for (int k = 0; k < N; ++k)
#pragma unroll
            for (int i = 0; i < 3; ++i) acc[k][i] = make_float2(0.f, 0.f);
        Unit vb[2];
        gather(vb[0], 0, s.nbr[0]);
        const int tn = t + W;
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            if (d == 0) { ring_wait(bar0, ph0); ph0 ^= 1u; }
            if (d == 4) {
                // every lane has read its last packet of stage 0: refill it with the next tile's first half
                __syncwarp();
                if (tn < ntiles && lane == 0) ring_issue(stage0, bar0, links + (size_t)tn * (size_t)(PPS * TILE));
                ring_wait(bar1, ph1); ph1 ^= 1u;
            }
            const float4 *st = (d < 4) ? stage0 : stage1;
            C m[9];
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                const float4 q = st[(3 * (d & 3) + i) * TILE + lane];
                m[2 * i] = make_float2(q.x, q.y);
                m[2 * i + 1] = make_float2(q.z, q.w);
            }
            rebuild_row2<float>(m, (neg >> d) & 1u);
#pragma unroll
            for (int u = 0; u < NU; ++u) {
                const int step = d * NU + u;
                if (step + 1 < 8 * NU) gather(vb[(step + 1) & 1], (u + 1) % NU, s.nbr[(step + 1) / NU]);
                const Unit &v = vb[step & 1];
                if (2 * u + 1 < N) {
#pragma unroll
                    for (int i = 0; i < 3; ++i)
#pragma unroll
                        for (int j = 0; j < 3; ++j) {
                            cfma(acc[2 * u][i], m[3 * i + j], make_float2(v.q[j].x, v.q[j].y));
                            cfma(acc[2 * u + 1][i], m[3 * i + j], make_float2(v.q[j].z, v.q[j].w));
                        }
                } else {
#pragma unroll
                    for (int i = 0; i < 3; ++i)
#pragma unroll
                        for (int j = 0; j < 3; ++j) cfma(acc[N - 1][i], m[3 * i + j], make_float2(v.q[j].x, v.q[j].y));
                }
            }
        }
        __syncwarp();
        if (tn < ntiles && lane == 0) ring_issue(stage1, bar1, links + (size_t)tn * (size_t)(PPS * TILE) + RING_HALF_PACKETS * TILE);
#pragma unroll
        for (int j = 0; j < N / 2; ++j)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                st_keep((float4 *)(out + 2 * j * rs) + (size_t)c * g.Vh_pad + cb,
                        make_float4(acc[2 * j][c].x, acc[2 * j][c].y, acc[2 * j + 1][c].x, acc[2 * j + 1][c].y));
        if (N & 1) {
#pragma unroll
            for (int c = 0; c < 3; ++c) st_keep(out + (N - 1) * rs + (size_t)c * g.Vh_pad + cb, acc[N - 1][c]);
        }
    }
}

}  // namespace stag
