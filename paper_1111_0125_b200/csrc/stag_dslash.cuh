// stag_dslash.cuh -- the staggered Dslash parity hop (eq. 2.5) on sm_100a.
//
// One thread per output site, one warp per 32-site link tile.  Per site the kernel
// streams eight link matrices from the gathered, tiled field (include/stag.h,
// stag_links_create) in 16-byte packets with evict-first loads -- the gauge field is read
// exactly once per hop and must not push the spinors out of L2 -- gathers the eight
// neighbour colour vectors through L1/L2 (each is needed by eight output sites, the farthest
// reuse one time slice away), and accumulates eight 3x3 complex matrix-vector products:
// 8*(66+6) = 576 flop.  HBM-bound: 8*18 + 6 + 6 reals per site
// compulsory.
//
// The link stream is issued in GROUPS of K*GM independent 16-byte loads per thread (K = 9 or
// 6 packets) before the first of them is used; with __launch_bounds__(128, MINB) giving
// ptxas the registers to keep a group in flight this is what moves the kernel from 0.94 to
// 1.05 of the measured copy bandwidth (profiles/README.md, round-1 sweep).
#pragma once
#include "stag_common.cuh"
#include "stag_mem.cuh"

namespace stag {

constexpr int DSLASH_BLOCK = 128;

enum { HOP_PLAIN = 0,    // out = D in
       HOP_XPAY = 1,     // out = a*own - D in                        (second hop of A, eq. 2.3: a = m^2)
       HOP_XPAY_DOT = 2, // same, plus per-block partial sums of <own,out>  (Fig. 1)
       HOP_AXPBY = 3     // out = a*own - cD * D in                   ((D+m) psi = h wrapper, Q23)
};

// 16-byte link packets: two complex numbers in fp32, one in fp64.
template <typename T> struct Pkt;
template <> struct Pkt<float>  { using type = float4;  static constexpr int CPP = 2; };
template <> struct Pkt<double> { using type = double2; static constexpr int CPP = 1; };
template <typename T> using pkt_t = typename Pkt<T>::type;

// complex number c of a run of packets held in registers (c is a compile-time constant
// after unrolling)
__device__ __forceinline__ float2 pk_get(const float4 *pk, int c)
{
    return (c & 1) ? make_float2(pk[c >> 1].z, pk[c >> 1].w) : make_float2(pk[c >> 1].x, pk[c >> 1].y);
}
__device__ __forceinline__ double2 pk_get(const double2 *pk, int c) { return pk[c]; }

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

// The 8-parameter form (P:L113 names it and rejects it for its round-off; Ref. [6] of the paper
// defines it).  A matrix M = s*U, U in SU(3) with rows a, b, c, s = det M = +-1, is stored as four
// complex slots  a2, a3, b1, (theta1, theta2)  with theta1 = arg a1, theta2 = arg c1, and rebuilt:
//   |a1|^2 = 1 - |a2|^2 - |a3|^2            (row a has unit norm)
//   |c1|^2 = 1 - |a1|^2 - |b1|^2            (column 1 has unit norm)
//   N = |a2|^2 + |a3|^2
//   b2 = -(a3* c1* + a1* a2 b1)/N    b3 =  (a2* c1* - a1* a3 b1)/N
//   c2 =  (a3* b1* - a1* a2 c1)/N    c3 = -(a2* b1* + a1* a3 c1)/N
// (unitarity and det U = 1 solved for the four unknowns).  1/N amplifies rounding when the first
// row is nearly (a1,0,0): that is the round-off the paper means, and N = 0 (unit links) has no
// 8-parameter form at all; stag_links_create measures the rebuilt error and refuses such fields.
// On entry m[0..3] hold the four slots; on exit m[0..8] the matrix M.
// fp32: the hardware sine / cosine (arguments are in [-pi, pi], absolute error ~5e-7, the size
// of an fp32 rounding of the stored phase itself) and reciprocal; the library sincosf with its
// range reduction made the fp32 hop ALU-bound (94.8 us against 70.0 us for 12-real on 28^3 x 96).
__device__ __forceinline__ void sincos_fast(float x, float *s, float *c) { __sincosf(x, s, c); }
__device__ __forceinline__ void sincos_fast(double x, double *s, double *c) { sincos(x, s, c); }
__device__ __forceinline__ float recip_fast(float x) { return __frcp_rn(x); }
__device__ __forceinline__ double recip_fast(double x) { return 1.0 / x; }

template <typename T>
__device__ __forceinline__ void rebuild_from8(cplx_t<T> *m, bool neg)
{
    using C = cplx_t<T>;
    const C a2 = m[0], a3 = m[1], b1 = m[2];
    T s1, c1r, s2, c2r;
    sincos_fast(m[3].x, &s1, &c1r);
    sincos_fast(m[3].y, &s2, &c2r);
    const T n = a2.x * a2.x + a2.y * a2.y + a3.x * a3.x + a3.y * a3.y;
    const T r1 = sqrt(fmax((T)0, (T)1 - n));
    const C a1 = mk<T>(r1 * c1r, r1 * s1);
    const T r2 = sqrt(fmax((T)0, (T)1 - r1 * r1 - (b1.x * b1.x + b1.y * b1.y)));
    const C c1 = mk<T>(r2 * c2r, r2 * s2);
    const T inv = recip_fast(n);
    const C a1c = mk<T>(a1.x, -a1.y), a2c = mk<T>(a2.x, -a2.y), a3c = mk<T>(a3.x, -a3.y);
    const C b1c = mk<T>(b1.x, -b1.y), c1c = mk<T>(c1.x, -c1.y);
    const C a1c_a2 = cmul(a1c, a2), a1c_a3 = cmul(a1c, a3);
    const C t1 = cmul(a3c, c1c), t2 = cmul(a1c_a2, b1);      // b2 = -(t1 + t2)/N
    const C t3 = cmul(a2c, c1c), t4 = cmul(a1c_a3, b1);      // b3 =  (t3 - t4)/N
    const C t5 = cmul(a3c, b1c), t6 = cmul(a1c_a2, c1);      // c2 =  (t5 - t6)/N
    const C t7 = cmul(a2c, b1c), t8 = cmul(a1c_a3, c1);      // c3 = -(t7 + t8)/N
    const T sg = neg ? (T)-1 : (T)1, si = sg * inv;
    m[0] = mk<T>(sg * a1.x, sg * a1.y);
    m[1] = mk<T>(sg * a2.x, sg * a2.y);
    m[2] = mk<T>(sg * a3.x, sg * a3.y);
    m[3] = mk<T>(sg * b1.x, sg * b1.y);
    m[4] = mk<T>(-si * (t1.x + t2.x), -si * (t1.y + t2.y));
    m[5] = mk<T>(si * (t3.x - t4.x), si * (t3.y - t4.y));
    m[6] = mk<T>(sg * c1.x, sg * c1.y);
    m[7] = mk<T>(si * (t5.x - t6.x), si * (t5.y - t6.y));
    m[8] = mk<T>(-si * (t7.x + t8.x), -si * (t7.y + t8.y));
}

// complex numbers stored per link for NR: 3 = all nine, 2 = rows 0,1, 1 = the 8-parameter form
__host__ __device__ constexpr int link_slots(int NR) { return NR == 1 ? 4 : 3 * NR; }

// Launch shape per precision / storage / right-hand sides, from the sweeps on 28^3 x 96
// (profiles/README.md): MINB = resident blocks per SM promised to ptxas, GM = directions' worth
// of packets loaded ahead (group = K*GM packets).  With N > 1 right-hand sides the registers go
// to the N accumulators and the N neighbour vectors of one group instead.
template <typename T, int NR, int N> struct HopTune { static constexpr int MINB = 4, GM = 1; };
template <> struct HopTune<float, 2, 1>            { static constexpr int MINB = 4, GM = 2; };
// 8-parameter fp32: ALU-bound (two sincos, two sqrt, a reciprocal and eight complex products per
// link); 4 blocks/SM with two directions in flight measured best (70.2 us; 6 blocks: 76.8 us)
template <> struct HopTune<float, 1, 1>            { static constexpr int MINB = 4, GM = 2; };
template <int N> struct HopTune<double, 3, N>      { static constexpr int MINB = (N == 1) ? 4 : 2, GM = 1; };
template <int N> struct HopTune<double, 2, N>      { static constexpr int MINB = (N == 1) ? 4 : 2, GM = 1; };

// Largest N instantiated per precision: more right-hand sides go through in chunks.
template <typename T> struct HopMaxRhs;
template <> struct HopMaxRhs<float>  { static constexpr int value = 4; };
template <> struct HopMaxRhs<double> { static constexpr int value = 2; };

// ---- T-slab halo (stag_slab_*) ------------------------------------
// A slab is time slices [t0, t0+X3) of a larger lattice held by one GPU.  The neighbour slices
// x3 = -1 and x3 = X3 of the INPUT spinor live in two halo buffers, [colour][s3] complex each,
// that the neighbouring GPUs fill with peer-to-peer stores (face_push_kernel) and then mark by
// storing the exchange's epoch into flag_back / flag_fwd with system-scope release.
// The kernel reads the number of the current exchange from the region's header (device memory,
// so a graph replay sees the right one) and derives the halo buffers of that parity from it.
template <typename T> struct HaloArgs {
    char *xch;           // this slab's exchange region
    // HOP_PLAIN only, may be null: push the faces of OUT as the next exchange while computing it
    // (the hop that produces the second hop's input stores its first / last time slice straight
    // into the neighbours' halo buffers; its last block then bumps the count and sets their flags)
    char *peer_fwd, *peer_bwd;
    unsigned n_push_blocks;   // blocks of this launch that own boundary-slice sites (they alone take the ticket)
};

// hdr: the header of the slab whose flag f belongs to (for the watchdog, stag_common.cuh).
// Returns false when the wait gave up: the slab is then marked (hdr->timed_out, sticky until
// stag_slab_reset) and the caller must not publish anything derived from the data it waited for.
__device__ __forceinline__ bool wait_flag(const unsigned long long *f, unsigned long long epoch, XchHeader *hdr)
{
    unsigned long long v, polls = 0;
    unsigned long long limit = __ldcg(&hdr->wait_limit);
    if (limit == 0) limit = XCH_DEFAULT_WAIT_POLLS;
    for (;;) {
        asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(f) : "memory");
        if (v >= epoch) {
            if (polls) { atomicAdd(&hdr->waits_spun, 1ull); atomicAdd(&hdr->polls_spent, polls); }
            return true;
        }
        if (++polls >= limit || __ldcg(&hdr->timed_out) != 0u) {
            *(volatile unsigned *)&hdr->timed_out = 1u;
            return false;
        }
        __nanosleep(200);
    }
}
// One thread, after it has observed (at gpu scope: ticket or barrier) every block's stores into the
// neighbours' halo buffers: make them visible at system scope, then set the neighbours' flags to e.
// STAG_FLAG_FENCE selects how (measured on B200, profiles/README.md round 2): 0 = two release
// stores, 1 = one fence.acq_rel.sys + two relaxed stores, 2 = __threadfence_system (fence.sc.sys).
#ifndef STAG_FLAG_FENCE
#define STAG_FLAG_FENCE 1
#endif
__device__ __forceinline__ void raise_halo_flags(char *peer_fwd, char *peer_bwd, unsigned long long e)
{
    unsigned long long *ff = &((XchHeader *)peer_fwd)->flag_back, *fb = &((XchHeader *)peer_bwd)->flag_fwd;
#if STAG_FLAG_FENCE == 0
    asm volatile("st.release.sys.global.u64 [%0], %1;" :: "l"(ff), "l"(e) : "memory");
    asm volatile("st.release.sys.global.u64 [%0], %1;" :: "l"(fb), "l"(e) : "memory");
#else
#if STAG_FLAG_FENCE == 1
    asm volatile("fence.acq_rel.sys;" ::: "memory");
#else
    __threadfence_system();
#endif
    asm volatile("st.relaxed.sys.global.u64 [%0], %1;" :: "l"(ff), "l"(e) : "memory");
    asm volatile("st.relaxed.sys.global.u64 [%0], %1;" :: "l"(fb), "l"(e) : "memory");
#endif
}

// A slab whose watchdog fired is dead until stag_slab_reset: every kernel of the slab path begins with
// this test (uniform over the grid when the mark predates the launch) and leaves without storing to a
// peer, bumping a count or setting a flag, so the neighbours' waits run into their own limit and every
// rank reports STAG_ETIMEOUT instead of consuming stale data.
__device__ __forceinline__ bool slab_dead(const char *xch)
{
    return __ldcg(&((const XchHeader *)xch)->timed_out) != 0u;
}

// One output site, one right-hand side: acc[i] = sum_d (M_d(x) chi(nbr_d(x)))_i -- the arithmetic of
// eq. 2.5 and its order, shared by dslash_kernel (N = 1) and the persistent iteration kernel
// (stag_persist.cuh), so that the two produce the same bits per site.  All 24 neighbour loads are
// issued before the link stream; the links arrive in groups of KG 16-byte packets (HopTune).
// HALO: the +-t neighbours of the slab's first / last time slice come from the halo buffers of
// exchange epoch() once the slab's own flag shows it (decode_site wrapped them onto the slab's other
// end; their in-slice index addresses the buffers).  epoch() is only evaluated by boundary threads.
// NC: the input spinor is read-only for the whole kernel (non-coherent loads, the plain kernels);
// false inside the persistent kernel, where another phase of the same launch wrote it.
// LRES: the gauge field is small enough to stay in L2 next to the vectors (persistent kernel on
// small lattices): its packets are then loaded with the keep policy instead of streamed through.
// Returns false when a halo wait of this site gave up (HALO only; the slab is then marked dead): acc
// was computed from a halo that never arrived, and the caller must not store it into a peer's buffers
// (wait_flag's contract: a timed-out slab publishes nothing).  Always true otherwise.
template <typename T, int NR, bool HALO, bool NC = true, bool LRES = false, typename EpochFn>
__device__ __forceinline__ bool hop_site(cplx_t<T> (&acc)[3], const cplx_t<T> *__restrict__ in,
                                         const pkt_t<T> *__restrict__ links, const Geom &g, const int cb,
                                         const Site &s, const unsigned neg, char *xch, EpochFn epoch)
{
    using C = cplx_t<T>;
    using P = pkt_t<T>;
    constexpr int K = link_slots(NR);
    constexpr int GM = HopTune<T, NR, 1>::GM;
    constexpr int DPG = Pkt<T>::CPP * GM;     // directions per group
    constexpr int NG = 8 / DPG;               // groups per site
    constexpr int KG = K * GM;                // packets per group
    static_assert(8 % DPG == 0, "group must divide the eight directions");
    const P *L = links + (size_t)(cb >> 5) * (size_t)(NG * KG * TILE) + (cb & 31);
    C v1[8][3];
#pragma unroll
    for (int d = 0; d < 8; ++d)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            if constexpr (NC) v1[d][c] = ld_keep_nc(in + (size_t)c * g.Vh_pad + s.nbr[d]);
            else v1[d][c] = ld_keep(in + (size_t)c * g.Vh_pad + s.nbr[d]);
        }
    bool fresh = true;
    if constexpr (HALO) {
        XchHeader *hdr = (XchHeader *)xch;
        if (s.x3 == g.X3 - 1) {
            const unsigned long long e = epoch();
            const C *fwd = (const C *)(xch + xch_halo_offset(g.s3, e, 1));
            fresh = wait_flag(&hdr->flag_fwd, e, hdr);
#pragma unroll
            for (int c = 0; c < 3; ++c) v1[3][c] = __ldcg(fwd + (size_t)c * g.s3 + s.nbr[3]);
        }
        if (s.x3 == 0) {
            const unsigned long long e = epoch();
            const C *back = (const C *)(xch + xch_halo_offset(g.s3, e, 0));
            fresh = wait_flag(&hdr->flag_back, e, hdr) && fresh;
#pragma unroll
            for (int c = 0; c < 3; ++c)
                v1[7][c] = __ldcg(back + (size_t)c * g.s3 + (s.nbr[7] - (g.X3 - 1) * g.s3));
        }
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) acc[i] = mk<T>(0, 0);
#pragma unroll
    for (int grp = 0; grp < NG; ++grp) {
        P pk[KG];
#pragma unroll
        for (int i = 0; i < KG; ++i) {
            if constexpr (LRES) pk[i] = ld_keep_nc(L + (grp * KG + i) * TILE);
            else pk[i] = ld_stream(L + (grp * KG + i) * TILE);
        }
#pragma unroll
        for (int dd = 0; dd < DPG; ++dd) {
            const int d = grp * DPG + dd;
            C m[9];
#pragma unroll
            for (int k = 0; k < K; ++k) m[k] = pk_get(pk, dd * K + k);
            if (NR == 2) rebuild_row2<T>(m, (neg >> d) & 1u);
            if (NR == 1) rebuild_from8<T>(m, (neg >> d) & 1u);
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = 0; j < 3; ++j) cfma(acc[i], m[3 * i + j], v1[d][j]);
        }
    }
    return fresh;
}

// T: float or double.  NR: storage of each link (3 = 18-real, 2 = 12-real rows 0,1, 1 = 8-parameter).
// N: right-hand sides handled by one thread.  Two batch layouts (include/stag.h "batch layouts"):
//   blocked (PAIRED = false): spinor k of a batch starts rs complex numbers after spinor k-1
//           (rs = 3*Vh_pad: the batch is N device spinors back to back);
//   paired  (PAIRED = true, fp32 only): right-hand sides 2j and 2j+1 are interleaved per complex
//           number, v[j][c][cb] = (re_2j, im_2j, re_2j+1, im_2j+1), one float4 plane triple per pair
//           (it occupies the 2*rs float2 slots the two spinors would), an odd last right-hand side
//           is an ordinary spinor after the pairs.  A neighbour colour of a pair is then ONE
//           16-byte gather instead of two 8-byte ones: half the gather instructions and address
//           arithmetic of the batch hop, which is bound by issue slots and loads in flight, not
//           by DRAM.  The arithmetic per right-hand side is unchanged.
// links: the gathered field of the OUTPUT parity as packets, L[tile][j][lane], packet j holding
// complex numbers CPP*j .. CPP*j+CPP-1 of the site's run c = d*K + k (d = direction 0..7,
// k = 3*row+col).  in: the other parity's spinor planes; out / own: this parity's.
// MODE HOP_XPAY*: out = a*own - D in;  HOP_AXPBY: out = a*own - cD * D in.
// partials: HOP_XPAY_DOT writes sum over the block of Re<own,out> (fp64) of right-hand
// side k to partials[k*gridDim.x + blockIdx.x]; the kernel that needs <d,Ad> adds them in index
// order (stag_blas.cuh).
// HALO (N = 1 only): the lattice is a T-slab; the +-t neighbours of the first and last time
// slice come from the halo buffers once their flag shows this exchange's epoch.  Sites are
// visited rotated by one time slice (slices 1 .. X3-1, then slice 0), so the blocks that may
// have to wait for a neighbouring GPU run last and the interior overlaps the exchange.
template <typename T, int NR, int MODE, int N, bool HALO = false, bool PAIRED = false>
__global__ void __launch_bounds__(DSLASH_BLOCK, HopTune<T, NR, N>::MINB)
dslash_kernel(cplx_t<T> *__restrict__ out, const cplx_t<T> *__restrict__ in,
              const pkt_t<T> *__restrict__ links, const Geom g, const int p, const T a, const T cD,
              const cplx_t<T> *__restrict__ own, double *__restrict__ partials,
              const CgCtrl *__restrict__ ctrl, const HaloArgs<T> halo)
{
    static_assert(!HALO || N == 1, "slab hops carry one right-hand side");
    static_assert(!PAIRED || (N > 1 && sizeof(T) == 4), "paired batches are fp32 with at least two right-hand sides");
    using C = cplx_t<T>;
    using P = pkt_t<T>;
    constexpr int K = link_slots(NR);
    constexpr int GM = HopTune<T, NR, N>::GM;
    constexpr int DPG = Pkt<T>::CPP * GM;     // directions per group
    constexpr int NG = 8 / DPG;               // groups per site
    constexpr int KG = K * GM;                // packets per group
    static_assert(8 % DPG == 0, "group must divide the eight directions");
    if (ctrl != nullptr && ctrl->state != CG_RUN) return;
    if constexpr (HALO) {
        if (slab_dead(halo.xch)) return;
    }

    int cb = blockIdx.x * DSLASH_BLOCK + threadIdx.x;
    if constexpr (HALO) {
        if (cb < g.Vh_pad) {
            cb += g.s3;
            if (cb >= g.Vh_pad) cb -= g.Vh_pad;
        }
    }
    const size_t rs = (size_t)3 * g.Vh_pad;
    bool pushing = false, pushed = false;
    unsigned long long e_in = 0;
    if constexpr (HALO && MODE == HOP_PLAIN) {
        pushing = halo.peer_fwd != nullptr;
    }
    double dot[N];
#pragma unroll
    for (int k = 0; k < N; ++k) dot[k] = 0.0;
    if (cb < g.Vh_pad) {
        // pad lanes (cb >= Vh) read zero links, so they produce zeros without a branch
        Site s;
        decode_site(g, p, cb < g.Vh ? cb : 0, s);
        const P *L = links + (size_t)(cb >> 5) * (size_t)(NG * KG * TILE) + (cb & 31);

        unsigned neg = 0;
        if (NR != 3) neg = det_sign_mask(g, s);

        C acc[N][3];
        bool fresh = true;      // false: a halo wait of this site timed out, its result is not pushed to a peer
        if constexpr (N == 1) {
            fresh = hop_site<T, NR, HALO, true>(acc[0], in, links, g, cb, s, neg, halo.xch,
                                  [&]() { return __ldcg(&((const XchHeader *)halo.xch)->epoch); });
        } else {
            // several right-hand sides: the neighbours of one group of directions at a time (register budget)
#pragma unroll
            for (int k = 0; k < N; ++k)
#pragma unroll
                for (int i = 0; i < 3; ++i) acc[k][i] = mk<T>(0, 0);
#pragma unroll
            for (int grp = 0; grp < NG; ++grp) {
                P pk[KG];
#pragma unroll
                for (int i = 0; i < KG; ++i) pk[i] = ld_stream(L + (grp * KG + i) * TILE);
                C vg[N][DPG][3];
                if constexpr (!PAIRED) {
#pragma unroll
                    for (int k = 0; k < N; ++k)
#pragma unroll
                        for (int dd = 0; dd < DPG; ++dd)
#pragma unroll
                            for (int c = 0; c < 3; ++c)
                                vg[k][dd][c] = ld_keep_nc(in + k * rs + (size_t)c * g.Vh_pad + s.nbr[grp * DPG + dd]);
                }
                if constexpr (PAIRED) {
#pragma unroll
                    for (int j = 0; j < N / 2; ++j)
#pragma unroll
                        for (int dd = 0; dd < DPG; ++dd)
#pragma unroll
                            for (int c = 0; c < 3; ++c) {
                                const float4 v = ld_keep_nc((const float4 *)(in + 2 * j * rs) + (size_t)c * g.Vh_pad + s.nbr[grp * DPG + dd]);
                                vg[2 * j][dd][c] = mk<T>(v.x, v.y);
                                vg[2 * j + 1][dd][c] = mk<T>(v.z, v.w);
                            }
                    if constexpr (N & 1) {
#pragma unroll
                        for (int dd = 0; dd < DPG; ++dd)
#pragma unroll
                            for (int c = 0; c < 3; ++c)
                                vg[N - 1][dd][c] = ld_keep_nc(in + (N - 1) * rs + (size_t)c * g.Vh_pad + s.nbr[grp * DPG + dd]);
                    }
                }
#pragma unroll
                for (int dd = 0; dd < DPG; ++dd) {
                    const int d = grp * DPG + dd;
                    C m[9];
#pragma unroll
                    for (int k = 0; k < K; ++k) m[k] = pk_get(pk, dd * K + k);
                    if (NR == 2) rebuild_row2<T>(m, (neg >> d) & 1u);
                    if (NR == 1) rebuild_from8<T>(m, (neg >> d) & 1u);
#pragma unroll
                    for (int k = 0; k < N; ++k)
#pragma unroll
                        for (int i = 0; i < 3; ++i)
#pragma unroll
                            for (int j = 0; j < 3; ++j) cfma(acc[k][i], m[3 * i + j], vg[k][dd][j]);
                }
            }
        }

        if (NR == 1 && cb >= g.Vh) {
            // a rebuilt 8-parameter matrix is unitary, never zero: pad lanes are zeroed here
            // (the 18- and 12-real forms get their zeros from the zero links of the pad lanes)
#pragma unroll
            for (int k = 0; k < N; ++k)
#pragma unroll
                for (int i = 0; i < 3; ++i) acc[k][i] = mk<T>(0, 0);
        }
        if constexpr (PAIRED) {
            // a pair's three colours leave as three 16-byte stores; its own-site vector arrives the same way
#pragma unroll
            for (int j = 0; j < N / 2; ++j)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    float4 *po = (float4 *)(out + 2 * j * rs) + (size_t)c * g.Vh_pad + cb;
                    if (MODE == HOP_PLAIN) {
                        st_keep(po, make_float4(acc[2 * j][c].x, acc[2 * j][c].y, acc[2 * j + 1][c].x, acc[2 * j + 1][c].y));
                    } else {
                        const float4 o = ld_keep_nc((const float4 *)(own + 2 * j * rs) + (size_t)c * g.Vh_pad + cb);
                        float4 r;
                        if (MODE == HOP_AXPBY) {
                            r.x = fma(a, o.x, -cD * acc[2 * j][c].x);     r.y = fma(a, o.y, -cD * acc[2 * j][c].y);
                            r.z = fma(a, o.z, -cD * acc[2 * j + 1][c].x); r.w = fma(a, o.w, -cD * acc[2 * j + 1][c].y);
                        } else {
                            r.x = fma(a, o.x, -acc[2 * j][c].x);     r.y = fma(a, o.y, -acc[2 * j][c].y);
                            r.z = fma(a, o.z, -acc[2 * j + 1][c].x); r.w = fma(a, o.w, -acc[2 * j + 1][c].y);
                        }
                        st_keep(po, r);
                        if (MODE == HOP_XPAY_DOT) {
                            dot[2 * j] += (double)o.x * (double)r.x + (double)o.y * (double)r.y;
                            dot[2 * j + 1] += (double)o.z * (double)r.z + (double)o.w * (double)r.w;
                        }
                    }
                }
        }
#pragma unroll
        for (int k = PAIRED ? (N / 2) * 2 : 0; k < N; ++k) {
            if (MODE == HOP_PLAIN) {
#pragma unroll
                for (int c = 0; c < 3; ++c) st_keep(out + k * rs + (size_t)c * g.Vh_pad + cb, acc[k][c]);
                if constexpr (HALO) {
                    if (pushing && fresh && cb < g.Vh && (s.x3 == 0 || s.x3 == g.X3 - 1)) {
                        // first slice -> the backward neighbour's "fwd" halo, last slice -> the
                        // forward neighbour's "back" halo, buffers of exchange e_in + 1.  Only the
                        // boundary threads read the count, and only their blocks take the ticket
                        // whose last holder bumps it: no reader can see the bumped value.
                        e_in = __ldcg(&((const XchHeader *)halo.xch)->epoch);
                        C *dst = (s.x3 == 0)
                            ? (C *)(halo.peer_bwd + xch_halo_offset(g.s3, e_in + 1, 1)) + cb
                            : (C *)(halo.peer_fwd + xch_halo_offset(g.s3, e_in + 1, 0)) + (cb - (g.Vh - g.s3));
#pragma unroll
                        for (int c = 0; c < 3; ++c) dst[(size_t)c * g.s3] = acc[k][c];
                        pushed = true;
                    }
                }
            } else {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const C o = ld_keep_nc(own + k * rs + (size_t)c * g.Vh_pad + cb);
                    C r;
                    if (MODE == HOP_AXPBY) {
                        r.x = fma(a, o.x, -cD * acc[k][c].x);
                        r.y = fma(a, o.y, -cD * acc[k][c].y);
                    } else {
                        r.x = fma(a, o.x, -acc[k][c].x);
                        r.y = fma(a, o.y, -acc[k][c].y);
                    }
                    st_keep(out + k * rs + (size_t)c * g.Vh_pad + cb, r);
                    if (MODE == HOP_XPAY_DOT)
                        dot[k] += (double)o.x * (double)r.x + (double)o.y * (double)r.y;
                }
            }
        }
    }

    if constexpr (HALO && MODE == HOP_PLAIN) {
        if (pushing) {       // uniform over the grid
            // one system-scope fence per block that stored to a peer (thread 0, after the block
            // barrier: cumulative over the block's stores), none in the interior blocks
            // Interior blocks leave without touching the ticket: a returning atomic per block held
            // every block ~1 us longer (14 waves: +14 us on 28^3 x 96).
            __shared__ unsigned long long s_e;
            if (pushed) s_e = e_in;                     // the same value from every boundary thread
            const int any = __syncthreads_or(pushed ? 1 : 0);
            XchHeader *hdr = (XchHeader *)halo.xch;
            if (any && threadIdx.x == 0) {
                e_in = s_e;
                __threadfence();      // release at gpu scope; the ticket's last holder fences at system scope
            }
            // every boundary block waited for its own halo before it got here, so the ticket's last
            // holder sees a timeout of any of them (their marks precede their gpu-scope fences)
            if (any && threadIdx.x == 0 && atomicAdd(&hdr->ticket, 1u) == halo.n_push_blocks - 1 && !slab_dead(halo.xch)) {
                hdr->ticket = 0;
                hdr->epoch = e_in + 1;
                raise_halo_flags(halo.peer_fwd, halo.peer_bwd, e_in + 1);   // cumulative: every block's peer stores precede the flags
            }
        }
    }

    if (MODE == HOP_XPAY_DOT) {
        // No ticket, no fence here: a gpu-scope fence invalidates the SM's L1 under the
        // neighbour gathers of the co-resident blocks.  The kernel boundary orders the
        // partials for their reader.  One block barrier for all N sums; the four warp totals are
        // added as block_sum's shuffle tree adds them, (w0 + w2) + (w1 + w3).
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
