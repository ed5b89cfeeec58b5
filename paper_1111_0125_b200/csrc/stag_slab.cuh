// stag_slab.cuh -- T-slab domain decomposition of the hop: the halo exchange over peer memory.
//
// The paper's multi-GPU Dirac operation is kernel -> boundary collect -> memcpy to host -> MPI ->
// memcpy to device (Table 1), and it plans peer-to-peer copies.  Here a
// slab's two boundary time slices of the hop's INPUT spinor are stored straight into the
// neighbouring GPUs' halo buffers (peer-to-peer stores over NVLink; the buffers are ordinary device
// memory mapped into this process with CUDA IPC or, for slabs that share a process, used directly)
// by the kernel that PRODUCES that spinor -- slab_xpay_push_kernel for the direction d, the
// boundary-slice threads of hop 1 for its output (stag_dslash.cuh) -- or, stand-alone, by
// face_push_kernel; the exchange's number is then stored into each neighbour's flag behind one
// system-scope fence (raise_halo_flags, stag_dslash.cuh).  The consuming hop (dslash_kernel<..., HALO = true>) waits on
// its own two flags only in the threads of the first and last time slice, which it visits last.
//
// The slab CG's global sums go through the same region: a rank stores its local total into slot
// [seq & 1][its rank] of EVERY rank's XchReduce and then release-stores seq into flag[its rank];
// whoever needs the sum acquire-waits for all nranks flags and adds the slots in rank order, so
// every rank forms bit-identical alpha, beta and stopping decisions.  The wait always sits in a
// kernel launched AFTER the publishing one on every rank, never in the same kernel.
//
// Exchange region of one slab (one allocation = one IPC handle), XCH_HDR bytes of header, then
// halo buffers [epoch & 1][dir][colour][s3] of 16-byte complex slots (fp32 uses the front half):
//   dir 0 = "back":  the neighbour slice x3 = -1,  written by rank-1 from its LAST slice
//   dir 1 = "fwd":   the neighbour slice x3 = X3,  written by rank+1 from its FIRST slice
// Ordering of a push: every storing block's thread 0, after the block barrier, fences at gpu scope and
// takes a ticket; the ticket's last holder has thereby observed all of them, fences at SYSTEM scope
// (cumulative over everything that happens-before it, i.e. every block's peer stores) and only then
// stores the flags (raise_halo_flags: fence.acq_rel.sys, then two relaxed system-scope stores).  One system-scope fence per launch instead of one per storing block:
// those sat at the tail of the kernel and cost ~8 us.
// Double buffering by epoch parity is enough: a rank cannot start exchange e+2 before both its
// neighbours have finished consuming exchange e (its own hop e+1 waits for their push e+1, which
// follows their hop e in stream order).
#pragma once
#include "stag_blas.cuh"
#include "stag_common.cuh"

namespace stag {

constexpr int MAX_RANKS = STAG_MAX_RANKS;
struct XchReduce {
    unsigned long long flag[MAX_RANKS];   // flag[r]: last reduction number rank r has published here
    double slot[2][MAX_RANKS];            // slot[seq & 1][r]: rank r's local total of reduction seq
};
static_assert(XCH_RED + sizeof(XchReduce) <= XCH_HDR, "reduction slots must fit the header area");
inline size_t xch_bytes(int s3) { return XCH_HDR + (size_t)4 * 3 * s3 * 16; }

// in: one parity's device spinor of the slab (planes of Vh_pad).  Stores its last time slice into
// fwd_back (the forward neighbour's "back" halo) and its first time slice into bwd_fwd (the
// backward neighbour's "fwd" halo), then marks both neighbours' flags with the epoch.
template <typename T>
__global__ void __launch_bounds__(256)
face_push_kernel(const cplx_t<T> *__restrict__ in, const int Vh, const int Vh_pad, const int s3,
                 char *mine, char *peer_fwd, char *peer_bwd)
{
    XchHeader *hdr = (XchHeader *)mine;
    if (slab_dead(mine)) return;              // watchdog fired earlier: publish nothing (stag_dslash.cuh)
    // every block reads the count before it takes its ticket; the last block bumps it afterwards
    const unsigned long long epoch = __ldcg(&hdr->epoch) + 1;
    cplx_t<T> *fwd_back = (cplx_t<T> *)(peer_fwd + xch_halo_offset(s3, epoch, 0));
    cplx_t<T> *bwd_fwd = (cplx_t<T> *)(peer_bwd + xch_halo_offset(s3, epoch, 1));
    const long i = blockIdx.x * 256L + threadIdx.x;
    const long face = 3L * s3;
    if (i < 2 * face) {
        const long r = i % face;
        const int c = (int)(r / s3), j = (int)(r % s3);
        if (i < face) fwd_back[(size_t)c * s3 + j] = in[(size_t)c * Vh_pad + (Vh - s3) + j];
        else          bwd_fwd[(size_t)c * s3 + j] = in[(size_t)c * Vh_pad + j];
    }
    __syncthreads();
    if (threadIdx.x == 0) __threadfence();    // gpu-scope release of the block's peer stores (after the block barrier)
    if (threadIdx.x == 0 && atomicAdd(&hdr->ticket, 1u) == gridDim.x - 1) {
        hdr->ticket = 0;
        hdr->epoch = epoch;
        raise_halo_flags(peer_fwd, peer_bwd, epoch);   // cumulative: every block's stores precede the flags
    }
}

// d = r + beta d (xpay_kernel) that also pushes the faces of the new d: the producer of the first
// hop's input stores the packets of its first / last time slice straight into the neighbours'
// halo buffers.  Vectors are flat (3 colour planes of Vh_pad complex); a 16-byte packet never
// straddles a slice because s3 and Vh are even.
template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK)
slab_xpay_push_kernel(T *__restrict__ d, const T *__restrict__ r, long n, const CgCtrl *__restrict__ ctrl,
                      const int Vh, const int Vh_pad, const int s3, char *mine, char *peer_fwd, char *peer_bwd)
{
    if (ctrl->state != CG_RUN || !ctrl->active[0]) return;     // the same in every block: no ticket taken
    if (slab_dead(mine)) return;
    using V = typename Vec4<T>::type;
    constexpr int N = Vec4<T>::N;
    constexpr int CPK = N / 2;                                 // complex numbers per packet
    XchHeader *hdr = (XchHeader *)mine;
    const unsigned long long epoch = __ldcg(&hdr->epoch) + 1;
    V *fwd_back = (V *)(peer_fwd + xch_halo_offset(s3, epoch, 0));
    V *bwd_fwd = (V *)(peer_bwd + xch_halo_offset(s3, epoch, 1));
    const T beta = (T)ctrl->beta[0];
    const long nv = n / N;
    V *dv = reinterpret_cast<V *>(d);
    const V *rv = reinterpret_cast<const V *>(r);
    bool stored = false;
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < nv; i += (long)gridDim.x * BLAS_BLOCK) {
        T a[N], b[N];
        unpack<T>(ld_keep(rv + i), a);
        unpack<T>(ld_keep(dv + i), b);
        if (beta == (T)0) {
#pragma unroll
            for (int j = 0; j < N; ++j) b[j] = a[j];
        } else {
#pragma unroll
            for (int j = 0; j < N; ++j) b[j] = fma(beta, b[j], a[j]);
        }
        const V pk = pack(b);
        st_keep(dv + i, pk);
        const long ci = i * CPK;                               // first complex number of the packet
        const int c = (ci >= 2L * Vh_pad) ? 2 : (ci >= Vh_pad ? 1 : 0);      // colour plane, no division
        const int cb = (int)(ci - (long)c * Vh_pad);
        if (cb < s3) {                                         // first time slice
            bwd_fwd[((long)c * s3 + cb) / CPK] = pk;
            stored = true;
        } else if (cb >= Vh - s3 && cb < Vh) {                 // last time slice
            fwd_back[((long)c * s3 + (cb - (Vh - s3))) / CPK] = pk;
            stored = true;
        }
    }
    const int any = __syncthreads_or(stored ? 1 : 0);
    if (threadIdx.x == 0 && any) __threadfence();      // gpu-scope release of the block's peer stores (after the block barrier)
    if (threadIdx.x == 0 && atomicAdd(&hdr->ticket, 1u) == gridDim.x - 1) {
        hdr->ticket = 0;
        hdr->epoch = epoch;
        raise_halo_flags(peer_fwd, peer_bwd, epoch);
    }
}

// ---- global sums of the slab CG ---------------------------------------------------------
// Both are called by ALL 32 LANES OF ONE WARP; lane r talks to rank r, so the system-scope round
// trips to the nranks regions overlap instead of queueing behind one another.
// Publish: lane r stores my local total of reduction seq into rank r's slot and release-stores
// seq into my flag there (the release orders the lane's own slot store before it).
static_assert(MAX_RANKS <= 32, "one lane per rank");
__device__ __forceinline__ void publish_total(char *const *peers, int nranks, int myrank,
                                              unsigned long long seq, double value)
{
    const int r = threadIdx.x & 31;
    if (r < nranks) {
        XchReduce *R = (XchReduce *)(peers[r] + XCH_RED);
        *(volatile double *)&R->slot[seq & 1ull][myrank] = value;
        asm volatile("st.release.sys.global.u64 [%0], %1;" :: "l"(&R->flag[myrank]), "l"(seq) : "memory");
    }
}

// The sum over ranks of reduction seq, added in rank order (same bits on every rank), returned
// to every lane.  *ok = false when a wait gave up (the slab is then marked dead; the sum is not to
// be used).  Lane r acquire-waits for rank r's flag and reads rank r's slot.
__device__ __forceinline__ double gather_total(char *mine, int nranks, unsigned long long seq, bool *ok)
{
    const XchReduce *R = (const XchReduce *)(mine + XCH_RED);
    const int r = threadIdx.x & 31;
    bool good = true;
    double mine_v = 0.0;
    if (r < nranks) {
        good = wait_flag(&R->flag[r], seq, (XchHeader *)mine);
        mine_v = __ldcg(&R->slot[seq & 1ull][r]);
    }
    good = __all_sync(0xffffffffu, good);
    double t = 0.0;
    for (int k = 0; k < nranks; ++k) t += __shfl_sync(0xffffffffu, mine_v, k);     // rank order
    *ok = good;
    return good ? t : 0.0;
}

// Comm: what a kernel of the slab CG needs to publish / gather (passed by value).  The number of
// a reduction is not an argument: the publisher takes red_seq + 1 from its own header and stores
// it back, the gatherer (a LATER kernel on the same stream) reads red_seq, so a captured graph of
// iterations can be replayed.
struct Comm {
    char *const *peers;     // device array of nranks pointers to every rank's exchange region
    char *mine;
    int nranks, myrank;
};

// one warp (all 32 lanes)
__device__ __forceinline__ void publish_next(const Comm &c, double value)
{
    XchHeader *hdr = (XchHeader *)c.mine;
    const unsigned long long seq = __ldcg(&hdr->red_seq) + 1;
    __syncwarp();
    publish_total(c.peers, c.nranks, c.myrank, seq, value);
    if ((threadIdx.x & 31) == 0) hdr->red_seq = seq;
}
// one warp (all 32 lanes) of a kernel launched after the publishing one
__device__ __forceinline__ double gather_current(const Comm &c, bool *ok)
{
    return gather_total(c.mine, c.nranks, __ldcg(&((const XchHeader *)c.mine)->red_seq), ok);
}

// Local fixed-order sum of the second hop's per-block partials of <d,Ad>, published to all ranks.
__global__ void __launch_bounds__(1024)
slab_publish_partials_kernel(const double *__restrict__ partials, int n, const Comm c,
                             const CgCtrl *__restrict__ ctrl)
{
    if (ctrl->state != CG_RUN || slab_dead(c.mine)) return;
    __shared__ double red[32];
    const double t = block_total_fixed(partials, n, red);
    if (threadIdx.x < 32) publish_next(c, t);
}

// update_kernel for one right-hand side of a slab: <d,Ad> is the all-rank sum of reduction
// last published; the local |r|^2 is published as the next one instead of running the epilogue.
template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK)
slab_update_kernel(T *__restrict__ y, T *__restrict__ r, const T *__restrict__ d,
                   const T *__restrict__ q, long n, double *__restrict__ partials,
                   CgCtrl *__restrict__ ctrl, const Comm c)
{
    if (ctrl->state != CG_RUN || slab_dead(c.mine)) return;
    using V = typename Vec4<T>::type;
    constexpr int N = Vec4<T>::N;
    __shared__ double red[32];
    __shared__ double totals[MAX_RHS];
    __shared__ double s_dAd;
    __shared__ bool s_ok;
    if (threadIdx.x < 32) {                                     // every block reads red_seq before the last one bumps it
        bool ok;
        const double t = gather_current(c, &ok);
        if (threadIdx.x == 0) { s_dAd = t; s_ok = ok; }
    }
    __syncthreads();
    if (!s_ok) return;            // a peer never published <d,Ad>: leave y, r alone and publish nothing
    const double dAd = s_dAd;
    const bool ok = dAd > 0.0;
    const double alpha_d = ok ? ctrl->delta[0] / dAd : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) { ctrl->dAd[0] = dAd; ctrl->alpha[0] = alpha_d; }
    const T alpha = (T)alpha_d;
    const long nv = n / N;
    V *yk = reinterpret_cast<V *>(y);
    V *rk = reinterpret_cast<V *>(r);
    const V *dk = reinterpret_cast<const V *>(d);
    const V *qk = reinterpret_cast<const V *>(q);
    double s = 0.0;
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < nv; i += (long)gridDim.x * BLAS_BLOCK) {
        T yy[N], rr[N], dd[N], qq[N];
        unpack<T>(ld_pass(yk + i), yy);
        unpack<T>(ld_keep(rk + i), rr);
        unpack<T>(ld_keep(dk + i), dd);
        unpack<T>(ld_keep(qk + i), qq);
#pragma unroll
        for (int j = 0; j < N; ++j) {
            yy[j] = fma(alpha, dd[j], yy[j]);
            rr[j] = fma(-alpha, qq[j], rr[j]);
            s += (double)rr[j] * (double)rr[j];
        }
        st_pass(yk + i, pack(yy));
        st_keep(rk + i, pack(rr));
    }
    const double bs = block_sum(s, red);
    if (!finish_reduction(bs, partials, &ctrl->ticket[1], red, totals)) return;
    if (threadIdx.x < 32) publish_next(c, totals[0]);
}

// residual_kernel for one right-hand side of a slab: publishes the local |r|^2 (or |b|^2).
template <typename T, int WHAT>
__global__ void __launch_bounds__(BLAS_BLOCK)
slab_residual_kernel(double *__restrict__ r, const double *__restrict__ b,
                     const double *__restrict__ q, T *__restrict__ r_lo, long n, long n_plane, long n_valid,
                     double *__restrict__ partials, CgCtrl *__restrict__ ctrl, const Comm c)
{
    if (slab_dead(c.mine)) return;
    double s = 0.0;
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < n; i += (long)gridDim.x * BLAS_BLOCK) {
        const double bi = (n_valid == n_plane || i % n_plane < n_valid) ? b[i] : 0.0;   // b's pad lanes count as zero
        if (WHAT == RES_NORM) {
            const double v = bi;
            s += v * v;
        } else {
            const double v = bi - q[i];
            r[i] = v;
            if (r_lo != nullptr) r_lo[i] = (T)v;
            s += v * v;
        }
    }
    __shared__ double red[32];
    __shared__ double totals[MAX_RHS];
    const double bs = block_sum(s, red);
    if (!finish_reduction(bs, partials, &ctrl->ticket[2], red, totals)) return;
    if (threadIdx.x < 32) publish_next(c, totals[0]);
}

// The scalar step that follows a published reduction: gather the all-rank sum and run the same
// epilogue the one-GPU kernels run in their last block.  WHAT: RES_* or SCALAR_ITER.
enum { SCALAR_ITER = 100 };
template <int WHAT>
__global__ void slab_scalar_kernel(CgCtrl *__restrict__ ctrl, const Comm c)
{
    if (threadIdx.x >= 32 || blockIdx.x != 0) return;            // one warp
    if (WHAT == SCALAR_ITER && ctrl->state != CG_RUN) return;
    if (slab_dead(c.mine)) return;
    bool ok;
    double total = gather_current(c, &ok);
    if (!ok || threadIdx.x != 0) return;   // on a timeout the scalars stay as they were; the host reads STAG_ETIMEOUT
    if (WHAT == SCALAR_ITER) cg_iteration_epilogue(ctrl, &total);
    else residual_epilogue<WHAT>(ctrl, &total);
}

}  // namespace stag
