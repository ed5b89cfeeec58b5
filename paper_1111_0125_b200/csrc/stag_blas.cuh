// stag_blas.cuh -- the CG vector algebra of Fig. 1 as fused, streaming kernels.
//
// Vectors are the flat device spinors (n = 6*Vh_pad reals, pads zero); a solve carries nrhs of
// them back to back (right-hand side k starts k*n reals in) and every kernel here runs on a
// 2-D grid: blockIdx.y = k, blockIdx.x strides over the packets of that one vector, so each
// block works with the scalars of a single right-hand side.  Every inner product is accumulated
// in fp64 whatever the vector precision.  Reductions are two-stage and fixed-order:
// each block writes one partial, the last block of the whole grid to finish (ticket) adds the
// partials of every right-hand side in index order and runs the scalar epilogue (alpha, beta,
// stopping tests) on the device, so the host never reads a scalar inside the iteration.
#pragma once
#include "stag_common.cuh"
#include "stag_mem.cuh"

namespace stag {

constexpr int BLAS_BLOCK = 256;

template <typename T> struct Vec4;                       // 16-byte packets
template <> struct Vec4<float>  { using type = float4;  static constexpr int N = 4; };
template <> struct Vec4<double> { using type = double2; static constexpr int N = 2; };

template <typename T> __device__ __forceinline__ void unpack(const float4 &v, T *a)
{ a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w; }
template <typename T> __device__ __forceinline__ void unpack(const double2 &v, T *a)
{ a[0] = v.x; a[1] = v.y; }
__device__ __forceinline__ float4 pack(const float *a) { return make_float4(a[0], a[1], a[2], a[3]); }
__device__ __forceinline__ double2 pack(const double *a) { return make_double2(a[0], a[1]); }

// Second stage shared by all reducing kernels.  Every block calls it with its partial of
// right-hand side blockIdx.y; in the LAST block of the grid to arrive it returns true (to all
// threads) with totals[k] = sum of partials[k*gridDim.x .. +gridDim.x) in index order for every
// k < gridDim.y (totals is shared memory, MAX_RHS doubles).
__device__ __forceinline__ bool finish_reduction(double block_value, double *partials,
                                                 unsigned *ticket, double *red, double *totals)
{
    __shared__ bool last;
    if (threadIdx.x == 0) {
        partials[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = block_value;
        __threadfence();
        last = (atomicAdd(ticket, 1u) == gridDim.x * gridDim.y - 1);
    }
    __syncthreads();
    if (!last) return false;
    for (unsigned k = 0; k < gridDim.y; ++k) {
        double t = 0.0;
        for (unsigned i = threadIdx.x; i < gridDim.x; i += blockDim.x)
            t += __ldcg(partials + (size_t)k * gridDim.x + i);
        t = block_sum(t, red);
        if (threadIdx.x == 0) totals[k] = t;
    }
    if (threadIdx.x == 0) *ticket = 0;
    __syncthreads();
    return true;
}

// ---- paired fp32 batches (stag_dslash.cuh; include/stag.h "batch layouts") -----------------------
// The fp32 vectors of a solve with nrhs >= 2 are kept paired: unit u = blockIdx.y of the vector
// kernels is, for u < nrhs/2, right-hand sides 2u and 2u+1 interleaved per complex number (16-byte
// packets (re_a, im_a, re_b, im_b), 2n reals starting 2u*n reals in), and, for odd nrhs, one last
// unit that is the ordinary spinor nrhs-1.  Each half of a packet is updated with the scalars of
// its own right-hand side; a frozen half is written back unchanged.
// Position of real i of right-hand side k inside a batch of nrhs spinors of n reals each:
__host__ __device__ inline size_t batch_index(int k, long i, long n, int nrhs, bool paired)
{
    if (!paired || k >= (nrhs / 2) * 2) return (size_t)k * n + i;
    return (size_t)(k / 2) * 2 * n + (size_t)(i >> 1) * 4 + (size_t)(k & 1) * 2 + (size_t)(i & 1);
}

// d = r + beta d   (Fig. 1; eq. 3.1 P:L91 when it follows an update).  beta = 0
// makes it d = r, which is how the iteration starts and restarts.
template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK)
xpay_kernel(T *__restrict__ d, const T *__restrict__ r, long n, const CgCtrl *__restrict__ ctrl)
{
    const int k = blockIdx.y;
    if (ctrl->state != CG_RUN || !ctrl->active[k]) return;
    using V = typename Vec4<T>::type;
    constexpr int N = Vec4<T>::N;
    const T beta = (T)ctrl->beta[k];
    const long nv = n / N;
    V *dk = reinterpret_cast<V *>(d + (size_t)k * n);
    const V *rk = reinterpret_cast<const V *>(r + (size_t)k * n);
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < nv; i += (long)gridDim.x * BLAS_BLOCK) {
        T a[N], b[N];
        unpack<T>(ld_keep(rk + i), a);
        unpack<T>(ld_keep(dk + i), b);
        if (beta == (T)0) {
#pragma unroll
            for (int j = 0; j < N; ++j) b[j] = a[j];
        } else {
#pragma unroll
            for (int j = 0; j < N; ++j) b[j] = fma(beta, b[j], a[j]);
        }
        st_keep(dk + i, pack(b));
    }
}

// ---- the vector kernels on a paired fp32 batch ------------------------------------------------
// One-dimensional grid of nrhs*B blocks, every block the same number of packets: pair u (twice the
// data of a single right-hand side) owns blocks [u*2B, (u+1)*2B), an odd last right-hand side the
// last B blocks.  (A 2-D grid with as many blocks per pair as per single leaves half the SMs idle
// while the pairs finish.)
struct PairedUnit {
    int k0;        // first right-hand side of the unit
    bool pair;     // two right-hand sides interleaved per complex number, or one ordinary spinor
    int lb, nb;    // this block's index inside the unit, blocks in the unit
};
__device__ __forceinline__ PairedUnit paired_unit(int nrhs)
{
    const int B = gridDim.x / nrhs, npairs = nrhs / 2, b = blockIdx.x;
    PairedUnit u;
    if (b < npairs * 2 * B) { u.k0 = 2 * (b / (2 * B)); u.pair = true; u.lb = b % (2 * B); u.nb = 2 * B; }
    else { u.k0 = 2 * npairs; u.pair = false; u.lb = b - npairs * 2 * B; u.nb = B; }
    return u;
}

__global__ void __launch_bounds__(BLAS_BLOCK)
xpay_paired_kernel(float *__restrict__ d, const float *__restrict__ r, long n, const CgCtrl *__restrict__ ctrl)
{
    if (ctrl->state != CG_RUN) return;
    const PairedUnit u = paired_unit(ctrl->nrhs);
    float4 *dk = reinterpret_cast<float4 *>(d + (size_t)u.k0 * n);
    const float4 *rk = reinterpret_cast<const float4 *>(r + (size_t)u.k0 * n);
    if (u.pair) {
        const bool act_a = ctrl->active[u.k0], act_b = ctrl->active[u.k0 + 1];
        if (!act_a && !act_b) return;
        const float beta_a = (float)ctrl->beta[u.k0], beta_b = (float)ctrl->beta[u.k0 + 1];
        const long nv = n / 2;                       // packets of the pair: one complex number of each
        for (long i = u.lb * (long)BLAS_BLOCK + threadIdx.x; i < nv; i += (long)u.nb * BLAS_BLOCK) {
            const float4 a = ld_keep(rk + i);
            float4 b = ld_keep(dk + i);
            if (act_a) {
                b.x = (beta_a == 0.f) ? a.x : fma(beta_a, b.x, a.x);
                b.y = (beta_a == 0.f) ? a.y : fma(beta_a, b.y, a.y);
            }
            if (act_b) {
                b.z = (beta_b == 0.f) ? a.z : fma(beta_b, b.z, a.z);
                b.w = (beta_b == 0.f) ? a.w : fma(beta_b, b.w, a.w);
            }
            st_keep(dk + i, b);
        }
        return;
    }
    if (!ctrl->active[u.k0]) return;
    const float beta = (float)ctrl->beta[u.k0];
    const long nv = n / 4;
    for (long i = u.lb * (long)BLAS_BLOCK + threadIdx.x; i < nv; i += (long)u.nb * BLAS_BLOCK) {
        const float4 a = ld_keep(rk + i);
        float4 b = ld_keep(dk + i);
        if (beta == 0.f) b = a;
        else { b.x = fma(beta, b.x, a.x); b.y = fma(beta, b.y, a.y); b.z = fma(beta, b.z, a.z); b.w = fma(beta, b.w, a.w); }
        st_keep(dk + i, b);
    }
}

// Sum of v[0..n) in a fixed order, the same in every block, returned to ALL threads of the
// block: every block that calls it with the same arguments gets the same bits.
__device__ __forceinline__ double block_total_fixed(const double *__restrict__ v, int n, double *red)
{
    // eight independent loads in flight per thread (a one-load-per-trip loop costs one L2
    // round trip per element: 13 us of the 37 us update_kernel took on 28^3 x 96); the adds
    // stay in index order, and an out-of-range slot adds +0.0, which changes nothing
    double t = 0.0;
    for (int base = threadIdx.x; base < n; base += 8 * blockDim.x) {
        double e[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int i = base + u * blockDim.x;
            e[u] = (i < n) ? __ldcg(v + i) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) t += e[u];
    }
    t = block_sum(t, red);
    __shared__ double total;
    if (threadIdx.x == 0) total = t;
    __syncthreads();
    return total;
}

// The scalar part of one pass of Fig. 1's loop plus the stopping / trigger tests
// (Q9-Q11), for every right-hand side, given totals[j] = the new |r_j|^2.  One thread.
// Shared by update_kernel (one GPU) and the slab path's scalar kernel (stag_slab.cuh), where
// totals are sums over all ranks and every rank runs this on identical inputs.
__device__ __forceinline__ void cg_iteration_epilogue(CgCtrl *__restrict__ ctrl, const double *totals)
{
    const int it = ctrl->iter + 1, mode = ctrl->mode, nrhs = ctrl->nrhs;
    ctrl->iter = it;
    bool breakdown = false, trigger = false;
    unsigned conv = 0;
    for (int j = 0; j < nrhs; ++j) {
        if (!ctrl->active[j]) continue;
        ctrl->iters[j] += 1;
        const double dn = totals[j];
        ctrl->sum1[j] = dn;
        // dAd[j] was written by another block of this launch: read it past L1
        if (!(__ldcg(&ctrl->dAd[j]) > 0.0) || !(dn == dn)) { breakdown = true; continue; }
        if (mode == STAG_CG_RELIABLE) {
            const double rn = sqrt(dn);
            if (dn <= ctrl->tol2b[j] || rn < ctrl->eps_in * ctrl->maxr[j]) trigger = true;   // P:L97, Q11
            else ctrl->maxr[j] = fmax(ctrl->maxr[j], rn);                                    // Q9
        } else if (mode == STAG_CG_DEFECT) {
            if (dn <= ctrl->inner2[j]) conv |= 1u << j;                                      // Fig. 2 inner
        } else {
            if (dn <= ctrl->tol2b[j]) conv |= 1u << j;                                       // Fig. 1
        }
    }
    int st = CG_RUN;
    if (breakdown) st = CG_BREAKDOWN;
    else if (trigger) st = CG_UPDATE;     // beta is then formed from the corrected residuals (Q10)
    else {
        bool any = false;
        for (int j = 0; j < nrhs; ++j) {
            if (!ctrl->active[j]) continue;
            const double dn = totals[j];
            ctrl->beta[j] = dn / ctrl->delta[j];
            ctrl->delta[j] = dn;
            if (conv & (1u << j)) ctrl->active[j] = 0;      // this right-hand side is done: freeze it
            else any = true;
        }
        if (!any) st = CG_CONVERGED;
    }
    if (st == CG_RUN && it >= ctrl->maxiter) st = CG_MAXITER;
    ctrl->state = st;
}

// alpha = delta / <d,Ad> ; y += alpha d ; r -= alpha q ; delta' = |r|^2 ; then the scalar part
// of the iteration (P:L51-54 and the trigger of P:L97) in the last block, for every right-hand
// side.  <d,Ad> arrives as the per-block partial sums of the second hop (stag_dslash.cuh): every
// block of right-hand side k adds the n_hop partials of k in the same order, so all of them use
// the same alpha and no extra launch or device-wide fence is needed between the hop and this
// kernel.  A frozen right-hand side (active == 0) is not touched.
template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK)
update_kernel(T *__restrict__ y, T *__restrict__ r, const T *__restrict__ d,
              const T *__restrict__ q, long n, const double *__restrict__ hop_partials,
              int n_hop, double *__restrict__ partials, CgCtrl *__restrict__ ctrl)
{
    if (ctrl->state != CG_RUN) return;
    using V = typename Vec4<T>::type;
    constexpr int N = Vec4<T>::N;
    __shared__ double red[32];
    __shared__ double totals[MAX_RHS];
    const int k = blockIdx.y;
    double s = 0.0;
    if (ctrl->active[k]) {
        const double dAd = block_total_fixed(hop_partials + (size_t)k * n_hop, n_hop, red);
        const bool ok = dAd > 0.0;                       // false also for NaN
        const double alpha_d = ok ? ctrl->delta[k] / dAd : 0.0;   // alpha = delta_new / d^dag A d
        if (blockIdx.x == 0 && threadIdx.x == 0) { ctrl->dAd[k] = dAd; ctrl->alpha[k] = alpha_d; }
        const T alpha = (T)alpha_d;
        const long nv = n / N;
        V *yk = reinterpret_cast<V *>(y + (size_t)k * n);
        V *rk = reinterpret_cast<V *>(r + (size_t)k * n);
        const V *dk = reinterpret_cast<const V *>(d + (size_t)k * n);
        const V *qk = reinterpret_cast<const V *>(q + (size_t)k * n);
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
    }
    const double bs = block_sum(s, red);
    if (!finish_reduction(bs, partials, &ctrl->ticket[1], red, totals)) return;
    if (threadIdx.x != 0) return;

    cg_iteration_epilogue(ctrl, totals);
}

// The same on a paired fp32 batch (grid and units: paired_unit above).  Partial sums of right-hand
// side k sit in partials[k*S + block-in-unit], S = 2B slots per right-hand side.
__global__ void __launch_bounds__(BLAS_BLOCK)
update_paired_kernel(float *__restrict__ y, float *__restrict__ r, const float *__restrict__ d,
                     const float *__restrict__ q, long n, const double *__restrict__ hop_partials,
                     int n_hop, double *__restrict__ partials, CgCtrl *__restrict__ ctrl)
{
    if (ctrl->state != CG_RUN) return;
    __shared__ double red[32];
    __shared__ double totals[MAX_RHS];
    __shared__ bool last;
    const int nrhs = ctrl->nrhs;
    const PairedUnit u = paired_unit(nrhs);
    const int S = 2 * (gridDim.x / nrhs);
    const int ka = u.k0, kb = u.k0 + 1;
    const bool act_a = ctrl->active[ka], act_b = u.pair && ctrl->active[kb];
    double s2[2] = {0.0, 0.0};
    if (act_a || act_b) {
        double ad[2] = {0.0, 0.0};
        if (act_a) {
            const double dAd = block_total_fixed(hop_partials + (size_t)ka * n_hop, n_hop, red);
            ad[0] = (dAd > 0.0) ? ctrl->delta[ka] / dAd : 0.0;                       // P:L51; 0 also for NaN
            if (u.lb == 0 && threadIdx.x == 0) { ctrl->dAd[ka] = dAd; ctrl->alpha[ka] = ad[0]; }
        }
        if (act_b) {
            const double dAd = block_total_fixed(hop_partials + (size_t)kb * n_hop, n_hop, red);
            ad[1] = (dAd > 0.0) ? ctrl->delta[kb] / dAd : 0.0;
            if (u.lb == 0 && threadIdx.x == 0) { ctrl->dAd[kb] = dAd; ctrl->alpha[kb] = ad[1]; }
        }
        float4 *yk = reinterpret_cast<float4 *>(y + (size_t)ka * n);
        float4 *rk = reinterpret_cast<float4 *>(r + (size_t)ka * n);
        const float4 *dk = reinterpret_cast<const float4 *>(d + (size_t)ka * n);
        const float4 *qk = reinterpret_cast<const float4 *>(q + (size_t)ka * n);
        // pair: halves .xy / .zw belong to ka / kb; single: the whole packet belongs to ka
        const float al_a = (float)ad[0], al_b = u.pair ? (float)ad[1] : al_a;
        const bool upd_xy = act_a, upd_zw = u.pair ? act_b : act_a;
        const long nv = u.pair ? n / 2 : n / 4;
        for (long i = u.lb * (long)BLAS_BLOCK + threadIdx.x; i < nv; i += (long)u.nb * BLAS_BLOCK) {
            float4 yy = ld_pass(yk + i), rr = ld_keep(rk + i);
            const float4 dd = ld_keep(dk + i), qq = ld_keep(qk + i);
            double sxy = 0.0, szw = 0.0;
            if (upd_xy) {
                yy.x = fma(al_a, dd.x, yy.x); yy.y = fma(al_a, dd.y, yy.y);
                rr.x = fma(-al_a, qq.x, rr.x); rr.y = fma(-al_a, qq.y, rr.y);
                sxy = (double)rr.x * (double)rr.x + (double)rr.y * (double)rr.y;
            }
            if (upd_zw) {
                yy.z = fma(al_b, dd.z, yy.z); yy.w = fma(al_b, dd.w, yy.w);
                rr.z = fma(-al_b, qq.z, rr.z); rr.w = fma(-al_b, qq.w, rr.w);
                szw = (double)rr.z * (double)rr.z + (double)rr.w * (double)rr.w;
            }
            s2[0] += sxy;
            if (u.pair) s2[1] += szw; else s2[0] += szw;
            st_pass(yk + i, yy);
            st_keep(rk + i, rr);
        }
    }
    double bs[2];
    bs[0] = block_sum(s2[0], red);
    bs[1] = block_sum(s2[1], red);
    if (threadIdx.x == 0) {
        partials[(size_t)ka * S + u.lb] = bs[0];
        if (u.pair) partials[(size_t)kb * S + u.lb] = bs[1];
        __threadfence();
        last = (atomicAdd(&ctrl->ticket[1], 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    for (int k = 0; k < nrhs; ++k) {       // fixed order; a frozen right-hand side's slots hold old values nobody reads
        const int nbk = (k < (nrhs / 2) * 2) ? S : S / 2;
        double t = 0.0;
        for (int i = threadIdx.x; i < nbk; i += blockDim.x) t += __ldcg(partials + (size_t)k * S + i);
        t = block_sum(t, red);
        if (threadIdx.x == 0) totals[k] = t;
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    ctrl->ticket[1] = 0;
    cg_iteration_epilogue(ctrl, totals);
}

// x64 += y ; y = 0  (group-wise update); the vectors are nrhs*n reals long
template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK)
accumulate_kernel(double *__restrict__ x, T *__restrict__ y, long n)
{
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < n; i += (long)gridDim.x * BLAS_BLOCK) {
        x[i] += (double)y[i];
        y[i] = (T)0;
    }
}
// The same for the pairs of a paired fp32 batch (y) against the blocked fp64 batch (x): one thread
// per (pair, complex number); npairs*n/2 packets.
__global__ void __launch_bounds__(BLAS_BLOCK)
accumulate_paired_kernel(double *__restrict__ x, float *__restrict__ y, long n, int npairs)
{
    const long nv = n / 2;
    float4 *yp = reinterpret_cast<float4 *>(y);
    for (long t = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; t < nv * npairs; t += (long)gridDim.x * BLAS_BLOCK) {
        const long j = t / nv, i = t % nv;
        const float4 v = yp[t];
        double2 *xa = reinterpret_cast<double2 *>(x + (size_t)(2 * j) * n) + i;
        double2 *xb = reinterpret_cast<double2 *>(x + (size_t)(2 * j + 1) * n) + i;
        double2 a = *xa, b = *xb;
        a.x += (double)v.x; a.y += (double)v.y;
        b.x += (double)v.z; b.y += (double)v.w;
        *xa = a; *xb = b;
        yp[t] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// Zero the pad lanes cb in [Vh, Vh_pad) of the three colour planes of spinor blockIdx.y of a batch.
template <typename C>
__global__ void zero_pads_kernel(C *__restrict__ v, int Vh, int Vh_pad)
{
    C *vk = v + (size_t)blockIdx.y * 3 * Vh_pad;
    const int npad = Vh_pad - Vh;
    for (int i = threadIdx.x; i < 3 * npad; i += blockDim.x) {
        C z; z.x = 0; z.y = 0;
        vk[(size_t)(i / npad) * Vh_pad + Vh + i % npad] = z;
    }
}

enum { RES_INIT = 0, RES_UPDATE = 1, RES_FINAL = 2, RES_NORM = 3 };

// Scalar part of residual_kernel (see there), given totals[k] = |r_k|^2 (or |b_k|^2).  One thread.
template <int WHAT>
__device__ __forceinline__ void residual_epilogue(CgCtrl *__restrict__ ctrl, const double *totals)
{
    const int nrhs = ctrl->nrhs;
    bool any = false, bad = false;
    for (int k = 0; k < nrhs; ++k) {
        const double dn = totals[k];
        if (WHAT == RES_NORM) { ctrl->bnorm2[k] = dn; continue; }
        ctrl->sum0[k] = dn;
        if (WHAT == RES_FINAL) continue;
        if (!(dn == dn)) { bad = true; continue; }
        if (WHAT == RES_INIT) {
            ctrl->delta[k] = dn;
            ctrl->beta[k] = 0.0;
            ctrl->maxr[k] = sqrt(dn);
            ctrl->inner2[k] = fmax(ctrl->eps_in * ctrl->eps_in * dn, ctrl->tol2b[k]);   // Fig. 2, Q8
            ctrl->active[k] = dn > ctrl->tol2b[k];
        } else if (ctrl->active[k]) {                     // RES_UPDATE
            ctrl->maxr[k] = sqrt(dn);                                                   // Q9
            if (dn <= ctrl->tol2b[k]) ctrl->active[k] = 0;
            else {
                ctrl->beta[k] = dn / ctrl->delta[k];                                    // Q10
                ctrl->delta[k] = dn;
            }
        }
        any = any || ctrl->active[k];
    }
    if (WHAT == RES_NORM || WHAT == RES_FINAL) return;
    if (WHAT == RES_UPDATE) ctrl->n_updates += 1;
    int st = any ? CG_RUN : CG_CONVERGED;
    if (bad) st = CG_BREAKDOWN;
    else if (any && ctrl->iter >= ctrl->maxiter) st = CG_MAXITER;
    ctrl->state = st;
}

// r = b - q in fp64, |r|^2, and optionally the fp32 copy of r (reliable update), for
// every right-hand side.  With WHAT == RES_NORM it only computes |b|^2.  The last block then
// sets the solver scalars of each right-hand side k:
//   RES_INIT   start, restart or outer step: delta = |r|^2, beta = 0, maxr = |r|, and k is
//              active iff |r|^2 > tol^2 |b|^2
//   RES_UPDATE after x += y (eq. 3.1): beta = |r|^2 / delta_old, delta = |r|^2;
//              an active k whose true residual meets the target is frozen
//   RES_FINAL  exit: only report |r|^2
// b is the caller's and read-only: its pad lanes (reals [n_valid, n_plane) of each colour plane,
// n_plane = 2 Vh_pad, n_valid = 2 Vh) are taken as zero whatever they hold, so no stray value can
// enter |b|^2, |r|^2 or the stopping tests.
template <typename T, int WHAT>
__global__ void __launch_bounds__(BLAS_BLOCK)
residual_kernel(double *__restrict__ r, const double *__restrict__ b,
                const double *__restrict__ q, T *__restrict__ r_lo, long n, long n_plane, long n_valid,
                double *__restrict__ partials, CgCtrl *__restrict__ ctrl, const bool lo_paired = false)
{
    const size_t off = (size_t)blockIdx.y * n;
    double s = 0.0;
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < n; i += (long)gridDim.x * BLAS_BLOCK) {
        const double bi = (n_valid == n_plane || i % n_plane < n_valid) ? b[off + i] : 0.0;
        if (WHAT == RES_NORM) {
            const double v = bi;
            s += v * v;
        } else {
            const double v = bi - q[off + i];
            r[off + i] = v;
            if (r_lo != nullptr) r_lo[batch_index((int)blockIdx.y, i, n, (int)gridDim.y, lo_paired)] = (T)v;   // the fp32 copy in its batch layout
            s += v * v;
        }
    }
    __shared__ double red[32];
    __shared__ double totals[MAX_RHS];
    const double bs = block_sum(s, red);
    if (!finish_reduction(bs, partials, &ctrl->ticket[2], red, totals)) return;
    if (threadIdx.x != 0) return;

    residual_epilogue<WHAT>(ctrl, totals);
}

}  // namespace stag
