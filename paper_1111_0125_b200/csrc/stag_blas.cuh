// stag_blas.cuh -- the CG vector algebra of Fig. 1 as fused, streaming kernels.
//
// Vectors are the flat device spinors (6*Vh_pad reals, pads zero).  Every inner product is
// accumulated in fp64 whatever the vector precision.  Reductions are two-stage and
// fixed-order: each block writes one partial, the last block to finish (ticket) adds the
// partials in index order and runs the scalar epilogue (alpha, beta, stopping tests) on the
// device, so the host never reads a scalar inside the iteration.
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

// Second stage shared by all reducing kernels: returns true in thread 0 of the last block with
// *total = sum of partials[0..gridDim.x) in fixed order.
__device__ __forceinline__ bool finish_reduction(double block_value, double *partials,
                                                 unsigned *ticket, double *red, double *total)
{
    __shared__ bool last;
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = block_value;
        __threadfence();
        last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return false;
    double t = 0.0;
    for (unsigned i = threadIdx.x; i < gridDim.x; i += blockDim.x) t += __ldcg(partials + i);
    t = block_sum(t, red);
    if (threadIdx.x == 0) { *total = t; *ticket = 0; return true; }
    return false;
}

// d = r + beta d   (Fig. 1; eq. 3.1 P:L91 when it follows an update).  beta = 0
// makes it d = r, which is how the iteration starts and restarts.
template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK)
xpay_kernel(T *__restrict__ d, const T *__restrict__ r, long n, const CgCtrl *__restrict__ ctrl)
{
    if (ctrl->state != CG_RUN) return;
    using V = typename Vec4<T>::type;
    constexpr int N = Vec4<T>::N;
    const T beta = (T)ctrl->beta;
    const long nv = n / N;
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < nv; i += (long)gridDim.x * BLAS_BLOCK) {
        T a[N], b[N];
        unpack<T>(ld_keep(reinterpret_cast<const V *>(r) + i), a);
        unpack<T>(ld_keep(reinterpret_cast<const V *>(d) + i), b);
        if (beta == (T)0) {
#pragma unroll
            for (int k = 0; k < N; ++k) b[k] = a[k];
        } else {
#pragma unroll
            for (int k = 0; k < N; ++k) b[k] = fma(beta, b[k], a[k]);
        }
        st_keep(reinterpret_cast<V *>(d) + i, pack(b));
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

// alpha = delta / <d,Ad> ; y += alpha d ; r -= alpha q ; delta' = |r|^2 ; then the scalar part
// of the iteration (P:L51-54 and the trigger of P:L97) in the last block.
// <d,Ad> arrives as the per-block partial sums of the second hop (stag_dslash.cuh); every block
// adds them in the same order, so all blocks use the same alpha and no extra launch or
// device-wide fence is needed between the hop and this kernel.
template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK)
update_kernel(T *__restrict__ y, T *__restrict__ r, const T *__restrict__ d,
              const T *__restrict__ q, long n, const double *__restrict__ hop_partials,
              int n_hop_partials, double *__restrict__ partials, CgCtrl *__restrict__ ctrl)
{
    if (ctrl->state != CG_RUN) return;
    using V = typename Vec4<T>::type;
    constexpr int N = Vec4<T>::N;
    __shared__ double red[32];
    const double dAd = block_total_fixed(hop_partials, n_hop_partials, red);
    const bool ok = dAd > 0.0;                       // false also for NaN
    const double alpha_d = ok ? ctrl->delta / dAd : 0.0;   // alpha = delta_new / d^dag A d
    const T alpha = (T)alpha_d;
    const long nv = n / N;
    double s = 0.0;
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < nv; i += (long)gridDim.x * BLAS_BLOCK) {
        T yy[N], rr[N], dd[N], qq[N];
        unpack<T>(ld_pass(reinterpret_cast<const V *>(y) + i), yy);
        unpack<T>(ld_keep(reinterpret_cast<const V *>(r) + i), rr);
        unpack<T>(ld_keep(reinterpret_cast<const V *>(d) + i), dd);
        unpack<T>(ld_keep(reinterpret_cast<const V *>(q) + i), qq);
#pragma unroll
        for (int k = 0; k < N; ++k) {
            yy[k] = fma(alpha, dd[k], yy[k]);
            rr[k] = fma(-alpha, qq[k], rr[k]);
            s += (double)rr[k] * (double)rr[k];
        }
        st_pass(reinterpret_cast<V *>(y) + i, pack(yy));
        st_keep(reinterpret_cast<V *>(r) + i, pack(rr));
    }
    double bs = block_sum(s, red), dn;
    if (!finish_reduction(bs, partials, &ctrl->ticket[1], red, &dn)) return;

    // ---- scalar epilogue, one thread ------------------------------------------------
    const int it = ctrl->iter + 1;
    ctrl->iter = it;
    ctrl->dAd = dAd;
    ctrl->alpha = alpha_d;
    int st = CG_RUN;
    if (!ok || !(dn == dn)) st = CG_BREAKDOWN;
    else if (ctrl->mode == STAG_CG_RELIABLE) {
        const double rn = sqrt(dn);
        if (dn <= ctrl->tol2b || rn < ctrl->eps_in * ctrl->maxr) st = CG_UPDATE;   // P:L97, Q11
        else ctrl->maxr = fmax(ctrl->maxr, rn);                                    // Q9
    } else if (ctrl->mode == STAG_CG_DEFECT) {
        if (dn <= ctrl->inner2) st = CG_CONVERGED;                                 // Fig. 2 inner
    } else {
        if (dn <= ctrl->tol2b) st = CG_CONVERGED;                                  // Fig. 1
    }
    if (st != CG_UPDATE) {            // on an update beta is formed from the corrected residual
        ctrl->beta = dn / ctrl->delta;
        ctrl->delta = dn;
    }
    if (st == CG_RUN && it >= ctrl->maxiter) st = CG_MAXITER;
    ctrl->sum1 = dn;
    ctrl->state = st;
}

// x64 += y ; y = 0  (group-wise update)
template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK)
accumulate_kernel(double *__restrict__ x, T *__restrict__ y, long n)
{
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < n; i += (long)gridDim.x * BLAS_BLOCK) {
        x[i] += (double)y[i];
        y[i] = (T)0;
    }
}

enum { RES_INIT = 0, RES_UPDATE = 1, RES_FINAL = 2, RES_NORM = 3 };

// r = b - q in fp64, |r|^2, and optionally the fp32 copy of r (reliable update).
// With WHAT == RES_NORM it only computes |b|^2.  The last block then sets the solver scalars:
//   RES_INIT   start or restart: delta = |r|^2, beta = 0, maxr = |r|
//   RES_UPDATE after x += y (eq. 3.1): beta = |r|^2 / delta_old, delta = |r|^2
//   RES_FINAL  exit: only report |r|^2
template <typename T, int WHAT>
__global__ void __launch_bounds__(BLAS_BLOCK)
residual_kernel(double *__restrict__ r, const double *__restrict__ b,
                const double *__restrict__ q, T *__restrict__ r_lo, long n,
                double *__restrict__ partials, CgCtrl *__restrict__ ctrl)
{
    double s = 0.0;
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < n; i += (long)gridDim.x * BLAS_BLOCK) {
        if (WHAT == RES_NORM) {
            const double v = b[i];
            s += v * v;
        } else {
            const double v = b[i] - q[i];
            r[i] = v;
            if (r_lo != nullptr) r_lo[i] = (T)v;
            s += v * v;
        }
    }
    __shared__ double red[32];
    double bs = block_sum(s, red), dn;
    if (!finish_reduction(bs, partials, &ctrl->ticket[2], red, &dn)) return;

    ctrl->sum0 = dn;
    if (WHAT == RES_NORM) {
        ctrl->bnorm2 = dn;
    } else if (WHAT == RES_INIT) {
        ctrl->delta = dn;
        ctrl->beta = 0.0;
        ctrl->maxr = sqrt(dn);
        ctrl->inner2 = fmax(ctrl->eps_in * ctrl->eps_in * dn, ctrl->tol2b);   // Fig. 2, Q8
        int st = CG_RUN;
        if (!(dn == dn)) st = CG_BREAKDOWN;
        else if (dn <= ctrl->tol2b) st = CG_CONVERGED;
        else if (ctrl->iter >= ctrl->maxiter) st = CG_MAXITER;
        ctrl->state = st;
    } else if (WHAT == RES_UPDATE) {
        ctrl->n_updates += 1;
        ctrl->maxr = sqrt(dn);                                                // Q9
        int st = CG_RUN;
        if (!(dn == dn)) st = CG_BREAKDOWN;
        else if (dn <= ctrl->tol2b) st = CG_CONVERGED;
        else {
            ctrl->beta = dn / ctrl->delta;                                    // Q10
            ctrl->delta = dn;
            if (ctrl->iter >= ctrl->maxiter) st = CG_MAXITER;
        }
        ctrl->state = st;
    }
}

// dst = (T) src, elementwise (precision change of a device spinor)
template <typename TD, typename TS>
__global__ void __launch_bounds__(BLAS_BLOCK)
convert_kernel(TD *__restrict__ dst, const TS *__restrict__ src, long n)
{
    for (long i = blockIdx.x * (long)BLAS_BLOCK + threadIdx.x; i < n; i += (long)gridDim.x * BLAS_BLOCK)
        dst[i] = (TD)src[i];
}

}  // namespace stag
