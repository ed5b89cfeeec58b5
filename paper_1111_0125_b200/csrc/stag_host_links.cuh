// stag_host_links.cuh -- setup step S0 (gather / derive kernels), the hop launchers and the C ABI of links, spinors and the operator
//
// A section of libstag's single translation unit: included by stag_lib.cu, which holds the
// per-thread state, the error / launch-count helpers and the link handle these sections share.
// Not a stand-alone header.

namespace {

size_t links_elems(const stag_links *L, int rows)   // complex numbers in one gathered field
{
    return (size_t)2 * L->ntiles * 8 * link_slots(rows) * TILE;
}

// ---- S0 kernels ----------------------------------------------------------------------

// canonical W[mu][p][cb][3][3] (fp64) -> gathered fp64/18 field L[p][tile][d][k][lane]; also
// measures how well row 2 is rebuilt from rows 0,1 (Q12).  fold = 0: W already carries
// eta*bc (the caller folded it); fold = 1: W is the bare U and each link is multiplied
// here by eta_mu(x') bc_mu(x') of ITS OWN site x' (x for the forward link, x - mu^ for the
// backward one), the device-side form of the paper's "gauge link preconditioning".
// The sign comes from det_sign_mask: det M_d = eta bc for d < 4 and -(eta bc) for d >= 4.
// g is the geometry of the lattice the handle covers, gg that of the whole lattice: the same
// for a whole-lattice handle; for a T-slab g is the slab (time slices [g.t0, g.t0 + g.X3) of gg).
// src says where the canonical links are: the whole field (stag_links_create, stag_slab_create from
// device memory), or only the slab's own time slices plus the t-links of the slice before it, which
// are the backward t-links of the slab's first slice and belong to the neighbouring slab
// (stag_slab_create_local): no rank then ever holds the whole lattice.
struct LinkSrc {
    const double *W;       // [mu][p][vh][3][3], cb index = global cb - off
    const double *Wback;   // [p][s3][3][3]: W_3 on time slice t0-1 (mod X3g); null when W holds it
    long vh;               // sites per (mu, p) plane of W
    long off;              // t0*s3 for a slab's own part, 0 for the whole field
};

__global__ void __launch_bounds__(128)
gather_links_kernel(double2 *__restrict__ L, const LinkSrc src_, const Geom g,
                    const Geom gg, unsigned long long *__restrict__ err_bits, const int fold)
{
    const double *__restrict__ W = src_.W;
    const long idx = blockIdx.x * 128L + threadIdx.x;
    if (idx >= 2L * g.Vh_pad) return;
    const int p = (int)(idx / g.Vh_pad);
    const int cb = (int)(idx % g.Vh_pad);
    double2 *dst = L + ((size_t)p * (g.Vh_pad / TILE) + (cb >> 5)) * (size_t)(8 * 9 * TILE) + (cb & 31);
    if (cb >= g.Vh) {
        for (int k = 0; k < 72; ++k) dst[k * TILE] = make_double2(0.0, 0.0);
        return;
    }
    // time slices are contiguous in the checkerboard index: global cb = local cb + t0 * s3
    const int cbg = cb + g.t0 * g.s3;
    Site s;
    decode_site(gg, p, cbg, s);                 // global coordinates and global neighbours
    const unsigned neg = det_sign_mask(gg, s);
    double worst = 0.0;
    for (int d = 0; d < 8; ++d) {
        double2 m[9];
        if (d < 4) {
            const double *src = W + (((size_t)d * 2 + p) * src_.vh + (cbg - src_.off)) * 18;
            for (int k = 0; k < 9; ++k) m[k] = make_double2(src[2 * k], src[2 * k + 1]);
        } else {
            const long at = (long)s.nbr[d] - src_.off;
            const double *src = W + (((size_t)(d - 4) * 2 + (1 - p)) * src_.vh + at) * 18;
            if (at < 0 || at >= src_.vh)      // only d = 7 on the slab's first slice: the neighbour slab's t-link
                src = src_.Wback + ((size_t)(1 - p) * gg.s3 + (s.nbr[d] % gg.s3)) * 18;
            for (int i = 0; i < 3; ++i)
                for (int j = 0; j < 3; ++j)   // M = -W^dag : M_ij = -conj(W_ji)
                    m[3 * i + j] = make_double2(-src[2 * (3 * j + i)], src[2 * (3 * j + i) + 1]);
        }
        if (fold) {
            const bool det_neg = (neg >> d) & 1u;
            const double sg = (d < 4) ? (det_neg ? -1.0 : 1.0) : (det_neg ? 1.0 : -1.0);
            for (int k = 0; k < 9; ++k) { m[k].x *= sg; m[k].y *= sg; }
        }
        for (int k = 0; k < 9; ++k) dst[(d * 9 + k) * TILE] = m[k];
        double2 t[9];
        for (int k = 0; k < 6; ++k) t[k] = m[k];
        rebuild_row2<double>(t, (neg >> d) & 1u);
        for (int j = 0; j < 3; ++j) {
            const double ex = fabs(t[6 + j].x - m[6 + j].x), ey = fabs(t[6 + j].y - m[6 + j].y);
            if (!(ex == ex) || !(ey == ey)) worst = 1e300;   // fmax would drop a NaN
            else worst = fmax(worst, fmax(ex, ey));
        }
    }
    atomicMax(err_bits, (unsigned long long)__double_as_longlong(worst));   // worst >= 0
}

// fp64/18 gathered field -> another precision / row count, in the packet layout of
// stag_dslash.cuh: dst[tile][j][lane], packet j = complex numbers CPP*j .. CPP*j+CPP-1 of the
// site's run c = d*K + k.  n_pkt = packets in dst (both parities).
template <typename TD, int ROWS>
__global__ void __launch_bounds__(256)
derive_links_kernel(pkt_t<TD> *__restrict__ dst, const double2 *__restrict__ src, long n_pkt)
{
    constexpr int K = 3 * ROWS;
    constexpr int CPP = Pkt<TD>::CPP;
    constexpr int PPS = 8 * K / CPP;             // packets per site
    const long i = blockIdx.x * 256L + threadIdx.x;
    if (i >= n_pkt) return;
    const int lane = (int)(i % TILE);
    const long r = i / TILE;
    const int j = (int)(r % PPS);
    const long tile = r / PPS;                   // p*ntiles + tile
    TD v[2 * CPP];
#pragma unroll
    for (int h = 0; h < CPP; ++h) {
        const int c = CPP * j + h, d = c / K, k = c % K;
        const double2 w = src[((tile * 8 + d) * 9 + k) * TILE + lane];
        v[2 * h] = (TD)w.x;
        v[2 * h + 1] = (TD)w.y;
    }
    dst[i] = pack(v);
}

// fp64/18 gathered field -> the 8-parameter form in precision TD (stag_dslash.cuh, rebuild_from8):
// one thread per (parity, site, direction) stores the four slots a2, a3, b1, (arg a1, arg c1) of
// U = s*M (s = det M from the site's coordinates), then rebuilds M from what it stored, in TD
// arithmetic, exactly as the hop will, and records the largest entry error against the fp64 M.
template <typename TD>
__global__ void __launch_bounds__(128)
derive_links8_kernel(pkt_t<TD> *__restrict__ dst, const double2 *__restrict__ src, const Geom g,
                     unsigned long long *__restrict__ err_bits)
{
    constexpr int CPP = Pkt<TD>::CPP;
    constexpr int PPS = 8 * 4 / CPP;             // packets per site
    const long idx = blockIdx.x * 128L + threadIdx.x;
    if (idx >= 2L * g.Vh_pad * 8) return;
    const int d = (int)(idx & 7);
    const long site = idx >> 3;                  // p * Vh_pad + cb
    const int p = (int)(site / g.Vh_pad);
    const int cb = (int)(site % g.Vh_pad);
    const long tile = site >> 5;
    const int lane = cb & 31;
    double2 M[9];
    for (int k = 0; k < 9; ++k) M[k] = src[((tile * 8 + d) * 9 + k) * TILE + lane];
    bool neg = false;
    if (cb < g.Vh) {
        Site s;
        decode_site(g, p, cb, s);
        neg = (det_sign_mask(g, s) >> d) & 1u;
    }
    const double sg = neg ? -1.0 : 1.0;
    cplx_t<TD> slot[9];
    slot[0] = mk<TD>((TD)(sg * M[1].x), (TD)(sg * M[1].y));      // a2
    slot[1] = mk<TD>((TD)(sg * M[2].x), (TD)(sg * M[2].y));      // a3
    slot[2] = mk<TD>((TD)(sg * M[3].x), (TD)(sg * M[3].y));      // b1
    slot[3] = mk<TD>((TD)atan2(sg * M[0].y, sg * M[0].x), (TD)atan2(sg * M[6].y, sg * M[6].x));
    if (cb >= g.Vh) {      // pad lanes: slots whose rebuild is finite (N = 1); the hop zeroes their output
        slot[0] = mk<TD>((TD)1, (TD)0);
        slot[1] = slot[2] = slot[3] = mk<TD>((TD)0, (TD)0);
    }
    TD v[2 * CPP];
    for (int j = 0; j < 4 / CPP; ++j) {
        for (int h = 0; h < CPP; ++h) { v[2 * h] = slot[CPP * j + h].x; v[2 * h + 1] = slot[CPP * j + h].y; }
        dst[(tile * PPS + (d * 4 / CPP + j)) * TILE + lane] = pack(v);
    }
    if (cb >= g.Vh) return;                      // pad lanes: no error to take
    rebuild_from8<TD>(slot, neg);
    double worst = 0.0;
    for (int k = 0; k < 9; ++k) {
        const double ex = fabs((double)slot[k].x - M[k].x), ey = fabs((double)slot[k].y - M[k].y);
        if (!(ex == ex) || !(ey == ey)) worst = 1e300;       // fmax would drop a NaN (0 * 1/0 at N = 0)
        else worst = fmax(worst, fmax(ex, ey));
    }
    atomicMax(err_bits, (unsigned long long)__double_as_longlong(worst));
}

template <typename T>
__global__ void __launch_bounds__(128)
spinor_pack_kernel(cplx_t<T> *__restrict__ dst, const double *__restrict__ src, int Vh, int Vh_pad)
{
    const int cb = blockIdx.x * 128 + threadIdx.x;
    if (cb >= Vh_pad) return;
    for (int c = 0; c < 3; ++c) {
        cplx_t<T> v = mk<T>(0, 0);
        if (cb < Vh) v = mk<T>((T)src[(size_t)cb * 6 + 2 * c], (T)src[(size_t)cb * 6 + 2 * c + 1]);
        dst[(size_t)c * Vh_pad + cb] = v;
    }
}

template <typename T>
__global__ void __launch_bounds__(128)
spinor_unpack_kernel(double *__restrict__ dst, const cplx_t<T> *__restrict__ src, int Vh, int Vh_pad)
{
    const int cb = blockIdx.x * 128 + threadIdx.x;
    if (cb >= Vh) return;
    for (int c = 0; c < 3; ++c) {
        const cplx_t<T> v = src[(size_t)c * Vh_pad + cb];
        dst[(size_t)cb * 6 + 2 * c] = (double)v.x;
        dst[(size_t)cb * 6 + 2 * c + 1] = (double)v.y;
    }
}

// Build (once) the gathered field of precision `prec` from the fp64/18 one.  Thread-safe: the
// first caller builds under the handle's mutex and synchronises its stream before the pointer is
// published, so a second thread (on another stream) never sees a field still being written.
int ensure_links_locked(const stag_links *L, int prec);
int ensure_links(const stag_links *L, int prec)
{
    if (!prec_ok(prec)) return STAG_EINVAL;
    if (L->L_ready[prec].load(std::memory_order_acquire)) return STAG_OK;
    std::lock_guard<std::mutex> lk(L->mu_links);
    if (L->L_ready[prec].load(std::memory_order_relaxed)) return STAG_OK;
    const int rc = ensure_links_locked(L, prec);
    if (rc == STAG_OK) L->L_ready[prec].store(1, std::memory_order_release);
    return rc;
}

int ensure_links_locked(const stag_links *L, int prec)
{
    const int rows = prec_rows(prec);
    if (rows == 2 && !(L->recon_err <= 1e-10)) {
        snprintf(t_errbuf, sizeof(t_errbuf),
                 "12-real links refused: row 2 is not s*conj(row0 x row1) (max error %.3g)", L->recon_err);
        t_errbuf_status = STAG_EINVAL;
        return STAG_EINVAL;
    }
    const size_t bytes = links_elems(L, rows) * (prec_is_f32(prec) ? sizeof(float2) : sizeof(double2));
    const size_t n = bytes / 16;                 // 16-byte packets
    void *dst = nullptr;
    if (rows == 1) {
        // the 8-parameter form has no representation for a first row (a1,0,0) and loses accuracy
        // near it: build it, measure the rebuilt error in the arithmetic of the hop,
        // and refuse the field if it is beyond what that precision can mean
        const int f32 = prec_is_f32(prec) ? 1 : 0;
        const double limit = f32 ? 1e-3 : 1e-9;
        if (!(L->recon_err <= 1e-10)) {
            snprintf(t_errbuf, sizeof(t_errbuf), "8-parameter links refused: the links are not +-SU(3) (max error %.3g)", L->recon_err);
            t_errbuf_status = STAG_EINVAL;
            return STAG_EINVAL;
        }
        if (L->recon8_err[f32] >= 0.0 && !(L->recon8_err[f32] <= limit)) {     // refused before: same answer, no rebuild
            snprintf(t_errbuf, sizeof(t_errbuf),
                     "8-parameter links refused: rebuilt entries are off by up to %.3g (limit %.1g); a link with a first row near (a1,0,0) has no usable 8-parameter form",
                     L->recon8_err[f32], limit);
            t_errbuf_status = STAG_EINVAL;
            return STAG_EINVAL;
        }
        unsigned long long *err = nullptr;
        CU(cudaMalloc(&dst, bytes));
        if (cudaMalloc(&err, sizeof(*err)) != cudaSuccess) { cudaFree(dst); return STAG_ENOMEM; }
        cudaMemsetAsync(err, 0, sizeof(*err), t_stream);
        const unsigned g8 = (unsigned)((2L * L->g.Vh_pad * 8 + 127) / 128);
        const double2 *src8 = (const double2 *)L->L[STAG_PREC_F64];
        if (f32) derive_links8_kernel<float><<<g8, 128, 0, t_stream>>>((float4 *)dst, src8, L->g, err);
        else derive_links8_kernel<double><<<g8, 128, 0, t_stream>>>((double2 *)dst, src8, L->g, err);
        count_launch();
        unsigned long long bits = 0;
        cudaError_t e8 = cudaGetLastError();
        if (e8 == cudaSuccess) e8 = cudaMemcpyAsync(&bits, err, sizeof(bits), cudaMemcpyDeviceToHost, t_stream);
        if (e8 == cudaSuccess) e8 = cudaStreamSynchronize(t_stream);
        cudaFree(err);
        if (e8 != cudaSuccess) { cudaFree(dst); return cuda_fail(e8, "derive_links8_kernel", __LINE__); }
        memcpy(&L->recon8_err[f32], &bits, sizeof(double));
        if (!(L->recon8_err[f32] <= limit)) {
            cudaFree(dst);
            snprintf(t_errbuf, sizeof(t_errbuf),
                     "8-parameter links refused: rebuilt entries are off by up to %.3g (limit %.1g); a link with a first row near (a1,0,0) has no usable 8-parameter form",
                     L->recon8_err[f32], limit);
            t_errbuf_status = STAG_EINVAL;
            return STAG_EINVAL;
        }
        L->L[prec] = dst;
        return STAG_OK;
    }
    CU(cudaMalloc(&dst, bytes));
    const unsigned grid = (unsigned)((n + 255) / 256);
    const double2 *src = (const double2 *)L->L[STAG_PREC_F64];
    switch (prec) {
    case STAG_PREC_F32:     derive_links_kernel<float, 3><<<grid, 256, 0, t_stream>>>((float4 *)dst, src, (long)n); break;
    case STAG_PREC_F64_R12: derive_links_kernel<double, 2><<<grid, 256, 0, t_stream>>>((double2 *)dst, src, (long)n); break;
    case STAG_PREC_F32_R12: derive_links_kernel<float, 2><<<grid, 256, 0, t_stream>>>((float4 *)dst, src, (long)n); break;
    default: cudaFree(dst); return STAG_EINVAL;
    }
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(t_stream);     // published only once it is complete
    if (e != cudaSuccess) { cudaFree(dst); return cuda_fail(e, "derive_links_kernel", __LINE__); }
    L->L[prec] = dst;
    return STAG_OK;
}

// ---- Dslash launcher ---------------------------------------------------------------------
template <typename T, int NR, int N, bool PAIRED>
int launch_hop_n(const stag_links *L, int prec, int hop, cplx_t<T> *out, const cplx_t<T> *in,
                 int parity, double a, double cD, const cplx_t<T> *own, double *partials,
                 const CgCtrl *ctrl, cudaStream_t s)
{
    const Geom &g = L->g;
    const pkt_t<T> *field = (const pkt_t<T> *)L->L[prec] +
                            (size_t)parity * L->ntiles * (8 * link_slots(NR) / Pkt<T>::CPP) * TILE;
    const unsigned grid = (unsigned)((g.Vh_pad + DSLASH_BLOCK - 1) / DSLASH_BLOCK);
    switch (hop) {
    case HOP_PLAIN:
        dslash_kernel<T, NR, HOP_PLAIN, N, false, PAIRED><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)cD, own, partials, ctrl, HaloArgs<T>{});
        break;
    case HOP_XPAY:
        dslash_kernel<T, NR, HOP_XPAY, N, false, PAIRED><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)cD, own, partials, ctrl, HaloArgs<T>{});
        break;
    case HOP_AXPBY:   // only the fp64 wrapper steps use it
        if constexpr (std::is_same<T, double>::value)
            dslash_kernel<T, NR, HOP_AXPBY, N, false, PAIRED><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)cD, own, partials, ctrl, HaloArgs<T>{});
        else
            return STAG_EINVAL;
        break;
    default:
        dslash_kernel<T, NR, HOP_XPAY_DOT, N, false, PAIRED><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)cD, own, partials, ctrl, HaloArgs<T>{});
        break;
    }
    count_launch();
    KCHECK();
    return STAG_OK;
}

// fp32, 2..4 right-hand sides: the batch kernel with its explicit load pipeline (stag_dslash_batch.cuh).
template <int NR, int MODE, int N, bool PAIRED>
int launch_batch_mode(const float4 *field, unsigned grid, float2 *out, const float2 *in, const Geom &g, int parity,
                      double a, double cD, const float2 *own, double *partials, const CgCtrl *ctrl, cudaStream_t s)
{
    dslash_batch_kernel<NR, MODE, N, PAIRED><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (float)a, (float)cD, own, partials, ctrl);
    count_launch();
    KCHECK();
    return STAG_OK;
}

template <int NR, int N, bool PAIRED>
int launch_batch_n(const stag_links *L, int prec, int hop, float2 *out, const float2 *in, int parity,
                   double a, double cD, const float2 *own, double *partials, const CgCtrl *ctrl, cudaStream_t s)
{
    const Geom &g = L->g;
    const float4 *field = (const float4 *)L->L[prec] + (size_t)parity * L->ntiles * (8 * link_slots(NR) / 2) * TILE;
    const unsigned grid = (unsigned)((g.Vh_pad + DSLASH_BLOCK - 1) / DSLASH_BLOCK);
    switch (hop) {
    case HOP_PLAIN:    return launch_batch_mode<NR, HOP_PLAIN, N, PAIRED>(field, grid, out, in, g, parity, a, cD, own, partials, ctrl, s);
    case HOP_XPAY:     return launch_batch_mode<NR, HOP_XPAY, N, PAIRED>(field, grid, out, in, g, parity, a, cD, own, partials, ctrl, s);
    case HOP_XPAY_DOT: return launch_batch_mode<NR, HOP_XPAY_DOT, N, PAIRED>(field, grid, out, in, g, parity, a, cD, own, partials, ctrl, s);
    }
    return STAG_EINVAL;      // HOP_AXPBY: only the fp64 wrapper steps use it
}

// nrhs right-hand sides in chunks of at most HopMaxRhs<T>: each chunk is one pass over the links.
// layout: STAG_BATCH_BLOCKED or STAG_BATCH_PAIRED (fp32 only; a chunk starts at an even right-hand
// side, so chunk k0 of a paired batch begins k0*rs complex numbers in, like a blocked one).
template <typename T, int NR>
int launch_hop_t(const stag_links *L, int prec, int hop, cplx_t<T> *out, const cplx_t<T> *in,
                 int parity, double a, double cD, const cplx_t<T> *own, double *partials,
                 const CgCtrl *ctrl, int nrhs, int layout, cudaStream_t s)
{
    constexpr int NB = HopMaxRhs<T>::value;
    constexpr bool F32 = std::is_same<T, float>::value;
    if (layout != STAG_BATCH_BLOCKED && !(F32 && layout == STAG_BATCH_PAIRED)) return STAG_EINVAL;
    const size_t rs = (size_t)3 * L->g.Vh_pad;
    const size_t n_hop = ((size_t)L->g.Vh_pad + DSLASH_BLOCK - 1) / DSLASH_BLOCK;
    for (int k0 = 0; k0 < nrhs; k0 += NB) {
        const int nb = nrhs - k0 < NB ? nrhs - k0 : NB;
        cplx_t<T> *o = out + k0 * rs;
        const cplx_t<T> *i = in + k0 * rs;
        const cplx_t<T> *w = own ? own + k0 * rs : nullptr;
        double *pp = partials ? partials + k0 * n_hop : nullptr;
        int rc = STAG_EINVAL;
        if (nb == 1) rc = launch_hop_n<T, NR, 1, false>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s);
        if constexpr (F32) {
            if (nb >= 2) {
                const bool pr = layout == STAG_BATCH_PAIRED;
                if (nb == 2) rc = pr ? launch_batch_n<NR, 2, true>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s)
                                     : launch_batch_n<NR, 2, false>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s);
                if (nb == 3) rc = pr ? launch_batch_n<NR, 3, true>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s)
                                     : launch_batch_n<NR, 3, false>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s);
                if (nb == 4) rc = pr ? launch_batch_n<NR, 4, true>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s)
                                     : launch_batch_n<NR, 4, false>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s);
            }
        } else {
            if (nb == 2) rc = launch_hop_n<T, NR, 2, false>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s);
        }
        if (rc) return rc;
    }
    return STAG_OK;
}

int launch_hop(const stag_links *L, int prec, int hop, void *out, const void *in, int parity,
               double a, double cD, const void *own, double *partials, const CgCtrl *ctrl,
               int nrhs, cudaStream_t s, int layout = STAG_BATCH_BLOCKED)
{
    switch (prec) {
    case STAG_PREC_F64:
        return launch_hop_t<double, 3>(L, prec, hop, (double2 *)out, (const double2 *)in, parity, a, cD, (const double2 *)own, partials, ctrl, nrhs, layout, s);
    case STAG_PREC_F32:
        return launch_hop_t<float, 3>(L, prec, hop, (float2 *)out, (const float2 *)in, parity, a, cD, (const float2 *)own, partials, ctrl, nrhs, layout, s);
    case STAG_PREC_F64_R12:
        return launch_hop_t<double, 2>(L, prec, hop, (double2 *)out, (const double2 *)in, parity, a, cD, (const double2 *)own, partials, ctrl, nrhs, layout, s);
    case STAG_PREC_F32_R12:
        return launch_hop_t<float, 2>(L, prec, hop, (float2 *)out, (const float2 *)in, parity, a, cD, (const float2 *)own, partials, ctrl, nrhs, layout, s);
    case STAG_PREC_F64_R8:
        return launch_hop_t<double, 1>(L, prec, hop, (double2 *)out, (const double2 *)in, parity, a, cD, (const double2 *)own, partials, ctrl, nrhs, layout, s);
    case STAG_PREC_F32_R8:
        return launch_hop_t<float, 1>(L, prec, hop, (float2 *)out, (const float2 *)in, parity, a, cD, (const float2 *)own, partials, ctrl, nrhs, layout, s);
    }
    return STAG_EINVAL;
}

bool same_dims(const stag_links *L, const int dims[4])
{
    return dims && dims[0] == L->dims[0] && dims[1] == L->dims[1] && dims[2] == L->dims[2] &&
           dims[3] == L->dims[3];
}

}  // namespace

// ------------------------------------------------------------------------------------
// C ABI: state
// ------------------------------------------------------------------------------------
extern "C" int stag_set_stream(void *cuda_stream)
{
    t_stream = (cudaStream_t)cuda_stream;
    return STAG_OK;
}

extern "C" const char *stag_strerror(int status)
{
    switch (status) {
    case STAG_OK: return "ok";
    case STAG_EINVAL: return (t_errbuf_status == STAG_EINVAL) ? t_errbuf : "invalid argument";
    case STAG_ECUDA: return t_errbuf;
    case STAG_ENOMEM: return (t_errbuf_status == STAG_ENOMEM) ? t_errbuf : "out of memory";
    case STAG_ETIMEOUT: return "a T-slab kernel gave up waiting for a neighbour's exchange or global sum";
    case STAG_ENOCONV: return "maxiter reached before the true residual met tol";
    case STAG_EBREAKDOWN: return "CG breakdown (NaN or <d,Ad> <= 0)";
    }
    return "unknown status";
}

extern "C" unsigned long long stag_launch_count(void) { return g_launches.load(); }
extern "C" void stag_reset_launch_count(void) { g_launches.store(0); }

// ------------------------------------------------------------------------------------
// C ABI: links
// ------------------------------------------------------------------------------------
static int links_create(stag_links_t **links_out, const int dims[4], int antiperiodic_t,
                        const double *W, int on_device, int fold, int rank, int nranks,
                        const double *W_back = nullptr, bool local = false);

extern "C" int stag_links_create(stag_links_t **links_out, const int dims[4], int antiperiodic_t,
                                 const double *W, int on_device)
{
    return links_create(links_out, dims, antiperiodic_t, W, on_device, 0, 0, 1);
}

extern "C" int stag_links_create_unfolded(stag_links_t **links_out, const int dims[4],
                                          int antiperiodic_t, const double *U, int on_device)
{
    return links_create(links_out, dims, antiperiodic_t, U, on_device, 1, 0, 1);
}

// dims: the whole lattice.  nranks > 1: the handle covers time slices [rank*X3/nranks, (rank+1)*X3/nranks)
// only.  local: W is the slab's own part and W_back the t-links of the slice before it (LinkSrc);
// otherwise W is the whole field, and from HOST memory only those same sub-ranges are copied to the
// device (8 + 2 contiguous ranges: time slices are contiguous in cb), never the whole lattice.
static int links_create(stag_links_t **links_out, const int dims[4], int antiperiodic_t,
                        const double *W, int on_device, int fold, int rank, int nranks,
                        const double *W_back, bool local)
{
    if (!links_out || !W) return STAG_EINVAL;
    *links_out = nullptr;
    Geom gg, g;
    if (!make_geom(gg, dims, antiperiodic_t)) return STAG_EINVAL;
    if (nranks < 1 || rank < 0 || rank >= nranks || dims[3] % nranks) return STAG_EINVAL;
    const int ldims[4] = { dims[0], dims[1], dims[2], dims[3] / nranks };
    if (!make_geom(g, ldims, antiperiodic_t)) return STAG_EINVAL;     // local extent even, >= 2
    if (local && nranks > 1 && !W_back) return STAG_EINVAL;
    g.t0 = rank * ldims[3];
    g.X3g = dims[3];
    stag_links *L = new (std::nothrow) stag_links();
    if (!L) return STAG_ENOMEM;
    L->uid = g_next_uid.fetch_add(1, std::memory_order_relaxed);
    L->g = g;
    for (int m = 0; m < 4; ++m) { L->dims[m] = ldims[m]; L->gdims[m] = dims[m]; }
    L->rank = rank;
    L->nranks = nranks;
    L->ntiles = g.Vh_pad / TILE;

    const size_t plane_l = (size_t)g.Vh * 18, plane_g = (size_t)gg.Vh * 18;      // doubles per (mu, p)
    const size_t slice = (size_t)gg.s3 * 18;
    const bool part = local || (nranks > 1 && !on_device);    // the device sees only the slab's part
    double *Wd = nullptr, *Wbd = nullptr;
    unsigned long long *err = nullptr;
    int rc = STAG_OK;
    cudaError_t e = cudaSuccess;
    LinkSrc src;
    src.W = W; src.Wback = W_back;
    src.vh = part ? g.Vh : gg.Vh;
    src.off = part ? (long)g.t0 * gg.s3 : 0;
    do {
        if (!on_device) {
            if ((e = cudaMalloc(&Wd, 8 * (part ? plane_l : plane_g) * sizeof(double))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(staging)", __LINE__); break; }
            if (local || !part) {
                e = cudaMemcpyAsync(Wd, W, 8 * (part ? plane_l : plane_g) * sizeof(double), cudaMemcpyHostToDevice, t_stream);
            } else {
                for (int mp = 0; mp < 8 && e == cudaSuccess; ++mp)
                    e = cudaMemcpyAsync(Wd + mp * plane_l, W + mp * plane_g + (size_t)src.off * 18, plane_l * sizeof(double), cudaMemcpyHostToDevice, t_stream);
            }
            if (e != cudaSuccess) { rc = cuda_fail(e, "cudaMemcpyAsync(W)", __LINE__); break; }
            src.W = Wd;
            if (part && nranks > 1) {
                if ((e = cudaMalloc(&Wbd, 2 * slice * sizeof(double))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(staging)", __LINE__); break; }
                if (local) {
                    e = cudaMemcpyAsync(Wbd, W_back, 2 * slice * sizeof(double), cudaMemcpyHostToDevice, t_stream);
                } else {
                    const size_t tb = (size_t)((g.t0 + dims[3] - 1) % dims[3]) * slice;
                    for (int pp = 0; pp < 2 && e == cudaSuccess; ++pp)
                        e = cudaMemcpyAsync(Wbd + pp * slice, W + (size_t)(6 + pp) * plane_g + tb, slice * sizeof(double), cudaMemcpyHostToDevice, t_stream);
                }
                if (e != cudaSuccess) { rc = cuda_fail(e, "cudaMemcpyAsync(W_back)", __LINE__); break; }
                src.Wback = Wbd;
            }
        }
        if ((e = cudaMalloc(&L->L[STAG_PREC_F64], links_elems(L, 3) * sizeof(double2))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(links)", __LINE__); break; }
        if ((e = cudaMalloc(&err, sizeof(*err))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(err)", __LINE__); break; }
        if ((e = cudaMemsetAsync(err, 0, sizeof(*err), t_stream)) != cudaSuccess) { rc = cuda_fail(e, "cudaMemsetAsync", __LINE__); break; }
        const unsigned grid = (unsigned)((2L * g.Vh_pad + 127) / 128);
        gather_links_kernel<<<grid, 128, 0, t_stream>>>((double2 *)L->L[STAG_PREC_F64], src, g, gg, err, fold);
        count_launch();
        if ((e = cudaGetLastError()) != cudaSuccess) { rc = cuda_fail(e, "gather_links_kernel", __LINE__); break; }
        unsigned long long bits = 0;
        if ((e = cudaMemcpyAsync(&bits, err, sizeof(bits), cudaMemcpyDeviceToHost, t_stream)) != cudaSuccess) { rc = cuda_fail(e, "cudaMemcpyAsync(err)", __LINE__); break; }
        if ((e = cudaStreamSynchronize(t_stream)) != cudaSuccess) { rc = cuda_fail(e, "cudaStreamSynchronize", __LINE__); break; }
        memcpy(&L->recon_err, &bits, sizeof(double));
        L->L_ready[STAG_PREC_F64].store(1, std::memory_order_release);
    } while (0);
    if (Wd) cudaFree(Wd);
    if (Wbd) cudaFree(Wbd);
    if (err) cudaFree(err);
    if (rc != STAG_OK) { stag_links_destroy(L); return rc; }
    *links_out = L;
    return STAG_OK;
}

static void stag_slab_cg_free(struct stag_slab_cg *c);

extern "C" void stag_links_destroy(stag_links_t *L)
{
    if (!L) return;
    for (int i = 0; i < N_PREC; ++i) if (L->L[i]) cudaFree(L->L[i]);
    L->own.release();
    if (L->xch) cudaFree(L->xch);
    if (L->peers_dev) cudaFree(L->peers_dev);
    stag_slab_cg_free(L->cg);
    delete L;
}

extern "C" int stag_links_recon8_error(const stag_links_t *L, int prec, double *err_out)
{
    if (!L || !err_out || (prec != STAG_PREC_F64_R8 && prec != STAG_PREC_F32_R8)) return STAG_EINVAL;
    const int rc = ensure_links(L, prec);        // builds (or refuses) and measures
    *err_out = L->recon8_err[prec_is_f32(prec) ? 1 : 0];
    return rc;
}

extern "C" int stag_links_recon_error(const stag_links_t *L, double *err_out)
{
    if (!L || !err_out) return STAG_EINVAL;
    *err_out = L->recon_err;
    return STAG_OK;
}

// ------------------------------------------------------------------------------------
// C ABI: spinors
// ------------------------------------------------------------------------------------
extern "C" size_t stag_spinor_bytes(const int dims[4], int prec)
{
    Geom g;
    if (!prec_ok(prec) || !make_geom(g, dims, 0)) return 0;
    return (size_t)3 * g.Vh_pad * (prec_is_f32(prec) ? sizeof(float2) : sizeof(double2));
}

extern "C" int stag_spinor_pack(void *dst, const double *src, const int dims[4], int prec)
{
    Geom g;
    if (!dst || !src || !prec_ok(prec) || !make_geom(g, dims, 0)) return STAG_EINVAL;
    const unsigned grid = (unsigned)((g.Vh_pad + 127) / 128);
    if (prec_is_f32(prec)) spinor_pack_kernel<float><<<grid, 128, 0, t_stream>>>((float2 *)dst, src, g.Vh, g.Vh_pad);
    else spinor_pack_kernel<double><<<grid, 128, 0, t_stream>>>((double2 *)dst, src, g.Vh, g.Vh_pad);
    count_launch();
    KCHECK();
    return STAG_OK;
}

extern "C" int stag_spinor_unpack(double *dst, const void *src, const int dims[4], int prec)
{
    Geom g;
    if (!dst || !src || !prec_ok(prec) || !make_geom(g, dims, 0)) return STAG_EINVAL;
    const unsigned grid = (unsigned)((g.Vh + 127) / 128);
    if (prec_is_f32(prec)) spinor_unpack_kernel<float><<<grid, 128, 0, t_stream>>>(dst, (const float2 *)src, g.Vh, g.Vh_pad);
    else spinor_unpack_kernel<double><<<grid, 128, 0, t_stream>>>(dst, (const double2 *)src, g.Vh, g.Vh_pad);
    count_launch();
    KCHECK();
    return STAG_OK;
}

// ------------------------------------------------------------------------------------
// C ABI: the operator
// ------------------------------------------------------------------------------------
extern "C" int stag_dslash_batch(void *out, const void *in, const stag_links_t *links, int parity,
                                 const int dims[4], int prec, int nrhs, int layout)
{
    const stag_links *L = links;
    if (!out || !in || !L || out == in || (parity & ~1) || !prec_ok(prec) || !same_dims(L, dims) ||
        nrhs < 1 || L->is_slab)      // a slab's hop needs its halo: stag_slab_hop
        return STAG_EINVAL;
    if (layout != STAG_BATCH_BLOCKED && !(layout == STAG_BATCH_PAIRED && prec_is_f32(prec))) return STAG_EINVAL;
    int rc = ensure_links(L, prec);
    if (rc) return rc;
    return launch_hop(L, prec, HOP_PLAIN, out, in, parity, 0.0, 1.0, nullptr, nullptr, nullptr, nrhs, t_stream, layout);
}

extern "C" int stag_dslash_mrhs(void *out, const void *in, const stag_links_t *links, int parity,
                                const int dims[4], int prec, int nrhs)
{
    return stag_dslash_batch(out, in, links, parity, dims, prec, nrhs, STAG_BATCH_BLOCKED);
}

// blocked <-> paired: rhs 2j, 2j+1 of an fp32 batch interleaved per complex number
__global__ void __launch_bounds__(256)
batch_convert_kernel(float4 *__restrict__ dst, const float4 *__restrict__ src, long rs, int npairs, int to_paired)
{
    // one thread per (pair, complex index i): blocked holds a[i] at 2j*rs + i and b[i] at (2j+1)*rs + i
    // (float2 units); paired holds (a[i], b[i]) as the float4 number i of the pair.  Two complex
    // numbers per thread so that both sides move 16-byte packets (rs is even).
    const long half = rs / 2;
    const long t = blockIdx.x * 256L + threadIdx.x;
    if (t >= (long)npairs * half) return;
    const long j = t / half, i2 = t % half;                 // complex numbers 2*i2, 2*i2+1
    const float4 *sj = src + j * rs;                        // the pair's 2*rs float2 = rs float4
    float4 *dj = dst + j * rs;
    if (to_paired) {
        const float4 a = sj[i2], b = sj[half + i2];         // a[2i2], a[2i2+1] ; b[2i2], b[2i2+1]
        dj[2 * i2] = make_float4(a.x, a.y, b.x, b.y);
        dj[2 * i2 + 1] = make_float4(a.z, a.w, b.z, b.w);
    } else {
        const float4 p = sj[2 * i2], q = sj[2 * i2 + 1];
        dj[i2] = make_float4(p.x, p.y, q.x, q.y);
        dj[half + i2] = make_float4(p.z, p.w, q.z, q.w);
    }
}

extern "C" int stag_batch_convert(void *dst, const void *src, const int dims[4], int prec, int nrhs,
                                  int to_layout)
{
    Geom g;
    if (!dst || !src || dst == src || !prec_ok(prec) || !make_geom(g, dims, 0) || nrhs < 1 ||
        (to_layout != STAG_BATCH_BLOCKED && to_layout != STAG_BATCH_PAIRED))
        return STAG_EINVAL;
    const size_t sb = stag_spinor_bytes(dims, prec);
    if (!prec_is_f32(prec)) {     // fp64 batches have one layout
        CU(cudaMemcpyAsync(dst, src, sb * nrhs, cudaMemcpyDeviceToDevice, t_stream));
        return STAG_OK;
    }
    const long rs = 3L * g.Vh_pad;
    const int npairs = nrhs / 2;
    if (npairs) {
        const long n = (long)npairs * (rs / 2);
        batch_convert_kernel<<<(unsigned)((n + 255) / 256), 256, 0, t_stream>>>((float4 *)dst, (const float4 *)src, rs, npairs, to_layout == STAG_BATCH_PAIRED);
        count_launch();
        KCHECK();
    }
    if (nrhs & 1)                 // the odd last right-hand side is an ordinary spinor in both layouts
        CU(cudaMemcpyAsync((char *)dst + sb * (nrhs - 1), (const char *)src + sb * (nrhs - 1), sb, cudaMemcpyDeviceToDevice, t_stream));
    return STAG_OK;
}

extern "C" int stag_dslash(void *out, const void *in, const stag_links_t *links, int parity,
                           const int dims[4], int prec)
{
    return stag_dslash_mrhs(out, in, links, parity, dims, prec, 1);
}

extern "C" int stag_apply_A_batch(void *out_even, const void *in_even, const stag_links_t *links,
                                  double mass, int prec, int nrhs, int layout)
{
    const stag_links *L = links;
    if (!out_even || !in_even || !L || out_even == in_even || !prec_ok(prec) || nrhs < 1 || nrhs > MAX_RHS || L->is_slab)
        return STAG_EINVAL;
    if (layout != STAG_BATCH_BLOCKED && !(layout == STAG_BATCH_PAIRED && prec_is_f32(prec))) return STAG_EINVAL;
    int rc = ensure_links(L, prec);
    if (rc) return rc;
    // the odd-site intermediate lives in the workspace (the caller's, or the handle's own)
    const WsLayout lay = ws_layout(L->g, -1, nrhs);
    WsLease lease;
    if ((rc = lease_workspace(L, lay.total, lease))) return rc;
    void *tmp_odd = lease.ws->base + lay.scratch;
    // tmp_o = D_oe in_e ;  out_e = m^2 in_e - D_eo tmp_o      (eq. 2.3)
    if ((rc = launch_hop(L, prec, HOP_PLAIN, tmp_odd, in_even, 1, 0.0, 1.0, nullptr, nullptr, nullptr, nrhs, t_stream, layout))) return rc;
    return launch_hop(L, prec, HOP_XPAY, out_even, tmp_odd, 0, mass * mass, 1.0, in_even, nullptr, nullptr, nrhs, t_stream, layout);
}

extern "C" int stag_apply_A_mrhs(void *out_even, const void *in_even, const stag_links_t *links,
                                 double mass, int prec, int nrhs)
{
    return stag_apply_A_batch(out_even, in_even, links, mass, prec, nrhs, STAG_BATCH_BLOCKED);
}

extern "C" int stag_apply_A(void *out_even, const void *in_even, const stag_links_t *links,
                            double mass, int prec)
{
    return stag_apply_A_mrhs(out_even, in_even, links, mass, prec, 1);
}

