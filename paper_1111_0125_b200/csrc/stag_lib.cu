// stag_lib.cu -- host side of libstag: the C ABI of include/stag.h, the link handle and its
// setup kernels (step S0), kernel launchers, and the CG drivers (Fig. 1, Fig. 2, section 3.2).
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <type_traits>

#include "stag_blas.cuh"
#include "stag_common.cuh"
#include "stag_dslash.cuh"
#include "stag_slab.cuh"

using namespace stag;

// ------------------------------------------------------------------------------------
// per-thread state, errors, launch counting
// ------------------------------------------------------------------------------------
namespace {

thread_local cudaStream_t t_stream = nullptr;
thread_local char t_errbuf[256] = "no error recorded";
thread_local int t_errbuf_status = 0;   // which status t_errbuf describes
std::atomic<unsigned long long> g_launches{0};
thread_local bool t_capturing = false;
thread_local unsigned long long t_captured_nodes = 0;

inline void count_launch(unsigned long long n = 1)
{
    if (t_capturing) t_captured_nodes += n;
    else g_launches.fetch_add(n, std::memory_order_relaxed);
}

int cuda_fail(cudaError_t e, const char *what, int line)
{
    snprintf(t_errbuf, sizeof(t_errbuf), "%s (line %d): %s", what, line, cudaGetErrorString(e));
    (void)cudaGetLastError();
    t_errbuf_status = (e == cudaErrorMemoryAllocation) ? STAG_ENOMEM : STAG_ECUDA;
    return t_errbuf_status;
}

#define CU(call)                                                     \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call, __LINE__); \
    } while (0)

#define KCHECK() CU(cudaGetLastError())

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

constexpr int N_PREC = 6;
inline bool prec_ok(int prec) { return prec >= 0 && prec < N_PREC; }
inline bool prec_is_f32(int prec) { return prec == STAG_PREC_F32 || prec == STAG_PREC_F32_R12 || prec == STAG_PREC_F32_R8; }
// storage of a link: 3 = 18-real, 2 = 12-real (rows 0,1), 1 = 8-parameter
inline int prec_rows(int prec)
{
    if (prec == STAG_PREC_F64_R8 || prec == STAG_PREC_F32_R8) return 1;
    return (prec == STAG_PREC_F64_R12 || prec == STAG_PREC_F32_R12) ? 2 : 3;
}

// Grid of the streaming vector kernels: 4 resident blocks of 256 threads per SM (a multiple of
// the SM count) shared among the nrhs right-hand sides (grid.y = nrhs), fewer when the vector
// is too short to feed them.  Returns grid.x, the blocks per right-hand side.
int blas_full_grid()
{
    static int full = 0;
    if (full == 0) {
        int dev = 0, sms = 148;
        if (cudaGetDevice(&dev) == cudaSuccess)
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        full = sms * 4;
    }
    return full;
}
int blas_grid(long n_reals, int nrhs)
{
    const long per = blas_full_grid() / (nrhs < 1 ? 1 : nrhs);
    const long need = (n_reals / 2 + BLAS_BLOCK - 1) / BLAS_BLOCK;
    const long g = need < per ? need : per;
    return (int)(g < 1 ? 1 : g);
}

}  // namespace

// ------------------------------------------------------------------------------------
// the link handle
// ------------------------------------------------------------------------------------
struct stag_slab_cg;
struct stag_links {
    Geom g;
    int dims[4];           // extents of the lattice this handle covers (the slab's, for a slab)
    int gdims[4];          // extents of the whole lattice
    int rank, nranks;      // T-slab: time slices [rank*X3, (rank+1)*X3) of nranks*X3; else 0, 1
    int is_slab;           // made by stag_slab_create: operator calls go through stag_slab_*
    int ntiles;            // Vh_pad / TILE
    void *L[6];            // gathered link fields by precision enum; L[STAG_PREC_F64] always set
    double recon8_err[2];  // 8-parameter forms: largest rebuilt-entry error, [0] fp64, [1] fp32 (-1: not built)
    double recon_err;
    void *tmp_odd[2];      // scratch odd-parity spinors for stag_apply_A: [0] fp64, [1] fp32
    int tmp_odd_rhs[2];    // how many right-hand sides each holds
    // CG workspace (lazy)
    char *ws;
    size_t ws_bytes;
    int ws_rhs;            // right-hand sides the workspace was sized for
    CgCtrl *h_ctrl;        // pinned mirror
    cudaStream_t cap_stream;
    // staging for stag_cg_solve_host (lazy)
    double *stage_dev;     // 2 canonical spinors + 2 device-layout fp64 spinors
    // T-slab exchange (stag_slab_*): my exchange region, the neighbours' (peer memory), and the
    // number of exchanges started so far
    char *xch;
    char *peer_bwd, *peer_fwd;
    unsigned long long epoch;
    unsigned n_push_blocks; // blocks of a HALO hop that own boundary-slice sites (cached)
    char **peers_dev;      // device array: every rank's exchange region (stag_slab_connect_all)
    int all_connected;
    struct stag_slab_cg *cg;   // state of the slab CG in progress (stag_slab_cg_*)
    void *wrap_b;          // stag_solve_M: b_e of the even-site system, wrap_b_rhs spinors (lazy)
    int wrap_b_rhs;
    cudaEvent_t ev0, ev1;
};

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
// g is the geometry of the lattice the handle covers, gg that of the lattice W covers: the same
// for a whole-lattice handle; for a T-slab (stag_slab_create) g is the slab (time slices
// [g.t0, g.t0 + g.X3) of gg) and every link, including the backward t-links of the slab's first
// slice that belong to the neighbouring slab, is read from the whole field.
__global__ void __launch_bounds__(128)
gather_links_kernel(double2 *__restrict__ L, const double *__restrict__ W, const Geom g,
                    const Geom gg, unsigned long long *__restrict__ err_bits, const int fold)
{
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
            const double *src = W + (((size_t)d * 2 + p) * gg.Vh + cbg) * 18;
            for (int k = 0; k < 9; ++k) m[k] = make_double2(src[2 * k], src[2 * k + 1]);
        } else {
            const double *src = W + (((size_t)(d - 4) * 2 + (1 - p)) * gg.Vh + s.nbr[d]) * 18;
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

// Build (once) the gathered field of precision `prec` from the fp64/18 one.
int ensure_links(stag_links *L, int prec)
{
    if (L->L[prec]) return STAG_OK;
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
    if (e != cudaSuccess) { cudaFree(dst); return cuda_fail(e, "derive_links_kernel", __LINE__); }
    L->L[prec] = dst;
    return STAG_OK;
}

int ensure_tmp(stag_links *L, int f32, int nrhs)
{
    if (L->tmp_odd[f32] && L->tmp_odd_rhs[f32] >= nrhs) return STAG_OK;
    if (L->tmp_odd[f32]) { CU(cudaFree(L->tmp_odd[f32])); L->tmp_odd[f32] = nullptr; }
    CU(cudaMalloc(&L->tmp_odd[f32], (size_t)nrhs * 3 * L->g.Vh_pad * (f32 ? sizeof(float2) : sizeof(double2))));
    L->tmp_odd_rhs[f32] = nrhs;
    return STAG_OK;
}

// ---- Dslash launcher ---------------------------------------------------------------------
template <typename T, int NR, int N>
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
        dslash_kernel<T, NR, HOP_PLAIN, N><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)cD, own, partials, ctrl, HaloArgs<T>{});
        break;
    case HOP_XPAY:
        dslash_kernel<T, NR, HOP_XPAY, N><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)cD, own, partials, ctrl, HaloArgs<T>{});
        break;
    case HOP_AXPBY:   // only the fp64 wrapper steps use it
        if constexpr (std::is_same<T, double>::value)
            dslash_kernel<T, NR, HOP_AXPBY, N><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)cD, own, partials, ctrl, HaloArgs<T>{});
        else
            return STAG_EINVAL;
        break;
    default:
        dslash_kernel<T, NR, HOP_XPAY_DOT, N><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)cD, own, partials, ctrl, HaloArgs<T>{});
        break;
    }
    count_launch();
    KCHECK();
    return STAG_OK;
}

// nrhs right-hand sides in chunks of at most HopMaxRhs<T>: each chunk is one pass over the links.
template <typename T, int NR>
int launch_hop_t(const stag_links *L, int prec, int hop, cplx_t<T> *out, const cplx_t<T> *in,
                 int parity, double a, double cD, const cplx_t<T> *own, double *partials,
                 const CgCtrl *ctrl, int nrhs, cudaStream_t s)
{
    constexpr int NB = HopMaxRhs<T>::value;
    const size_t rs = (size_t)3 * L->g.Vh_pad;
    const size_t n_hop = ((size_t)L->g.Vh_pad + DSLASH_BLOCK - 1) / DSLASH_BLOCK;
    for (int k0 = 0; k0 < nrhs; k0 += NB) {
        const int nb = nrhs - k0 < NB ? nrhs - k0 : NB;
        cplx_t<T> *o = out + k0 * rs;
        const cplx_t<T> *i = in + k0 * rs;
        const cplx_t<T> *w = own ? own + k0 * rs : nullptr;
        double *pp = partials ? partials + k0 * n_hop : nullptr;
        int rc = STAG_EINVAL;
        if (nb == 1) rc = launch_hop_n<T, NR, 1>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s);
        if (nb == 2) rc = launch_hop_n<T, NR, 2>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s);
        if constexpr (NB >= 4) {
            if (nb == 3) rc = launch_hop_n<T, NR, 3>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s);
            if (nb == 4) rc = launch_hop_n<T, NR, 4>(L, prec, hop, o, i, parity, a, cD, w, pp, ctrl, s);
        }
        if (rc) return rc;
    }
    return STAG_OK;
}

int launch_hop(const stag_links *L, int prec, int hop, void *out, const void *in, int parity,
               double a, double cD, const void *own, double *partials, const CgCtrl *ctrl,
               int nrhs, cudaStream_t s)
{
    switch (prec) {
    case STAG_PREC_F64:
        return launch_hop_t<double, 3>(L, prec, hop, (double2 *)out, (const double2 *)in, parity, a, cD, (const double2 *)own, partials, ctrl, nrhs, s);
    case STAG_PREC_F32:
        return launch_hop_t<float, 3>(L, prec, hop, (float2 *)out, (const float2 *)in, parity, a, cD, (const float2 *)own, partials, ctrl, nrhs, s);
    case STAG_PREC_F64_R12:
        return launch_hop_t<double, 2>(L, prec, hop, (double2 *)out, (const double2 *)in, parity, a, cD, (const double2 *)own, partials, ctrl, nrhs, s);
    case STAG_PREC_F32_R12:
        return launch_hop_t<float, 2>(L, prec, hop, (float2 *)out, (const float2 *)in, parity, a, cD, (const float2 *)own, partials, ctrl, nrhs, s);
    case STAG_PREC_F64_R8:
        return launch_hop_t<double, 1>(L, prec, hop, (double2 *)out, (const double2 *)in, parity, a, cD, (const double2 *)own, partials, ctrl, nrhs, s);
    case STAG_PREC_F32_R8:
        return launch_hop_t<float, 1>(L, prec, hop, (float2 *)out, (const float2 *)in, parity, a, cD, (const float2 *)own, partials, ctrl, nrhs, s);
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
                        const double *W, int on_device, int fold, int rank, int nranks);

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

// dims: the lattice W covers.  nranks > 1 (or slab != 0): the handle covers time slices
// [rank*X3/nranks, (rank+1)*X3/nranks) only and is a T-slab (exchange region allocated).
static int links_create(stag_links_t **links_out, const int dims[4], int antiperiodic_t,
                        const double *W, int on_device, int fold, int rank, int nranks)
{
    if (!links_out || !W) return STAG_EINVAL;
    *links_out = nullptr;
    Geom gg, g;
    if (!make_geom(gg, dims, antiperiodic_t)) return STAG_EINVAL;
    if (nranks < 1 || rank < 0 || rank >= nranks || dims[3] % nranks) return STAG_EINVAL;
    const int ldims[4] = { dims[0], dims[1], dims[2], dims[3] / nranks };
    if (!make_geom(g, ldims, antiperiodic_t)) return STAG_EINVAL;     // local extent even, >= 2
    g.t0 = rank * ldims[3];
    g.X3g = dims[3];
    stag_links *L = new (std::nothrow) stag_links();
    if (!L) return STAG_ENOMEM;
    memset(L, 0, sizeof(*L));
    L->g = g;
    for (int m = 0; m < 4; ++m) { L->dims[m] = ldims[m]; L->gdims[m] = dims[m]; }
    L->rank = rank;
    L->nranks = nranks;
    L->ntiles = g.Vh_pad / TILE;

    const size_t canon_bytes = (size_t)4 * 2 * gg.Vh * 18 * sizeof(double);
    double *Wd = nullptr;
    unsigned long long *err = nullptr;
    int rc = STAG_OK;
    cudaError_t e;
    do {
        if (!on_device) {
            if ((e = cudaMalloc(&Wd, canon_bytes)) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(staging)", __LINE__); break; }
            if ((e = cudaMemcpyAsync(Wd, W, canon_bytes, cudaMemcpyHostToDevice, t_stream)) != cudaSuccess) { rc = cuda_fail(e, "cudaMemcpyAsync(W)", __LINE__); break; }
        }
        if ((e = cudaMalloc(&L->L[STAG_PREC_F64], links_elems(L, 3) * sizeof(double2))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(links)", __LINE__); break; }
        if ((e = cudaMalloc(&err, sizeof(*err))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(err)", __LINE__); break; }
        if ((e = cudaMemsetAsync(err, 0, sizeof(*err), t_stream)) != cudaSuccess) { rc = cuda_fail(e, "cudaMemsetAsync", __LINE__); break; }
        const unsigned grid = (unsigned)((2L * g.Vh_pad + 127) / 128);
        gather_links_kernel<<<grid, 128, 0, t_stream>>>((double2 *)L->L[STAG_PREC_F64], on_device ? W : Wd, g, gg, err, fold);
        count_launch();
        if ((e = cudaGetLastError()) != cudaSuccess) { rc = cuda_fail(e, "gather_links_kernel", __LINE__); break; }
        unsigned long long bits = 0;
        if ((e = cudaMemcpyAsync(&bits, err, sizeof(bits), cudaMemcpyDeviceToHost, t_stream)) != cudaSuccess) { rc = cuda_fail(e, "cudaMemcpyAsync(err)", __LINE__); break; }
        if ((e = cudaStreamSynchronize(t_stream)) != cudaSuccess) { rc = cuda_fail(e, "cudaStreamSynchronize", __LINE__); break; }
        memcpy(&L->recon_err, &bits, sizeof(double));
        if ((e = cudaStreamCreateWithFlags(&L->cap_stream, cudaStreamNonBlocking)) != cudaSuccess) { rc = cuda_fail(e, "cudaStreamCreate", __LINE__); break; }
        if ((e = cudaEventCreate(&L->ev0)) != cudaSuccess || (e = cudaEventCreate(&L->ev1)) != cudaSuccess) { rc = cuda_fail(e, "cudaEventCreate", __LINE__); break; }
    } while (0);
    if (Wd) cudaFree(Wd);
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
    for (int i = 0; i < 2; ++i) if (L->tmp_odd[i]) cudaFree(L->tmp_odd[i]);
    if (L->ws) cudaFree(L->ws);
    if (L->h_ctrl) cudaFreeHost(L->h_ctrl);
    if (L->stage_dev) cudaFree(L->stage_dev);
    if (L->wrap_b) cudaFree(L->wrap_b);
    if (L->xch) cudaFree(L->xch);
    if (L->peers_dev) cudaFree(L->peers_dev);
    stag_slab_cg_free(L->cg);
    if (L->cap_stream) cudaStreamDestroy(L->cap_stream);
    if (L->ev0) cudaEventDestroy(L->ev0);
    if (L->ev1) cudaEventDestroy(L->ev1);
    delete L;
}

extern "C" int stag_links_recon8_error(const stag_links_t *links, int prec, double *err_out)
{
    stag_links *L = const_cast<stag_links *>(links);
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
extern "C" int stag_dslash_mrhs(void *out, const void *in, const stag_links_t *links, int parity,
                                const int dims[4], int prec, int nrhs)
{
    stag_links *L = const_cast<stag_links *>(links);
    if (!out || !in || !L || out == in || (parity & ~1) || !prec_ok(prec) || !same_dims(L, dims) ||
        nrhs < 1 || L->is_slab)      // a slab's hop needs its halo: stag_slab_hop
        return STAG_EINVAL;
    int rc = ensure_links(L, prec);
    if (rc) return rc;
    return launch_hop(L, prec, HOP_PLAIN, out, in, parity, 0.0, 1.0, nullptr, nullptr, nullptr, nrhs, t_stream);
}

extern "C" int stag_dslash(void *out, const void *in, const stag_links_t *links, int parity,
                           const int dims[4], int prec)
{
    return stag_dslash_mrhs(out, in, links, parity, dims, prec, 1);
}

extern "C" int stag_apply_A_mrhs(void *out_even, const void *in_even, const stag_links_t *links,
                                 double mass, int prec, int nrhs)
{
    stag_links *L = const_cast<stag_links *>(links);
    if (!out_even || !in_even || !L || out_even == in_even || !prec_ok(prec) || nrhs < 1 || L->is_slab)
        return STAG_EINVAL;
    int rc = ensure_links(L, prec);
    if (rc) return rc;
    const int f32 = prec_is_f32(prec) ? 1 : 0;
    if ((rc = ensure_tmp(L, f32, nrhs))) return rc;
    // tmp_o = D_oe in_e ;  out_e = m^2 in_e - D_eo tmp_o      (eq. 2.3)
    if ((rc = launch_hop(L, prec, HOP_PLAIN, L->tmp_odd[f32], in_even, 1, 0.0, 1.0, nullptr, nullptr, nullptr, nrhs, t_stream))) return rc;
    return launch_hop(L, prec, HOP_XPAY, out_even, L->tmp_odd[f32], 0, mass * mass, 1.0, in_even, nullptr, nullptr, nrhs, t_stream);
}

extern "C" int stag_apply_A(void *out_even, const void *in_even, const stag_links_t *links,
                            double mass, int prec)
{
    return stag_apply_A_mrhs(out_even, in_even, links, mass, prec, 1);
}

// ------------------------------------------------------------------------------------
// the CG drivers
// ------------------------------------------------------------------------------------
namespace {

struct Workspace {
    CgCtrl *ctrl;
    double *partials;       // block partials of the vector kernels' reductions, [rhs][block]
    double *hop_partials;   // block partials of <d,Ad> written by the second hop, [rhs][block]
    int n_hop;              // = grid of the hop
    double *r64, *q64, *tmp64, *d64;          // nrhs spinors each
    float *y32, *r32, *d32, *q32, *tmp32;
};

// One allocation on the handle, sized for nrhs right-hand sides (grown when a later solve
// carries more).  Right-hand side k of every vector starts k*n reals in (n = 6*Vh_pad).
int ensure_workspace(stag_links *L, Workspace &w, int nrhs)
{
    const size_t n = (size_t)6 * L->g.Vh_pad;
    if (L->ws && L->ws_rhs < nrhs) { CU(cudaFree(L->ws)); L->ws = nullptr; }
    const int cap = L->ws ? L->ws_rhs : nrhs;
    const size_t nb64 = align_up(cap * n * sizeof(double), 256), nb32 = align_up(cap * n * sizeof(float), 256);
    const size_t n_hop = ((size_t)L->g.Vh_pad + DSLASH_BLOCK - 1) / DSLASH_BLOCK;
    const size_t pb = align_up((size_t)MAX_RHS * blas_full_grid() * sizeof(double), 256);
    const size_t hb = align_up((size_t)cap * n_hop * sizeof(double), 256);
    const size_t total = CTRL_SLOT + pb + hb + 4 * nb64 + 5 * nb32;
    if (!L->ws) {
        CU(cudaMalloc((void **)&L->ws, total));
        L->ws_bytes = total;
        L->ws_rhs = cap;
    }
    if (!L->h_ctrl) CU(cudaMallocHost((void **)&L->h_ctrl, sizeof(CgCtrl)));
    char *p = L->ws;
    w.ctrl = (CgCtrl *)p; p += CTRL_SLOT;
    w.partials = (double *)p; p += pb;
    w.hop_partials = (double *)p; p += hb;
    w.n_hop = (int)n_hop;
    w.r64 = (double *)p; p += nb64;
    w.q64 = (double *)p; p += nb64;
    w.tmp64 = (double *)p; p += nb64;
    w.d64 = (double *)p; p += nb64;
    w.y32 = (float *)p; p += nb32;
    w.r32 = (float *)p; p += nb32;
    w.d32 = (float *)p; p += nb32;
    w.q32 = (float *)p; p += nb32;
    w.tmp32 = (float *)p; p += nb32;
    return STAG_OK;
}

struct Solver {
    stag_links *L;
    Workspace w;
    cudaStream_t s;
    double m2;
    int mode;
    int nrhs;
    int prec_lo;     // precision enum of the iteration's Dslash
    int prec_hi;     // precision enum of the fp64 corrections
    long n;          // reals per spinor
    int gb;          // blas grid.x (blocks per right-hand side)
    int applies_f64;

    dim3 grid2() const { return dim3((unsigned)gb, (unsigned)nrhs); }

    // q64 = A x  in fp64 (two hops), outside the iteration
    int apply_A64(const double *x)
    {
        int rc = launch_hop(L, prec_hi, HOP_PLAIN, w.tmp64, x, 1, 0.0, 1.0, nullptr, nullptr, nullptr, nrhs, s);
        if (rc) return rc;
        ++applies_f64;
        return launch_hop(L, prec_hi, HOP_XPAY, w.q64, w.tmp64, 0, m2, 1.0, x, nullptr, nullptr, nrhs, s);
    }

    template <int WHAT>
    int residual(const double *b, bool lo_copy)
    {
        residual_kernel<float, WHAT><<<grid2(), BLAS_BLOCK, 0, s>>>(w.r64, b, w.q64, lo_copy ? w.r32 : nullptr, n, w.partials, w.ctrl);
        count_launch();
        KCHECK();
        return STAG_OK;
    }

    int accumulate(double *x)
    {
        accumulate_kernel<float><<<blas_grid(n * nrhs, 1), BLAS_BLOCK, 0, s>>>(x, w.y32, n * nrhs);
        count_launch();
        KCHECK();
        return STAG_OK;
    }

    // one pass of the loop body of Fig. 1, four launches (the hops: one launch per
    // chunk of right-hand sides)
    template <typename T>
    int iteration(T *y, T *r, T *d, T *q, T *tmp, cudaStream_t st)
    {
        xpay_kernel<T><<<grid2(), BLAS_BLOCK, 0, st>>>(d, r, n, w.ctrl);                     // d = r + beta d
        count_launch();
        KCHECK();
        int rc = launch_hop(L, prec_lo, HOP_PLAIN, tmp, d, 1, 0.0, 1.0, nullptr, nullptr, w.ctrl, nrhs, st);   // D_oe d
        if (rc) return rc;
        rc = launch_hop(L, prec_lo, HOP_XPAY_DOT, q, tmp, 0, m2, 1.0, d, w.hop_partials, w.ctrl, nrhs, st);  // q = A d, <d,q>
        if (rc) return rc;
        update_kernel<T><<<grid2(), BLAS_BLOCK, 0, st>>>(y, r, d, q, n, w.hop_partials, w.n_hop, w.partials, w.ctrl);  // alpha, y, r, delta, beta
        count_launch();
        KCHECK();
        return STAG_OK;
    }

    int iteration_mode(double *x, cudaStream_t st)
    {
        if (mode == STAG_CG_F64) return iteration<double>(x, w.r64, w.d64, w.q64, w.tmp64, st);
        return iteration<float>(w.y32, w.r32, w.d32, w.q32, w.tmp32, st);
    }

    int read_ctrl()
    {
        CU(cudaMemcpyAsync(L->h_ctrl, w.ctrl, sizeof(CgCtrl), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        return STAG_OK;
    }
};

// nrhs right-hand sides in lockstep.  x, b: nrhs fp64 device spinors
// back to back.  stats: nrhs entries, or null.
int cg_solve_device(double *x, const double *b, stag_links *L, double mass, double tol, int maxiter,
                    int mode, int nrhs, const stag_cg_params_t *prm, stag_cg_stats_t *stats)
{
    stag_cg_params_t P;
    memset(&P, 0, sizeof(P));
    if (prm) P = *prm;
    if (!(P.eps_in > 0.0)) P.eps_in = (mode == STAG_CG_DEFECT) ? 1e-2 : 0.1;
    if (P.graph_chunk == 0) P.graph_chunk = 32;

    Solver S;
    S.L = L;
    S.s = t_stream;
    S.m2 = mass * mass;
    S.mode = mode;
    S.nrhs = nrhs;
    S.prec_lo = (mode == STAG_CG_F64) ? (P.recon8 ? STAG_PREC_F64_R8 : P.recon12 ? STAG_PREC_F64_R12 : STAG_PREC_F64)
                                       : (P.recon8 ? STAG_PREC_F32_R8 : P.recon12 ? STAG_PREC_F32_R12 : STAG_PREC_F32);
    S.prec_hi = P.recon12_f64 ? STAG_PREC_F64_R12 : STAG_PREC_F64;
    S.n = (long)6 * L->g.Vh_pad;
    S.gb = blas_grid(S.n, nrhs);
    S.applies_f64 = 0;
    int rc;
    if ((rc = ensure_links(L, S.prec_lo))) return rc;
    if ((rc = ensure_links(L, S.prec_hi))) return rc;
    if ((rc = ensure_workspace(L, S.w, nrhs))) return rc;
    Workspace &w = S.w;
    cudaStream_t s = S.s;
    const bool lo = (mode != STAG_CG_F64);
    const size_t vec_bytes = (size_t)S.n * sizeof(double);

    CU(cudaEventRecord(L->ev0, s));

    // ---- |b_k|^2 and the solver scalars ---------------------------------------------------
    CgCtrl *h = L->h_ctrl;
    memset(h, 0, sizeof(*h));
    h->mode = mode;
    h->maxiter = maxiter;
    h->eps_in = P.eps_in;
    h->nrhs = nrhs;
    CU(cudaMemcpyAsync(w.ctrl, h, sizeof(CgCtrl), cudaMemcpyHostToDevice, s));
    residual_kernel<float, RES_NORM><<<S.grid2(), BLAS_BLOCK, 0, s>>>(nullptr, b, nullptr, nullptr, S.n, w.partials, w.ctrl);
    count_launch();
    KCHECK();
    if ((rc = S.read_ctrl())) return rc;
    double bnorm2[MAX_RHS];
    bool all_zero = true, bad = false;
    for (int k = 0; k < nrhs; ++k) {
        bnorm2[k] = h->bnorm2[k];
        if (bnorm2[k] != 0.0) all_zero = false;
        if (!(bnorm2[k] == bnorm2[k]) || std::isinf(bnorm2[k])) bad = true;
    }

    stag_cg_stats_t zero;
    memset(&zero, 0, sizeof(zero));
    if (bad) {
        for (int k = 0; stats && k < nrhs; ++k) { stats[k] = zero; stats[k].true_resid = NAN; }
        return STAG_EBREAKDOWN;
    }
    // b_k = 0  =>  x_k = 0 exactly, nothing to iterate for k (no 0/0)
    for (int k = 0; k < nrhs; ++k)
        if (bnorm2[k] == 0.0) CU(cudaMemsetAsync(x + (size_t)k * S.n, 0, vec_bytes, s));
    if (all_zero) {
        CU(cudaEventRecord(L->ev1, s));
        CU(cudaStreamSynchronize(s));
        for (int k = 0; stats && k < nrhs; ++k) stats[k] = zero;
        return STAG_OK;
    }
    for (int k = 0; k < nrhs; ++k) h->tol2b[k] = tol * tol * bnorm2[k];
    CU(cudaMemcpyAsync(w.ctrl, h, sizeof(CgCtrl), cudaMemcpyHostToDevice, s));

    // ---- r = b - A x0 (P:L46 / Fig. 2), in fp64 -------------------------------------
    if ((rc = S.apply_A64(x))) return rc;
    if ((rc = S.residual<RES_INIT>(b, lo))) return rc;
    if (lo) CU(cudaMemsetAsync(w.y32, 0, (size_t)nrhs * S.n * sizeof(float), s));
    // beta = 0 makes the first xpay d = r without reading d, so d needs no initial value

    // ---- the iteration as a CUDA graph of `chunk` passes ----------------------------------
    const int chunk = P.graph_chunk;
    cudaGraphExec_t gexec = nullptr;
    unsigned long long graph_nodes = 0;
    if (chunk > 0) {
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamBeginCapture(L->cap_stream, cudaStreamCaptureModeThreadLocal);
        if (e != cudaSuccess) return cuda_fail(e, "cudaStreamBeginCapture", __LINE__);
        t_capturing = true;
        t_captured_nodes = 0;
        rc = STAG_OK;
        for (int i = 0; i < chunk && rc == STAG_OK; ++i) rc = S.iteration_mode(x, L->cap_stream);
        t_capturing = false;
        graph_nodes = t_captured_nodes;
        e = cudaStreamEndCapture(L->cap_stream, &graph);
        if (rc != STAG_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture", __LINE__);
        e = cudaGraphInstantiate(&gexec, graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) return cuda_fail(e, "cudaGraphInstantiate", __LINE__);
    }
    struct GraphGuard { cudaGraphExec_t g; ~GraphGuard() { if (g) cudaGraphExecDestroy(g); } } guard{gexec};

    int n_restarts = 0, n_outer = 0;
    int final_state = CG_RUN;
    bool have_true = true;      // ctrl->sum0[k] holds |b_k - A x_k|^2 for the current x
    bool verifying = false;     // mode 0: the last launch was the true-residual check of Q6b
    for (;;) {
        if ((rc = S.read_ctrl())) return rc;
        const int state = h->state;
        if (state == CG_RUN) {
            if (verifying) ++n_restarts;
            verifying = false;
            if (gexec) {
                CU(cudaGraphLaunch(gexec, s));
                count_launch(graph_nodes);
            } else {
                for (int i = 0; i < 8; ++i) if ((rc = S.iteration_mode(x, s))) return rc;
            }
            have_true = false;
            continue;
        }
        if (state == CG_UPDATE) {                      // section 3.2: mode 3 only
            if ((rc = S.accumulate(x))) return rc;                 // x += y ; y = 0
            if ((rc = S.apply_A64(x))) return rc;
            if ((rc = S.residual<RES_UPDATE>(b, true))) return rc; // r = b - A x -> r32, beta
            have_true = true;
            continue;
        }
        if (state == CG_CONVERGED && !have_true) {
            if (mode == STAG_CG_F64) {                 // Q6b: verify on the true residual
                if ((rc = S.apply_A64(x))) return rc;
                if ((rc = S.residual<RES_INIT>(b, false))) return rc;
                have_true = true;
                verifying = true;
                continue;
            }
            if (mode == STAG_CG_DEFECT) {              // Fig. 2 outer step
                if ((rc = S.accumulate(x))) return rc;
                if ((rc = S.apply_A64(x))) return rc;
                if ((rc = S.residual<RES_INIT>(b, true))) return rc;
                have_true = true;
                ++n_outer;
                continue;
            }
            if (mode == STAG_CG_F32) {
                if ((rc = S.accumulate(x))) return rc;
                if ((rc = S.apply_A64(x))) return rc;
                if ((rc = S.residual<RES_FINAL>(b, false))) return rc;
                have_true = true;
                final_state = CG_CONVERGED;
                if ((rc = S.read_ctrl())) return rc;
                break;
            }
        }
        if (state == CG_CONVERGED) { final_state = CG_CONVERGED; break; }
        // CG_MAXITER or CG_BREAKDOWN: fold y into x, report the true residual
        final_state = state;
        if (!have_true) {
            if (lo && (rc = S.accumulate(x))) return rc;
            if ((rc = S.apply_A64(x))) return rc;
            if ((rc = S.residual<RES_FINAL>(b, false))) return rc;
            if ((rc = S.read_ctrl())) return rc;
        }
        break;
    }
    CU(cudaEventRecord(L->ev1, s));
    CU(cudaStreamSynchronize(s));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, L->ev0, L->ev1));

    bool all_met = true;
    for (int k = 0; k < nrhs; ++k) {
        stag_cg_stats_t st = zero;
        st.iters = h->iters[k];
        st.n_updates = (mode == STAG_CG_DEFECT) ? n_outer : h->n_updates;
        st.n_restarts = n_restarts;
        st.iters_f32 = lo ? h->iters[k] : 0;
        st.applies_f64 = S.applies_f64;
        st.true_resid = bnorm2[k] > 0.0 ? sqrt(h->sum0[k] / bnorm2[k]) : 0.0;
        st.iter_resid = bnorm2[k] > 0.0 ? sqrt(h->sum1[k] / bnorm2[k]) : 0.0;
        st.seconds = ms * 1e-3;
        if (!(st.true_resid <= tol)) all_met = false;
        if (stats) stats[k] = st;
    }
    if (final_state == CG_BREAKDOWN) return STAG_EBREAKDOWN;
    if (!all_met) return STAG_ENOCONV;
    return STAG_OK;
}

}  // namespace

extern "C" int stag_cg_solve_mrhs(void *x_even, const void *b_even, const stag_links_t *links,
                                  double mass, double tol, int maxiter, int mode, int nrhs,
                                  const stag_cg_params_t *params, stag_cg_stats_t *stats_out)
{
    stag_links *L = const_cast<stag_links *>(links);
    if (!x_even || !b_even || !L || x_even == b_even || !(tol > 0.0) || maxiter < 0 || mode < 0 ||
        mode > 3 || nrhs < 1 || nrhs > MAX_RHS || L->is_slab)
        return STAG_EINVAL;
    return cg_solve_device((double *)x_even, (const double *)b_even, L, mass, tol, maxiter, mode,
                           nrhs, params, stats_out);
}

extern "C" int stag_cg_solve_ex(void *x_even, const void *b_even, const stag_links_t *links,
                                double mass, double tol, int maxiter, int mode,
                                const stag_cg_params_t *params, stag_cg_stats_t *stats_out)
{
    return stag_cg_solve_mrhs(x_even, b_even, links, mass, tol, maxiter, mode, 1, params, stats_out);
}

extern "C" int stag_cg_solve(void *x_even, const void *b_even, const stag_links_t *links,
                             double mass, double tol, int maxiter, int mode, int *iters_out,
                             double *true_resid_out)
{
    stag_cg_stats_t st;
    memset(&st, 0, sizeof(st));
    int rc = stag_cg_solve_ex(x_even, b_even, links, mass, tol, maxiter, mode, nullptr, &st);
    if (rc < 0) return rc;
    if (iters_out) *iters_out = st.iters;
    if (true_resid_out) *true_resid_out = st.true_resid;
    return rc;
}

extern "C" int stag_cg_solve_host(double *x_host, const double *b_host, const stag_links_t *links,
                                  double mass, double tol, int maxiter, int mode,
                                  const stag_cg_params_t *params, stag_cg_stats_t *stats_out)
{
    stag_links *L = const_cast<stag_links *>(links);
    if (!x_host || !b_host || !L || x_host == b_host) return STAG_EINVAL;
    const size_t nc = (size_t)L->g.Vh * 6;         // canonical doubles
    const size_t nd = (size_t)L->g.Vh_pad * 6;     // device-layout doubles
    if (!L->stage_dev) CU(cudaMalloc((void **)&L->stage_dev, (2 * nc + 2 * nd) * sizeof(double)));
    double *cx = L->stage_dev, *cb = cx + nc, *dx = cb + nc, *db = dx + nd;
    CU(cudaMemcpyAsync(cb, b_host, nc * sizeof(double), cudaMemcpyHostToDevice, t_stream));
    CU(cudaMemcpyAsync(cx, x_host, nc * sizeof(double), cudaMemcpyHostToDevice, t_stream));
    int rc;
    if ((rc = stag_spinor_pack(db, cb, L->dims, STAG_PREC_F64))) return rc;
    if ((rc = stag_spinor_pack(dx, cx, L->dims, STAG_PREC_F64))) return rc;
    const int solve_rc = stag_cg_solve_ex(dx, db, L, mass, tol, maxiter, mode, params, stats_out);
    if (solve_rc < 0) return solve_rc;
    if ((rc = stag_spinor_unpack(cx, dx, L->dims, STAG_PREC_F64))) return rc;
    CU(cudaMemcpyAsync(x_host, cx, nc * sizeof(double), cudaMemcpyDeviceToHost, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    return solve_rc;
}

// (D + m) psi = h on the whole lattice through the even-site solve (Q23):
//   b_e = m h_e - D_eo h_o ;  A psi_e = b_e ;  psi_o = (h_o - D_oe psi_e) / m
// The two extra hops run in fp64 on the 18-real links; b_e lives in scratch on the handle.
extern "C" int stag_solve_M(void *psi_even, void *psi_odd, const void *h_even, const void *h_odd,
                            const stag_links_t *links, double mass, double tol, int maxiter,
                            int mode, int nrhs, const stag_cg_params_t *params,
                            stag_cg_stats_t *stats_out)
{
    stag_links *L = const_cast<stag_links *>(links);
    if (!psi_even || !psi_odd || !h_even || !h_odd || !L || psi_even == h_even ||
        psi_odd == h_odd || !(tol > 0.0) || maxiter < 0 || mode < 0 || mode > 3 || nrhs < 1 ||
        nrhs > MAX_RHS || mass == 0.0 || L->is_slab)
        return STAG_EINVAL;
    int rc;
    if ((rc = ensure_links(L, STAG_PREC_F64))) return rc;
    const size_t bytes = (size_t)nrhs * 6 * L->g.Vh_pad * sizeof(double);
    if (L->wrap_b && L->wrap_b_rhs < nrhs) { CU(cudaFree(L->wrap_b)); L->wrap_b = nullptr; }
    if (!L->wrap_b) { CU(cudaMalloc(&L->wrap_b, bytes)); L->wrap_b_rhs = nrhs; }
    // step 1: b_e = m h_e - D_eo h_o
    if ((rc = launch_hop(L, STAG_PREC_F64, HOP_XPAY, L->wrap_b, h_odd, 0, mass, 1.0, h_even, nullptr, nullptr, nrhs, t_stream))) return rc;
    // step 2: A psi_e = b_e (psi_even holds the initial guess on entry)
    const int solve_rc = cg_solve_device((double *)psi_even, (const double *)L->wrap_b, L, mass, tol,
                                         maxiter, mode, nrhs, params, stats_out);
    if (solve_rc < 0) return solve_rc;
    // step 3: psi_o = (1/m) h_o - (1/m) D_oe psi_e
    if ((rc = launch_hop(L, STAG_PREC_F64, HOP_AXPBY, psi_odd, psi_even, 1, 1.0 / mass, 1.0 / mass, h_odd, nullptr, nullptr, nrhs, t_stream))) return rc;
    return solve_rc;
}

// ------------------------------------------------------------------------------------
// C ABI: T-slab decomposition (include/stag.h "T-slabs"; stag_slab.cuh)
// ------------------------------------------------------------------------------------
extern "C" int stag_slab_connect_all(stag_links_t *L, void *const *regions);

extern "C" int stag_slab_create(stag_links_t **slab_out, const int global_dims[4], int antiperiodic_t,
                                const double *W_global, int on_device, int rank, int nranks)
{
    int rc = links_create(slab_out, global_dims, antiperiodic_t, W_global, on_device, 0, rank, nranks);
    if (rc) return rc;
    stag_links *L = *slab_out;
    L->is_slab = 1;
    const size_t bytes = xch_bytes(L->g.s3);
    cudaError_t e = cudaMalloc((void **)&L->xch, bytes);
    if (e == cudaSuccess) e = cudaMemsetAsync(L->xch, 0, bytes, t_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(t_stream);
    if (e != cudaSuccess) { rc = cuda_fail(e, "slab exchange region", __LINE__); stag_links_destroy(L); *slab_out = nullptr; return rc; }
    if (nranks == 1) {                                       // periodic wrap through my own halo
        void *self[1] = { L->xch };
        return stag_slab_connect_all(L, self);
    }
    return STAG_OK;
}

extern "C" int stag_slab_info(const stag_links_t *L, int local_dims_out[4], int *rank_out,
                              int *nranks_out, void **exchange_ptr_out, size_t *exchange_bytes_out)
{
    if (!L || !L->is_slab) return STAG_EINVAL;
    if (local_dims_out) for (int m = 0; m < 4; ++m) local_dims_out[m] = L->dims[m];
    if (rank_out) *rank_out = L->rank;
    if (nranks_out) *nranks_out = L->nranks;
    if (exchange_ptr_out) *exchange_ptr_out = L->xch;
    if (exchange_bytes_out) *exchange_bytes_out = xch_bytes(L->g.s3);
    return STAG_OK;
}

static_assert(sizeof(cudaIpcMemHandle_t) == STAG_IPC_HANDLE_BYTES, "IPC handle size");

extern "C" int stag_slab_ipc_handle(const stag_links_t *L, unsigned char handle_out[STAG_IPC_HANDLE_BYTES])
{
    if (!L || !L->is_slab || !handle_out) return STAG_EINVAL;
    cudaIpcMemHandle_t h;
    CU(cudaIpcGetMemHandle(&h, L->xch));
    memcpy(handle_out, &h, sizeof(h));
    return STAG_OK;
}

extern "C" int stag_slab_ipc_open(const unsigned char handle[STAG_IPC_HANDLE_BYTES], void **ptr_out)
{
    if (!handle || !ptr_out) return STAG_EINVAL;
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, sizeof(h));
    CU(cudaIpcOpenMemHandle(ptr_out, h, cudaIpcMemLazyEnablePeerAccess));
    return STAG_OK;
}

extern "C" int stag_slab_ipc_close(void *ptr)
{
    if (!ptr) return STAG_EINVAL;
    CU(cudaIpcCloseMemHandle(ptr));
    return STAG_OK;
}

extern "C" int stag_slab_connect(stag_links_t *L, void *bwd_exchange, void *fwd_exchange)
{
    if (!L || !L->is_slab || !bwd_exchange || !fwd_exchange) return STAG_EINVAL;
    L->peer_bwd = (char *)bwd_exchange;
    L->peer_fwd = (char *)fwd_exchange;
    return STAG_OK;
}

namespace {

template <typename T>
int slab_push_t(stag_links *L, const cplx_t<T> *in, cudaStream_t s)
{
    const Geom &g = L->g;
    ++L->epoch;            // host mirror, only for "has anything been pushed yet"; the kernels count for themselves
    const unsigned grid = (unsigned)((2L * 3 * g.s3 + 255) / 256);
    face_push_kernel<T><<<grid, 256, 0, s>>>(in, g.Vh, g.Vh_pad, g.s3, L->xch, L->peer_fwd, L->peer_bwd);
    count_launch();
    KCHECK();
    return STAG_OK;
}

template <typename T, int NR>
int slab_hop_t(stag_links *L, int prec, cplx_t<T> *out, const cplx_t<T> *in, int parity, double a,
               const cplx_t<T> *own, cudaStream_t s)
{
    const Geom &g = L->g;
    const pkt_t<T> *field = (const pkt_t<T> *)L->L[prec] +
                            (size_t)parity * L->ntiles * (8 * link_slots(NR) / Pkt<T>::CPP) * TILE;
    const unsigned grid = (unsigned)((g.Vh_pad + DSLASH_BLOCK - 1) / DSLASH_BLOCK);
    HaloArgs<T> h;
    h.xch = L->xch;
    h.peer_fwd = h.peer_bwd = nullptr;
    h.n_push_blocks = 0;
    if (own)
        dslash_kernel<T, NR, HOP_XPAY, 1, true><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)1, own, nullptr, nullptr, h);
    else
        dslash_kernel<T, NR, HOP_PLAIN, 1, true><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)0, (T)1, nullptr, nullptr, nullptr, h);
    count_launch();
    KCHECK();
    return STAG_OK;
}

}  // namespace

extern "C" int stag_slab_push(const void *in, stag_links_t *L, int prec)
{
    if (!in || !L || !L->is_slab || !prec_ok(prec) || !L->peer_bwd || !L->peer_fwd) return STAG_EINVAL;
    if (prec_is_f32(prec)) return slab_push_t<float>(L, (const float2 *)in, t_stream);
    return slab_push_t<double>(L, (const double2 *)in, t_stream);
}

extern "C" int stag_slab_hop(void *out, const void *in, stag_links_t *L, int parity, int prec,
                             double a, const void *own)
{
    if (!out || !in || !L || !L->is_slab || out == in || (parity & ~1) || !prec_ok(prec) ||
        L->epoch == 0)
        return STAG_EINVAL;
    int rc = ensure_links(L, prec);
    if (rc) return rc;
    switch (prec) {
    case STAG_PREC_F64:     return slab_hop_t<double, 3>(L, prec, (double2 *)out, (const double2 *)in, parity, a, (const double2 *)own, t_stream);
    case STAG_PREC_F32:     return slab_hop_t<float, 3>(L, prec, (float2 *)out, (const float2 *)in, parity, a, (const float2 *)own, t_stream);
    case STAG_PREC_F64_R12: return slab_hop_t<double, 2>(L, prec, (double2 *)out, (const double2 *)in, parity, a, (const double2 *)own, t_stream);
    case STAG_PREC_F32_R12: return slab_hop_t<float, 2>(L, prec, (float2 *)out, (const float2 *)in, parity, a, (const float2 *)own, t_stream);
    default: break;       // the 8-parameter forms are whole-lattice only
    }
    return STAG_EINVAL;
}

extern "C" int stag_slab_dslash(void *out, const void *in, stag_links_t *L, int parity, int prec)
{
    int rc = stag_slab_push(in, L, prec);
    if (rc) return rc;
    return stag_slab_hop(out, in, L, parity, prec, 0.0, nullptr);
}

// ------------------------------------------------------------------------------------
// C ABI: CG over T-slabs (include/stag.h "CG over T-slabs")
// ------------------------------------------------------------------------------------
struct stag_slab_cg {
    double *x;
    const double *b;
    double mass, m2, tol;
    int maxiter, mode;
    stag_cg_params_t P;
    Workspace w;
    int prec_lo, prec_hi;
    long n;
    int gb;
    bool lo;
    cudaGraphExec_t iter_graph;      // stag_slab_cg_run: one ACT_ITER (graph_chunk passes) captured
    unsigned long long iter_graph_nodes;
    int stage;                       // 0: nothing done, 1: |b|^2 on its way, 2: in the loop, 3: done
    bool have_true, verifying;
    int n_restarts, applies_f64, final_state;
    double bnorm2;
    int rc_final;
};

extern "C" int stag_slab_connect_all(stag_links_t *L, void *const *regions)
{
    if (!L || !L->is_slab || !regions || L->nranks > MAX_RANKS) return STAG_EINVAL;
    for (int r = 0; r < L->nranks; ++r) if (!regions[r]) return STAG_EINVAL;
    if (!L->peers_dev) CU(cudaMalloc((void **)&L->peers_dev, MAX_RANKS * sizeof(char *)));
    CU(cudaMemcpyAsync(L->peers_dev, regions, L->nranks * sizeof(char *), cudaMemcpyHostToDevice, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    L->peer_bwd = (char *)regions[(L->rank + L->nranks - 1) % L->nranks];
    L->peer_fwd = (char *)regions[(L->rank + 1) % L->nranks];
    L->all_connected = 1;
    return STAG_OK;
}

namespace {

Comm make_comm(const stag_links *L)
{
    Comm c;
    c.peers = L->peers_dev;
    c.mine = L->xch;
    c.nranks = L->nranks;
    c.myrank = L->rank;
    return c;
}

// Blocks of a HALO hop launch that own at least one site of the first or last time slice (the hop
// visits sites rotated by one slice: thread t of block b owns cb = (b*128 + t + s3) mod Vh_pad).
unsigned push_block_count(const Geom &g)
{
    const unsigned grid = (unsigned)((g.Vh_pad + DSLASH_BLOCK - 1) / DSLASH_BLOCK);
    unsigned n = 0;
    for (unsigned b = 0; b < grid; ++b) {
        bool any = false;
        for (int t = 0; t < DSLASH_BLOCK && !any; ++t) {
            int cb = (int)b * DSLASH_BLOCK + t;
            if (cb >= g.Vh_pad) break;
            cb += g.s3;
            if (cb >= g.Vh_pad) cb -= g.Vh_pad;
            if (cb < g.Vh) {
                const int x3 = cb / g.s3;
                any = (x3 == 0 || x3 == g.X3 - 1);
            }
        }
        n += any ? 1u : 0u;
    }
    return n;
}

template <typename T, int NR>
int slab_hop_mode_t(stag_links *L, int prec, int hop, cplx_t<T> *out, const cplx_t<T> *in, int parity,
                    double a, const cplx_t<T> *own, double *partials, const CgCtrl *ctrl, cudaStream_t s,
                    bool push_out = false)
{
    const Geom &g = L->g;
    const pkt_t<T> *field = (const pkt_t<T> *)L->L[prec] +
                            (size_t)parity * L->ntiles * (8 * link_slots(NR) / Pkt<T>::CPP) * TILE;
    const unsigned grid = (unsigned)((g.Vh_pad + DSLASH_BLOCK - 1) / DSLASH_BLOCK);
    HaloArgs<T> h;
    h.xch = L->xch;
    h.peer_fwd = h.peer_bwd = nullptr;
    h.n_push_blocks = 0;
    if (push_out && hop == HOP_PLAIN) {      // the faces of out go to the neighbours as the next exchange
        h.peer_fwd = L->peer_fwd;
        h.peer_bwd = L->peer_bwd;
        if (L->n_push_blocks == 0) L->n_push_blocks = push_block_count(g);    // once per handle
        h.n_push_blocks = L->n_push_blocks;
        ++L->epoch;
    }
    switch (hop) {
    case HOP_PLAIN:
        dslash_kernel<T, NR, HOP_PLAIN, 1, true><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)0, (T)1, nullptr, nullptr, ctrl, h);
        break;
    case HOP_XPAY:
        dslash_kernel<T, NR, HOP_XPAY, 1, true><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)1, own, nullptr, ctrl, h);
        break;
    default:
        dslash_kernel<T, NR, HOP_XPAY_DOT, 1, true><<<grid, DSLASH_BLOCK, 0, s>>>(out, in, field, g, parity, (T)a, (T)1, own, partials, ctrl, h);
        break;
    }
    count_launch();
    KCHECK();
    return STAG_OK;
}

int slab_hop_mode(stag_links *L, int prec, int hop, void *out, const void *in, int parity, double a,
                  const void *own, double *partials, const CgCtrl *ctrl, cudaStream_t s, bool push_out = false)
{
    switch (prec) {
    case STAG_PREC_F64:     return slab_hop_mode_t<double, 3>(L, prec, hop, (double2 *)out, (const double2 *)in, parity, a, (const double2 *)own, partials, ctrl, s, push_out);
    case STAG_PREC_F32:     return slab_hop_mode_t<float, 3>(L, prec, hop, (float2 *)out, (const float2 *)in, parity, a, (const float2 *)own, partials, ctrl, s, push_out);
    case STAG_PREC_F64_R12: return slab_hop_mode_t<double, 2>(L, prec, hop, (double2 *)out, (const double2 *)in, parity, a, (const double2 *)own, partials, ctrl, s, push_out);
    case STAG_PREC_F32_R12: return slab_hop_mode_t<float, 2>(L, prec, hop, (float2 *)out, (const float2 *)in, parity, a, (const float2 *)own, partials, ctrl, s, push_out);
    default: break;
    }
    return STAG_EINVAL;
}

int slab_push_prec(stag_links *L, const void *in, int prec, cudaStream_t s)
{
    if (prec_is_f32(prec)) return slab_push_t<float>(L, (const float2 *)in, s);
    return slab_push_t<double>(L, (const double2 *)in, s);
}

// r64 = b - A64 x and its global |r|^2 in four phases (0..3); WHAT selects the scalar step.
template <int WHAT>
int slab_residual_phase(stag_links *L, stag_slab_cg *C, int ph, bool accumulate_first, bool lo_copy, bool *more, cudaStream_t s)
{
    Workspace &w = C->w;
    int rc = STAG_OK;
    *more = ph < 3;
    switch (ph) {
    case 0:
        if (accumulate_first) {
            accumulate_kernel<float><<<blas_grid(C->n, 1), BLAS_BLOCK, 0, s>>>(C->x, w.y32, C->n);   // x += y ; y = 0
            count_launch();
            KCHECK();
        }
        return slab_push_prec(L, C->x, C->prec_hi, s);
    case 1:
        if ((rc = slab_hop_mode(L, C->prec_hi, HOP_PLAIN, w.tmp64, C->x, 1, 0.0, nullptr, nullptr, nullptr, s))) return rc;
        ++C->applies_f64;
        return slab_push_prec(L, w.tmp64, C->prec_hi, s);
    case 2:
        if ((rc = slab_hop_mode(L, C->prec_hi, HOP_XPAY, w.q64, w.tmp64, 0, C->m2, C->x, nullptr, nullptr, s))) return rc;
        slab_residual_kernel<float, WHAT><<<C->gb, BLAS_BLOCK, 0, s>>>(w.r64, C->b, w.q64, lo_copy ? w.r32 : nullptr, C->n, w.partials, w.ctrl, make_comm(L));
        count_launch();
        KCHECK();
        return STAG_OK;
    case 3:
        slab_scalar_kernel<WHAT><<<1, 32, 0, s>>>(w.ctrl, make_comm(L));
        count_launch();
        KCHECK();
        return STAG_OK;
    }
    return STAG_EINVAL;
}

// phase ph of iteration chunk: five phases per pass of Fig. 1's loop
template <typename T>
int slab_iteration_phase(stag_links *L, stag_slab_cg *C, int sub, T *y, T *r, T *d, T *q, T *tmp, cudaStream_t s)
{
    Workspace &w = C->w;
    int rc;
    switch (sub) {
    case 0:   // d = r + beta d, its faces stored into the neighbours' halos by the same kernel
        ++L->epoch;
        slab_xpay_push_kernel<T><<<C->gb, BLAS_BLOCK, 0, s>>>(d, r, C->n, w.ctrl, L->g.Vh, L->g.Vh_pad, L->g.s3,
                                                             L->xch, L->peer_fwd, L->peer_bwd);
        count_launch();
        KCHECK();
        return STAG_OK;
    case 1:   // tmp = D_oe d, the faces of tmp pushed by the boundary-slice threads of the same kernel
        return slab_hop_mode(L, C->prec_lo, HOP_PLAIN, tmp, d, 1, 0.0, nullptr, nullptr, w.ctrl, s, true);
    case 2:   // q = m^2 d - D_eo tmp, local <d,q> published
        if ((rc = slab_hop_mode(L, C->prec_lo, HOP_XPAY_DOT, q, tmp, 0, C->m2, d, w.hop_partials, w.ctrl, s))) return rc;
        slab_publish_partials_kernel<<<1, 1024, 0, s>>>(w.hop_partials, w.n_hop, make_comm(L), w.ctrl);
        count_launch();
        KCHECK();
        return STAG_OK;
    case 3:   // alpha from the global <d,Ad>; y, r; local |r|^2 published
        slab_update_kernel<T><<<C->gb, BLAS_BLOCK, 0, s>>>(y, r, d, q, C->n, w.partials, w.ctrl, make_comm(L));
        count_launch();
        KCHECK();
        return STAG_OK;
    case 4:   // beta, stopping tests, trigger: the same epilogue on every rank
        slab_scalar_kernel<SCALAR_ITER><<<1, 32, 0, s>>>(w.ctrl, make_comm(L));
        count_launch();
        KCHECK();
        return STAG_OK;
    }
    return STAG_EINVAL;
}

}  // namespace

extern "C" int stag_slab_cg_begin(stag_links_t *L, void *x_even, const void *b_even, double mass,
                                  double tol, int maxiter, int mode, const stag_cg_params_t *params)
{
    if (!L || !L->is_slab || !L->all_connected || !x_even || !b_even || x_even == b_even ||
        !(tol > 0.0) || maxiter < 0 || (mode != STAG_CG_F64 && mode != STAG_CG_RELIABLE))
        return STAG_EINVAL;
    if (!L->cg) {
        L->cg = new (std::nothrow) stag_slab_cg();
        if (!L->cg) return STAG_ENOMEM;
    }
    stag_slab_cg *C = L->cg;
    if (C->iter_graph) cudaGraphExecDestroy(C->iter_graph);
    memset(C, 0, sizeof(*C));
    if (params) C->P = *params;
    if (!(C->P.eps_in > 0.0)) C->P.eps_in = 0.1;
    if (C->P.graph_chunk <= 0) C->P.graph_chunk = 32;    // iterations between host checks (plain launches)
    C->x = (double *)x_even;
    C->b = (const double *)b_even;
    C->mass = mass;
    C->m2 = mass * mass;
    C->tol = tol;
    C->maxiter = maxiter;
    C->mode = mode;
    C->lo = (mode != STAG_CG_F64);
    C->prec_lo = C->lo ? (C->P.recon12 ? STAG_PREC_F32_R12 : STAG_PREC_F32)
                       : (C->P.recon12 ? STAG_PREC_F64_R12 : STAG_PREC_F64);
    C->prec_hi = C->P.recon12_f64 ? STAG_PREC_F64_R12 : STAG_PREC_F64;
    C->n = (long)6 * L->g.Vh_pad;
    C->gb = blas_grid(C->n, 1);
    int rc;
    if ((rc = ensure_links(L, C->prec_lo))) return rc;
    if ((rc = ensure_links(L, C->prec_hi))) return rc;
    if ((rc = ensure_workspace(L, C->w, 1))) return rc;
    CgCtrl *h = L->h_ctrl;
    memset(h, 0, sizeof(*h));
    h->mode = mode;
    h->maxiter = maxiter;
    h->eps_in = C->P.eps_in;
    h->nrhs = 1;
    CU(cudaMemcpyAsync(C->w.ctrl, h, sizeof(CgCtrl), cudaMemcpyHostToDevice, t_stream));
    CU(cudaEventRecord(L->ev0, t_stream));
    C->stage = 0;
    return STAG_OK;
}

// Decide what every rank does next.  Synchronises the stream and reads the control block; all
// ranks hold identical scalars, so all ranks get the same answer.
extern "C" int stag_slab_cg_control(stag_links_t *L, int *action_out)
{
    if (!L || !L->is_slab || !L->cg || !action_out) return STAG_EINVAL;
    stag_slab_cg *C = L->cg;
    CgCtrl *h = L->h_ctrl;
    if (C->stage == 0) { C->stage = 1; *action_out = STAG_SLAB_ACT_NORM; return STAG_OK; }
    if (C->stage == 3) { *action_out = STAG_SLAB_ACT_DONE; return STAG_OK; }
    CU(cudaMemcpyAsync(h, C->w.ctrl, sizeof(CgCtrl), cudaMemcpyDeviceToHost, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    if (C->stage == 1) {                       // |b|^2 (global) has arrived
        C->bnorm2 = h->bnorm2[0];
        if (C->bnorm2 == 0.0) {                // b = 0  =>  x = 0, nothing to iterate
            CU(cudaMemsetAsync(C->x, 0, (size_t)C->n * sizeof(double), t_stream));
            C->final_state = CG_CONVERGED;
            C->stage = 3;
            *action_out = STAG_SLAB_ACT_DONE;
            return STAG_OK;
        }
        if (!(C->bnorm2 == C->bnorm2) || std::isinf(C->bnorm2)) {
            C->final_state = CG_BREAKDOWN;
            h->sum0[0] = NAN;
            C->stage = 3;
            *action_out = STAG_SLAB_ACT_DONE;
            return STAG_OK;
        }
        h->tol2b[0] = C->tol * C->tol * C->bnorm2;
        CU(cudaMemcpyAsync(C->w.ctrl, h, sizeof(CgCtrl), cudaMemcpyHostToDevice, t_stream));
        C->stage = 2;
        C->have_true = true;
        *action_out = STAG_SLAB_ACT_INIT;      // r = b - A x0, also sets y = 0
        return STAG_OK;
    }
    const int state = h->state;
    if (state == CG_RUN) {
        if (C->verifying) ++C->n_restarts;
        C->verifying = false;
        C->have_true = false;
        *action_out = STAG_SLAB_ACT_ITER;
        return STAG_OK;
    }
    if (state == CG_UPDATE) {                  // section 3.2
        C->have_true = true;
        *action_out = STAG_SLAB_ACT_UPDATE;
        return STAG_OK;
    }
    if (state == CG_CONVERGED && !C->have_true && C->mode == STAG_CG_F64) {   // Q6b
        C->have_true = true;
        C->verifying = true;
        *action_out = STAG_SLAB_ACT_VERIFY;
        return STAG_OK;
    }
    if (state == CG_CONVERGED && C->have_true) {
        C->final_state = CG_CONVERGED;
        C->stage = 3;
        *action_out = STAG_SLAB_ACT_DONE;
        return STAG_OK;
    }
    // CG_MAXITER or CG_BREAKDOWN (or a converged state without a true residual): report it
    C->final_state = state;
    if (!C->have_true) {
        C->have_true = true;
        *action_out = STAG_SLAB_ACT_FINAL;
        return STAG_OK;
    }
    C->stage = 3;
    *action_out = STAG_SLAB_ACT_DONE;
    return STAG_OK;
}

// Enqueue phase `phase` of `action`.  *more_out = 1 while the action has further phases.  Within a
// phase no kernel waits for a peer's kernel of the SAME phase, so ranks that share a device may be
// stepped one after the other, phase by phase.
static int slab_cg_step_on(stag_links_t *L, int action, int phase, int *more_out, cudaStream_t t_stream);

extern "C" int stag_slab_cg_step(stag_links_t *L, int action, int phase, int *more_out)
{
    return slab_cg_step_on(L, action, phase, more_out, t_stream);
}

static int slab_cg_step_on(stag_links_t *L, int action, int phase, int *more_out, cudaStream_t t_stream)
{
    if (!L || !L->is_slab || !L->cg || phase < 0 || !more_out) return STAG_EINVAL;
    stag_slab_cg *C = L->cg;
    Workspace &w = C->w;
    bool more = false;
    int rc = STAG_EINVAL;
    switch (action) {
    case STAG_SLAB_ACT_NORM:
        if (phase == 0) {
                slab_residual_kernel<float, RES_NORM><<<C->gb, BLAS_BLOCK, 0, t_stream>>>(nullptr, C->b, nullptr, nullptr, C->n, w.partials, w.ctrl, make_comm(L));
            count_launch();
            KCHECK();
            more = true;
            rc = STAG_OK;
        } else if (phase == 1) {
            slab_scalar_kernel<RES_NORM><<<1, 32, 0, t_stream>>>(w.ctrl, make_comm(L));
            count_launch();
            KCHECK();
            rc = STAG_OK;
        }
        break;
    case STAG_SLAB_ACT_INIT:
        if (phase == 0 && C->lo) CU(cudaMemsetAsync(w.y32, 0, (size_t)C->n * sizeof(float), t_stream));
        rc = slab_residual_phase<RES_INIT>(L, C, phase, false, C->lo, &more, t_stream);
        break;
    case STAG_SLAB_ACT_VERIFY:
        rc = slab_residual_phase<RES_INIT>(L, C, phase, false, false, &more, t_stream);
        break;
    case STAG_SLAB_ACT_UPDATE:
        rc = slab_residual_phase<RES_UPDATE>(L, C, phase, true, true, &more, t_stream);
        break;
    case STAG_SLAB_ACT_FINAL:
        rc = slab_residual_phase<RES_FINAL>(L, C, phase, C->lo, false, &more, t_stream);
        break;
    case STAG_SLAB_ACT_ITER: {
        const int total = 5 * C->P.graph_chunk;
        if (phase >= total) return STAG_EINVAL;
        more = phase + 1 < total;
        if (C->lo) rc = slab_iteration_phase<float>(L, C, phase % 5, w.y32, w.r32, w.d32, w.q32, w.tmp32, t_stream);
        else rc = slab_iteration_phase<double>(L, C, phase % 5, C->x, w.r64, w.d64, w.q64, w.tmp64, t_stream);
        break;
    }
    default:
        return STAG_EINVAL;
    }
    *more_out = more ? 1 : 0;
    return rc;
}

extern "C" int stag_slab_cg_finish(stag_links_t *L, stag_cg_stats_t *stats_out)
{
    if (!L || !L->is_slab || !L->cg || L->cg->stage != 3) return STAG_EINVAL;
    stag_slab_cg *C = L->cg;
    CgCtrl *h = L->h_ctrl;
    CU(cudaEventRecord(L->ev1, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, L->ev0, L->ev1));
    stag_cg_stats_t st;
    memset(&st, 0, sizeof(st));
    st.iters = h->iters[0];
    st.n_updates = h->n_updates;
    st.n_restarts = C->n_restarts;
    st.iters_f32 = C->lo ? h->iters[0] : 0;
    st.applies_f64 = C->applies_f64;
    st.true_resid = C->bnorm2 > 0.0 ? sqrt(h->sum0[0] / C->bnorm2) : 0.0;
    st.iter_resid = C->bnorm2 > 0.0 ? sqrt(h->sum1[0] / C->bnorm2) : 0.0;
    st.seconds = ms * 1e-3;
    if (stats_out) *stats_out = st;
    if (C->final_state == CG_BREAKDOWN) return STAG_EBREAKDOWN;
    if (!(st.true_resid <= C->tol)) return STAG_ENOCONV;
    return STAG_OK;
}

// begin + the control / step loop + finish in one call: what each process of a one-process-per-GPU
// run uses (every rank calls it at the same time; kernels of a phase may wait for peers' kernels
// of earlier phases, which are running or queued on the OTHER devices).
extern "C" int stag_slab_cg_run(stag_links_t *L, void *x_even, const void *b_even, double mass,
                                double tol, int maxiter, int mode, const stag_cg_params_t *params,
                                stag_cg_stats_t *stats_out)
{
    int rc = stag_slab_cg_begin(L, x_even, b_even, mass, tol, maxiter, mode, params);
    if (rc) return rc;
    for (;;) {
        int act = STAG_SLAB_ACT_DONE;
        if ((rc = stag_slab_cg_control(L, &act))) return rc;
        if (act == STAG_SLAB_ACT_DONE) break;
        if (act == STAG_SLAB_ACT_ITER) {
            // the chunk of iterations as ONE graph launch: possible because the exchange and
            // reduction numbers live in device memory, not in the kernels' arguments
            stag_slab_cg *C = L->cg;
            if (!C->iter_graph) {
                cudaGraph_t graph = nullptr;
                cudaError_t e = cudaStreamBeginCapture(L->cap_stream, cudaStreamCaptureModeThreadLocal);
                if (e != cudaSuccess) return cuda_fail(e, "cudaStreamBeginCapture", __LINE__);
                t_capturing = true;
                t_captured_nodes = 0;
                int more = 1;
                rc = STAG_OK;
                for (int ph = 0; more && rc == STAG_OK; ++ph) rc = slab_cg_step_on(L, act, ph, &more, L->cap_stream);
                t_capturing = false;
                C->iter_graph_nodes = t_captured_nodes;
                e = cudaStreamEndCapture(L->cap_stream, &graph);
                if (rc != STAG_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
                if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture", __LINE__);
                e = cudaGraphInstantiate(&C->iter_graph, graph, 0);
                cudaGraphDestroy(graph);
                if (e != cudaSuccess) return cuda_fail(e, "cudaGraphInstantiate", __LINE__);
            }
            CU(cudaGraphLaunch(C->iter_graph, t_stream));
            count_launch(C->iter_graph_nodes);
            continue;
        }
        int more = 1;
        for (int ph = 0; more; ++ph)
            if ((rc = stag_slab_cg_step(L, act, ph, &more))) return rc;
    }
    return stag_slab_cg_finish(L, stats_out);
}

static void stag_slab_cg_free(struct stag_slab_cg *c)
{
    if (c && c->iter_graph) cudaGraphExecDestroy(c->iter_graph);
    delete c;
}
