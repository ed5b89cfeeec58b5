// stag_host_slab.cuh -- the C ABI of the T-slab decomposition: exchange wiring, push / hop, and the CG over slabs
//
// A section of libstag's single translation unit: included by stag_lib.cu, which holds the
// per-thread state, the error / launch-count helpers and the link handle these sections share.
// Not a stand-alone header.

// ------------------------------------------------------------------------------------
// C ABI: T-slab decomposition (include/stag.h "T-slabs"; stag_slab.cuh)
// ------------------------------------------------------------------------------------
extern "C" int stag_slab_connect_all(stag_links_t *L, void *const *regions);

static int slab_finish_create(stag_links_t **slab_out, int rc, int nranks);

extern "C" int stag_slab_create(stag_links_t **slab_out, const int global_dims[4], int antiperiodic_t,
                                const double *W_global, int on_device, int rank, int nranks)
{
    return slab_finish_create(slab_out, links_create(slab_out, global_dims, antiperiodic_t, W_global, on_device, 0, rank, nranks), nranks);
}

extern "C" int stag_slab_create_local(stag_links_t **slab_out, const int global_dims[4], int antiperiodic_t,
                                      const double *W_local, const double *W_back, int on_device,
                                      int rank, int nranks)
{
    return slab_finish_create(slab_out, links_create(slab_out, global_dims, antiperiodic_t, W_local, on_device, 0, rank, nranks, W_back, true), nranks);
}

static int slab_finish_create(stag_links_t **slab_out, int rc, int nranks)
{
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
    if (prec_rows(prec) == 1) return STAG_EINVAL;      // the 8-parameter forms are whole-lattice only
    return slab_hop_mode(L, prec, own ? HOP_XPAY : HOP_PLAIN, out, in, parity, a, own, nullptr, nullptr, t_stream);
}

extern "C" int stag_slab_set_wait_limit(stag_links_t *L, unsigned long long polls)
{
    if (!L || !L->is_slab) return STAG_EINVAL;
    CU(cudaMemcpyAsync(&((XchHeader *)L->xch)->wait_limit, &polls, sizeof(polls), cudaMemcpyHostToDevice, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    return STAG_OK;
}

extern "C" int stag_slab_wait_stats(stag_links_t *L, unsigned long long *waits_spun_out, unsigned long long *polls_out)
{
    if (!L || !L->is_slab) return STAG_EINVAL;
    unsigned long long v[2] = {0, 0};
    CU(cudaMemcpyAsync(v, &((XchHeader *)L->xch)->waits_spun, sizeof(v), cudaMemcpyDeviceToHost, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    if (waits_spun_out) *waits_spun_out = v[0];
    if (polls_out) *polls_out = v[1];
    return STAG_OK;
}

extern "C" int stag_slab_reset(stag_links_t *L)
{
    if (!L || !L->is_slab) return STAG_EINVAL;
    CU(cudaStreamSynchronize(t_stream));
    unsigned long long limit = 0;
    XchHeader *hdr = (XchHeader *)L->xch;
    CU(cudaMemcpyAsync(&limit, &hdr->wait_limit, sizeof(limit), cudaMemcpyDeviceToHost, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    CU(cudaMemsetAsync(L->xch, 0, XCH_HDR, t_stream));        // flags, counts, tickets, the mark, reduction slots and flags
    CU(cudaMemcpyAsync(&hdr->wait_limit, &limit, sizeof(limit), cudaMemcpyHostToDevice, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    L->epoch = 0;
    return STAG_OK;
}

extern "C" int stag_slab_status(stag_links_t *L)
{
    if (!L || !L->is_slab) return STAG_EINVAL;
    unsigned flag = 0;
    CU(cudaMemcpyAsync(&flag, &((XchHeader *)L->xch)->timed_out, sizeof(flag), cudaMemcpyDeviceToHost, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    return flag ? STAG_ETIMEOUT : STAG_OK;
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
    bool persist;                    // stag_slab_cg_run iterates in the persistent kernel (stag_persist.cuh)
    bool persist_ran;                // the last action was a persistent launch: ctrl->have_true says whether sum0 is current
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
        slab_residual_kernel<float, WHAT><<<C->gb, BLAS_BLOCK, 0, s>>>(w.r64, C->b, w.q64, lo_copy ? w.r32 : nullptr, C->n, 2L * L->g.Vh_pad, 2L * L->g.Vh, w.partials, w.ctrl, make_comm(L));
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
    if (C->P.persist_chunk <= 0) C->P.persist_chunk = 1024;
    if (C->P.persist_chunk > PERSIST_MAX_CHUNK) C->P.persist_chunk = PERSIST_MAX_CHUNK;
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
    {   // a slab handle belongs to one host thread and owns its workspace
        const WsLayout lay = ws_layout(L->g, mode, 1);
        WsLease lease;
        WsHost *saved = t_ws.p;
        t_ws.p = nullptr;                           // never the caller's: the solve spans several calls
        rc = lease_workspace(L, lay.total, lease);
        t_ws.p = saved;
        if (rc) return rc;
        carve(L->own.base, lay, C->w);
    }
    if (L->g.Vh_pad != L->g.Vh) {
        zero_pads_kernel<<<dim3(1, 1), 128, 0, t_stream>>>((double2 *)x_even, L->g.Vh, L->g.Vh_pad);
        count_launch();
        KCHECK();
    }
    CgCtrl *h = L->own.h_ctrl;
    memset(h, 0, sizeof(*h));
    h->mode = mode;
    h->maxiter = maxiter;
    h->eps_in = C->P.eps_in;
    h->nrhs = 1;
    CU(cudaMemcpyAsync(C->w.ctrl, h, sizeof(CgCtrl), cudaMemcpyHostToDevice, t_stream));
    // persistent = 0 (the library decides) takes the persistent kernel only for a lattice held by ONE
    // slab.  Across several GPUs its peer stores, system-scope flags and replicated scalars have never
    // executed on hardware and its volume threshold was measured with all ranks on one device (same
    // L2, no NVLink): until tests/test_gpu_slab_multi.py and a timing have run on >= 2 GPUs it is
    // opt-in there (persistent = 1) and the default is the kernel-per-step graph.
    C->persist = persist_prec_ok(C->prec_lo) &&
                 (C->P.persistent > 0 || (C->P.persistent == 0 && L->nranks == 1 && persist_by_volume(L->g, true)));
    CU(cudaEventRecord(L->own.ev0, t_stream));
    C->stage = 0;
    return STAG_OK;
}

// One ACT_ITER of the slabs given, all of them in ONE cooperative launch of the persistent kernel
// (stag_persist.cuh): every slab is a rank group of the grid.  n = 1 is what a process of a
// one-process-per-GPU run launches for itself; n = nranks with every slab on this device is the
// single-GPU emulation of the multi-GPU run, the ranks concurrent by construction.
namespace {
template <typename T>
int slab_iter_all_t(stag_links_t *const *slabs, int n, cudaStream_t s)
{
    IterArgs<T> A;
    const stag_slab_cg *C0 = slabs[0]->cg;
    for (int i = 0; i < n; ++i) {
        stag_links *L = slabs[i];
        stag_slab_cg *C = L->cg;
        Workspace &w = C->w;
        if (std::is_same<T, float>::value) {
            persist_fill<T>(A.rk[i], L, w, C->prec_lo, C->m2, (T *)w.y32, (T *)w.r32, (T *)w.d32, (T *)w.q32, (T *)w.tmp32);
            if (C->mode == STAG_CG_RELIABLE && C->prec_hi == STAG_PREC_F64) persist_fill_update(A.rk[i].up, L, w, C->x, C->b, C->m2);
        } else
            persist_fill<T>(A.rk[i], L, w, C->prec_lo, C->m2, (T *)C->x, (T *)w.r64, (T *)w.d64, (T *)w.q64, (T *)w.tmp64);
        ++L->epoch;
        C->persist_ran = true;
    }
    A.nlocal = n;
    A.max_iters = C0->P.persist_chunk;
    return persist_launch<T>(A, C0->prec_lo, true, s);
}
}  // namespace

extern "C" int stag_slab_cg_iter_all(stag_links_t *const *slabs, int n)
{
    if (!slabs || n < 1 || n > MAX_RANKS) return STAG_EINVAL;
    for (int i = 0; i < n; ++i) {
        const stag_links *L = slabs[i];
        if (!L || !L->is_slab || !L->cg || L->cg->stage != 2 || !persist_prec_ok(L->cg->prec_lo)) return STAG_EINVAL;
        if (L->cg->prec_lo != slabs[0]->cg->prec_lo || L->cg->P.persist_chunk != slabs[0]->cg->P.persist_chunk) return STAG_EINVAL;
        for (int j = 0; j < i; ++j) if (slabs[j] == L) return STAG_EINVAL;
    }
    return slabs[0]->cg->lo ? slab_iter_all_t<float>(slabs, n, t_stream) : slab_iter_all_t<double>(slabs, n, t_stream);
}

// Decide what every rank does next.  Synchronises the stream and reads the control block; all
// ranks hold identical scalars, so all ranks get the same answer.
extern "C" int stag_slab_cg_control(stag_links_t *L, int *action_out)
{
    if (!L || !L->is_slab || !L->cg || !action_out) return STAG_EINVAL;
    stag_slab_cg *C = L->cg;
    CgCtrl *h = L->own.h_ctrl;
    if (C->stage == 0) { C->stage = 1; *action_out = STAG_SLAB_ACT_NORM; return STAG_OK; }
    if (C->stage == 3) { *action_out = STAG_SLAB_ACT_DONE; return STAG_OK; }
    CU(cudaMemcpyAsync(h, C->w.ctrl, sizeof(CgCtrl), cudaMemcpyDeviceToHost, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    { const int ws = stag_slab_status(L); if (ws != STAG_OK) return ws; }      // a wait gave up: nothing below is valid
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
    if (C->persist_ran) { C->have_true = h->have_true != 0; C->persist_ran = false; }
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
            slab_residual_kernel<float, RES_NORM><<<C->gb, BLAS_BLOCK, 0, t_stream>>>(nullptr, C->b, nullptr, nullptr, C->n, 2L * L->g.Vh_pad, 2L * L->g.Vh, w.partials, w.ctrl, make_comm(L));
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
    CgCtrl *h = L->own.h_ctrl;
    CU(cudaEventRecord(L->own.ev1, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    { const int ws = stag_slab_status(L); if (ws != STAG_OK) return ws; }
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, L->own.ev0, L->own.ev1));
    stag_cg_stats_t st;
    memset(&st, 0, sizeof(st));
    st.iters = h->iters[0];
    st.n_updates = h->n_updates;
    st.n_restarts = C->n_restarts;
    st.iters_f32 = C->lo ? h->iters[0] : 0;
    st.applies_f64 = C->applies_f64 + h->n_inkernel;
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
            if (C->persist) {
                stag_links_t *one[1] = { L };
                if ((rc = stag_slab_cg_iter_all(one, 1))) return rc;
                continue;
            }
            if (!C->iter_graph) {
                cudaGraph_t graph = nullptr;
                cudaError_t e = cudaStreamBeginCapture(L->own.cap_stream, cudaStreamCaptureModeThreadLocal);
                if (e != cudaSuccess) return cuda_fail(e, "cudaStreamBeginCapture", __LINE__);
                t_capturing = true;
                t_captured_nodes = 0;
                int more = 1;
                rc = STAG_OK;
                for (int ph = 0; more && rc == STAG_OK; ++ph) rc = slab_cg_step_on(L, act, ph, &more, L->own.cap_stream);
                t_capturing = false;
                C->iter_graph_nodes = t_captured_nodes;
                e = cudaStreamEndCapture(L->own.cap_stream, &graph);
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

