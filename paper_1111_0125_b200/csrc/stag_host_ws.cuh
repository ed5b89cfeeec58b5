// stag_host_ws.cuh -- the CG workspace: its layout, who owns it, and the C ABI stag_cg_workspace_bytes / stag_set_workspace
//
// A section of libstag's single translation unit: included by stag_lib.cu, which holds the
// per-thread state, the error / launch-count helpers and the link handle these sections share.
// Not a stand-alone header.
//
// What a workspace holds ("the caller owns every spinor buffer and the
// workspace"): the vectors of Fig. 1 other than x and b -- r, d, Ad = q and the odd-site
// intermediate of A (eq. 2.3) in fp64 -- the fp32 iteration's y, r, d, q, tmp (section 3.2,
// P:L88-101), the device-resident scalars (CgCtrl), the partial sums of the inner products, and
// the scratch of the wrapper entry points.  One layout function serves stag_cg_workspace_bytes and
// the carving, so the two cannot disagree.

namespace {

struct WsLayout {
    size_t ctrl, partials, hop_partials;   // offsets
    size_t scratch;                        // stag_apply_A's odd-site intermediate (aliases wrap_b .. r64: no solve runs meanwhile)
    size_t wrap_b;                         // stag_solve_M: b_e, nrhs fp64 spinors
    size_t stage;                          // stag_cg_solve_host: x and b in the device layout, 2 fp64 spinors
    size_t r64, q64, tmp64, d64;           // nrhs fp64 spinors each (d64: mode 0 only)
    size_t y32, r32, d32, q32, tmp32;      // nrhs fp32 spinors each (modes 1-3 only)
    size_t total;
    int n_hop;
};

// mode < 0: the operator entry points only (stag_apply_A*): control block + nrhs fp64 spinors.
WsLayout ws_layout(const Geom &g, int mode, int nrhs)
{
    WsLayout w;
    const size_t n = (size_t)6 * g.Vh_pad;
    const size_t nb64 = align_up((size_t)nrhs * n * sizeof(double), 256);
    const size_t nb32 = align_up((size_t)nrhs * n * sizeof(float), 256);
    const size_t one64 = align_up(n * sizeof(double), 256);
    w.n_hop = (int)(((size_t)g.Vh_pad + DSLASH_BLOCK - 1) / DSLASH_BLOCK);
    size_t p = 0;
    w.ctrl = p;         p += CTRL_SLOT;
    w.partials = p;     p += align_up((size_t)MAX_RHS * MAX_BLAS_GRID * sizeof(double), 256);
    w.hop_partials = p; p += align_up((size_t)nrhs * w.n_hop * sizeof(double), 256);
    w.scratch = p;
    w.wrap_b = p;       p += nb64;
    if (mode < 0) { w.stage = w.r64 = w.q64 = w.tmp64 = w.d64 = w.y32 = w.r32 = w.d32 = w.q32 = w.tmp32 = p; w.total = p; return w; }
    w.stage = p;        p += 2 * one64;
    w.r64 = p;          p += nb64;
    w.q64 = p;          p += nb64;
    w.tmp64 = p;        p += nb64;
    w.d64 = p;          if (mode == STAG_CG_F64) p += nb64;
    w.y32 = w.r32 = w.d32 = w.q32 = w.tmp32 = p;
    if (mode != STAG_CG_F64) {
        w.y32 = p;   p += nb32;
        w.r32 = p;   p += nb32;
        w.d32 = p;   p += nb32;
        w.q32 = p;   p += nb32;
        w.tmp32 = p; p += nb32;
    }
    w.total = p;
    return w;
}

struct Workspace {
    CgCtrl *ctrl;
    double *partials;       // block partials of the vector kernels' reductions, [rhs][block]
    double *hop_partials;   // block partials of <d,Ad> written by the second hop, [rhs][block]
    int n_hop;              // = grid of the hop
    double *wrap_b, *stage;
    double *r64, *q64, *tmp64, *d64;          // nrhs spinors each
    float *y32, *r32, *d32, *q32, *tmp32;
};

void carve(char *base, const WsLayout &l, Workspace &w)
{
    w.ctrl = (CgCtrl *)(base + l.ctrl);
    w.partials = (double *)(base + l.partials);
    w.hop_partials = (double *)(base + l.hop_partials);
    w.n_hop = l.n_hop;
    w.wrap_b = (double *)(base + l.wrap_b);
    w.stage = (double *)(base + l.stage);
    w.r64 = (double *)(base + l.r64);
    w.q64 = (double *)(base + l.q64);
    w.tmp64 = (double *)(base + l.tmp64);
    w.d64 = (double *)(base + l.d64);
    w.y32 = (float *)(base + l.y32);
    w.r32 = (float *)(base + l.r32);
    w.d32 = (float *)(base + l.d32);
    w.q32 = (float *)(base + l.q32);
    w.tmp32 = (float *)(base + l.tmp32);
}

// The workspace one call runs on, for the duration of the call.  With a caller-owned workspace
// (this thread called stag_set_workspace) nothing of the link handle is touched.  Otherwise the
// handle's own workspace is used under the handle's mutex (held until the lease ends), grown on
// demand; a call arriving on another stream than the previous one first waits, on the device, for
// that one's work (the event `busy`; the same on a caller-owned workspace whose thread changed its
// stream), so the default path is safe -- merely serialised -- from any number of threads and streams.
struct WsLease {
    WsHost *ws = nullptr;
    std::unique_lock<std::mutex> lock;
    WsLease() = default;
    WsLease(const WsLease &) = delete;
    WsLease &operator=(const WsLease &) = delete;
    ~WsLease()
    {
        if (!ws) return;
        if (ws->busy && cudaEventRecord(ws->busy, t_stream) == cudaSuccess) {
            ws->busy_recorded = true;
            ws->last_stream = t_stream;
        } else {
            (void)cudaGetLastError();
        }
        ws->in_use = false;
    }
};

int lease_workspace(const stag_links *L, size_t need, WsLease &out)
{
    if (t_ws.p) {
        WsHost *w = t_ws.p;
        if (w->bytes < need) {
            snprintf(t_errbuf, sizeof(t_errbuf), "workspace too small: %zu bytes set, this call needs %zu (stag_cg_workspace_bytes)", w->bytes, need);
            t_errbuf_status = STAG_EINVAL;
            return STAG_EINVAL;
        }
        if (w->in_use) return STAG_EINVAL;
        if (w->busy_recorded && w->last_stream != t_stream) CU(cudaStreamWaitEvent(t_stream, w->busy, 0));
        w->in_use = true;
        out.ws = w;
        return STAG_OK;
    }
    out.lock = std::unique_lock<std::mutex>(L->mu_ws);
    WsHost *w = &L->own;
    int rc = w->init_host_objects();
    if (rc) return rc;
    if (w->bytes < need) {
        w->drop_graphs();                       // they bake the old addresses
        if (w->base) CU(cudaFree(w->base));     // cudaFree waits for the device: no kernel still uses it
        w->base = nullptr; w->bytes = 0;
        CU(cudaMalloc((void **)&w->base, need));
        w->bytes = need;
        w->owned = true;
        w->busy_recorded = false;
    } else if (w->busy_recorded && w->last_stream != t_stream) {
        CU(cudaStreamWaitEvent(t_stream, w->busy, 0));
    }
    w->in_use = true;
    out.ws = w;
    return STAG_OK;
}

}  // namespace

extern "C" size_t stag_cg_workspace_bytes(const int dims[4], int mode, int nrhs)
{
    Geom g;
    if (!make_geom(g, dims, 0) || mode > 3 || nrhs < 1 || nrhs > MAX_RHS) return 0;
    return ws_layout(g, mode, nrhs).total;
}

extern "C" int stag_set_workspace(void *ws, size_t bytes)
{
    if (t_ws.p) {
        if (t_ws.p->in_use) return STAG_EINVAL;
        if (ws && t_ws.p->base == (char *)ws && t_ws.p->bytes == bytes) return STAG_OK;   // unchanged: keep the cached graphs
        t_ws.p->release();
        delete t_ws.p;
        t_ws.p = nullptr;
    }
    if (!ws) return bytes == 0 ? STAG_OK : STAG_EINVAL;
    if (bytes < CTRL_SLOT || ((uintptr_t)ws & 255u)) return STAG_EINVAL;     // 256-byte aligned (any cudaMalloc / torch allocation is)
    WsHost *w = new (std::nothrow) WsHost();
    if (!w) return STAG_ENOMEM;
    const int rc = w->init_host_objects();
    if (rc) { w->release(); delete w; return rc; }
    w->base = (char *)ws;
    w->bytes = bytes;
    w->owned = false;
    t_ws.p = w;
    return STAG_OK;
}
