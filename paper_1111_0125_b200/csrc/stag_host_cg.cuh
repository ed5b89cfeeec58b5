// stag_host_cg.cuh -- the CG drivers of one GPU (Fig. 1, Fig. 2, section 3.2; several right-hand sides; the (D+m) wrapper) and their C ABI
//
// A section of libstag's single translation unit: included by stag_lib.cu, which holds the
// per-thread state, the error / launch-count helpers and the link handle these sections share.
// Not a stand-alone header.

// ------------------------------------------------------------------------------------
// the CG drivers
// ------------------------------------------------------------------------------------
namespace {

struct Solver {
    const stag_links *L;
    WsHost *ws;
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
    bool paired;     // the fp32 vectors are a paired batch (nrhs >= 2, fp32 modes)
    int gb_lo;       // grid.x of the iteration's vector kernels: blocks per unit (pair or single)

    dim3 grid2() const { return dim3((unsigned)gb, (unsigned)nrhs); }
    // paired: 1-D grid of nrhs*gb_lo equal blocks (stag_blas.cuh, paired_unit); else (blocks, right-hand sides)
    dim3 grid_lo() const { return paired ? dim3((unsigned)(gb_lo * nrhs), 1u) : dim3((unsigned)gb_lo, (unsigned)nrhs); }

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
        residual_kernel<float, WHAT><<<grid2(), BLAS_BLOCK, 0, s>>>(w.r64, b, w.q64, lo_copy ? w.r32 : nullptr, n, 2L * L->g.Vh_pad, 2L * L->g.Vh, w.partials, w.ctrl, paired);
        count_launch();
        KCHECK();
        return STAG_OK;
    }

    int accumulate(double *x)
    {
        if (!paired) {
            accumulate_kernel<float><<<blas_grid(n * nrhs, 1), BLAS_BLOCK, 0, s>>>(x, w.y32, n * nrhs);
            count_launch();
            KCHECK();
            return STAG_OK;
        }
        const int npairs = nrhs / 2;
        accumulate_paired_kernel<<<blas_grid(n * npairs, 1), BLAS_BLOCK, 0, s>>>(x, w.y32, n, npairs);
        count_launch();
        KCHECK();
        if (nrhs & 1) {
            const size_t off = (size_t)(nrhs - 1) * n;
            accumulate_kernel<float><<<blas_grid(n, 1), BLAS_BLOCK, 0, s>>>(x + off, w.y32 + off, n);
            count_launch();
            KCHECK();
        }
        return STAG_OK;
    }

    // one pass of the loop body of Fig. 1, four launches (the hops: one launch per
    // chunk of right-hand sides)
    template <typename T>
    int iteration(T *y, T *r, T *d, T *q, T *tmp, cudaStream_t st)
    {
        constexpr bool F32 = std::is_same<T, float>::value;
        const int layout = (F32 && paired) ? STAG_BATCH_PAIRED : STAG_BATCH_BLOCKED;
        if (F32 && paired) xpay_paired_kernel<<<grid_lo(), BLAS_BLOCK, 0, st>>>((float *)d, (const float *)r, n, w.ctrl);
        else xpay_kernel<T><<<grid_lo(), BLAS_BLOCK, 0, st>>>(d, r, n, w.ctrl);             // d = r + beta d
        count_launch();
        KCHECK();
        int rc = launch_hop(L, prec_lo, HOP_PLAIN, tmp, d, 1, 0.0, 1.0, nullptr, nullptr, w.ctrl, nrhs, st, layout);   // D_oe d
        if (rc) return rc;
        rc = launch_hop(L, prec_lo, HOP_XPAY_DOT, q, tmp, 0, m2, 1.0, d, w.hop_partials, w.ctrl, nrhs, st, layout);  // q = A d, <d,q>
        if (rc) return rc;
        if (F32 && paired) update_paired_kernel<<<grid_lo(), BLAS_BLOCK, 0, st>>>((float *)y, (float *)r, (const float *)d, (const float *)q, n, w.hop_partials, w.n_hop, w.partials, w.ctrl);
        else update_kernel<T><<<grid_lo(), BLAS_BLOCK, 0, st>>>(y, r, d, q, n, w.hop_partials, w.n_hop, w.partials, w.ctrl);  // alpha, y, r, delta, beta
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
        CU(cudaMemcpyAsync(ws->h_ctrl, w.ctrl, sizeof(CgCtrl), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        return STAG_OK;
    }
};

// nrhs right-hand sides in lockstep.  x, b: nrhs fp64 device spinors
// back to back.  stats: nrhs entries, or null.
// ws: the leased workspace (at least ws_layout(g, mode, nrhs).total bytes).
int cg_solve_device(double *x, const double *b, const stag_links *L, WsHost *ws, double mass, double tol,
                    int maxiter, int mode, int nrhs, const stag_cg_params_t *prm, stag_cg_stats_t *stats)
{
    stag_cg_params_t P;
    memset(&P, 0, sizeof(P));
    if (prm) P = *prm;
    if (!(P.eps_in > 0.0)) P.eps_in = (mode == STAG_CG_DEFECT) ? 1e-2 : 0.1;
    if (P.graph_chunk == 0) P.graph_chunk = 32;
    if (P.persist_chunk <= 0) P.persist_chunk = 1024;
    if (P.persist_chunk > PERSIST_MAX_CHUNK) P.persist_chunk = PERSIST_MAX_CHUNK;

    Solver S;
    S.L = L;
    S.ws = ws;
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
    S.paired = (mode != STAG_CG_F64) && nrhs >= 2;
    S.gb_lo = S.gb;      // blocks per right-hand side: a pair gets twice as many
    int rc;
    if ((rc = ensure_links(L, S.prec_lo))) return rc;
    if ((rc = ensure_links(L, S.prec_hi))) return rc;
    carve(ws->base, ws_layout(L->g, mode, nrhs), S.w);
    Workspace &w = S.w;
    cudaStream_t s = S.s;
    const bool lo = (mode != STAG_CG_F64);
    const size_t vec_bytes = (size_t)S.n * sizeof(double);

    CU(cudaEventRecord(ws->ev0, s));

    // Pad lanes (Vh not a multiple of 32) must be zero in every vector that enters a reduction:
    // x is the caller's to overwrite, so its pads are zeroed here; b is read-only, its pads are
    // masked where b is read (residual_kernel).
    if (L->g.Vh_pad != L->g.Vh) {
        zero_pads_kernel<<<dim3(1, (unsigned)nrhs), 128, 0, s>>>((double2 *)x, L->g.Vh, L->g.Vh_pad);
        count_launch();
        KCHECK();
    }

    // ---- |b_k|^2 and the solver scalars ---------------------------------------------------
    CgCtrl *h = ws->h_ctrl;
    memset(h, 0, sizeof(*h));
    h->mode = mode;
    h->maxiter = maxiter;
    h->eps_in = P.eps_in;
    h->nrhs = nrhs;
    CU(cudaMemcpyAsync(w.ctrl, h, sizeof(CgCtrl), cudaMemcpyHostToDevice, s));
    residual_kernel<float, RES_NORM><<<S.grid2(), BLAS_BLOCK, 0, s>>>(nullptr, b, nullptr, nullptr, S.n, 2L * L->g.Vh_pad, 2L * L->g.Vh, w.partials, w.ctrl);
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
        CU(cudaEventRecord(ws->ev1, s));
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
    // Instantiated once per (handle, mode, link form, nrhs, chunk, mass[, x]) and kept with the
    // workspace: everything else the nodes bake in (vector addresses, control block) is a
    // function of the workspace's base address and those.
    // Or, for one right-hand side, as one persistent kernel per chunk (stag_persist.cuh).
    bool persist = nrhs == 1 && persist_prec_ok(S.prec_lo) &&
                   (P.persistent > 0 || (P.persistent == 0 && persist_by_volume(L->g, false)));
    IterArgs<float> pa32;
    IterArgs<double> pa64;
    if (persist) {
        if (lo) {
            persist_fill<float>(pa32.rk[0], L, w, S.prec_lo, S.m2, w.y32, w.r32, w.d32, w.q32, w.tmp32);
            if ((mode == STAG_CG_RELIABLE || mode == STAG_CG_DEFECT) && S.prec_hi == STAG_PREC_F64) persist_fill_update(pa32.rk[0].up, L, w, x, b, S.m2);
            pa32.nlocal = 1; pa32.max_iters = P.persist_chunk;
        } else {
            persist_fill<double>(pa64.rk[0], L, w, S.prec_lo, S.m2, x, w.r64, w.d64, w.q64, w.tmp64);
            pa64.nlocal = 1; pa64.max_iters = P.persist_chunk;
        }
    }
    const int chunk = P.graph_chunk;
    cudaGraphExec_t gexec = nullptr;
    unsigned long long graph_nodes = 0;
    // (a lambda: the persistent path needs the graph only if its launch is refused, see the loop)
    auto acquire_graph = [&]() -> int {
        if (chunk <= 0 || gexec) return STAG_OK;
        const void *xkey = (mode == STAG_CG_F64) ? (const void *)x : nullptr;
        GraphSlot *slot = nullptr, *victim = &ws->graphs[0];
        for (GraphSlot &gs : ws->graphs) {
            if (gs.exec && gs.uid == L->uid && gs.mode == mode && gs.prec_lo == S.prec_lo && gs.nrhs == nrhs &&
                gs.chunk == chunk && gs.m2 == S.m2 && gs.x == xkey) { slot = &gs; break; }
            if (!gs.exec || (victim->exec && gs.stamp < victim->stamp)) victim = &gs;
        }
        if (!slot) {
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamBeginCapture(ws->cap_stream, cudaStreamCaptureModeThreadLocal);
            if (e != cudaSuccess) return cuda_fail(e, "cudaStreamBeginCapture", __LINE__);
            t_capturing = true;
            t_captured_nodes = 0;
            rc = STAG_OK;
            for (int i = 0; i < chunk && rc == STAG_OK; ++i) rc = S.iteration_mode(x, ws->cap_stream);
            t_capturing = false;
            e = cudaStreamEndCapture(ws->cap_stream, &graph);
            if (rc != STAG_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture", __LINE__);
            cudaGraphExec_t ge = nullptr;
            e = cudaGraphInstantiate(&ge, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) return cuda_fail(e, "cudaGraphInstantiate", __LINE__);
            if (victim->exec) cudaGraphExecDestroy(victim->exec);
            *victim = GraphSlot{L->uid, mode, S.prec_lo, nrhs, chunk, S.m2, xkey, ge, t_captured_nodes, 0};
            slot = victim;
        }
        slot->stamp = ++ws->stamp;
        gexec = slot->exec;
        graph_nodes = slot->nodes;
        return STAG_OK;
    };
    if (!persist && (rc = acquire_graph())) return rc;

    int n_restarts = 0, n_outer = 0;
    int final_state = CG_RUN;
    bool have_true = true;      // ctrl->sum0[k] holds |b_k - A x_k|^2 for the current x
    bool verifying = false;     // mode 0: the last launch was the true-residual check of Q6b
    bool persist_ran = false;   // the last thing launched was the persistent kernel: it says whether sum0 is current
    bool persist_any = false;   // a persistent launch has been accepted in this solve
    for (;;) {
        if ((rc = S.read_ctrl())) return rc;
        const int state = h->state;
        if (persist_ran) { have_true = h->have_true != 0; persist_ran = false; }
        if (state == CG_RUN) {
            if (verifying) ++n_restarts;
            verifying = false;
            if (persist) {
                rc = lo ? persist_launch<float>(pa32, S.prec_lo, false, s) : persist_launch<double>(pa64, S.prec_lo, false, s);
                if (rc == STAG_OK) {
                    persist_ran = persist_any = true;
                    continue;
                }
                // The library chose this path itself (persistent = 0) and the device refuses the
                // cooperative launch (an MPS thread limit, MIG, a green context, no cooperative
                // launch at all) before any pass has run: nothing was changed, so take the
                // kernel-per-step path these lattices ran on before.  An explicit persistent = 1
                // keeps the hard error.
                if (P.persistent != 0 || persist_any) return rc;
                (void)cudaGetLastError();
                persist = false;
                if ((rc = acquire_graph())) return rc;
            }
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
    CU(cudaEventRecord(ws->ev1, s));
    CU(cudaStreamSynchronize(s));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, ws->ev0, ws->ev1));

    bool all_met = true;
    for (int k = 0; k < nrhs; ++k) {
        stag_cg_stats_t st = zero;
        st.iters = h->iters[k];
        st.n_updates = (mode == STAG_CG_DEFECT) ? n_outer + h->n_inkernel : h->n_updates;
        st.n_restarts = n_restarts;
        st.iters_f32 = lo ? h->iters[k] : 0;
        st.applies_f64 = S.applies_f64 + h->n_inkernel;
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

extern "C" int stag_cg_solve_mrhs(void *x_even, const void *b_even, const stag_links_t *L,
                                  double mass, double tol, int maxiter, int mode, int nrhs,
                                  const stag_cg_params_t *params, stag_cg_stats_t *stats_out)
{
    if (!x_even || !b_even || !L || x_even == b_even || !(tol > 0.0) || maxiter < 0 || mode < 0 ||
        mode > 3 || nrhs < 1 || nrhs > MAX_RHS || L->is_slab)
        return STAG_EINVAL;
    WsLease lease;
    int rc = lease_workspace(L, ws_layout(L->g, mode, nrhs).total, lease);
    if (rc) return rc;
    return cg_solve_device((double *)x_even, (const double *)b_even, L, lease.ws, mass, tol, maxiter, mode,
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

// The canonical copies of b and x0 pass through the workspace's r64 / q64 (dead until the solve
// starts, and again once it has finished); x and b in the device layout have their own two slots.
extern "C" int stag_cg_solve_host(double *x_host, const double *b_host, const stag_links_t *L,
                                  double mass, double tol, int maxiter, int mode,
                                  const stag_cg_params_t *params, stag_cg_stats_t *stats_out)
{
    if (!x_host || !b_host || !L || x_host == b_host || !(tol > 0.0) || maxiter < 0 || mode < 0 ||
        mode > 3 || L->is_slab)
        return STAG_EINVAL;
    const size_t nc = (size_t)L->g.Vh * 6;         // canonical doubles
    const size_t nd = (size_t)L->g.Vh_pad * 6;     // device-layout doubles
    const WsLayout lay = ws_layout(L->g, mode, 1);
    WsLease lease;
    int rc = lease_workspace(L, lay.total, lease);
    if (rc) return rc;
    Workspace w;
    carve(lease.ws->base, lay, w);
    double *cb = w.r64, *cx = w.q64, *dx = w.stage, *db = w.stage + nd;
    CU(cudaMemcpyAsync(cb, b_host, nc * sizeof(double), cudaMemcpyHostToDevice, t_stream));
    CU(cudaMemcpyAsync(cx, x_host, nc * sizeof(double), cudaMemcpyHostToDevice, t_stream));
    if ((rc = stag_spinor_pack(db, cb, L->dims, STAG_PREC_F64))) return rc;
    if ((rc = stag_spinor_pack(dx, cx, L->dims, STAG_PREC_F64))) return rc;
    const int solve_rc = cg_solve_device(dx, db, L, lease.ws, mass, tol, maxiter, mode, 1, params, stats_out);
    if (solve_rc < 0) return solve_rc;
    if ((rc = stag_spinor_unpack(cx, dx, L->dims, STAG_PREC_F64))) return rc;
    CU(cudaMemcpyAsync(x_host, cx, nc * sizeof(double), cudaMemcpyDeviceToHost, t_stream));
    CU(cudaStreamSynchronize(t_stream));
    return solve_rc;
}

// (D + m) psi = h on the whole lattice through the even-site solve (Q23):
//   b_e = m h_e - D_eo h_o ;  A psi_e = b_e ;  psi_o = (h_o - D_oe psi_e) / m
// The two extra hops run in fp64 on the 18-real links; b_e lives in the workspace.
extern "C" int stag_solve_M(void *psi_even, void *psi_odd, const void *h_even, const void *h_odd,
                            const stag_links_t *L, double mass, double tol, int maxiter,
                            int mode, int nrhs, const stag_cg_params_t *params,
                            stag_cg_stats_t *stats_out)
{
    if (!psi_even || !psi_odd || !h_even || !h_odd || !L || psi_even == h_even ||
        psi_odd == h_odd || !(tol > 0.0) || maxiter < 0 || mode < 0 || mode > 3 || nrhs < 1 ||
        nrhs > MAX_RHS || mass == 0.0 || L->is_slab)
        return STAG_EINVAL;
    int rc;
    if ((rc = ensure_links(L, STAG_PREC_F64))) return rc;
    const WsLayout lay = ws_layout(L->g, mode, nrhs);
    WsLease lease;
    if ((rc = lease_workspace(L, lay.total, lease))) return rc;
    Workspace w;
    carve(lease.ws->base, lay, w);
    // step 1: b_e = m h_e - D_eo h_o
    if ((rc = launch_hop(L, STAG_PREC_F64, HOP_XPAY, w.wrap_b, h_odd, 0, mass, 1.0, h_even, nullptr, nullptr, nrhs, t_stream))) return rc;
    // step 2: A psi_e = b_e (psi_even holds the initial guess on entry)
    const int solve_rc = cg_solve_device((double *)psi_even, w.wrap_b, L, lease.ws, mass, tol,
                                         maxiter, mode, nrhs, params, stats_out);
    if (solve_rc < 0) return solve_rc;
    // step 3: psi_o = (1/m) h_o - (1/m) D_oe psi_e
    if ((rc = launch_hop(L, STAG_PREC_F64, HOP_AXPBY, psi_odd, psi_even, 1, 1.0 / mass, 1.0 / mass, h_odd, nullptr, nullptr, nrhs, t_stream))) return rc;
    if (L->g.Vh_pad != L->g.Vh) {       // psi_o's pad lanes hold h_o's / m: zero them (every output keeps zero pads)
        zero_pads_kernel<<<dim3(1, (unsigned)nrhs), 128, 0, t_stream>>>((double2 *)psi_odd, L->g.Vh, L->g.Vh_pad);
        count_launch();
        KCHECK();
    }
    return solve_rc;
}
