// stag_host_persist.cuh -- launching the persistent iteration kernel (stag_persist.cuh)
//
// A section of libstag's single translation unit: included by stag_lib.cu, which holds the
// per-thread state, the error / launch-count helpers and the link handle these sections share.
// Not a stand-alone header.

namespace {

// offset of the rank group's barrier words inside the workspace's control slot (behind CgCtrl)
constexpr size_t PERSIST_BAR_OFF = 1792;
static_assert(sizeof(CgCtrl) <= PERSIST_BAR_OFF && PERSIST_BAR_OFF + sizeof(unsigned) <= CTRL_SLOT, "barrier words must fit the control slot");

// persistent = 0 picks the persistent kernel for whole lattices of at most this many sites per parity
// (28^3 x 24 = 263 424: 47.8 us per pass against 50.4 on the kernel-per-step path; at 28^3 x 48 the
// two are level and beyond it the stand-alone hops win, profiles/README.md round 2).  T-slabs, whose
// kernel-per-step pass has six launches, gain up to a larger volume: 28^3 x 48 (526 848 sites) 101.0 us
// per pass against 107.5, 28^3 x 96 199.0-200.2 against 193.9-197.7.
constexpr int PERSIST_AUTO_MAX_VH = 300000;
constexpr int PERSIST_AUTO_MAX_VH_SLAB = 800000;

// Most passes one persistent launch carries (params.persist_chunk is clamped to it).  The group
// barrier compares a 32-bit arrival counter, reset at every launch, with a target that grows by the
// group's block count at each of the <= 7 barriers of a pass: 65 536 passes x 7 x 296 blocks = 1.4e8,
// far from wrapping -- an unchecked user value of a few million passes would wrap it and leave the
// cooperative grid spinning for ever (the whole-lattice path has no watchdog).
constexpr int PERSIST_MAX_CHUNK = 65536;

inline bool persist_prec_ok(int prec)     // the 8-parameter forms stay on the kernel-per-step path
{
    return prec == STAG_PREC_F64 || prec == STAG_PREC_F32 || prec == STAG_PREC_F64_R12 || prec == STAG_PREC_F32_R12;
}

// Blocks of the persistent kernel that can be resident at once on this device (the cooperative
// launch refuses more).  One query per instantiation and device.
template <typename T, int NR, bool SLAB, bool LRES>
int persist_capacity()
{
    constexpr int MAX_DEV = 64;                  // cached per device ordinal; beyond that, asked every time
    static std::atomic<int> cap[MAX_DEV];        // zero-initialised
    int dev = 0, sms = 0, per = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    const bool cached = dev >= 0 && dev < MAX_DEV;
    int c = cached ? cap[dev].load(std::memory_order_relaxed) : 0;
    if (c == 0) {
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, cg_iter_persistent_kernel<T, NR, SLAB, LRES>, PERSIST_THREADS, 0) != cudaSuccess)
            return -1;
        c = sms * per;
        if (cached) cap[dev].store(c, std::memory_order_relaxed);
    }
    return c;
}

// persistent = 0: which lattices iterate in the persistent kernel.  The kernel boundaries it removes
// cost a fixed ~5 us per pass; its hops end with 4-8 us of stragglers at the barrier on lattices
// that stream from HBM, so on one GPU it pays for small volumes only.
inline bool persist_by_volume(const Geom &g, bool is_slab)
{
    return g.Vh <= (is_slab ? PERSIST_AUTO_MAX_VH_SLAB : PERSIST_AUTO_MAX_VH);
}

// Bytes of links + vectors up to which the persistent kernel keeps the links in L2: 5/8 of the
// device's L2 (126 MB on B200), which leaves room for the two dies' duplicates and the fp64 vectors.
inline size_t persist_l2_budget()
{
    static std::atomic<size_t> budget{0};
    size_t b = budget.load(std::memory_order_relaxed);
    if (b == 0) {
        int dev = 0, l2 = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev) != cudaSuccess) l2 = 0;
        b = (size_t)l2 / 8 * 5;
        if (b == 0) b = 1;
        budget.store(b, std::memory_order_relaxed);
    }
    return b;
}

// Blocks a rank group of this volume can use: one site per thread per trip at most.
inline int persist_want(const Geom &g) { return (g.Vh_pad + PERSIST_THREADS - 1) / PERSIST_THREADS; }

template <typename T>
void persist_fill(IterRank<T> &R, const stag_links *L, const Workspace &w, int prec, double m2,
                  T *y, T *r, T *d, T *q, T *tmp)
{
    const int rows = prec_rows(prec);
    const size_t per_parity = (size_t)L->ntiles * (8 * link_slots(rows) / Pkt<T>::CPP) * TILE;
    R.y = y; R.r = r; R.d = d; R.q = q; R.tmp = tmp;
    R.links_even = (const pkt_t<T> *)L->L[prec];
    R.links_odd = R.links_even + per_parity;
    R.g = L->g;
    R.ctrl = w.ctrl;
    R.partials = w.partials;
    R.bar = (unsigned *)((char *)w.ctrl + PERSIST_BAR_OFF);
    R.m2 = (T)m2;
    R.block0 = 0; R.nblocks = 0;
    R.xch = L->is_slab ? L->xch : nullptr;
    R.peer_fwd = L->peer_fwd; R.peer_bwd = L->peer_bwd;
    R.peers = L->peers_dev;
    R.nranks = L->nranks; R.myrank = L->rank;
    memset(&R.up, 0, sizeof(R.up));          // reliable updates are the host's unless persist_fill_update follows
}

// Mode 3 with the fp64 corrections on 18-real links: the kernel does the reliable + group-wise update
// itself (x += y, r = b - A x in fp64), so a whole solve is one launch per persist_chunk passes.
inline void persist_fill_update(IterUpdate &U, const stag_links *L, const Workspace &w, double *x, const double *b, double m2)
{
    const size_t per_parity = (size_t)L->ntiles * (8 * link_slots(3)) * TILE;
    U.x = x; U.b = b; U.tmp = w.tmp64;
    U.links_even = (const double2 *)L->L[STAG_PREC_F64];
    U.links_odd = U.links_even + per_parity;
    U.m2 = m2;
}

template <typename T, int NR, bool SLAB, bool LRES>
int persist_launch_t(IterArgs<T> &A, cudaStream_t s)
{
    const int cap = persist_capacity<T, NR, SLAB, LRES>();
    if (cap < A.nlocal) {
        snprintf(t_errbuf, sizeof(t_errbuf), "persistent kernel: %d rank group(s) but only %d block(s) can be resident on this device", A.nlocal, cap);
        t_errbuf_status = STAG_ECUDA;
        (void)cudaGetLastError();
        return STAG_ECUDA;
    }
    // split the resident blocks evenly among the rank groups, no group larger than its volume needs
    const int share = cap / A.nlocal;
    int grid = 0;
    for (int i = 0; i < A.nlocal; ++i) {
        int nb = persist_want(A.rk[i].g);
        if (nb > share) nb = share;
        if (nb < 1) nb = 1;
        A.rk[i].block0 = grid;
        A.rk[i].nblocks = nb;
        grid += nb;
    }
    for (int i = 0; i < A.nlocal; ++i) CU(cudaMemsetAsync(A.rk[i].bar, 0, sizeof(unsigned), s));
    void *args[] = { (void *)&A };
    CU(cudaLaunchCooperativeKernel((const void *)cg_iter_persistent_kernel<T, NR, SLAB, LRES>, dim3((unsigned)grid),
                                   dim3(PERSIST_THREADS), args, 0, s));
    count_launch();
#ifdef STAG_PERSIST_TIMING
    {
        unsigned long long h[16];
        cudaStreamSynchronize(s);
        if (cudaMemcpyFromSymbol(h, g_persist_stamps, sizeof(h)) == cudaSuccess) {
            static const char *what[10] = { "P0 xpay", "barrier", "P1 hop", "barrier", "P2 hop+dot", "barrier", "sum <d,Ad>", "P3 update", "barrier", "sum |r|^2" };
            fprintf(stderr, "[persist pass 20, ns]");
            for (int k = 0; k < 10; ++k) fprintf(stderr, " %s %llu |", what[k], h[k + 1] - h[k]);
            fprintf(stderr, " total %llu\n", h[10] - h[0]);
        }
    }
#endif
    return STAG_OK;
}

template <typename T>
int persist_launch(IterArgs<T> &A, int prec, bool slab, cudaStream_t s)
{
    const int rows = prec_rows(prec);
    // do the links of both parities and the five vectors of every rank group fit L2 together?
    size_t bytes = 0;
    for (int i = 0; i < A.nlocal; ++i)
        bytes += (size_t)A.rk[i].g.Vh_pad * (2 * 8 * link_slots(rows) * 2 + 5 * 6) * sizeof(T);
    const bool lres = bytes <= persist_l2_budget();
    if (rows == 3) {
        if (lres) return slab ? persist_launch_t<T, 3, true, true>(A, s) : persist_launch_t<T, 3, false, true>(A, s);
        return slab ? persist_launch_t<T, 3, true, false>(A, s) : persist_launch_t<T, 3, false, false>(A, s);
    }
    if (rows == 2) {
        if (lres) return slab ? persist_launch_t<T, 2, true, true>(A, s) : persist_launch_t<T, 2, false, true>(A, s);
        return slab ? persist_launch_t<T, 2, true, false>(A, s) : persist_launch_t<T, 2, false, false>(A, s);
    }
    return STAG_EINVAL;
}

}  // namespace
