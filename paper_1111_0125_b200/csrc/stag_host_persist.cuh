// stag_host_persist.cuh -- launching the persistent iteration kernel (stag_persist.cuh)
//
// A section of libstag's single translation unit: included by stag_lib.cu, which holds the
// per-thread state, the error / launch-count helpers and the link handle these sections share.
// Not a stand-alone header.

namespace {

// offset of the rank group's barrier words inside the workspace's control slot (behind CgCtrl)
constexpr size_t PERSIST_BAR_OFF = 1792;
static_assert(sizeof(CgCtrl) <= PERSIST_BAR_OFF && PERSIST_BAR_OFF + 2 * sizeof(unsigned) <= CTRL_SLOT, "barrier words must fit the control slot");

constexpr int PERSIST_AUTO_MAX_VH = 0;     // set from the measurements (profiles/README.md)

inline bool persist_prec_ok(int prec)     // the 8-parameter forms stay on the kernel-per-step path
{
    return prec == STAG_PREC_F64 || prec == STAG_PREC_F32 || prec == STAG_PREC_F64_R12 || prec == STAG_PREC_F32_R12;
}

// Blocks of the persistent kernel that can be resident at once on this device (the cooperative
// launch refuses more).  One query per instantiation.
template <typename T, int NR, bool SLAB>
int persist_capacity()
{
    static std::atomic<int> cap{0};
    int c = cap.load(std::memory_order_relaxed);
    if (c == 0) {
        int dev = 0, sms = 0, per = 0;
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, cg_iter_persistent_kernel<T, NR, SLAB>, PERSIST_THREADS, 0) != cudaSuccess)
            return -1;
        c = sms * per;
        cap.store(c, std::memory_order_relaxed);
    }
    return c;
}

// persistent = 0: which lattices iterate in the persistent kernel.  The kernel boundaries it removes
// cost a fixed ~12 us per pass; its own hop is a few per cent slower than the stand-alone kernel
// on lattices that stream from HBM, so it pays for small volumes only.
inline bool persist_by_volume(const Geom &g, bool lo)
{
    (void)lo;
    return g.Vh <= PERSIST_AUTO_MAX_VH;
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
}

template <typename T, int NR, bool SLAB>
int persist_launch_t(IterArgs<T> &A, cudaStream_t s)
{
    const int cap = persist_capacity<T, NR, SLAB>();
    if (cap < A.nlocal) return STAG_ECUDA;
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
    void *args[] = { (void *)&A };
    CU(cudaLaunchCooperativeKernel((const void *)cg_iter_persistent_kernel<T, NR, SLAB>, dim3((unsigned)grid),
                                   dim3(PERSIST_THREADS), args, 0, s));
    count_launch();
    return STAG_OK;
}

template <typename T>
int persist_launch(IterArgs<T> &A, int prec, bool slab, cudaStream_t s)
{
    const int rows = prec_rows(prec);
    if (rows == 3) return slab ? persist_launch_t<T, 3, true>(A, s) : persist_launch_t<T, 3, false>(A, s);
    if (rows == 2) return slab ? persist_launch_t<T, 2, true>(A, s) : persist_launch_t<T, 2, false>(A, s);
    return STAG_EINVAL;
}

}  // namespace
