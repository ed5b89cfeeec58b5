// stag_lib.cu -- host side of libstag: the C ABI of include/stag.h, the link handle and its
// setup kernels (step S0), kernel launchers, and the CG drivers (Fig. 1, Fig. 2, section 3.2).
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <type_traits>

#include "stag_blas.cuh"
#include "stag_common.cuh"
#include "stag_dslash.cuh"
#include "stag_dslash_batch.cuh"
#include "stag_slab.cuh"
#include "stag_persist.cuh"

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
// is too short to feed them.  Returns grid.x, the blocks per right-hand side.  Never more than
// MAX_BLAS_GRID, which is what a workspace reserves partial-sum slots for.
constexpr int MAX_BLAS_GRID = 1024;
int blas_full_grid()
{
    static std::atomic<int> full{0};
    int f = full.load(std::memory_order_relaxed);
    if (f == 0) {
        int dev = 0, sms = 148;
        if (cudaGetDevice(&dev) == cudaSuccess)
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        f = sms * 4;
        if (f > MAX_BLAS_GRID) f = MAX_BLAS_GRID;
        if (f < 1) f = 1;
        full.store(f, std::memory_order_relaxed);
    }
    return f;
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
// CG workspace: device memory for Fig. 1's vectors r, d, Ad and the mixed driver's
// y, fp32 copies and scalars, plus the host-side objects that go with one solve in flight.
// Either caller-owned (stag_set_workspace, one per host thread) or owned by a link handle and
// shared, behind the handle's mutex, by every call that finds no caller workspace.
// ------------------------------------------------------------------------------------
struct GraphSlot {           // one instantiated CUDA graph of `chunk` CG iterations, and what it baked in
    unsigned long long uid;  // the link handle's unique id (not its address: handles come and go)
    int mode, prec_lo, nrhs, chunk;
    double m2;
    const void *x;           // mode 0 iterates on the caller's x itself; null for the fp32 modes
    cudaGraphExec_t exec;
    unsigned long long nodes, stamp;
};
constexpr int N_GRAPH_SLOTS = 4;

struct WsHost {
    char *base = nullptr;
    size_t bytes = 0;
    bool owned = false;          // base was cudaMalloc'ed by the library (handle-owned workspace)
    bool in_use = false;         // a call is running on it (re-entry guard)
    CgCtrl *h_ctrl = nullptr;    // pinned mirror of the control block
    cudaStream_t cap_stream = nullptr;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr, busy = nullptr;
    cudaStream_t last_stream = nullptr;
    bool busy_recorded = false;
    GraphSlot graphs[N_GRAPH_SLOTS] = {};
    unsigned long long stamp = 0;

    int init_host_objects()
    {
        if (h_ctrl) return STAG_OK;
        CU(cudaMallocHost((void **)&h_ctrl, sizeof(CgCtrl)));
        CU(cudaStreamCreateWithFlags(&cap_stream, cudaStreamNonBlocking));
        CU(cudaEventCreate(&ev0));
        CU(cudaEventCreate(&ev1));
        CU(cudaEventCreateWithFlags(&busy, cudaEventDisableTiming));
        return STAG_OK;
    }
    void drop_graphs()
    {
        for (GraphSlot &g : graphs) {
            if (g.exec) cudaGraphExecDestroy(g.exec);
            g = GraphSlot{};
        }
    }
    void release()
    {
        drop_graphs();
        if (owned && base) cudaFree(base);
        base = nullptr; bytes = 0; owned = false;
        if (h_ctrl) cudaFreeHost(h_ctrl);
        if (cap_stream) cudaStreamDestroy(cap_stream);
        if (ev0) cudaEventDestroy(ev0);
        if (ev1) cudaEventDestroy(ev1);
        if (busy) cudaEventDestroy(busy);
        h_ctrl = nullptr; cap_stream = nullptr; ev0 = ev1 = busy = nullptr;
        busy_recorded = false;
    }
};

namespace {
// the caller-owned workspace of this host thread (stag_set_workspace), if any
struct ThreadWs {
    WsHost *p = nullptr;
    ~ThreadWs() { if (p) { p->release(); delete p; p = nullptr; } }
};
thread_local ThreadWs t_ws;
std::atomic<unsigned long long> g_next_uid{1};
}  // namespace

// ------------------------------------------------------------------------------------
// the link handle
// ------------------------------------------------------------------------------------
// Immutable after creation for every caller of the `const stag_links_t *` entry points, with two
// exceptions that are invisible to them and internally synchronised (hence `mutable`):
//   * the derived link forms (fp32, 12-real, 8-parameter), built once on first use under mu_links
//     and published only after the building stream has been synchronised;
//   * the handle-owned workspace `own`, used only when the calling thread has set none, under mu_ws
//     for the whole call.
struct stag_slab_cg;
struct stag_links {
    Geom g{};
    int dims[4] = {0, 0, 0, 0};    // extents of the lattice this handle covers (the slab's, for a slab)
    int gdims[4] = {0, 0, 0, 0};   // extents of the whole lattice
    int rank = 0, nranks = 1;      // T-slab: time slices [rank*X3, (rank+1)*X3) of nranks*X3; else 0, 1
    int is_slab = 0;               // made by stag_slab_create: operator calls go through stag_slab_*
    int ntiles = 0;                // Vh_pad / TILE
    unsigned long long uid = 0;
    double recon_err = 0.0;
    mutable std::mutex mu_links;
    mutable void *L[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // gathered link fields by precision enum
    mutable std::atomic<int> L_ready[6];
    mutable double recon8_err[2] = {-1.0, -1.0};   // 8-parameter forms: largest rebuilt-entry error, [0] fp64, [1] fp32
    mutable std::mutex mu_ws;
    mutable WsHost own;
    // T-slab exchange (stag_slab_*; slab handles are not const in the ABI and belong to one host
    // thread): my exchange region, the neighbours' (peer memory), exchanges started so far
    char *xch = nullptr;
    char *peer_bwd = nullptr, *peer_fwd = nullptr;
    unsigned long long epoch = 0;
    unsigned n_push_blocks = 0;    // blocks of a HALO hop that own boundary-slice sites (cached)
    char **peers_dev = nullptr;    // device array: every rank's exchange region (stag_slab_connect_all)
    int all_connected = 0;
    struct stag_slab_cg *cg = nullptr;   // state of the slab CG in progress (stag_slab_cg_*)

    stag_links() { for (auto &r : L_ready) r.store(0, std::memory_order_relaxed); }
};

// The rest of the translation unit, in six sections (they see everything above):
#include "stag_host_ws.cuh"      // the CG workspace: layout, lease; C ABI: stag_cg_workspace_bytes, stag_set_workspace
#include "stag_host_links.cuh"   // S0 kernels, hop launchers; C ABI: state, links, spinors, operator
#include "stag_host_persist.cuh" // launching the persistent iteration kernel (stag_persist.cuh)
#include "stag_host_cg.cuh"      // one-GPU CG drivers; C ABI: stag_cg_solve*, stag_solve_M
#include "stag_host_slab.cuh"    // T-slabs: wiring, push / hop, CG over slabs; C ABI: stag_slab_*
#include "stag_host_noalloc.cuh" // A with its intermediate in a static device array; C ABI: stag_apply_A_noalloc
