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

// The rest of the translation unit, in three sections (they see everything above):
#include "stag_host_links.cuh"   // S0 kernels, hop launchers; C ABI: state, links, spinors, operator
#include "stag_host_cg.cuh"      // one-GPU CG drivers; C ABI: stag_cg_solve*, stag_solve_M
#include "stag_host_slab.cuh"    // T-slabs: wiring, push / hop, CG over slabs; C ABI: stag_slab_*
