/*
 * stag.h -- C ABI of libstag: the single-GPU hot path of the mixed-precision
 * staggered-fermion CG inverter of arXiv:1111.0125 (Jang, Kim, Lee, Lattice
 * 2011), written for NVIDIA B200 (sm_100a).
 *
 * Citations "P:Lnn" are lines of the paper text; "Qn" are the
 * readings listed in DESIGN.md where the paper is silent.
 *
 * What the library computes
 *   D chi(x) = sum_mu [ W_mu(x) chi(x+mu) - W_mu(x-mu)^dag chi(x-mu) ]   eq. 2.5
 *   A        = -D^2 + m^2 on the even sites = m^2 - D_eo D_oe             eq. 2.3
 *   A x = b  by conjugate gradient (Fig. 1), in fp64, in fp32, by
 *            iterative refinement (Fig. 2) or with the corrected
 *            restart + reliable + group-wise updates of section 3.2
 * W_mu(x) = eta_mu(x) * bc_mu(x) * U_mu(x): the staggered phases (and the
 * antiperiodic time boundary) are folded into the links by the caller before
 * the solver is entered, as the paper does.
 *
 * Geometry (all entry points)
 *   dims = (X0,X1,X2,X3), every extent even and >= 2; mu = 3 is time.
 *   site index   idx = x0 + X0*(x1 + X1*(x2 + X2*x3))
 *   parity       p = (x0+x1+x2+x3) & 1   (0 = even)
 *   checkerboard cb = idx >> 1,  Vh = X0*X1*X2*X3/2 sites per parity
 *
 * Canonical (interchange) layouts, fp64, C order -- what the caller hands in:
 *   links   W[mu][p][cb][i][j][re,im]   4*2*Vh*18 doubles
 *   spinor  chi[cb][i][re,im]           Vh*6 doubles, one parity
 *
 * Device (working) layouts -- what the kernels read and write:
 *   spinor, one parity, precision fp64 or fp32: three colour planes of
 *     complex numbers,  v[c][cb],  c = 0..2, cb = 0..Vh_pad-1, where
 *     Vh_pad = Vh rounded up to a multiple of 32.  Pad entries are zero and
 *     every kernel keeps them zero.  stag_spinor_bytes() gives the size.
 *   links: owned by the opaque handle, see stag_links_create().
 *
 * Pointers: every `void *` / `const void *` spinor argument is DEVICE memory
 * in the device layout unless the name ends in `_host`.  The caller owns all
 * spinor buffers and, once it has called stag_set_workspace(), the solver's
 * workspace; the library owns only what hangs off a stag_links_t.
 * All calls are asynchronous on the stream set by stag_set_stream() except
 * where stated.  No call throws or aborts; every `int` return is a
 * stag_status (0 = OK, < 0 = failure, > 0 = solver outcome that still wrote
 * its results).
 *
 * Threads: the stream, the workspace and the error text are PER HOST THREAD.
 * A `const stag_links_t *` is immutable to its callers: any number of host
 * threads, each with its own stream and its own workspace, may apply the
 * operator and solve on one handle at the same time (the production pattern:
 * many sources per gauge field).  A thread that has set no workspace
 * uses one owned by the handle, under the handle's mutex: such calls are safe
 * from any thread but run one after the other.  Slab handles (stag_slab_*) are
 * not const and belong to one host thread.
 */
#ifndef STAG_H
#define STAG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes ------------------------------------------------------- */
enum {
    STAG_OK         = 0,
    STAG_EINVAL     = -1,  /* null pointer, odd or < 2 extent, dims != handle's, bad enum,
                              tol <= 0, maxiter < 0, out aliases in, 12-real unavailable     */
    STAG_ECUDA      = -2,  /* a CUDA call failed; text via stag_strerror(STAG_ECUDA)         */
    STAG_ENOMEM     = -3,  /* device or host allocation failed                               */
    STAG_ETIMEOUT   = -4,  /* T-slabs: a kernel gave up waiting for a neighbour's exchange or global
                              sum (missing, mis-ordered or dead peer); results are not valid     */
    STAG_ENOCONV    = 1,   /* maxiter reached; x, iters and the true residual ARE written    */
    STAG_EBREAKDOWN = 2    /* NaN or <d,Ad> <= 0; x, iters and the true residual ARE written */
};

/* ---- precision / storage of one Dslash ------------------------------------
 * 18-real: all nine complex entries of each link are stored.
 * 12-real: rows 0 and 1 are stored; row 2 = s * conj(row0 x row1) is rebuilt
 *          in registers, s = +-1 recomputed from the site coordinates (Q12). */
enum {
    STAG_PREC_F64    = 0,
    STAG_PREC_F32    = 1,
    STAG_PREC_F64_R12 = 2,
    STAG_PREC_F32_R12 = 3,
    /* 8-parameter form (the paper names and rejects it for its round-off; its Ref. [6]):
     * four complex slots per link, a2, a3, b1 and the phases of a1 and c1; the rest follows from
     * unitarity and det = +-1 with a division by |a2|^2+|a3|^2.  Whole-lattice handles only;
     * refused (STAG_EINVAL) for fields whose rebuilt entries are off by more than 1e-9 (fp64) /
     * 1e-3 (fp32), e.g. unit links.  A measured accuracy / bandwidth trade-off next to 12-real. */
    STAG_PREC_F64_R8  = 4,
    STAG_PREC_F32_R8  = 5
};

/* ---- CG modes ---------------------------------------------------------- */
enum {
    STAG_CG_F64      = 0,  /* Fig. 1 in fp64                                                 */
    STAG_CG_F32      = 1,  /* Fig. 1 in fp32 (diagnostic: stalls above 1e-10)                */
    STAG_CG_DEFECT   = 2,  /* Fig. 2: fp64 outer loop, fresh fp32 inner solve of A y = r_k   */
    STAG_CG_RELIABLE = 3   /* section 3.2: fp32 iteration, direction kept across restarts
                              (eq. 3.1), reliable + group-wise update on the trigger of P:L97 */
};

typedef struct stag_links stag_links_t;

/* ---- global state ------------------------------------------------------ */

/* Stream (a cudaStream_t cast to void*) every later call enqueues on; NULL = the legacy
 * default stream.  Per host thread. */
int stag_set_stream(void *cuda_stream);

/* ---- workspace ("the caller owns every spinor buffer and the
 * workspace") ----------------------------------------------------------------------------
 *
 * What lives there: Fig. 1's vectors other than x and b -- r, d and q = A d and the
 * odd-site intermediate of A (eq. 2.3) in fp64 -- the fp32 iteration's y, r, d, q, tmp of the
 * mixed modes (section 3.2), the device-resident scalars alpha, beta, delta, the
 * partial sums of the inner products, b_e of stag_solve_M and the two device-layout
 * spinors stag_cg_solve_host stages x and b in.
 *
 * stag_cg_workspace_bytes: bytes a workspace needs for any of stag_cg_solve*, stag_solve_M,
 * stag_cg_solve_host, stag_apply_A* on a lattice `dims` in CG mode `mode` with up to `nrhs`
 * right-hand sides (mode < 0: only stag_apply_A*).  Pure arithmetic, no device needed; 0 on bad
 * arguments.  A workspace sized for (mode, nrhs) also serves fewer right-hand sides; sizes for
 * different modes differ, take the largest of the modes you use.
 *
 * stag_set_workspace: from now on THIS host thread's calls keep every intermediate in
 * ws[0 .. bytes) (device memory, 256-byte aligned, caller-owned, must stay valid until replaced)
 * and write nothing to the link handle.  A call that needs more than `bytes` fails with
 * STAG_EINVAL (stag_strerror says how much).  Calls sharing a workspace must be issued from the
 * thread that set it; they are ordered on the device even if that thread changes its stream in
 * between.  The instantiated CUDA graph of the iteration is cached with the workspace per
 * (handle, mode, link form, nrhs, chunk, mass), so repeated solves do not re-capture.
 * ws = NULL, bytes = 0 returns to the handle-owned default.  Not asynchronous; no device work. */
size_t stag_cg_workspace_bytes(const int dims[4], int mode, int nrhs);
int stag_set_workspace(void *ws, size_t bytes);

/* Text for a status; for STAG_ECUDA, the text of the last CUDA error seen by this thread.
 * The pointer stays valid until the next failing call on this thread. */
const char *stag_strerror(int status);

/* Number of kernel launches (graph-replayed launches included) issued by this library since
 * the process started or since the last stag_reset_launch_count(). */
unsigned long long stag_launch_count(void);
void stag_reset_launch_count(void);

/* ---- links: setup step S0 (P:L60 eta folding is the caller's; "rearranging data
 * for the coalesced access" is this call) --------------------------------------------
 *
 * W: canonical fp64 links (layout above), with eta*bc already folded in; host memory when
 * on_device == 0, device memory otherwise.  The call reads W before it returns only when W
 * is host memory (it synchronises the stream in that case); a device W must stay valid until
 * the stream has passed this call.  antiperiodic_t says whether the caller folded a -1 into
 * the mu=3 links leaving x3 = X3-1; it is needed only to rebuild 12-real links (Q12).
 *
 * The handle keeps, per output parity p and per precision, the EIGHT matrices each output
 * site needs in one place ("gathered" form):
 *   M_d(x) = W_d(x)                      d = 0..3   (forward hop)
 *   M_d(x) = -W_{d-4}(x - (d-4)^)^dag    d = 4..7   (backward hop, sign folded)
 * so that D chi(x) = sum_d M_d(x) chi(nbr_d(x)), stored in tiles of 32 sites:
 *   L[p][tile][d][k][lane]  complex,  k = 3*row+col (18-real: 9 entries, 12-real: 6)
 * The fp64/18 form is built by this call; the other three are built on first use. */
int stag_links_create(stag_links_t **links_out, const int dims[4], int antiperiodic_t,
                      const double *W, int on_device);
/* The same from the BARE gauge field U_mu(x) (same layout, no phases): eta_mu(x) =
 * (-1)^(x0+..+x_{mu-1}) and, when antiperiodic_t, the -1 on the mu=3 links leaving x3 = X3-1
 * are folded in on the device while gathering -- the paper's "gauge link preconditioning"
 * done by the library instead of the caller.  Multiplication by +-1 is exact: the
 * handle is bit-identical to the one stag_links_create builds from the folded field. */
int stag_links_create_unfolded(stag_links_t **links_out, const int dims[4], int antiperiodic_t,
                               const double *U, int on_device);
void stag_links_destroy(stag_links_t *links);

/* Largest | row2 - s conj(row0 x row1) | over all links, measured when the handle was made.
 * 12-real precisions are refused (STAG_EINVAL) when it exceeds 1e-10. */
int stag_links_recon_error(const stag_links_t *links, double *err_out);
/* The same for the 8-parameter form of precision prec (STAG_PREC_F64_R8 / _F32_R8), rebuilt in
 * that precision's arithmetic exactly as the hop rebuilds it.  Builds the form on first use;
 * returns STAG_EINVAL (with *err_out still set) when the field is refused. */
int stag_links_recon8_error(const stag_links_t *links, int prec, double *err_out);

/* ---- spinors ----------------------------------------------------------- */

/* Bytes of one single-parity spinor in the device layout (prec: F64 or F32; the _R12
 * values are accepted and mean the same as their 18-real partner).  0 on bad arguments. */
size_t stag_spinor_bytes(const int dims[4], int prec);

/* canonical fp64 chi[cb][3][re,im] (device) -> device layout of precision prec, pads zeroed */
int stag_spinor_pack(void *dst, const double *src_canonical, const int dims[4], int prec);
/* device layout -> canonical fp64 (device) */
int stag_spinor_unpack(double *dst_canonical, const void *src, const int dims[4], int prec);

/* ---- the operator ------------------------------------------------------ */

/* One parity hop of eq. 2.5: out (sites of parity `parity`, 0 = even, 1 = odd)
 * = D in (sites of the other parity).  parity = 1 is D_oe, parity = 0 is D_eo.  576 flop per
 * output site.  dims must equal the handle's.  out must not alias in. */
int stag_dslash(void *out, const void *in, const stag_links_t *links, int parity,
                const int dims[4], int prec);

/* A = -D^2 + m^2 on the even sites (eq. 2.3):
 *   out_even = mass^2 * in_even - D_eo ( D_oe in_even ).
 * The odd-parity intermediate lives in the workspace.  out must not alias in. */
int stag_apply_A(void *out_even, const void *in_even, const stag_links_t *links, double mass,
                 int prec);

/* The same operator for callers that cannot allocate device memory.
 *
 * stag_apply_A needs somewhere to keep D_oe in_even between its two hops: the workspace, which
 * either you own (stag_set_workspace) or the handle cudaMallocs on first use.  That rules it out
 * for a program that gave all device memory to its own pool at start-up (a cudaMalloc from inside
 * a library then fails), for code running where cudaMalloc / cudaFree are banned because they
 * stall every stream on the device, and for a caller that holds nothing but the spinors it was
 * handed and cannot keep a workspace of ours alive.  This entry point is for them: the
 * intermediate lives in an array that is part of the library image, STAG_NOALLOC_SCRATCH_BYTES
 * (8 MiB) of it on every device that loads libstag.so, held until the process exits whether or
 * not this function is ever called.  The call itself issues two kernel launches and nothing
 * else: no cudaMalloc, no cudaFree, no workspace, no library routine that allocates.
 *
 * Arguments, layouts, result (eq. 2.3: out_even = mass^2 in_even - D_eo D_oe in_even, bit for bit
 * what stag_apply_A writes) and stream as stag_apply_A with one right-hand side; you still
 * supply in_even and out_even (device, device layout of `prec`, not aliased).  Limits:
 *   - size: 3 * Vh_pad complex numbers of `prec` must fit the array, i.e. Vh_pad <= 174 762
 *     sites per parity in fp64 (16^3 x 32, 16^3 x 64 fit; 28^3 x 96 does not) and <= 349 525 in
 *     fp32.  A larger lattice gets STAG_EINVAL and stag_strerror names both sizes; nothing is
 *     launched.
 *   - links: the gathered links of `prec` must exist already, because building them allocates.
 *     STAG_PREC_F64 always exists; any other form is built by the first stag_dslash /
 *     stag_apply_A / solve that uses it, so make one such call during set-up.  Otherwise
 *     STAG_EINVAL (the text says so).
 *   - first call on each device: looks up the array's device address (cudaGetSymbolAddress,
 *     with that device current) and remembers it.  It is host-side bookkeeping that may load the
 *     library's device code; make that first call during set-up, before any stream capture is
 *     begun.
 *   - sharing: there is ONE array per device and every call uses it.  Calls issued on one
 *     stream are ordered and safe.  Two calls that can overlap on the GPU (different streams,
 *     or different host threads on different streams) race on it and both results are garbage;
 *     the library does not detect this.  The array keeps whatever the last call left in it;
 *     no call depends on that, since the first hop overwrites every element the second reads. */
#define STAG_NOALLOC_SCRATCH_BYTES (8u << 20)
int stag_apply_A_noalloc(void *out_even, const void *in_even, const stag_links_t *links, double mass,
                         int prec);

/* ---- several right-hand sides sharing one pass over the links ------------------------
 *
 * The hop is bandwidth-bound on the gauge field, and the production use of the
 * solver inverts on several sources per gauge field (three colours per point source).
 * The *_mrhs entry points take nrhs spinors stored back to back -- spinor k starts
 * k * stag_spinor_bytes(dims, prec) bytes after spinor 0 -- and read each link once per chunk
 * of up to 4 (fp32) or 2 (fp64) right-hand sides instead of once per right-hand side
 * (DESIGN.md section 13).  nrhs = 1 is exactly the single entry point. */
#define STAG_MAX_RHS 12    /* most right-hand sides one solve carries */

int stag_dslash_mrhs(void *out, const void *in, const stag_links_t *links, int parity,
                     const int dims[4], int prec, int nrhs);
int stag_apply_A_mrhs(void *out_even, const void *in_even, const stag_links_t *links, double mass,
                      int prec, int nrhs);

/* Batch layouts.  BLOCKED is the layout above (nrhs spinors back to back) and the only one of fp64
 * batches.  PAIRED (fp32 only) interleaves right-hand sides 2j and 2j+1 per complex number:
 *     pair j:  p[j][c][cb] = (re_2j, im_2j, re_2j+1, im_2j+1)    one 16-byte element per (colour, site)
 * stored where spinors 2j and 2j+1 of the blocked batch would be (2 * stag_spinor_bytes per pair);
 * an odd last right-hand side stays an ordinary spinor after the pairs, so both layouts take
 * nrhs * stag_spinor_bytes and nrhs = 1 is the same in both.  In the paired layout a neighbour's
 * colour for two right-hand sides is ONE 16-byte gather: the batch hop, which is bound by issue
 * slots and loads in flight rather than by DRAM, needs half the gather
 * instructions.  The arithmetic per right-hand side, and so every result bit, is the same in both.
 * The fp32 iteration of stag_cg_solve_mrhs / stag_solve_M keeps its vectors paired internally;
 * their x and b (fp64) are blocked.  stag_batch_convert changes the layout of a batch (dst != src;
 * fp64: a copy); stag_dslash_batch / stag_apply_A_batch are the *_mrhs calls on a given layout. */
enum { STAG_BATCH_BLOCKED = 0, STAG_BATCH_PAIRED = 1 };
int stag_batch_convert(void *dst, const void *src, const int dims[4], int prec, int nrhs, int to_layout);
int stag_dslash_batch(void *out, const void *in, const stag_links_t *links, int parity,
                      const int dims[4], int prec, int nrhs, int layout);
int stag_apply_A_batch(void *out_even, const void *in_even, const stag_links_t *links, double mass,
                       int prec, int nrhs, int layout);

/* ---- T-slabs: the hop on a lattice split along time over several GPUs --------------------
 *
 * The paper's subject is the multi-GPU Dirac operation: kernel, boundary collect, memcpy to the
 * host, MPI, memcpy back (Table 1), with GPU-to-GPU copies planned.  Here
 * rank r of nranks holds time slices [r*X3/nranks, (r+1)*X3/nranks) of the global lattice
 * (X3/nranks even); one process per GPU.  A slab handle owns its gathered links (the backward
 * t-links of its first slice included, so links are never exchanged) and an EXCHANGE REGION: two
 * flags and double-buffered halo buffers for the neighbour slices x3 = -1 and x3 = X3 of a
 * hop's input spinor.  stag_slab_push stores the slab's last / first slice of `in` directly into
 * the forward / backward neighbour's halo (peer-to-peer stores) and then release-stores the
 * exchange number into their flags; stag_slab_hop computes the slab's hop, its boundary-slice
 * threads (visited last) acquire-waiting on the slab's own flags.  All ranks must issue the same
 * sequence of pushes and hops.  Spinors are ordinary device spinors of the LOCAL dims.
 *
 * Wiring: every rank publishes its region (stag_slab_ipc_handle, 64 bytes, to be exchanged by
 * any means, e.g. torch.distributed), opens its two neighbours' (stag_slab_ipc_open) and calls
 * stag_slab_connect.  Slabs living in one process connect with the raw pointers from
 * stag_slab_info.  nranks = 1 connects to itself.  DESIGN.md section 14. */
#define STAG_IPC_HANDLE_BYTES 64
#define STAG_MAX_RANKS 16       /* most slabs a lattice is split into */

/* W_global: canonical fp64 links of the WHOLE lattice global_dims (eta*bc folded).  From host
 * memory only the rank's own part is copied to the device (the sub-ranges stag_slab_create_local
 * takes); from device memory the field is read in place. */
int stag_slab_create(stag_links_t **slab_out, const int global_dims[4], int antiperiodic_t,
                     const double *W_global, int on_device, int rank, int nranks);
/* The same slab from the rank's OWN part of the field, so that no rank ever holds or moves the
 * whole lattice (per-rank setup memory and time shrink with nranks).  Time slices are contiguous
 * in the checkerboard index, so with s3 = X0*X1*X2/2, Tl = X3/nranks, t0 = rank*Tl:
 *   W_local[mu][p][cb'][3][3]  = W_global[mu][p][t0*s3 + cb'],  cb' = 0 .. Tl*s3-1
 *                                (the canonical layout of a lattice of the LOCAL dims);
 *   W_back[p][j][3][3]         = W_global[3][p][((t0-1) mod X3)*s3 + j],  j = 0 .. s3-1
 *                                (the t-links leaving the time slice before the slab: the
 *                                backward t-links of the slab's first slice, owned by rank-1).
 * eta*bc folded by the caller as in stag_links_create; both in host (on_device = 0) or both in
 * device memory.  The result is bit-identical to stag_slab_create on the whole field. */
int stag_slab_create_local(stag_links_t **slab_out, const int global_dims[4], int antiperiodic_t,
                           const double *W_local, const double *W_back, int on_device,
                           int rank, int nranks);
/* Any output pointer may be NULL. */
int stag_slab_info(const stag_links_t *slab, int local_dims_out[4], int *rank_out, int *nranks_out,
                   void **exchange_ptr_out, size_t *exchange_bytes_out);
int stag_slab_ipc_handle(const stag_links_t *slab, unsigned char handle_out[STAG_IPC_HANDLE_BYTES]);
int stag_slab_ipc_open(const unsigned char handle[STAG_IPC_HANDLE_BYTES], void **ptr_out);
int stag_slab_ipc_close(void *ptr);
/* bwd / fwd: device-accessible addresses of the exchange regions of ranks r-1 and r+1 (mod nranks) */
int stag_slab_connect(stag_links_t *slab, void *bwd_exchange, void *fwd_exchange);

/* Start exchange number e = (pushes so far) + 1 with the faces of `in` (one parity, precision of prec). */
int stag_slab_push(const void *in, stag_links_t *slab, int prec);
/* out (sites of `parity`) = D in on the slab, halo from the last exchange; with own != NULL,
 * out = a*own - D in (the second hop of A, a = m^2).  STAG_EINVAL before the first push. */
int stag_slab_hop(void *out, const void *in, stag_links_t *slab, int parity, int prec, double a,
                  const void *own);
/* push + hop: what each rank of a real multi-GPU run calls. */
int stag_slab_dslash(void *out, const void *in, stag_links_t *slab, int parity, int prec);

/* Watchdog.  A kernel that waits for a neighbour's flag polls it at most `polls` times (about a
 * microsecond each; 0 restores the default of 2^23, roughly ten seconds), then gives up and marks
 * the slab DEAD.  A dead slab publishes nothing any more: the kernel whose wait gave up finishes
 * its own stores but sets no neighbour's flag and bumps no count, and every later kernel of the
 * slab path returns at once, so the neighbours' waits run into their own limit in turn and EVERY
 * rank ends with STAG_ETIMEOUT instead of consuming stale data.  The limit counts rank skew too
 * (a peer that starts late is indistinguishable from a dead one): put a barrier before the first
 * exchange.  stag_slab_status synchronises the stream and returns STAG_ETIMEOUT for a dead slab
 * (also reported by stag_slab_cg_control / _finish), STAG_OK otherwise.
 * stag_slab_reset revives a slab: flags, counts, reduction slots and the mark are cleared (the wait
 * limit is kept).  Collective: ALL ranks must call it, with nothing of the slab path in flight
 * anywhere, and synchronise with each other (a barrier) both before and after the call; the
 * alternative is to destroy the handles. */
int stag_slab_set_wait_limit(stag_links_t *slab, unsigned long long polls);
int stag_slab_status(stag_links_t *slab);
int stag_slab_reset(stag_links_t *slab);
/* Diagnostics since creation / the last reset: how many acquire-waits of this slab's kernels did
 * not find their flag already set, and how many polls they spent (either pointer may be NULL).
 * Zero when every kernel found its peers' data waiting, as in a lockstep run. */
int stag_slab_wait_stats(stag_links_t *slab, unsigned long long *waits_spun_out, unsigned long long *polls_out);

/* ---- the solver -------------------------------------------------------- */

/* Optional knobs for stag_cg_solve_ex; zero-initialise, then set what you need
 * (a zero field means "library default"). */
typedef struct stag_cg_params {
    double eps_in;        /* inner tolerance eps^in of P:L82 / P:L97 (Q8).  Default 0.1 for
                             STAG_CG_RELIABLE, 1e-2 for STAG_CG_DEFECT.                       */
    int    recon12;       /* 1: the fp32 (and, in mode 0, fp64) Dslash uses 12-real links     */
    int    graph_chunk;   /* CG iterations per CUDA-graph replay between host checks
                             (default 32); < 0 disables graphs (plain launches)               */
    int    recon12_f64;   /* 1: the fp64 correction steps use 12-real links too               */
    int    recon8;        /* 1: the iteration's Dslash uses 8-parameter links (overrides recon12) */
    int    persistent;    /* the iteration as ONE persistent cooperative kernel per chunk of passes
                             (grid barriers instead of four kernel boundaries per pass; one
                             right-hand side, 18- or 12-real links; in mode 3 with 18-real fp64
                             corrections the reliable updates run inside the kernel too, so a
                             solve is one launch after the initial residual): 1 = yes, -1 = no,
                             0 = the library decides by lattice volume
                             and falls back to the kernel-per-step path if the device refuses
                             the cooperative launch (1 reports that as STAG_ECUDA instead);
                             for a lattice split over more than one T-slab 0 means "no": across
                             GPUs this kernel is opt-in until it has been run and timed there  */
    int    persist_chunk; /* passes per persistent launch between host checks (default 1024;
                             values above 65536 are taken as 65536)                            */
} stag_cg_params_t;

typedef struct stag_cg_stats {
    int    iters;         /* loop passes of Fig. 1 = applications of A to d (Q7)              */
    int    n_updates;     /* reliable/group-wise updates (mode 3) or outer steps (mode 2)     */
    int    n_restarts;    /* mode 0: restarts after the true residual missed tol (Q6b)        */
    int    iters_f32;     /* of iters, how many ran in fp32 (P:L84's "99.8 %")                */
    int    applies_f64;   /* fp64 applications of A (initial, updates, final residual)        */
    double true_resid;    /* |b - A x| / |b| in fp64 on exit                                  */
    double iter_resid;    /* the iterated residual norm / |b| on exit                         */
    double seconds;       /* device time of the solve (CUDA events around it)                 */
} stag_cg_stats_t;

/* Solve A x = b on the even sites (eq. 2.1 with A of eq. 2.3).  x (fp64 device layout) holds
 * the initial guess on entry and the solution on exit; b is fp64 device layout.  Convergence:
 * |r| <= tol * |b| (Q6), checked on the fp64 true residual before returning.  Synchronises
 * the stream before returning iterations and true residual.  b = 0 gives x = 0, 0 iterations,
 * residual 0.  Pad lanes of x are zeroed on entry, pad lanes of b are read as zero whatever
 * they hold.  Returns STAG_OK, STAG_ENOCONV, STAG_EBREAKDOWN or an error < 0. */
int stag_cg_solve(void *x_even, const void *b_even, const stag_links_t *links, double mass,
                  double tol, int maxiter, int mode, int *iters_out, double *true_resid_out);

int stag_cg_solve_ex(void *x_even, const void *b_even, const stag_links_t *links, double mass,
                     double tol, int maxiter, int mode, const stag_cg_params_t *params,
                     stag_cg_stats_t *stats_out);

/* nrhs <= STAG_MAX_RHS independent systems A x_k = b_k solved in lockstep: one Fig. 1
 * recurrence per right-hand side (its own alpha, beta, residual, stopping test), one shared
 * iteration loop, every hop applied to all of them at once.  A right-hand side that has met
 * its target is frozen (no longer updated) while the others finish; in mode 3 a reliable
 * update triggered by any right-hand side is carried out for all.  x_even / b_even: nrhs fp64
 * device spinors back to back.  stats_out: nrhs entries (or NULL); iters is the number of loop
 * passes during which that right-hand side was active.  Returns STAG_OK only if every
 * right-hand side met tol; STAG_ENOCONV / STAG_EBREAKDOWN / < 0 as stag_cg_solve. */
int stag_cg_solve_mrhs(void *x_even, const void *b_even, const stag_links_t *links, double mass,
                       double tol, int maxiter, int mode, int nrhs,
                       const stag_cg_params_t *params, stag_cg_stats_t *stats_out);

/* The staggered propagator: (D + m) psi = h on the WHOLE lattice (the system whose normal
 * equations are eq. 2.2-2.3: (D+m)^dag (D+m) = -D^2 + m^2 = A because D^dag = -D, eq. 2.4;
 * DESIGN.md Q23), for nrhs sources, through one even-site solve:
 *     b_e = m h_e - D_eo h_o ;   A psi_e = b_e (stag_cg_solve_mrhs) ;   psi_o = (h_o - D_oe psi_e) / m
 * All four spinor arguments are nrhs fp64 device spinors back to back, one parity each;
 * psi_even holds the initial guess of the even-site solve on entry.  tol applies to the
 * even-site system (|b_e - A psi_e| <= tol |b_e|), which bounds |h - (D+m) psi| <= tol |b_e| / m.
 * mass must be non-zero.  stats_out and the return value are those of the even-site solve. */
int stag_solve_M(void *psi_even, void *psi_odd, const void *h_even, const void *h_odd,
                 const stag_links_t *links, double mass, double tol, int maxiter, int mode,
                 int nrhs, const stag_cg_params_t *params, stag_cg_stats_t *stats_out);

/* The same solve from and to HOST memory in the canonical fp64 layout (Vh*6 doubles each):
 * copies b (and x as the initial guess) to the device, packs, solves, unpacks, copies x back.
 * This is the end-to-end entry bench.py times.  Pinned host memory makes the copies faster
 * but is not required. */
int stag_cg_solve_host(double *x_host, const double *b_host, const stag_links_t *links,
                       double mass, double tol, int maxiter, int mode,
                       const stag_cg_params_t *params, stag_cg_stats_t *stats_out);

/* ---- CG over T-slabs -----------------------------------------------------------------
 *
 * The paper's headline is the CG on several GPUs (title; Table 1; 36 / 19 GFLOPS per GPU once
 * the network is included).  Here every rank runs Fig. 1 (mode 0) or the mixed
 * driver of section 3.2 (mode 3) on its slab; the hops exchange faces as above, and the two
 * inner products of an iteration are summed over ranks through the exchange regions: each rank
 * stores its local total into every rank's slots, and every rank adds the nranks slots in rank
 * order, so alpha, beta and every stopping decision are bit-identical everywhere and no rank
 * ever talks to the host inside a chunk of iterations.  Needs stag_slab_connect_all.
 *
 * The solve is a sequence of ACTIONS, each a fixed sequence of PHASES:
 *     stag_slab_cg_begin(...);
 *     for (;;) { stag_slab_cg_control(slab, &act); if (act == STAG_SLAB_ACT_DONE) break;
 *                for (ph = 0, more = 1; more; ++ph) stag_slab_cg_step(slab, act, ph, &more); }
 *     stag_slab_cg_finish(slab, &stats);
 * One process per GPU runs exactly that loop.  No kernel of a phase waits for a peer's kernel of
 * the same phase, so slabs that share one device can instead be stepped rank after rank, phase
 * by phase (how the single-GPU tests run the multi-GPU data path).  x, b: fp64 device spinors of
 * the slab's local dims; x holds the initial guess.  Modes: STAG_CG_F64, STAG_CG_RELIABLE.
 * graph_chunk of the params = iterations per ACT_ITER (default 32): plain launches when stepped,
 * one CUDA-graph launch per ACT_ITER inside stag_slab_cg_run (the exchange and reduction numbers
 * live in device memory, so the captured chunk can be replayed). */
enum {
    STAG_SLAB_ACT_DONE = 0, STAG_SLAB_ACT_NORM = 1, STAG_SLAB_ACT_INIT = 2, STAG_SLAB_ACT_ITER = 3,
    STAG_SLAB_ACT_UPDATE = 4, STAG_SLAB_ACT_VERIFY = 5, STAG_SLAB_ACT_FINAL = 6
};
/* regions[r]: device-accessible address of rank r's exchange region, r = 0..nranks-1 (the
 * slab's own included); also sets the two neighbours.  Host array. */
int stag_slab_connect_all(stag_links_t *slab, void *const *regions);
int stag_slab_cg_begin(stag_links_t *slab, void *x_even, const void *b_even, double mass, double tol,
                       int maxiter, int mode, const stag_cg_params_t *params);
int stag_slab_cg_control(stag_links_t *slab, int *action_out);
int stag_slab_cg_step(stag_links_t *slab, int action, int phase, int *more_out);
/* Returns STAG_OK / STAG_ENOCONV / STAG_EBREAKDOWN like stag_cg_solve; stats as there. */
int stag_slab_cg_finish(stag_links_t *slab, stag_cg_stats_t *stats_out);
/* One STAG_SLAB_ACT_ITER (up to persist_chunk passes of the loop) of the n slabs given, in ONE
 * cooperative launch of the persistent iteration kernel: each slab's blocks form a rank group with
 * its own barrier, and the groups talk only through the exchange regions.  n = 1: what a process of
 * a one-process-per-GPU run launches for its own slab (stag_slab_cg_run does when
 * params->persistent = 1, or when it is 0 and the slab is the whole lattice, nranks = 1).  n = nranks with all slabs on the calling thread's device: the
 * single-GPU emulation of the multi-GPU run -- the ranks' kernels run concurrently and really wait
 * for each other, which separate launches on one device cannot promise.  Replaces the phases of
 * that action in the stepped loop; every slab must have been told STAG_SLAB_ACT_ITER by
 * stag_slab_cg_control.  18- and 12-real links. */
int stag_slab_cg_iter_all(stag_links_t *const *slabs, int n);
/* begin + the loop above + finish: the call of a one-process-per-GPU run (all ranks together).
 * Slabs sharing a device may call it too -- one host thread and one stream per slab -- as long as
 * all their kernels can be resident at the same time (small lattices; tests/test_gpu_slab_concurrent.py):
 * a waiting kernel that fills the device would block the kernel it waits for, and the watchdog
 * turns that into STAG_ETIMEOUT. */
int stag_slab_cg_run(stag_links_t *slab, void *x_even, const void *b_even, double mass, double tol,
                     int maxiter, int mode, const stag_cg_params_t *params, stag_cg_stats_t *stats_out);

#ifdef __cplusplus
}
#endif
#endif /* STAG_H */
