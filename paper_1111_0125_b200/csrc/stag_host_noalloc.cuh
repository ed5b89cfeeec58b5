// stag_host_noalloc.cuh -- sixth section of stag_lib.cu: stag_apply_A_noalloc, the operator
// A = m^2 - D_eo D_oe (eq. 2.3) for callers that must not allocate device memory.
//
// Who that is.  stag_apply_A keeps the odd-site intermediate D_oe chi in a workspace: the calling
// thread's (stag_set_workspace), or one the link handle cudaMallocs the first time it is needed.
// Some users of this library can offer neither:
//   * a program that handed the whole device to its own memory pool at start-up, so that a
//     cudaMalloc issued later from inside a library simply fails;
//   * a measurement or production loop that other streams run beside, where cudaMalloc and
//     cudaFree stall the device (they synchronise it) and are therefore banned after set-up;
//   * a caller that only holds the spinors it was given and has no way to size, own and keep
//     alive a workspace of ours.
// For them the intermediate lives in the array below: it is part of the loaded library image,
// so the driver places it when the library's module is loaded on a device and no call here ever
// asks for memory.  The price: every device that loads libstag.so carries these
// STAG_NOALLOC_SCRATCH_BYTES (8 MiB) until the process exits, used or not, and lattices whose
// odd-site spinor is larger are refused.
//
// The array and the only host code that takes its address are in this one file on purpose:
// the symbol is `static`, and in HOST code its name is just a host-side shadow the runtime uses
// as a lookup key -- not a device pointer.  Handing `g_noalloc_scratch` itself to a kernel
// would fault (or, on systems where the GPU can dereference host addresses, quietly work on the
// wrong memory).  The device address comes from cudaGetSymbolAddress, asked once per device
// with that device current, and only that pointer goes to the kernels.

static __device__ __align__(256) unsigned char g_noalloc_scratch[STAG_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mu;
void *g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};   // device address of g_noalloc_scratch, per device ordinal

// Device address of the scratch array on the CURRENT device; looked up on the first call per device.
int noalloc_scratch(void **ptr_out)
{
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) {
        snprintf(t_errbuf, sizeof(t_errbuf), "stag_apply_A_noalloc: device ordinal %d is beyond the %d this entry point keeps track of",
                 dev, NOALLOC_MAX_DEVICES);
        t_errbuf_status = STAG_EINVAL;
        return STAG_EINVAL;
    }
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress((void **)&p, g_noalloc_scratch));
        if (!p || ((size_t)p & 255)) {
            snprintf(t_errbuf, sizeof(t_errbuf), "stag_apply_A_noalloc: cudaGetSymbolAddress gave %p for the scratch array", p);
            t_errbuf_status = STAG_ECUDA;
            return STAG_ECUDA;
        }
        g_noalloc_ptr[dev] = p;
    }
    *ptr_out = g_noalloc_ptr[dev];
    return STAG_OK;
}

}  // namespace

// See include/stag.h for the contract.  The two launches are exactly stag_apply_A's (one
// right-hand side): tmp_o = D_oe in_e into the static array, then out_e = m^2 in_e - D_eo tmp_o.
// No cudaMalloc, cudaFree, workspace lease or link-form build happens on this path.
extern "C" int stag_apply_A_noalloc(void *out_even, const void *in_even, const stag_links_t *links,
                                    double mass, int prec)
{
    const stag_links *L = links;
    if (!out_even || !in_even || !L || out_even == in_even || !prec_ok(prec) || L->is_slab)
        return STAG_EINVAL;
    // building a derived link form allocates: this entry point only uses forms that exist already
    if (!L->L_ready[prec].load(std::memory_order_acquire)) {
        snprintf(t_errbuf, sizeof(t_errbuf),
                 "stag_apply_A_noalloc: the links of precision %d are not built yet and building them allocates; "
                 "call stag_dslash or stag_apply_A once in this precision during set-up (STAG_PREC_F64 always exists)", prec);
        t_errbuf_status = STAG_EINVAL;
        return STAG_EINVAL;
    }
    const size_t need = (size_t)3 * L->g.Vh_pad * (prec_is_f32(prec) ? sizeof(float2) : sizeof(double2));
    if (need > (size_t)STAG_NOALLOC_SCRATCH_BYTES) {
        snprintf(t_errbuf, sizeof(t_errbuf),
                 "stag_apply_A_noalloc: the odd-site intermediate of this lattice takes %zu bytes, the built-in scratch array holds %zu; use stag_apply_A with a workspace",
                 need, (size_t)STAG_NOALLOC_SCRATCH_BYTES);
        t_errbuf_status = STAG_EINVAL;
        return STAG_EINVAL;
    }
    void *tmp_odd = nullptr;
    int rc = noalloc_scratch(&tmp_odd);
    if (rc) return rc;
    // Nothing in the array has to start at zero: the first hop stores all 3*Vh_pad complex numbers
    // (pad lanes included, as zeros) before the second hop reads any of them, and bytes beyond
    // `need` are never touched.  What an earlier call left there is overwritten, not read.
    if ((rc = launch_hop(L, prec, HOP_PLAIN, tmp_odd, in_even, 1, 0.0, 1.0, nullptr, nullptr, nullptr, 1, t_stream))) return rc;
    return launch_hop(L, prec, HOP_XPAY, out_even, tmp_odd, 0, mass * mass, 1.0, in_even, nullptr, nullptr, 1, t_stream);
}
