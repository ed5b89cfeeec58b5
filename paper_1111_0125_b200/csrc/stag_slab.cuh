// stag_slab.cuh -- T-slab domain decomposition of the hop: the halo exchange over peer memory.
//
// The paper's multi-GPU Dirac operation is kernel -> boundary collect -> memcpy to host -> MPI ->
// memcpy to device (Table 1), and it plans peer-to-peer copies.  Here a
// slab's two boundary time slices of the hop's INPUT spinor are stored straight into the
// neighbouring GPUs' halo buffers by face_push_kernel (peer-to-peer stores over NVLink; the
// buffers are ordinary device memory mapped into this process with CUDA IPC or, for slabs that
// share a process, used directly), followed by one system-scope release store of the exchange's
// epoch into each neighbour's flag.  The consuming hop (dslash_kernel<..., HALO = true>) waits on
// its own two flags only in the threads of the first and last time slice, which it visits last.
//
// Exchange region of one slab (one allocation = one IPC handle), XCH_HDR bytes of header, then
// halo buffers [epoch & 1][dir][colour][s3] of 16-byte complex slots (fp32 uses the front half):
//   dir 0 = "back":  the neighbour slice x3 = -1,  written by rank-1 from its LAST slice
//   dir 1 = "fwd":   the neighbour slice x3 = X3,  written by rank+1 from its FIRST slice
// Double buffering by epoch parity is enough: a rank cannot start exchange e+2 before both its
// neighbours have finished consuming exchange e (its own hop e+1 waits for their push e+1, which
// follows their hop e in stream order).
#pragma once
#include "stag_common.cuh"

namespace stag {

constexpr size_t XCH_HDR = 256;
struct XchHeader {
    unsigned long long flag_back;   // epoch of the last completed push into my "back" halo
    unsigned long long flag_fwd;    // ... into my "fwd" halo
    unsigned ticket;                // last-block ticket of MY face_push_kernel (never peer-written)
};
static_assert(sizeof(XchHeader) <= XCH_HDR, "exchange header must fit its slot");

inline size_t xch_halo_offset(int s3, unsigned long long epoch, int dir)
{
    return XCH_HDR + ((size_t)((epoch & 1ull) * 2 + dir) * 3 * s3) * 16;
}
inline size_t xch_bytes(int s3) { return XCH_HDR + (size_t)4 * 3 * s3 * 16; }

// in: one parity's device spinor of the slab (planes of Vh_pad).  Stores its last time slice into
// fwd_back (the forward neighbour's "back" halo) and its first time slice into bwd_fwd (the
// backward neighbour's "fwd" halo), then marks both neighbours' flags with the epoch.
template <typename T>
__global__ void __launch_bounds__(256)
face_push_kernel(const cplx_t<T> *__restrict__ in, const int Vh, const int Vh_pad, const int s3,
                 cplx_t<T> *__restrict__ fwd_back, cplx_t<T> *__restrict__ bwd_fwd,
                 unsigned long long *fwd_flag_back, unsigned long long *bwd_flag_fwd,
                 const unsigned long long epoch, unsigned *ticket)
{
    const long i = blockIdx.x * 256L + threadIdx.x;
    const long face = 3L * s3;
    if (i < 2 * face) {
        const long r = i % face;
        const int c = (int)(r / s3), j = (int)(r % s3);
        if (i < face) fwd_back[(size_t)c * s3 + j] = in[(size_t)c * Vh_pad + (Vh - s3) + j];
        else          bwd_fwd[(size_t)c * s3 + j] = in[(size_t)c * Vh_pad + j];
    }
    __threadfence_system();       // my peer stores are ordered before what follows, system-wide
    __syncthreads();
    if (threadIdx.x == 0 && atomicAdd(ticket, 1u) == gridDim.x - 1) {
        *ticket = 0;
        __threadfence_system();   // cumulativity: every block's stores precede the flags
        asm volatile("st.release.sys.global.u64 [%0], %1;" :: "l"(fwd_flag_back), "l"(epoch) : "memory");
        asm volatile("st.release.sys.global.u64 [%0], %1;" :: "l"(bwd_flag_fwd), "l"(epoch) : "memory");
    }
}

}  // namespace stag
