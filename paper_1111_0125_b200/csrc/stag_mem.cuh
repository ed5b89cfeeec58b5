// stag_mem.cuh -- global-memory access with explicit L2 eviction policies (sm_100a).
//
// The hot path moves two kinds of data with opposite reuse:
//   links   read exactly once per hop, 607-1214 MB per launch on 28^3 x 96: must pass
//           THROUGH the 126 MB L2 without displacing anything  -> L2::evict_first
//   spinors 25-50 MB each, written by one kernel of the CG iteration and read by the next
//           (d: xpay -> hop 1, tmp: hop 1 -> hop 2, q: hop 2 -> update, r: update -> xpay)
//           -> L2::evict_last, so the producer's lines are still resident for the consumer
// Measured on B200 (28^3 x 96, CUDA events around each kernel of the running CG iteration):
// a 25 MB buffer written by one kernel survives a 607 MB `.cs` stream in L2, and the explicit
// hints buy a further 2.5 % of the fp32 iteration (240 -> 234 us); for fp64 spinors (four
// 50 MB vectors, more than L2 holds next to the stream) evict_last costs 4 %, so it is off.
// The policies are PTX `createpolicy` descriptors passed as `.L2::cache_hint` operands;
// ptxas folds them into the memory descriptor of the LDG/STG, no instruction is added.
#pragma once
#include <cuda_runtime.h>

#ifndef STAG_LINK_POLICY      // 0: ld.global.cs   1: cs + L2::evict_first hint
#define STAG_LINK_POLICY 1
#endif
#ifndef STAG_SPINOR_POLICY    // 0: default        1: L2::evict_last hint on fp32 spinor loads/stores
#define STAG_SPINOR_POLICY 1
#endif
#ifndef STAG_SPINOR_POLICY_F64   // the same for fp64 spinors: off, four 50 MB fp64 vectors do not fit
#define STAG_SPINOR_POLICY_F64 0 // L2 and pinning them measured 4 % slower (profiles/README.md)
#endif

namespace stag {

__device__ __forceinline__ unsigned long long policy_evict_first()
{
    unsigned long long p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long policy_evict_last()
{
    unsigned long long p;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}

// ---- streaming (read-once) 16-byte loads: the link packets ---------------------------
__device__ __forceinline__ float4 ld_stream(const float4 *p)
{
#if STAG_LINK_POLICY == 0
    return __ldcs(p);
#else
    float4 v;
    asm("ld.global.cs.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
        : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
        : "l"(p), "l"(policy_evict_first()));
    return v;
#endif
}
__device__ __forceinline__ double2 ld_stream(const double2 *p)
{
#if STAG_LINK_POLICY == 0
    return __ldcs(p);
#else
    double2 v;
    asm("ld.global.cs.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
        : "=d"(v.x), "=d"(v.y)
        : "l"(p), "l"(policy_evict_first()));
    return v;
#endif
}

// ---- resident (reused) data: spinor elements and 16-byte spinor packets ---------------
// read-only within the kernel (non-coherent path, cached in L1): the neighbour gather
__device__ __forceinline__ float2 ld_keep_nc(const float2 *p)
{
#if STAG_SPINOR_POLICY == 0
    return __ldg(p);
#else
    float2 v;
    asm("ld.global.nc.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;"
                 : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(policy_evict_last()));
    return v;
#endif
}
__device__ __forceinline__ double2 ld_keep_nc(const double2 *p)
{
#if STAG_SPINOR_POLICY_F64 == 0
    return __ldg(p);
#else
    double2 v;
    asm("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
                 : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(policy_evict_last()));
    return v;
#endif
}

// a pair of right-hand sides interleaved per complex number (stag_dslash.cuh, "paired" batches)
__device__ __forceinline__ float4 ld_keep_nc(const float4 *p)
{
#if STAG_SPINOR_POLICY == 0
    return __ldg(p);
#else
    float4 v;
    asm("ld.global.nc.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
        : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(policy_evict_last()));
    return v;
#endif
}

// coherent loads (the buffer may be written by this kernel)
__device__ __forceinline__ float2 ld_keep(const float2 *p)
{
#if STAG_SPINOR_POLICY == 0
    return *p;
#else
    float2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;"
                 : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(policy_evict_last()) : "memory");
    return v;
#endif
}
__device__ __forceinline__ double2 ld_keep(const double2 *p)
{
#if STAG_SPINOR_POLICY_F64 == 0
    return *p;
#else
    double2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
                 : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(policy_evict_last()) : "memory");
    return v;
#endif
}
__device__ __forceinline__ float4 ld_keep(const float4 *p)
{
#if STAG_SPINOR_POLICY == 0
    return *p;
#else
    float4 v;
    asm volatile("ld.global.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "l"(p), "l"(policy_evict_last()) : "memory");
    return v;
#endif
}

__device__ __forceinline__ void st_keep(float2 *p, const float2 v)
{
#if STAG_SPINOR_POLICY == 0
    *p = v;
#else
    asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1,%2}, %3;"
                 :: "l"(p), "f"(v.x), "f"(v.y), "l"(policy_evict_last()) : "memory");
#endif
}
__device__ __forceinline__ void st_keep(double2 *p, const double2 v)
{
#if STAG_SPINOR_POLICY_F64 == 0
    *p = v;
#else
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;"
                 :: "l"(p), "d"(v.x), "d"(v.y), "l"(policy_evict_last()) : "memory");
#endif
}
__device__ __forceinline__ void st_keep(float4 *p, const float4 v)
{
#if STAG_SPINOR_POLICY == 0
    *p = v;
#else
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(policy_evict_last())
                 : "memory");
#endif
}

// ---- pass-through vectors (y of the CG iteration: read and written once per iteration,
// never reused before the next iteration): evict-first both ways ------------------------
__device__ __forceinline__ float4 ld_pass(const float4 *p)
{
#if STAG_SPINOR_POLICY == 0
    return *p;
#endif
    float4 v;
    asm volatile("ld.global.cs.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "l"(p), "l"(policy_evict_first()) : "memory");
    return v;
}
__device__ __forceinline__ double2 ld_pass(const double2 *p)
{
#if STAG_SPINOR_POLICY_F64 == 0
    return *p;
#endif
    double2 v;
    asm volatile("ld.global.cs.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
                 : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(policy_evict_first()) : "memory");
    return v;
}
__device__ __forceinline__ void st_pass(float4 *p, const float4 v)
{
#if STAG_SPINOR_POLICY == 0
    *p = v;
    return;
#endif
    asm volatile("st.global.cs.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(policy_evict_first())
                 : "memory");
}
__device__ __forceinline__ void st_pass(double2 *p, const double2 v)
{
#if STAG_SPINOR_POLICY_F64 == 0
    *p = v;
    return;
#endif
    asm volatile("st.global.cs.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;"
                 :: "l"(p), "d"(v.x), "d"(v.y), "l"(policy_evict_first()) : "memory");
}

}  // namespace stag
