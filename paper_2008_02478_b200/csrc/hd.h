// hd.h — host/device portability shims.
//
// Every arithmetic routine of the library is written as a BD_HD inline function
// so that the same source compiles (a) with nvcc into the sm_100a kernels and
// (b) with g++ into the host-side emulation used by the CPU tests
// (tests/emu/emulate.cpp), which steps the kernels' phases thread by thread.
// The emulation is test infrastructure: libborisdemag.so never runs it.
#pragma once

#if defined(__CUDACC__)
#define BD_HD __host__ __device__ __forceinline__
#define BD_D __device__ __forceinline__
#else
#define BD_HD inline
#define BD_D inline
#endif

#if defined(__CUDA_ARCH__)
#define BD_LDG(p) __ldg(p)
#define BD_LDCG(p) __ldcg(p)
#define BD_STCG(p, v) __stcg((p), (v))
#if defined(BD_PLAIN_STS)
#define BD_STS(p, v) (*(p) = (v))
#else
#define BD_STS(p, v) bd_sts_pair((p), (v))
#endif
#define BD_UNROLL _Pragma("unroll")
#define BD_PRAGMA_(x) _Pragma(#x)
#define BD_UNROLL_N(n) BD_PRAGMA_(unroll n)
#else
#define BD_LDG(p) (*(p))
#define BD_LDCG(p) (*(p))
#define BD_STCG(p, v) (*(p) = (v))
#define BD_UNROLL
#define BD_UNROLL_N(n)
#define BD_STS(p, v) (*(p) = (v))
#endif

#include <vector_types.h>   // float2, float4, double2 (plain structs on the host)

BD_HD float2 bd_f2(float x, float y) { float2 r; r.x = x; r.y = y; return r; }

// hint: bring the 128-byte line at p into L2 (no-op in the host emulation)
BD_HD void bd_prefetch_l2(const void* p) {
#if defined(__CUDA_ARCH__)
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
#else
    (void)p;
#endif
}

// Store of a complex pair to SHARED memory (p must point into shared memory).  Written as st.shared.v2.f32: for the
// plain C++ store of a float2 that came out of a packed f32x2 operation nvcc emits st.shared.u64, and ptxas (12.9)
// then copies every such register pair into one fixed pair first (two MOVs per STS.64: 15 - 25 % of the
// instructions of a register-DFT pass, profiles/r02_plane.md).
#if defined(__CUDA_ARCH__)
__device__ __forceinline__ void bd_sts_pair(float2* p, float2 v) {
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"((unsigned)__cvta_generic_to_shared(p)), "f"(v.x), "f"(v.y) : "memory");
}
#endif
