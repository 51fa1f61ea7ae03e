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
#define BD_UNROLL _Pragma("unroll")
#define BD_PRAGMA_(x) _Pragma(#x)
#define BD_UNROLL_N(n) BD_PRAGMA_(unroll n)
#else
#define BD_LDG(p) (*(p))
#define BD_LDCG(p) (*(p))
#define BD_STCG(p, v) (*(p) = (v))
#define BD_UNROLL
#define BD_UNROLL_N(n)
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
