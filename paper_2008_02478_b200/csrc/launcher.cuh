// launcher.cuh — the __global__ wrapper that runs a kernel struct's phases, and the CUDA
// launch policy of bd::enqueue_apply (apply_seq.h).  Included by every translation unit of
// libborisdemag.so; the tiled paths are compiled in units of their own (tu_*.cu) so that
// the library builds in parallel.
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <cstdlib>
#include <type_traits>
#include <vector>

#include "apply_seq.h"

namespace bd {

// K::warp_local_after(PH) (optional): what phase PH + 1 reads of phase PH's shared-memory writes was written by threads of the
// same warp, and what it overwrites no other warp reads in either phase: the block barrier between them becomes a warp barrier
template <class K, class = void>
struct WarpLocal { static BD_HD constexpr bool after(int) { return false; } };
template <class K>
struct WarpLocal<K, std::void_t<decltype(K::warp_local_after(0))>> { static BD_HD constexpr bool after(int ph) { return K::warp_local_after(ph); } };

template <class K, int PH>
__device__ __forceinline__ void run_phases(const typename K::Args& a, float2* sm) {
    K::template phase<PH>(threadIdx.x, blockIdx.x, blockIdx.y, a, sm);
    if constexpr (PH + 1 < K::NPHASES) {
        if constexpr (WarpLocal<K>::after(PH)) __syncwarp();
        else __syncthreads();
        run_phases<K, PH + 1>(a, sm);
    }
}

template <class K, class = void>
struct MinBlocks { static constexpr int value = 1; };
template <class K>
struct MinBlocks<K, std::void_t<decltype(K::MINB)>> { static constexpr int value = K::MINB; };

// The kernels of one evaluation are launched with programmatic stream serialization: a kernel's blocks may
// become resident while the last blocks of its predecessor drain (launch_dependents at the top lets the
// successor's launch begin once every block of this grid has started), and wait here until the predecessor
// grid has completed and its writes are visible.  Every kernel of the library waits before it touches memory,
// so completion orders chain: nothing runs ahead of data it reads or overwrites.  Outside such a launch both
// instructions are no-ops.
template <class K, class = void>
struct HasPrologue : std::false_type {};
template <class K>
struct HasPrologue<K, std::void_t<decltype(&K::prologue)>> : std::true_type {};

template <class K>
__global__ void __launch_bounds__(K::NT, MinBlocks<K>::value) phase_kernel(const __grid_constant__ typename K::Args a) {
    extern __shared__ __align__(16) float2 bd_smem[];
    asm volatile("griddepcontrol.launch_dependents;");
    // what a block may do before its predecessor grid has finished: hints for data no kernel of the evaluation writes
    if constexpr (HasPrologue<K>::value) K::prologue(threadIdx.x, blockIdx.x, a);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    run_phases<K, 0>(a, bd_smem);
}

struct TimedLaunch { int kind; cudaEvent_t t0, t1; };

struct CudaLauncher;
// parts of the tiled paths, each defined in its own translation unit
int cu_tiled_2d(CudaLauncher& run, const PlanView& p, const float* M, float* H);          // tu_t2d.cu
int cu_yfused3(CudaLauncher& run, const PlanView& p);                                     // tu_y3.cu
int cu_xz_small(CudaLauncher& run, const PlanView& p, const float* M, float* H, bool fwd);  // tu_xz_a.cu  nz 2..16
int cu_xz_32(CudaLauncher& run, const PlanView& p, const float* M, float* H, bool fwd);     // tu_xz_b.cu  nz 32
int cu_xz_big(CudaLauncher& run, const PlanView& p, const float* M, float* H, bool fwd);    // tu_xz_c.cu  nz 64..256
int cu_plane_x(CudaLauncher& run, const PlanView& p, const float* M, float* H, bool fwd);   // tu_plane_x.cu
int cu_plane_yz(CudaLauncher& run, const PlanView& p);                                      // tu_plane_yz.cu

constexpr int kMaxDevices = 64;

// BORIS_DEMAG_NO_PDL=1 in the environment launches the kernels plainly (A/B measurements)
inline bool pdl_enabled() {
    static const bool on = [] { const char* v = getenv("BORIS_DEMAG_NO_PDL"); return !(v && v[0] == '1'); }();
    return on;
}

struct CudaLauncher {
    cudaStream_t st;
    int dev = 0;                                   // the plan's device (the current one: checked by the entry points)
    cudaError_t err = cudaSuccess;
    bool pdl = pdl_enabled();                      // programmatic dependent launch between the kernels of an evaluation
    std::vector<TimedLaunch>* timed = nullptr;     // boris_demag_apply_timed only
    template <class K>
    int run(Grid g, const typename K::Args& a) {
        if (timed) {
            TimedLaunch t{K::KIND, nullptr, nullptr};
            if ((err = cudaEventCreate(&t.t0)) != cudaSuccess) return -2;
            if ((err = cudaEventCreate(&t.t1)) != cudaSuccess) { cudaEventDestroy(t.t0); return -2; }
            timed->push_back(t);
            cudaEventRecord(t.t0, st);
            const int rc = launch<K>(g, a);
            cudaEventRecord(t.t1, st);
            return rc;
        }
        return launch<K>(g, a);
    }
    template <class K>
    int launch(Grid g, const typename K::Args& a) {
        const size_t smem = (size_t)K::smem_elems(a) * sizeof(float2);
        // the opt-in to more than 48 KB of dynamic shared memory is per kernel AND per device
        static std::atomic<size_t> opted[kMaxDevices];
        const int d = dev >= 0 && dev < kMaxDevices ? dev : 0;
        if (smem > 48 * 1024 && smem > opted[d].load(std::memory_order_relaxed)) {
            err = cudaFuncSetAttribute(phase_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (err != cudaSuccess) return -2;
            size_t seen = opted[d].load(std::memory_order_relaxed);
            while (seen < smem && !opted[d].compare_exchange_weak(seen, smem, std::memory_order_relaxed)) {}
        }
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(g.x, g.y);
        cfg.blockDim = dim3(K::NT);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = pdl ? 1 : 0;
        err = cudaLaunchKernelEx(&cfg, phase_kernel<K>, a);
        return err == cudaSuccess ? 0 : -2;
    }
    // hooks of enqueue_apply (apply_seq.h)
    int tiled_2d(const PlanView& p, const float* M, float* H) { return cu_tiled_2d(*this, p, M, H); }
    int yfused3(const PlanView& p) { return cu_yfused3(*this, p); }
    int plane_x(const PlanView& p, const float* M, float* H, bool fwd) { return cu_plane_x(*this, p, M, H, fwd); }
    int plane_yz(const PlanView& p) { return cu_plane_yz(*this, p); }
    int xz(const PlanView& p, const float* M, float* H, bool fwd) {
        if (p.nz <= 16) return cu_xz_small(*this, p, M, H, fwd);
        if (p.nz == 32) return cu_xz_32(*this, p, M, H, fwd);
        return cu_xz_big(*this, p, M, H, fwd);
    }
};

}  // namespace bd
