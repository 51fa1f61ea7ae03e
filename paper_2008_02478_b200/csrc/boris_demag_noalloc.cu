// boris_demag_noalloc.cu — boris_demag_energy_noalloc (include/boris_demag_noalloc.h): the demagnetizing energy of S8
// (E = -(mu0/2) dV sum M.H) by a variant of boris_demag.cu's energy kernel whose scratch memory is a
// file-scope device array: the entry point allocates nothing.
//
// The array is shared by every call on a device and keeps the last call's contents: the block sums are all
// overwritten before they are read, the ticket is cleared on the stream before every launch.  Calls that overlap on
// the GPU race (header).
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>

#include "../../include/boris_demag_noalloc.h"

namespace bd {
int micro_fail(cudaError_t e, const char* what);
int set_error(int code, const char* msg);
void clear_error();
}  // namespace bd

namespace {

constexpr int kThreads = 256, kUnroll = 8;                       // 16-byte load pairs in flight per thread
constexpr long long kValuesPerBlock = 4LL * kThreads * kUnroll;  // 8192 values of M.H per block
constexpr int kMaxBlocks = (int)(BORIS_DEMAG_NOALLOC_MAX_VALUES / kValuesPerBlock);   // 16384
constexpr int kTicketSlot = kMaxBlocks;                          // the ticket has a 256-byte line of its own
constexpr double kPi = 3.14159265358979323846264338327950288;
static_assert((size_t)(kMaxBlocks + 32) * sizeof(double) == BORIS_DEMAG_NOALLOC_SCRATCH_BYTES, "scratch size of the header");

// [0, kMaxBlocks): fp64 block sums; [kTicketSlot]: the ticket counter (an unsigned in the first 4 bytes).
// In HOST code this name is a stand-in, not a device address: host code uses scratch_of_current_device().
static __device__ __align__(256) double g_noalloc_scratch[kMaxBlocks + 32];

__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double block_sum(double v, double* sh) {
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    v = (threadIdx.x < (blockDim.x >> 5)) ? sh[threadIdx.x] : 0.0;
    if (wid == 0) v = warp_sum(v);
    return v;
}
// four products, each split exactly into its rounded fp32 value and the fma residual (boris_demag.cu dot4)
__device__ __forceinline__ double dot4(const float4& m, const float4& h) {
    const float p0 = m.x * h.x, p1 = m.y * h.y, p2 = m.z * h.z, p3 = m.w * h.w;
    const float e = (fmaf(m.x, h.x, -p0) + fmaf(m.y, h.y, -p1)) + (fmaf(m.z, h.z, -p2) + fmaf(m.w, h.w, -p3));
    return (((double)p0 + (double)p1) + ((double)p2 + (double)p3)) + (double)e;
}

// Block b sums the float4 items [b 2048, (b + 1) 2048) of M.H; the last block also takes the n % 4 trailing values.
// scratch: the device address of g_noalloc_scratch (passed by the host, which looked it up for this device).
__global__ void __launch_bounds__(kThreads) k_energy_noalloc(const float4* __restrict__ M, const float4* __restrict__ H, long long n4,
                                                             int tail, double* scratch, double factor, double* E) {
    __shared__ double sh[32];
    __shared__ bool last;
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch + kTicketSlot);
    const long long lo = (long long)blockIdx.x * (kThreads * kUnroll);
    double acc0 = 0.0, acc1 = 0.0;
    if (lo + kThreads * kUnroll <= n4) {
        float4 m[kUnroll], h[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) { m[u] = __ldcs(&M[lo + u * kThreads + threadIdx.x]); h[u] = __ldcs(&H[lo + u * kThreads + threadIdx.x]); }
#pragma unroll
        for (int u = 0; u < kUnroll; u += 2) { acc0 += dot4(m[u], h[u]); acc1 += dot4(m[u + 1], h[u + 1]); }
    } else {
        for (long long i = lo + threadIdx.x; i < n4; i += kThreads) acc0 += dot4(__ldcs(&M[i]), __ldcs(&H[i]));
    }
    if (blockIdx.x == gridDim.x - 1 && (int)threadIdx.x < tail) {
        const float* ms = reinterpret_cast<const float*>(M + n4);
        const float* hs = reinterpret_cast<const float*>(H + n4);
        acc1 += (double)ms[threadIdx.x] * (double)hs[threadIdx.x];
    }
    const double acc = block_sum(acc0 + acc1, sh);
    // second level in the same launch: the block that finishes last adds the block sums in index order
    // (the ticket decides WHO adds, not what: E is bit-identical across calls)
    if (threadIdx.x == 0) {
        scratch[blockIdx.x] = acc;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double tot = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += kThreads) tot += __ldcg(&scratch[i]);
    __syncthreads();                       // sh is reused
    tot = block_sum(tot, sh);
    if (threadIdx.x == 0) { *E = factor * tot; *ticket = 0u; }
}

constexpr int kMaxDevices = 64;
std::atomic<double*> g_scratch_addr[kMaxDevices];      // device address of g_noalloc_scratch, per device

// The device address of the array on the CURRENT device: looked up once per device (cudaGetSymbolAddress answers for
// the device that is current when it is called).
int scratch_of_current_device(double** out) {
    int dev = 0;
    if (cudaError_t e = cudaGetDevice(&dev); e != cudaSuccess)
        return bd::micro_fail(e, "cudaGetDevice (no CUDA device: this library has no CPU fallback)");
    if (dev < 0 || dev >= kMaxDevices) return bd::set_error(-1, "device ordinal above 63");
    double* p = g_scratch_addr[dev].load(std::memory_order_acquire);
    if (!p) {
        if (cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch); e != cudaSuccess)
            return bd::micro_fail(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
        if (!p) return bd::set_error(-2, "cudaGetSymbolAddress returned a null address");
        g_scratch_addr[dev].store(p, std::memory_order_release);   // two threads racing here store the same value
    }
    *out = p;
    return 0;
}

}  // namespace

extern "C" int boris_demag_energy_noalloc(const float* M, const float* H, long long n_values, double hx, double hy, double hz,
                                          double* E_dev, void* stream) {
    bd::clear_error();
    if (!M || !H || !E_dev) return bd::set_error(-1, "null argument");
    if (n_values < 1) return bd::set_error(-1, "n_values must be at least 1");
    if (n_values > BORIS_DEMAG_NOALLOC_MAX_VALUES)
        return bd::set_error(-1, "n_values above BORIS_DEMAG_NOALLOC_MAX_VALUES (2^27 = 134217728 values per field): the static scratch "
                                 "array holds 16384 block sums of 8192 values; use boris_demag_energy for larger meshes");
    if (!(hx > 0.0) || !(hy > 0.0) || !(hz > 0.0)) return bd::set_error(-1, "cell sizes must be positive");
    if (((uintptr_t)M | (uintptr_t)H) & 15u) return bd::set_error(-1, "M and H must be 16-byte aligned");
    if ((uintptr_t)E_dev & 7u) return bd::set_error(-1, "E_dev must be 8-byte aligned");
    double* scratch = nullptr;
    if (int rc = scratch_of_current_device(&scratch)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const long long n4 = n_values / 4;
    const int tail = (int)(n_values - 4 * n4);
    const long long nblk = (n_values + kValuesPerBlock - 1) / kValuesPerBlock;          // <= kMaxBlocks
    // the ticket must start at zero, whatever an earlier (possibly failed) call left in the shared array
    if (cudaError_t e = cudaMemsetAsync(scratch + kTicketSlot, 0, sizeof(unsigned), st); e != cudaSuccess)
        return bd::micro_fail(e, "cudaMemsetAsync(ticket)");
    const double factor = -0.5 * (4e-7 * kPi) * hx * hy * hz;
    k_energy_noalloc<<<(unsigned)nblk, kThreads, 0, st>>>(reinterpret_cast<const float4*>(M), reinterpret_cast<const float4*>(H), n4,
                                                         tail, scratch, factor, E_dev);
    if (cudaError_t e = cudaGetLastError(); e != cudaSuccess) return bd::micro_fail(e, "k_energy_noalloc launch");
    return 0;
}
