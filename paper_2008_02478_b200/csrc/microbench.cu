// microbench.cu — the two probes of include/boris_micro.h (FP32 lane rate, segment-size bandwidth).
// Measurement tooling: nothing on the hot path calls it.
#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/boris_micro.h"

namespace bd { int micro_fail(cudaError_t e, const char* what); }   // boris_demag.cu: sets the last-error text

namespace {

constexpr int kChains = 8;

template <int OP>
__global__ void __launch_bounds__(256) k_rate(float* out, int iters, float a, float b) {
    float2 v[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) v[i] = make_float2(threadIdx.x * 1e-3f + i, blockIdx.x * 1e-4f - i);
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < kChains; ++i) {
            if (OP == 0) { v[i].x = v[i].x + a; }
            if (OP == 1) { v[i].x = fmaf(v[i].x, a, b); }
            if (OP == 2) { v[i] = __fadd2_rn(v[i], a2); }
            if (OP == 3) { v[i] = __ffma2_rn(v[i], a2, b2); }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += v[i].x + v[i].y;
    if (s == 123.456f) out[0] = s;            // keeps the chains alive
}

// a warp touches 32 * 16 bytes per trip as 512 / SEG pieces of SEG contiguous bytes; the pieces of one
// trip lie `stride` bytes apart (different DRAM pages), successive trips walk through the buffer
template <int SEG, bool WRITE>
__global__ void __launch_bounds__(256) k_segments(uint4* buf, size_t n16, size_t stride16, uint4* sink) {
    constexpr int LPS = SEG / 16;                               // lanes per piece
    const size_t warps = (size_t)gridDim.x * (blockDim.x / 32);
    const size_t warp = (size_t)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
    const int lane = threadIdx.x & 31, piece = lane / LPS, in_piece = lane % LPS;
    const size_t pieces_per_row = stride16 / LPS;               // pieces of one "row" of stride16 units
    uint4 acc = make_uint4(0, 0, 0, 0);
    // piece index space: [n16 / stride16 rows][pieces_per_row]; a trip takes the same piece column of 32/LPS rows
    const size_t rows = n16 / stride16, row_groups = rows / (32 / LPS);
    for (size_t t = warp; t < row_groups * pieces_per_row; t += warps) {
        const size_t rg = t / pieces_per_row, pc = t % pieces_per_row;
        const size_t idx = (rg * (32 / LPS) + piece) * stride16 + pc * LPS + in_piece;
        if (WRITE) {
            __stcg(&buf[idx], make_uint4((unsigned)idx, 1u, 2u, 3u));
        } else {
            const uint4 x = __ldcg(&buf[idx]);
            acc.x ^= x.x; acc.y ^= x.y; acc.z ^= x.z; acc.w ^= x.w;
        }
    }
    if (!WRITE && acc.x == 0x12345678u && acc.y == 0x9abcdef0u) sink[0] = acc;
}

template <int OP>
int run_rate(double* out) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    float* d = nullptr;
    cudaError_t e = cudaMalloc((void**)&d, 16);
    if (e != cudaSuccess) return bd::micro_fail(e, "cudaMalloc");
    const int blocks = sms * 8, iters = 1 << 14;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    k_rate<OP><<<blocks, 256>>>(d, 64, 1.0001f, 1e-7f);
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(t0);
        k_rate<OP><<<blocks, 256>>>(d, iters, 1.0001f, 1e-7f);
        cudaEventRecord(t1);
        e = cudaEventSynchronize(t1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(t0); cudaEventDestroy(t1); cudaFree(d);
    if (e != cudaSuccess) return bd::micro_fail(e, "k_rate");
    const double per_thread = (double)iters * kChains * (OP >= 2 ? 2 : 1);
    *out = per_thread * 256.0 * blocks / (best * 1e-3);
    return 0;
}

template <int SEG>
int run_seg(int write, double* gbs) {
    const size_t bytes = (size_t)1 << 30, n16 = bytes / 16, stride16 = (size_t)(64 << 10) / 16;   // 64 KB between pieces
    uint4 *buf = nullptr, *sink = nullptr;
    cudaError_t e = cudaMalloc((void**)&buf, bytes);
    if (e != cudaSuccess) return bd::micro_fail(e, "cudaMalloc");
    e = cudaMalloc((void**)&sink, 16);
    if (e != cudaSuccess) { cudaFree(buf); return bd::micro_fail(e, "cudaMalloc"); }
    cudaMemset(buf, 1, bytes);
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(t0);
        if (write) k_segments<SEG, true><<<sms * 8, 256>>>(buf, n16, stride16, sink);
        else k_segments<SEG, false><<<sms * 8, 256>>>(buf, n16, stride16, sink);
        cudaEventRecord(t1);
        e = cudaEventSynchronize(t1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(t0); cudaEventDestroy(t1); cudaFree(buf); cudaFree(sink);
    if (e != cudaSuccess) return bd::micro_fail(e, "k_segments");
    *gbs = (double)bytes / (best * 1e-3) / 1e9;
    return 0;
}

}  // namespace

extern "C" {

int boris_micro_fp32_rate(int op, double* lane_ops_per_s) {
    if (!lane_ops_per_s) return -1;
    switch (op) {
        case 0: return run_rate<0>(lane_ops_per_s);
        case 1: return run_rate<1>(lane_ops_per_s);
        case 2: return run_rate<2>(lane_ops_per_s);
        case 3: return run_rate<3>(lane_ops_per_s);
        default: return -1;
    }
}

int boris_micro_segment_bw(int seg_bytes, int write, double* gbs) {
    if (!gbs) return -1;
    switch (seg_bytes) {
        case 16: return run_seg<16>(write, gbs);
        case 32: return run_seg<32>(write, gbs);
        case 64: return run_seg<64>(write, gbs);
        case 128: return run_seg<128>(write, gbs);
        case 256: return run_seg<256>(write, gbs);
        case 512: return run_seg<512>(write, gbs);
        default: return -1;
    }
}

}  // extern "C"
