// boris_demag.cu — C ABI (include/boris_demag.h), plan construction and kernel launches.
//
// Build: nvcc -std=c++17 -O3 -lineinfo -gencode arch=compute_100a,code=sm_100a
//             -shared -Xcompiler -fPIC -o libborisdemag.so boris_demag.cu
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <type_traits>
#include <vector>

#include "../../include/boris_demag.h"
#include "apply_seq.h"
#include "kernels.h"
#include "launcher.cuh"
#include "khat_layout.h"
#include "plan_math.h"

namespace {

using namespace bd;

thread_local std::string g_err;

int fail(int code, const std::string& msg) { g_err = msg; return code; }
int cuda_fail(cudaError_t e, const char* what) {
    const int code = (e == cudaErrorMemoryAllocation) ? -3 : -2;
    return fail(code, std::string(what) + ": " + cudaGetErrorString(e));
}
#define BD_CUDA(call)                                             \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);       \
    } while (0)


// ------------------------------------------------------------------ plan-time kernels (fp64)
struct Images { int per[3]; int img[3]; };      // period in cells and copies per side along x, y, z (plan_math.h)

__global__ void k_tensor(double* N, int ncomp, int nx, int ny, int nz, double hx, double hy, double hz, Images im) {
    const long total = (long)nx * ny * nz;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        const int i = (int)(idx % nx), j = (int)((idx / nx) % ny), k = (int)(idx / ((long)nx * ny));
        double out[6];
        tensor_point_images(i, j, k, im.per, im.img, hx, hy, hz, out);
        for (int c = 0; c < ncomp; ++c) N[c * total + idx] = out[c];
    }
}

// out[c][a2][a1][k] along dimension `dim` of an array in[c][d2][d1][d0]; the transformed
// dimension has n samples in and n+1 (or 1 if n == 1) frequencies out.
__global__ void k_real_transform(const double* in, double* out, int ncomp, int d0, int d1, int d2, int dim,
                                 const double2* cs) {
    const int n = dim == 0 ? d0 : (dim == 1 ? d1 : d2);
    const int nk = n > 1 ? n + 1 : 1;
    const int o0 = dim == 0 ? nk : d0, o1 = dim == 1 ? nk : d1, o2 = dim == 2 ? nk : d2;
    const long total = (long)ncomp * o2 * o1 * o0;
    const long stride = dim == 0 ? 1 : (dim == 1 ? d0 : (long)d0 * d1);
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        const int a0 = (int)(idx % o0), a1 = (int)((idx / o0) % o1), a2 = (int)((idx / ((long)o0 * o1)) % o2);
        const int c = (int)(idx / ((long)o0 * o1 * o2));
        const int k = dim == 0 ? a0 : (dim == 1 ? a1 : a2);
        const long base = (((long)c * d2 + (dim == 2 ? 0 : a2)) * d1 + (dim == 1 ? 0 : a1)) * d0 + (dim == 0 ? 0 : a0);
        out[idx] = real_transform(in + base, stride, n, k, comp_is_odd(c, dim), cs);
    }
}

__global__ void k_scale_sign(double* K, KLayout kl, double scale) {
    const long per = (long)kl.nzr() * kl.nyr() * kl.nxr(), total = kl.ncomp * per;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        const int c = (int)(idx / per);
        K[idx] *= (c >= 3 ? -scale : scale);      // (-i)^2 of the two odd coordinates
    }
}

__global__ void k_fill_storage(float* Kst, KLayout kl, const double* Kred) {
    const long total = kl.storage_elems();
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x)
        Kst[idx] = (float)storage_value(kl, idx, Kred);
}

__global__ void k_fill_plane(float* KP, PlaneK pk, const int* slot_ky, const double* Kred) {
    const long total = pk.storage_elems();
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x)
        KP[idx] = (float)plane_storage_value(pk, idx, slot_ky, Kred);
}
__global__ void k_gather_plane(const float* KP, PlaneK pk, const int* kidx, float* out) {
    const long total = 6L * (pk.nz + 1) * (pk.ny + 1) * (pk.nx + 1);
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        long r = idx;
        const int kx = (int)(r % (pk.nx + 1)); r /= (pk.nx + 1);
        const int ky = (int)(r % (pk.ny + 1)); r /= (pk.ny + 1);
        const int kz = (int)(r % (pk.nz + 1)); const int c = (int)(r / (pk.nz + 1));
        out[idx] = KP[plane_storage_index_of(pk, kidx, c, kz, ky, kx)];
    }
}

__global__ void k_gather_natural(const float* Kst, KLayout kl, float* out) {
    const long total = kl.reduced_elems();
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        long r = idx;
        const int kx = (int)(r % kl.nxr()); r /= kl.nxr();
        const int ky = (int)(r % kl.nyr()); r /= kl.nyr();
        const int kz = (int)(r % kl.nzr()); const int c = (int)(r / kl.nzr());
        float sign;
        const long s = storage_index_of(kl, c, kz, ky, kx, sign);
        out[idx] = sign * Kst[s];
    }
}

// ------------------------------------------------------------------ energy (S8)
constexpr int kEnergyBlocks = 1184, kEnergyThreads = 256;          // 8 blocks per SM of a 148-SM device
constexpr int kEnergyUnroll = 8;                                   // 16-byte load pairs in flight per thread
constexpr int kFusedEnergySlots = 8192;          // blocks of XInvT (3 ny / rb), ZXInv (3 ny) or XInvP (3 nz ny / 16)

__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double block_sum(double v, double* sh) {
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    const int nw = blockDim.x >> 5;
    v = (threadIdx.x < nw) ? sh[threadIdx.x] : 0.0;
    if (wid == 0) v = warp_sum(v);
    return v;
}

// sum of four products: each product m h is split exactly into its rounded fp32 value p and the residual
// e = fma(m, h, -p); the p are added in fp64, the residuals (2^-24 of the products) in fp32 and then to the fp64 sum:
// the result differs from the all-fp64 sum by 2^-48 of the terms, at one conversion per product instead of two
__device__ __forceinline__ double dot4(const float4& m, const float4& h) {
    const float p0 = m.x * h.x, p1 = m.y * h.y, p2 = m.z * h.z, p3 = m.w * h.w;
    const float e = (fmaf(m.x, h.x, -p0) + fmaf(m.y, h.y, -p1)) + (fmaf(m.z, h.z, -p2) + fmaf(m.w, h.w, -p3));
    return (((double)p0 + (double)p1) + ((double)p2 + (double)p3)) + (double)e;
}

__global__ void __launch_bounds__(kEnergyThreads) k_energy_partial(const float4* __restrict__ M, const float4* __restrict__ H,
                                                                    long n4, double* partial, unsigned* ticket,
                                                                    double factor, double* E) {
    __shared__ double sh[32];
    double acc0 = 0.0, acc1 = 0.0;
    // a block streams one contiguous piece of both arrays (whole DRAM pages), kEnergyUnroll load pairs in flight per thread
    const long per = (n4 + gridDim.x - 1) / gridDim.x;
    const long lo = blockIdx.x * per, hi = lo + per < n4 ? lo + per : n4;
    long i = lo + threadIdx.x;
    for (; i + (kEnergyUnroll - 1) * (long)kEnergyThreads < hi; i += kEnergyUnroll * (long)kEnergyThreads) {
        float4 m[kEnergyUnroll], h[kEnergyUnroll];
#pragma unroll
        for (int u = 0; u < kEnergyUnroll; ++u) { m[u] = __ldcs(&M[i + u * kEnergyThreads]); h[u] = __ldcs(&H[i + u * kEnergyThreads]); }
#pragma unroll
        for (int u = 0; u < kEnergyUnroll; u += 2) { acc0 += dot4(m[u], h[u]); acc1 += dot4(m[u + 1], h[u + 1]); }
    }
    for (; i < hi; i += kEnergyThreads) acc0 += dot4(__ldcs(&M[i]), __ldcs(&H[i]));
    double acc = block_sum(acc0 + acc1, sh);
    // second level in the same launch: the block that finishes last adds the partial sums in
    // index order (the ticket only decides WHO adds, so E is bit-identical across calls)
    __shared__ bool last;
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = acc;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double tot = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) tot += __ldcg(&partial[i]);
    __syncthreads();                       // sh is reused
    tot = block_sum(tot, sh);
    if (threadIdx.x == 0) { *E = factor * tot; *ticket = 0u; }
}
int grid_for(long total, int threads) {
    long g = (total + threads - 1) / threads;
    return (int)(g < 1 ? 1 : (g > 148L * 64 ? 148L * 64 : g));
}

}  // namespace

// the other translation units of the library report their failures through the same thread-local text
namespace bd {
int micro_fail(cudaError_t e, const char* what) { return cuda_fail(e, what); }
int set_error(int code, const char* msg) { return fail(code, msg); }
void clear_error() { g_err.clear(); }
}  // namespace bd

// ------------------------------------------------------------------ plan
struct boris_demag_plan {
    // nx, ny, nz: the mesh the kernels work on (powers of two).  ux, uy, uz: the caller's mesh; where it is
    // not one the kernels take, it sits in the corner of the next power-of-two mesh whose other cells
    // hold M = 0 (exact: empty cells add nothing to the sum of PAPER.md:L323), staged through Mp / Hp.
    int ux, uy, uz;
    int images[3] = {0, 0, 0};       // copies per side along x, y, z (periodic boundary conditions; 0: open)
    bool padmode = false;
    float* Mp = nullptr;             // [3][nz][ny][nx], zero outside the caller's cells
    float* Hp = nullptr;
    int nx, ny, nz;
    double hx, hy, hz;
    bd::KLayout kl;
    int device;
    // device memory
    float* Kst = nullptr;            // kernel spectrum, fused-pass order
    float2* tw_x = nullptr;          // exp(-2 pi i k / LX)
    float2* tw_xpost = nullptr;      // exp(-2 pi i k / Px), k <= LX/2
    float2* tw_y = nullptr;          // exp(-2 pi i k / Py)
    float2* tw_z = nullptr;          // exp(-2 pi i k / Pz)
    float2* W = nullptr;             // [3][NS][nz][ny]
    float2* T = nullptr;             // [3][cs][nz][Py]   (nz > 1)
    float2* V = nullptr;             // tiled path: [3][Pz][ntl][ny][cols]
    float2* ptw_x = nullptr;         // tiled path: per-pass twiddles of the x / y transforms
    float2* ptw_y = nullptr;
    float4* xpost = nullptr;         // tiled path: fill_xpost table
    // plane path (plane.h)
    float2* X = nullptr;             // [3 nz][nx+1][ny]
    float2* P = nullptr;             // [NQ][3 nz][nx+1][LSP]
    float* KP = nullptr;             // kernel spectrum, plane order
    int* kidx = nullptr;             // [NQ][LS]
    float2* pl_tw = nullptr;
    float2* pl_zt = nullptr;
    double* partial = nullptr;       // energy partial sums, followed by the ticket counter
    double* partial_f = nullptr;     // fused energy (apply_energy): one slot per block of the last kernel + ticket
    float* stage_M = nullptr;        // apply_host staging
    float* stage_H = nullptr;
    double* stage_E = nullptr;
    bd::LaunchCfg cfg;               // launch configuration (apply_seq.h)
    long bytes = 0;
};

namespace {

template <class T>
int dev_alloc(boris_demag_plan* p, T** ptr, size_t count) {
    const size_t bytes = count * sizeof(T);
    cudaError_t e = cudaMalloc((void**)ptr, bytes ? bytes : sizeof(T));
    if (e != cudaSuccess) { *ptr = nullptr; return cuda_fail(e, "cudaMalloc"); }
    p->bytes += (long)bytes;
    return 0;
}

int upload_twiddles(boris_demag_plan* p, float2** dst, int count, int denom) {
    std::vector<float2> h((size_t)count);
    bd::fill_twiddles(h.data(), count, denom);
    if (int rc = dev_alloc(p, dst, (size_t)count)) return rc;
    BD_CUDA(cudaMemcpy(*dst, h.data(), (size_t)count * sizeof(float2), cudaMemcpyHostToDevice));
    return 0;
}

int upload_pass_twiddles(boris_demag_plan* p, float2** dst, int L) {
    std::vector<float2> h((size_t)bd::ptw_total(L));
    bd::fill_pass_twiddles(h.data(), L);
    if (int rc = dev_alloc(p, dst, h.size())) return rc;
    BD_CUDA(cudaMemcpy(*dst, h.data(), h.size() * sizeof(float2), cudaMemcpyHostToDevice));
    return 0;
}

bd::PlanView plan_view(const boris_demag_plan* p) {
    bd::PlanView pv{p->nx, p->ny, p->nz, p->cfg, p->Kst, p->tw_x, p->tw_xpost, p->tw_y, p->tw_z, p->W, p->T};
    pv.ptw_x = p->ptw_x; pv.ptw_y = p->ptw_y; pv.V = p->V; pv.xpost = p->xpost;
    pv.X = p->X; pv.P = p->P; pv.KP = p->KP; pv.kidx = p->kidx; pv.pl_tw = p->pl_tw; pv.pl_zt = p->pl_zt;
    return pv;
}

int upload_cs_table(double2** dst, int P) {
    std::vector<double2> h((size_t)P);
    for (int m = 0; m < P; ++m) {
        const double a = 2.0 * bd::kPi * (double)m / (double)P;
        h[m].x = std::cos(a); h[m].y = std::sin(a);
        if ((4 * m) % P == 0) {
            const int quarter = (4 * m) / P % 4;
            const double cx[4] = {1, 0, -1, 0}, sy[4] = {0, 1, 0, -1};
            h[m].x = cx[quarter]; h[m].y = sy[quarter];
        }
    }
    BD_CUDA(cudaMalloc((void**)dst, (size_t)P * sizeof(double2)));
    BD_CUDA(cudaMemcpy(*dst, h.data(), (size_t)P * sizeof(double2), cudaMemcpyHostToDevice));
    return 0;
}

// The natural, symmetry-reduced spectrum Kred[c][kz][ky][kx] of khat_layout.h on the device (fp64), with the
// factor of reading R12 folded in.  *out is cudaMalloc'ed here; the caller frees it.
int build_reduced(const bd::KLayout& kl, double hx, double hy, double hz, const Images& im, double** out) {
    const int nx = kl.nx, ny = kl.ny, nz = kl.nz, nc = kl.ncomp;
    const long cells = (long)nx * ny * nz;
    double *dN = nullptr, *dA = nullptr, *dB = nullptr, *dC = nullptr;
    double2 *csx = nullptr, *csy = nullptr, *csz = nullptr;
    int rc = 0;
    auto cleanup = [&]() {
        cudaFree(dN); cudaFree(dA); cudaFree(dB); cudaFree(dC); cudaFree(csx); cudaFree(csy); cudaFree(csz);
    };
#define BD_TRY(call)                                                              \
    do {                                                                          \
        cudaError_t e_ = (call);                                                  \
        if (e_ != cudaSuccess) { rc = cuda_fail(e_, #call); cleanup(); return rc; } \
    } while (0)
    const long nA = (long)nc * nz * ny * kl.nxr(), nB = (long)nc * nz * kl.nyr() * kl.nxr(), nC = kl.reduced_elems();
    BD_TRY(cudaMalloc((void**)&dN, (size_t)nc * cells * sizeof(double)));
    BD_TRY(cudaMalloc((void**)&dA, (size_t)nA * sizeof(double)));
    k_tensor<<<grid_for(cells, 128), 128>>>(dN, nc, nx, ny, nz, hx, hy, hz, im);
    BD_TRY(cudaGetLastError());
    if ((rc = upload_cs_table(&csx, kl.Px))) { cleanup(); return rc; }
    if ((rc = upload_cs_table(&csy, kl.Py))) { cleanup(); return rc; }
    if ((rc = upload_cs_table(&csz, kl.Pz > 1 ? kl.Pz : 2))) { cleanup(); return rc; }
    k_real_transform<<<grid_for(nA, 128), 128>>>(dN, dA, nc, nx, ny, nz, 0, csx);
    BD_TRY(cudaGetLastError());
    BD_TRY(cudaDeviceSynchronize());
    cudaFree(dN); dN = nullptr;
    BD_TRY(cudaMalloc((void**)&dB, (size_t)nB * sizeof(double)));
    k_real_transform<<<grid_for(nB, 128), 128>>>(dA, dB, nc, kl.nxr(), ny, nz, 1, csy);
    BD_TRY(cudaGetLastError());
    BD_TRY(cudaDeviceSynchronize());
    cudaFree(dA); dA = nullptr;
    BD_TRY(cudaMalloc((void**)&dC, (size_t)nC * sizeof(double)));
    k_real_transform<<<grid_for(nC, 128), 128>>>(dB, dC, nc, kl.nxr(), kl.nyr(), nz, 2, csz);
    BD_TRY(cudaGetLastError());
    // fold -1/(2 Px Py Pz): minus sign of H = -N*M, FFT normalisation, and the factor 2
    // each of XFwd's post-pass and XInv's pre-pass leaves out (reading R12)
    const double scale = -1.0 / (2.0 * (double)kl.Px * (double)kl.Py * (double)kl.Pz);
    k_scale_sign<<<grid_for(nC, 256), 256>>>(dC, kl, scale);
    BD_TRY(cudaGetLastError());
    BD_TRY(cudaDeviceSynchronize());
#undef BD_TRY
    *out = dC;
    dC = nullptr;
    cleanup();
    return 0;
}

// Build the kernel spectrum on the device (fp64), store it as fp32 in fused-pass order.
int build_spectrum(boris_demag_plan* p) {
    const bd::KLayout& kl = p->kl;
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    double* dC = nullptr;
    const Images im{{p->ux, p->uy, p->uz}, {p->images[0], p->images[1], p->images[2]}};
    int rc = build_reduced(kl, p->hx, p->hy, p->hz, im, &dC);
    if (rc) return rc;
    auto cleanup = [&]() { cudaFree(dC); };
#define BD_TRY(call)                                                              \
    do {                                                                          \
        cudaError_t e_ = (call);                                                  \
        if (e_ != cudaSuccess) { rc = cuda_fail(e_, #call); cleanup(); return rc; } \
    } while (0)
    if (p->cfg.plane.on) {
        const bd::PlaneGeom& g = p->cfg.plane;
        const bd::PlaneK pk = bd::make_plane_k(nx, ny, nz, g);
        std::vector<int> kidx((size_t)g.nq * g.ls), slotky((size_t)g.nq * g.nsl);
        bd::plane_fill_tables(ny, g, kidx.data(), slotky.data());
        int* dslot = nullptr;
        if ((rc = dev_alloc(p, &p->kidx, kidx.size()))) { cleanup(); return rc; }
        if ((rc = dev_alloc(p, &p->KP, (size_t)pk.storage_elems()))) { cleanup(); return rc; }
        BD_TRY(cudaMalloc((void**)&dslot, slotky.size() * sizeof(int)));
        cudaMemcpy(dslot, slotky.data(), slotky.size() * sizeof(int), cudaMemcpyHostToDevice);
        cudaMemcpy(p->kidx, kidx.data(), kidx.size() * sizeof(int), cudaMemcpyHostToDevice);
        k_fill_plane<<<grid_for(pk.storage_elems(), 256), 256>>>(p->KP, pk, dslot, dC);
        cudaError_t e1 = cudaGetLastError();
        if (e1 == cudaSuccess) e1 = cudaDeviceSynchronize();
        cudaFree(dslot);
        BD_TRY(e1);
    } else {
        if ((rc = dev_alloc(p, &p->Kst, (size_t)kl.storage_elems()))) { cleanup(); return rc; }
        k_fill_storage<<<grid_for(kl.storage_elems(), 256), 256>>>(p->Kst, kl, dC);
        BD_TRY(cudaGetLastError());
        BD_TRY(cudaDeviceSynchronize());
    }
#undef BD_TRY
    cleanup();
    return 0;
}

int check_sizes(int nx, int ny, int nz, double hx, double hy, double hz) {
    if (!(hx > 0.0) || !(hy > 0.0) || !(hz > 0.0) || !std::isfinite(hx) || !std::isfinite(hy) || !std::isfinite(hz))
        return fail(-1, "cell sides must be positive and finite");
    if (nx < 1 || nx > 1024) return fail(-1, "nx must be in [1, 1024]");
    if (ny < 1 || ny > 1024) return fail(-1, "ny must be in [1, 1024]");
    if (nz < 1 || nz > 512) return fail(-1, "nz must be in [1, 512]");
    return 0;
}

int next_pow2(int n) { int p = 1; while (p < n) p <<= 1; return p; }
constexpr int kMaxImages = 1000;

// (used by the entry points below)
// caller's mesh [3][uz][uy][ux] <-> its corner of the kernels' mesh [3][nz][ny][nx]
// aos: the caller's array is [uz][uy][ux][3] (one float3 per cell) instead of planar [3][uz][uy][ux]
__global__ void k_pad(const float* __restrict__ src, float* __restrict__ dst, int ux, int uy, int uz, int nx, int ny, int nz,
                      bool aos) {
    const long cells = (long)ux * uy * uz, total = 3L * cells;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        long r = idx;
        const int x = (int)(r % ux); r /= ux;
        const int y = (int)(r % uy); r /= uy;
        const int z = (int)(r % uz); const int c = (int)(r / uz);
        const long cell = ((long)z * uy + y) * ux + x;
        dst[(((long)c * nz + z) * ny + y) * nx + x] = src[aos ? 3 * cell + c : idx];
    }
}
// accumulate: dst += the staged field instead of dst = it (additive effective-field contributions)
__global__ void k_crop(const float* __restrict__ src, float* __restrict__ dst, int ux, int uy, int uz, int nx, int ny, int nz,
                       bool aos, bool accumulate) {
    const long cells = (long)ux * uy * uz, total = 3L * cells;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        long r = idx;
        const int x = (int)(r % ux); r /= ux;
        const int y = (int)(r % uy); r /= uy;
        const int z = (int)(r % uz); const int c = (int)(r / uz);
        const long cell = ((long)z * uy + y) * ux + x;
        const long o = aos ? 3 * cell + c : idx;
        const float v = src[(((long)c * nz + z) * ny + y) * nx + x];
        dst[o] = accumulate ? dst[o] + v : v;
    }
}

}  // namespace

namespace bd {
// for the fp64 engine (boris_demag_f64.cu): the reduced fp64 spectrum of a power-of-two mesh nx x ny x nz whose
// copies repeat with period per[] cells, img[] copies a side; *out is cudaMalloc'ed, the caller frees it
int build_reduced_spectrum(int nx, int ny, int nz, double hx, double hy, double hz, const int per[3], const int img[3],
                           double** out) {
    const Images im{{per[0], per[1], per[2]}, {img[0], img[1], img[2]}};
    return build_reduced(bd::make_klayout(nx, ny, nz, 1), hx, hy, hz, im, out);
}
int check_mesh_args(int nx, int ny, int nz, double hx, double hy, double hz) { return check_sizes(nx, ny, nz, hx, hy, hz); }
}  // namespace bd

extern "C" {

const char* boris_demag_version(void) { return "boris-demag-b200 0.1 (sm_100a)"; }
const char* boris_demag_last_error(void) { return g_err.c_str(); }

void boris_demag_plan_destroy(boris_demag_plan* p) {
    if (!p) return;
    cudaFree(p->Kst); cudaFree(p->tw_x); cudaFree(p->tw_xpost); cudaFree(p->tw_y); cudaFree(p->tw_z);
    cudaFree(p->W); cudaFree(p->T); cudaFree(p->partial); cudaFree(p->partial_f);
    cudaFree(p->X); cudaFree(p->P); cudaFree(p->KP); cudaFree(p->kidx); cudaFree(p->pl_tw); cudaFree(p->pl_zt);
    cudaFree(p->V); cudaFree(p->ptw_x); cudaFree(p->ptw_y); cudaFree(p->xpost); cudaFree(p->Mp); cudaFree(p->Hp);
    cudaFree(p->stage_M); cudaFree(p->stage_H); cudaFree(p->stage_E);
    delete p;
}

boris_demag_plan* boris_demag_plan_create(int ux, int uy, int uz, double hx, double hy, double hz) {
    return boris_demag_plan_create_pbc(ux, uy, uz, hx, hy, hz, 0, 0, 0);
}

boris_demag_plan* boris_demag_plan_create_pbc(int ux, int uy, int uz, double hx, double hy, double hz, int images_x,
                                              int images_y, int images_z) {
    g_err.clear();
    if (check_sizes(ux, uy, uz, hx, hy, hz)) return nullptr;
    if (images_x < 0 || images_y < 0 || images_z < 0 || images_x > kMaxImages || images_y > kMaxImages ||
        images_z > kMaxImages) {
        fail(-1, "images per side must be in [0, 1000]");
        return nullptr;
    }
    // the kernels take power-of-two meshes: nx >= 4, ny >= 2, nz = 1 or >= 2
    const int nx = next_pow2(ux < 4 ? 4 : ux), ny = next_pow2(uy < 2 ? 2 : uy), nz = uz == 1 ? 1 : next_pow2(uz);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cuda_fail(e, "cudaGetDevice (no CUDA device: this library has no CPU fallback)"); return nullptr; }
    boris_demag_plan* p = new (std::nothrow) boris_demag_plan();
    if (!p) { fail(-3, "out of host memory"); return nullptr; }
    p->nx = nx; p->ny = ny; p->nz = nz; p->hx = hx; p->hy = hy; p->hz = hz; p->device = dev;
    p->ux = ux; p->uy = uy; p->uz = uz;
    p->images[0] = images_x; p->images[1] = images_y; p->images[2] = images_z;
    p->padmode = nx != ux || ny != uy || nz != uz;
    const int Py = 2 * ny, Pz = nz > 1 ? 2 * nz : 1;
    p->cfg = bd::make_launch_cfg(nx, ny, nz);
    if (const char* e = getenv("BORIS_DEMAG_NO_PLANE")) { if (e[0] == '1') p->cfg.plane.on = 0; }     // A/B measurements
    {
        int sms = 148;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        p->cfg.pf_y = sms / 2;          // measured: 8..148 blocks ahead are within 1 %, longer distances lose (profiles/r01_tiled.md)
        p->cfg.pf_xz = sms / 4;         // measured best of 0 / 8 / 32 / 74 / 110 / 148 / 296
    }
    p->kl = p->cfg.tiled ? bd::make_klayout_tiled(nx, ny, nz, p->cfg.cols) : bd::make_klayout(nx, ny, nz, p->cfg.ty);
    const bd::KLayout& kl = p->kl;

    int rc = build_spectrum(p);
    if (!rc) rc = upload_twiddles(p, &p->tw_x, nx, nx);
    if (!rc) rc = upload_twiddles(p, &p->tw_xpost, nx / 2 + 1, 2 * nx);
    if (!rc) rc = upload_twiddles(p, &p->tw_y, Py, Py);
    if (!rc && nz > 1) rc = upload_twiddles(p, &p->tw_z, Pz, Pz);
    if (p->cfg.plane.on) {
        const bd::PlaneGeom& g = p->cfg.plane;
        if (!rc) rc = dev_alloc(p, &p->X, (size_t)3 * nz * (nx + 1) * ny);
        if (!rc) rc = dev_alloc(p, &p->P, (size_t)g.nq * 3 * nz * (nx + 1) * g.lsp);
        if (!rc) rc = upload_pass_twiddles(p, &p->ptw_x, nx);
        if (!rc) {
            std::vector<float4> h((size_t)nx / 2 + 1);
            bd::fill_xpost(h.data(), nx);
            rc = dev_alloc(p, &p->xpost, h.size());
            if (!rc && cudaMemcpy(p->xpost, h.data(), h.size() * sizeof(float4), cudaMemcpyHostToDevice) != cudaSuccess)
                rc = fail(-2, "cudaMemcpy xpost");
        }
        if (!rc) {
            std::vector<float2> h((size_t)g.nq * g.ls);
            bd::plane_fill_tw(h.data(), ny, g);
            rc = dev_alloc(p, &p->pl_tw, h.size());
            if (!rc && cudaMemcpy(p->pl_tw, h.data(), h.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess)
                rc = fail(-2, "cudaMemcpy pl_tw");
        }
        if (!rc) {
            std::vector<float2> h((size_t)g.zs * 16);
            bd::plane_fill_zt(h.data(), nz, g);
            rc = dev_alloc(p, &p->pl_zt, h.size());
            if (!rc && cudaMemcpy(p->pl_zt, h.data(), h.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess)
                rc = fail(-2, "cudaMemcpy pl_zt");
        }
    } else if (p->cfg.tiled) {
        const size_t nv = (size_t)3 * Pz * kl.ntl * ny * kl.cols;
        if (!rc) rc = dev_alloc(p, &p->V, nv);
        // the padding columns of the last tile are transformed along with the rest: keep them finite
        if (!rc && cudaMemset(p->V, 0, nv * sizeof(float2)) != cudaSuccess) rc = fail(-2, "cudaMemset");
        if (!rc) rc = upload_pass_twiddles(p, &p->ptw_x, nx);
        if (!rc) rc = upload_pass_twiddles(p, &p->ptw_y, Py);
        if (!rc) {
            std::vector<float4> h((size_t)nx / 2 + 1);
            bd::fill_xpost(h.data(), nx);
            rc = dev_alloc(p, &p->xpost, h.size());
            if (!rc && cudaMemcpy(p->xpost, h.data(), h.size() * sizeof(float4), cudaMemcpyHostToDevice) != cudaSuccess)
                rc = fail(-2, "cudaMemcpy xpost");
        }
    } else {
        if (!rc) rc = dev_alloc(p, &p->W, (size_t)3 * kl.nxr() * nz * ny);
        if (!rc && nz > 1) rc = dev_alloc(p, &p->T, (size_t)3 * p->cfg.cs * nz * Py);
    }
    if (p->padmode) {
        const size_t np = (size_t)3 * nx * ny * nz;
        if (!rc) rc = dev_alloc(p, &p->Mp, np);
        if (!rc) rc = dev_alloc(p, &p->Hp, np);
        if (!rc && cudaMemset(p->Mp, 0, np * sizeof(float)) != cudaSuccess) rc = fail(-2, "cudaMemset");
        if (!rc && cudaMemset(p->Hp, 0, np * sizeof(float)) != cudaSuccess) rc = fail(-2, "cudaMemset");
    }
    if (!rc) rc = dev_alloc(p, &p->partial, (size_t)kEnergyBlocks + 1);
    if (!rc && cudaMemset(p->partial, 0, ((size_t)kEnergyBlocks + 1) * sizeof(double)) != cudaSuccess) rc = fail(-2, "cudaMemset");
    if (!rc) rc = dev_alloc(p, &p->partial_f, (size_t)kFusedEnergySlots + 1);
    if (!rc && cudaMemset(p->partial_f, 0, ((size_t)kFusedEnergySlots + 1) * sizeof(double)) != cudaSuccess) rc = fail(-2, "cudaMemset");
    if (rc) { std::string keep = g_err; boris_demag_plan_destroy(p); g_err = keep; return nullptr; }
    return p;
}

namespace {
// a plan belongs to the device it was created on (its tables, workspace and shared-memory opt-ins live there)
int check_device(const boris_demag_plan* p) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device)
        return fail(-1, "the current CUDA device is not the one the plan was created on");
    return 0;
}
int check_fields(const boris_demag_plan* p, const void* M, const void* H, bool alias_ok) {
    if (!p || !M || !H) return fail(-1, "null argument");
    if (!alias_ok && M == H) return fail(-1, "M and H must not alias");
    if (int rc = check_device(p)) return rc;
    // the kernels read rows as 16-byte vectors; a mesh staged through Mp / Hp is copied element by element
    if ((((uintptr_t)M | (uintptr_t)H) & (p->padmode ? 3 : 15)) != 0)
        return fail(-1, p->padmode ? "M and H must be 4-byte aligned" : "M and H must be 16-byte aligned");
    return 0;
}
int stage(const boris_demag_plan* p, bool in, const float* src, float* dst, cudaStream_t st, bool aos = false,
          bool accumulate = false) {
    const long total = 3L * p->ux * p->uy * p->uz;
    if (in) k_pad<<<grid_for(total, 256), 256, 0, st>>>(src, dst, p->ux, p->uy, p->uz, p->nx, p->ny, p->nz, aos);
    else k_crop<<<grid_for(total, 256), 256, 0, st>>>(src, dst, p->ux, p->uy, p->uz, p->nx, p->ny, p->nz, aos, accumulate);
    BD_CUDA(cudaGetLastError());
    return 0;
}
}  // namespace

int boris_demag_apply(boris_demag_plan* p, const float* M, float* H, void* stream) {
    if (int rc = check_fields(p, M, H, false)) return rc;
    if (p->padmode) {
        if (int rc = stage(p, true, M, p->Mp, (cudaStream_t)stream)) return rc;
        M = p->Mp;
    }
    float* Hu = H;
    if (p->padmode) H = p->Hp;
    CudaLauncher run{(cudaStream_t)stream, p->device};
    const bd::PlanView pv = plan_view(p);
    const int rc = bd::enqueue_apply(run, pv, M, H);
    if (rc == -2) return cuda_fail(run.err, "kernel launch");
    if (rc) return fail(rc, "unsupported size");
    if (p->padmode) return stage(p, false, p->Hp, Hu, (cudaStream_t)stream);
    return 0;
}

int boris_demag_apply_energy(boris_demag_plan* p, const float* M, float* H, double* E_dev, void* stream) {
    if (!E_dev) return fail(-1, "null argument");
    if (int rc = check_fields(p, M, H, false)) return rc;
    if (!p->cfg.tiled && !p->cfg.plane.on) {
        if (int rc = boris_demag_apply(p, M, H, stream)) return rc;
        return boris_demag_energy(p, M, H, E_dev, stream);
    }
    float* Hu = H;
    if (p->padmode) {            // the empty cells of Mp add nothing to sum M.H
        if (int rc = stage(p, true, M, p->Mp, (cudaStream_t)stream)) return rc;
        M = p->Mp; H = p->Hp;
    }
    CudaLauncher run{(cudaStream_t)stream, p->device};
    bd::PlanView pv = plan_view(p);
    pv.en = bd::EnergyArgs{M, p->partial_f, reinterpret_cast<unsigned*>(p->partial_f + kFusedEnergySlots), E_dev,
                           -0.5 * (4e-7 * bd::kPi) * p->hx * p->hy * p->hz};
    const int rc = bd::enqueue_apply(run, pv, M, H);
    if (rc == -2) return cuda_fail(run.err, "kernel launch");
    if (rc) return fail(rc, "unsupported size");
    if (p->padmode) return stage(p, false, p->Hp, Hu, (cudaStream_t)stream);
    return 0;
}

int boris_demag_apply_ex(boris_demag_plan* p, const float* M, float* H, unsigned flags, void* stream) {
    if (!p || !M || !H) return fail(-1, "null argument");
    if (M == H) return fail(-1, "M and H must not alias");
    if (flags & ~(unsigned)(BORIS_DEMAG_AOS | BORIS_DEMAG_ACCUMULATE)) return fail(-1, "unknown flag");
    if (flags == 0) return boris_demag_apply(p, M, H, stream);
    if (flags == BORIS_DEMAG_ACCUMULATE && !p->padmode && (p->cfg.tiled || p->cfg.plane.on)) {
        // planar fields on a mesh the tiled / plane kernels take as it is: the kernel that writes H adds to it
        if (int rc = check_fields(p, M, H, false)) return rc;
        CudaLauncher run{(cudaStream_t)stream, p->device};
        bd::PlanView pv = plan_view(p);
        pv.en.accumulate = 1;
        const int rc = bd::enqueue_apply(run, pv, M, H);
        if (rc == -2) return cuda_fail(run.err, "kernel launch");
        if (rc) return fail(rc, "unsupported size");
        return 0;
    }
    if (((uintptr_t)M | (uintptr_t)H) & 3) return fail(-1, "M and H must be 4-byte aligned");
    if (int rc = check_device(p)) return rc;
    if (!p->Mp || !p->Hp) {      // first use of a staged variant on a power-of-two mesh: both buffers or neither
        const size_t np = (size_t)3 * p->nx * p->ny * p->nz;
        float *mp = nullptr, *hp = nullptr;
        int rc = dev_alloc(p, &mp, np);
        if (!rc) rc = dev_alloc(p, &hp, np);
        if (!rc && cudaMemset(mp, 0, np * sizeof(float)) != cudaSuccess) rc = fail(-2, "cudaMemset");
        if (rc) { cudaFree(mp); cudaFree(hp); return rc; }
        p->Mp = mp; p->Hp = hp;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const bool aos = (flags & BORIS_DEMAG_AOS) != 0, acc = (flags & BORIS_DEMAG_ACCUMULATE) != 0;
    if (int rc = stage(p, true, M, p->Mp, st, aos)) return rc;
    CudaLauncher run{st, p->device};
    const bd::PlanView pv = plan_view(p);
    const int rc = bd::enqueue_apply(run, pv, p->Mp, p->Hp);
    if (rc == -2) return cuda_fail(run.err, "kernel launch");
    if (rc) return fail(rc, "unsupported size");
    return stage(p, false, p->Hp, H, st, aos, acc);
}

int boris_demag_apply_timed(boris_demag_plan* p, const float* M, float* H, void* stream, float ms_by_kind[6],
                            int launches_by_kind[6]) {
    if (!ms_by_kind || !launches_by_kind) return fail(-1, "null argument");
    if (int rc = check_fields(p, M, H, false)) return rc;
    float* Hu = H;
    std::vector<TimedLaunch> timed;
    auto timed_stage = [&](bool in, const float* src, float* dst, int kind) {
        TimedLaunch t{kind, nullptr, nullptr};
        if (cudaEventCreate(&t.t0) != cudaSuccess) return fail(-2, "cudaEventCreate");
        if (cudaEventCreate(&t.t1) != cudaSuccess) { cudaEventDestroy(t.t0); return fail(-2, "cudaEventCreate"); }
        timed.push_back(t);
        cudaEventRecord(t.t0, (cudaStream_t)stream);
        const int rc = stage(p, in, src, dst, (cudaStream_t)stream);
        cudaEventRecord(t.t1, (cudaStream_t)stream);
        return rc;
    };
    int rc = 0;
    if (p->padmode) {            // the staging copies count with the x kernels they feed (kinds 0 and 5)
        rc = timed_stage(true, M, p->Mp, 0);
        M = p->Mp; H = p->Hp;
    }
    CudaLauncher run{(cudaStream_t)stream, p->device};
    run.timed = &timed;
    run.pdl = false;             // every kernel alone between its two events
    const bd::PlanView pv = plan_view(p);
    if (!rc) rc = bd::enqueue_apply(run, pv, M, H);
    if (!rc && p->padmode) rc = timed_stage(false, p->Hp, Hu, 5);
    cudaError_t e = cudaStreamSynchronize((cudaStream_t)stream);
    for (int k = 0; k < bd::kNumKinds; ++k) { ms_by_kind[k] = 0.f; launches_by_kind[k] = 0; }
    for (const TimedLaunch& t : timed) {
        float ms = 0.f;
        if (rc == 0 && e == cudaSuccess && cudaEventElapsedTime(&ms, t.t0, t.t1) == cudaSuccess) {
            ms_by_kind[t.kind] += ms;
            launches_by_kind[t.kind] += 1;
        }
        cudaEventDestroy(t.t0); cudaEventDestroy(t.t1);
    }
    if (rc == -2) return cuda_fail(run.err, "kernel launch");
    if (rc) return fail(rc, "unsupported size");
    if (e != cudaSuccess) return cuda_fail(e, "cudaStreamSynchronize");
    return 0;
}

int boris_demag_energy(boris_demag_plan* p, const float* M, const float* H, double* E_dev, void* stream) {
    if (!E_dev) return fail(-1, "null argument");
    if (int rc = check_fields(p, M, H, true)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (p->padmode) {            // sum over the staged copies: the empty cells of Mp add nothing
        if (int rc = stage(p, true, M, p->Mp, st)) return rc;
        if (int rc = stage(p, true, H, p->Hp, st)) return rc;
        M = p->Mp; H = p->Hp;
    }
    const long n4 = 3L * p->nx * p->ny * p->nz / 4;
    const double factor = -0.5 * (4e-7 * bd::kPi) * p->hx * p->hy * p->hz;
    long nblk = (n4 + (long)kEnergyUnroll * kEnergyThreads - 1) / ((long)kEnergyUnroll * kEnergyThreads);   // fixed per plan: E stays reproducible
    nblk = nblk < 1 ? 1 : (nblk > kEnergyBlocks ? kEnergyBlocks : nblk);
    k_energy_partial<<<(unsigned)nblk, kEnergyThreads, 0, st>>>((const float4*)M, (const float4*)H, n4, p->partial,
                                                               reinterpret_cast<unsigned*>(p->partial + kEnergyBlocks), factor, E_dev);
    BD_CUDA(cudaGetLastError());
    return 0;
}

int boris_demag_apply_host(boris_demag_plan* p, const float* M_host, float* H_host, double* E_host, void* stream) {
    if (!p || !M_host || !H_host) return fail(-1, "null argument");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)3 * p->ux * p->uy * p->uz;
    if (!p->stage_M) {
        if (int rc = dev_alloc(p, &p->stage_M, n)) return rc;
        if (int rc = dev_alloc(p, &p->stage_H, n)) return rc;
        if (int rc = dev_alloc(p, &p->stage_E, 1)) return rc;
    }
    BD_CUDA(cudaMemcpyAsync(p->stage_M, M_host, n * sizeof(float), cudaMemcpyHostToDevice, st));
    if (E_host) {
        if (int rc = boris_demag_apply_energy(p, p->stage_M, p->stage_H, p->stage_E, stream)) return rc;
        BD_CUDA(cudaMemcpyAsync(E_host, p->stage_E, sizeof(double), cudaMemcpyDeviceToHost, st));
    } else {
        if (int rc = boris_demag_apply(p, p->stage_M, p->stage_H, stream)) return rc;
    }
    BD_CUDA(cudaMemcpyAsync(H_host, p->stage_H, n * sizeof(float), cudaMemcpyDeviceToHost, st));
    BD_CUDA(cudaStreamSynchronize(st));
    return 0;
}

int boris_demag_plan_info(const boris_demag_plan* p, long long* compulsory_bytes, long long* designed_hbm_bytes,
                          long long* workspace_bytes, int padded[3], int* kernel_launches) {
    if (!p) return fail(-1, "null plan");
    const bd::KLayout& kl = p->kl;
    const long long N = (long long)p->nx * p->ny * p->nz;
    const long long kred = 4LL * kl.ncomp * kl.nxr() * kl.nyr() * kl.nzr();
    const long long wbytes = 3LL * kl.nxr() * p->nz * p->ny * (long long)sizeof(float2);
    if (compulsory_bytes) *compulsory_bytes = 24 * N + kred;
    if (compulsory_bytes && p->padmode)      // of the caller's mesh: its cells and the reduced spectrum of its own 2n padding
        *compulsory_bytes = 24LL * p->ux * p->uy * p->uz +
                            4LL * kl.ncomp * (p->ux + 1) * (p->uy + 1) * (p->uz > 1 ? p->uz + 1 : 1);
    // M in, W out | W in, stored spectrum in, W out | W in, H out.  The scratch T of the
    // 3-D path is sized to stay in L2 and is not counted.
    if (designed_hbm_bytes) *designed_hbm_bytes = 24 * N + 4 * wbytes + 4LL * kl.storage_elems();
    if (designed_hbm_bytes && p->cfg.tiled) {
        // M in, V out | V in, stored spectrum in, V out | V in, H out
        const long long vbytes = 3LL * kl.Pz * kl.ntl * p->ny * kl.cols * (long long)sizeof(float2);
        *designed_hbm_bytes = 24 * N + 4 * vbytes + 4LL * kl.storage_elems();
    }
    if (designed_hbm_bytes && p->cfg.plane.on) {
        // M in, X out | X in, stored spectrum in, P out | P in, H out
        const bd::PlaneGeom& g = p->cfg.plane;
        const long long xb = 3LL * p->nz * (p->nx + 1) * p->ny * (long long)sizeof(float2);
        const long long pb = (long long)g.nq * 3 * p->nz * (p->nx + 1) * g.lsp * (long long)sizeof(float2);
        *designed_hbm_bytes = 24 * N + 2 * xb + 2 * pb + 4LL * bd::make_plane_k(p->nx, p->ny, p->nz, g).storage_elems();
    }
    if (designed_hbm_bytes && p->padmode) *designed_hbm_bytes += 48LL * p->ux * p->uy * p->uz;   // staging in and out
    if (workspace_bytes) *workspace_bytes = p->bytes;
    if (padded) { padded[0] = kl.Px; padded[1] = kl.Py; padded[2] = kl.Pz; }
    if (kernel_launches) *kernel_launches = bd::apply_launch_count(p->nx, p->nz, p->cfg) + (p->padmode ? 2 : 0);
    return 0;
}

int boris_demag_plan_mesh(const boris_demag_plan* p, int cells[3], double sides[3]) {
    if (!p) return fail(-1, "null plan");
    if (cells) { cells[0] = p->ux; cells[1] = p->uy; cells[2] = p->uz; }
    if (sides) { sides[0] = p->hx; sides[1] = p->hy; sides[2] = p->hz; }
    return 0;
}

int boris_demag_plan_layout(const boris_demag_plan* p, int* path, long long* spectrum_bytes,
                            long long* kernel_storage_bytes, int* cols) {
    if (!p) return fail(-1, "null plan");
    const bd::KLayout& kl = p->kl;
    if (p->cfg.plane.on) {
        const bd::PlaneGeom& g = p->cfg.plane;
        if (path) *path = 4;
        if (spectrum_bytes) *spectrum_bytes = 3LL * p->nz * (p->nx + 1) * p->ny * (long long)sizeof(float2);
        if (kernel_storage_bytes) *kernel_storage_bytes = 4LL * bd::make_plane_k(p->nx, p->ny, p->nz, g).storage_elems();
        if (cols) *cols = g.nq;
        return 0;
    }
    if (path) *path = p->cfg.tiled ? (p->nz == 1 ? 2 : 3) : 0;
    if (spectrum_bytes)
        *spectrum_bytes = p->cfg.tiled ? 3LL * kl.Pz * kl.ntl * p->ny * kl.cols * (long long)sizeof(float2)
                                       : 3LL * kl.nxr() * p->nz * p->ny * (long long)sizeof(float2);
    if (kernel_storage_bytes) *kernel_storage_bytes = 4LL * kl.storage_elems();
    if (cols) *cols = p->cfg.tiled ? kl.cols : 0;
    return 0;
}

int boris_demag_plan_kernel_spectrum(const boris_demag_plan* p, float* out_host) {
    if (!p || !out_host) return fail(-1, "null argument");
    const long n = p->kl.reduced_elems();
    float* d = nullptr;
    BD_CUDA(cudaMalloc((void**)&d, (size_t)n * sizeof(float)));
    if (p->cfg.plane.on)
        k_gather_plane<<<grid_for(n, 256), 256>>>(p->KP, bd::make_plane_k(p->nx, p->ny, p->nz, p->cfg.plane), p->kidx, d);
    else
        k_gather_natural<<<grid_for(n, 256), 256>>>(p->Kst, p->kl, d);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpy(out_host, d, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(e, "kernel spectrum read-back");
    return 0;
}

// ---- host-only entry points ----------------------------------------------------------
int boris_demag_tensor_host(int nx, int ny, int nz, double hx, double hy, double hz, double* out) {
    return boris_demag_tensor_host_pbc(nx, ny, nz, hx, hy, hz, 0, 0, 0, out);
}

int boris_demag_tensor_host_pbc(int nx, int ny, int nz, double hx, double hy, double hz, int images_x, int images_y,
                                int images_z, double* out) {
    if (!out || nx < 1 || ny < 1 || nz < 1 || !(hx > 0) || !(hy > 0) || !(hz > 0) || images_x < 0 || images_y < 0 ||
        images_z < 0)
        return fail(-1, "invalid argument");
    const long cells = (long)nx * ny * nz;
    const int per[3] = {nx, ny, nz}, img[3] = {images_x, images_y, images_z};
    for (long idx = 0; idx < cells; ++idx) {
        const int i = (int)(idx % nx), j = (int)((idx / nx) % ny), k = (int)(idx / ((long)nx * ny));
        double v[6];
        bd::tensor_point_images(i, j, k, per, img, hx, hy, hz, v);
        for (int c = 0; c < 6; ++c) out[c * cells + idx] = v[c];
    }
    return 0;
}

int boris_demag_spectrum_host(int nx, int ny, int nz, double hx, double hy, double hz, double* out) {
    if (!out || nx < 1 || ny < 1 || nz < 1 || !(hx > 0) || !(hy > 0) || !(hz > 0)) return fail(-1, "invalid argument");
    const int nc = nz > 1 ? 6 : 4;
    const int nxr = nx + 1, nyr = ny + 1, nzr = nz > 1 ? nz + 1 : 1;
    const long cells = (long)nx * ny * nz;
    std::vector<double> N6((size_t)6 * cells);
    boris_demag_tensor_host(nx, ny, nz, hx, hy, hz, N6.data());
    auto table = [](int P) {
        std::vector<double2> t((size_t)P);
        for (int m = 0; m < P; ++m) {
            const double a = 2.0 * bd::kPi * m / P;
            t[m].x = std::cos(a); t[m].y = std::sin(a);
        }
        return t;
    };
    const auto csx = table(2 * nx), csy = table(2 * ny), csz = table(nz > 1 ? 2 * nz : 2);
    std::vector<double> A((size_t)nc * nz * ny * nxr), B((size_t)nc * nz * nyr * nxr);
    for (int c = 0; c < nc; ++c)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int kx = 0; kx < nxr; ++kx)
                    A[(((size_t)c * nz + k) * ny + j) * nxr + kx] =
                        bd::real_transform(&N6[(((size_t)c * nz + k) * ny + j) * nx], 1, nx, kx, bd::comp_is_odd(c, 0), csx.data());
    for (int c = 0; c < nc; ++c)
        for (int k = 0; k < nz; ++k)
            for (int ky = 0; ky < nyr; ++ky)
                for (int kx = 0; kx < nxr; ++kx)
                    B[(((size_t)c * nz + k) * nyr + ky) * nxr + kx] =
                        bd::real_transform(&A[(((size_t)c * nz + k) * ny) * nxr + kx], nxr, ny, ky, bd::comp_is_odd(c, 1), csy.data());
    const double scale = -1.0 / (2.0 * (2.0 * nx) * (2.0 * ny) * (nz > 1 ? 2.0 * nz : 1.0));
    for (int c = 0; c < nc; ++c)
        for (int kz = 0; kz < nzr; ++kz)
            for (int ky = 0; ky < nyr; ++ky)
                for (int kx = 0; kx < nxr; ++kx)
                    out[(((size_t)c * nzr + kz) * nyr + ky) * nxr + kx] =
                        (c >= 3 ? -scale : scale) *
                        bd::real_transform(&B[(((size_t)c * nz) * nyr + ky) * nxr + kx], (long)nyr * nxr, nz, kz, bd::comp_is_odd(c, 2), csz.data());
    return 0;
}

}  // extern "C"
