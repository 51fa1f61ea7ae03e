// boris_demag_f64.cu — the double-precision variant of the demag convolution (include/boris_demag_f64.h;
// SURVEY.md section 8(f) NEXT-4; "either with single or double floating point precision").
//
// Same method as the fp32 engine — zero-padded convolution with the real, symmetry-reduced kernel spectrum
// of the plan-time code of boris_demag.cu (which is fp64 already) — organised exactly as PAPER.md:L275 words
// the pipelined convolution: x FFTs, y FFTs, then ONE launch that runs the z FFT, the point-by-point tensor
// multiplication and the inverse z FFT for all three components (the z-padded spectrum exists only in shared
// memory), then inverse y and inverse x FFTs: five launches.
//
//   x_fwd       S1     M [3][uz][uy][ux] real  -> X[3][nz][ny][nx+1]            (simple_engine.cuh; zero padding on load)
//   y_pass<fwd> S2     X -> Y[3][nz][Py][nx+1]                                   (y in bit-reversed order)
//   k64_z_mul   S3-S5  Y -> Y in place, per (ky, kx): z FFT, H^ = K^ M^, inverse z FFT, first nz kept   (this file)
//   y_pass<inv> S6     Y -> X, first ny kept
//   x_inv       S7     X -> H, Hermitian half spectrum -> real row, first ux kept
//
// Transforms: in-place radix-2 in shared memory, decimation in frequency forward (natural -> bit-reversed),
// decimation in time inverse (bit-reversed -> natural): nothing is reordered, the multiply looks the frequency of
// a position up by bit reversal.  Twiddles from fp64 tables.  A mesh that is not a power of two sits in the corner
// of the next power-of-two mesh (M = 0 elsewhere), as in the fp32 engine — here the first and last kernels read
// and write the caller's mesh directly.  FP64 is not the fast path of this chip; the variant exists for
// accuracy, not speed.
#include <cuda_runtime.h>

#include <cmath>
#include <new>
#include <vector>

#include "../../include/boris_demag_f64.h"
#include "simple_engine.cuh"

namespace bd {
int micro_fail(cudaError_t e, const char* what);
int set_error(int code, const char* msg);
void clear_error();
int build_reduced_spectrum(int nx, int ny, int nz, double hx, double hy, double hz, const int per[3], const int img[3],
                           double** out);
int check_mesh_args(int nx, int ny, int nz, double hx, double hy, double hz);
}  // namespace bd

namespace {

using namespace se;
constexpr double kPi64 = 3.14159265358979323846264338327950288;

// S3 + S4 + S5 (the pipelined step of PAPER.md:L275): block = tc consecutive kx at one y position, all 3 components.
// Kred[c][kz <= Pz/2][ky <= Py/2][kx]: real, with -1/(2 Px Py Pz) folded in (x 2 here: these are plain complex
// transforms, reading R12); a mirrored frequency reads the stored value with the sign of the odd components.
__global__ void __launch_bounds__(kThreads) k64_z_mul(double2* __restrict__ Y, const double* __restrict__ Kred, Geo g, int tc,
                                                      const double2* __restrict__ twz) {
    double2* sm64 = smem<double>();
    const int tiles = (g.nxr + tc - 1) / tc;
    const int pos_y = blockIdx.x / tiles, k0 = (blockIdx.x - pos_y * tiles) * tc;
    const int cols = min(tc, g.nxr - k0);
    const size_t zstride = (size_t)g.Py * g.nxr, cstride = zstride * g.nz;
    double2* base = Y + (size_t)pos_y * g.nxr + k0;
    // shared: s[c][col][Pz]
    for (int w = threadIdx.x; w < 3 * g.Pz * tc; w += blockDim.x) {
        const int col = w % tc, e = (w / tc) % g.Pz, c = w / (tc * g.Pz);
        sm64[((size_t)c * tc + col) * g.Pz + e] =
            (e < g.nz && col < cols) ? base[c * cstride + e * zstride + col] : make_double2(0.0, 0.0);
    }
    __syncthreads();
    if (g.Pz > 1) fft_dif(sm64, g.Pz, g.lz, 3 * tc, twz);
    const int ky = bitrev(pos_y, g.ly);
    const bool ymir = 2 * ky > g.Py;
    const int kyr = ymir ? g.Py - ky : ky;
    const double sy = ymir ? -1.0 : 1.0;
    const int nyr = g.ny + 1, nzr = g.nz > 1 ? g.nz + 1 : 1;
    const size_t kcs = (size_t)nzr * nyr * g.nxr;
    for (int w = threadIdx.x; w < g.Pz * tc; w += blockDim.x) {
        const int col = w % tc, e = w / tc;
        if (col >= cols) continue;
        const int kz = bitrev(e, g.lz);
        const bool zmir = 2 * kz > g.Pz;
        const int kzr = zmir ? g.Pz - kz : kz;
        const double sz = zmir ? -1.0 : 1.0;
        const double* kp = Kred + ((size_t)kzr * nyr + kyr) * g.nxr + k0 + col;
        const double kxx = 2.0 * kp[0], kyy = 2.0 * kp[kcs], kzz = 2.0 * kp[2 * kcs], kxy = 2.0 * sy * kp[3 * kcs];
        double kxz = 0.0, kyz = 0.0;
        if (g.nz > 1) { kxz = 2.0 * sz * kp[4 * kcs]; kyz = 2.0 * sy * sz * kp[5 * kcs]; }
        double2* px = sm64 + ((size_t)0 * tc + col) * g.Pz + e;
        double2* py = sm64 + ((size_t)1 * tc + col) * g.Pz + e;
        double2* pz = sm64 + ((size_t)2 * tc + col) * g.Pz + e;
        const double2 mx = *px, my = *py, mz = *pz;
        *px = make_double2(kxx * mx.x + kxy * my.x + kxz * mz.x, kxx * mx.y + kxy * my.y + kxz * mz.y);
        *py = make_double2(kxy * mx.x + kyy * my.x + kyz * mz.x, kxy * mx.y + kyy * my.y + kyz * mz.y);
        *pz = make_double2(kxz * mx.x + kyz * my.x + kzz * mz.x, kxz * mx.y + kyz * my.y + kzz * mz.y);
    }
    __syncthreads();
    if (g.Pz > 1) fft_dit_inv(sm64, g.Pz, g.lz, 3 * tc, twz);
    for (int w = threadIdx.x; w < 3 * g.nz * tc; w += blockDim.x) {
        const int col = w % tc, e = (w / tc) % g.nz, c = w / (tc * g.nz);
        if (col < cols) base[c * cstride + e * zstride + col] = sm64[((size_t)c * tc + col) * g.Pz + e];
    }
}

int upload_tw(double2** dst, int L) {
    const int n = L > 1 ? L / 2 : 1;
    std::vector<double2> h((size_t)n);
    for (int k = 0; k < n; ++k) {
        const double a = -2.0 * kPi64 * (double)k / (double)L;
        h[k] = make_double2(std::cos(a), std::sin(a));
        if (k == 0) h[k] = make_double2(1.0, 0.0);
        if (4 * k == L) h[k] = make_double2(0.0, -1.0);
    }
    cudaError_t e = cudaMalloc((void**)dst, (size_t)n * sizeof(double2));
    if (e == cudaSuccess) e = cudaMemcpy(*dst, h.data(), (size_t)n * sizeof(double2), cudaMemcpyHostToDevice);
    return e == cudaSuccess ? 0 : bd::micro_fail(e, "twiddle table");
}

}  // namespace

struct boris_demag_f64_plan {
    Geo g;
    double hx, hy, hz;
    int device;
    int tc_y, tc_z;                  // kx columns per block of the y / z kernels
    size_t smem_x, smem_y, smem_z;
    double* Kred = nullptr;
    double2 *twx = nullptr, *twy = nullptr, *twz = nullptr;
    double2 *X = nullptr, *Y = nullptr;
    double* partial = nullptr;       // energy partial sums + ticket
    long long bytes = 0;
};

extern "C" {

void boris_demag_f64_plan_destroy(boris_demag_f64_plan* p) {
    if (!p) return;
    cudaFree(p->Kred); cudaFree(p->twx); cudaFree(p->twy); cudaFree(p->twz); cudaFree(p->X); cudaFree(p->Y); cudaFree(p->partial);
    delete p;
}

boris_demag_f64_plan* boris_demag_f64_plan_create(int ux, int uy, int uz, double hx, double hy, double hz, int images_x,
                                                  int images_y, int images_z) {
    bd::clear_error();
    if (bd::check_mesh_args(ux, uy, uz, hx, hy, hz)) return nullptr;
    if (images_x < 0 || images_y < 0 || images_z < 0 || images_x > 1000 || images_y > 1000 || images_z > 1000) {
        bd::set_error(-1, "images per side must be in [0, 1000]");
        return nullptr;
    }
    int dev = 0;
    if (cudaError_t e = cudaGetDevice(&dev); e != cudaSuccess) {
        bd::micro_fail(e, "cudaGetDevice (no CUDA device: this library has no CPU fallback)");
        return nullptr;
    }
    boris_demag_f64_plan* p = new (std::nothrow) boris_demag_f64_plan();
    if (!p) { bd::set_error(-3, "out of host memory"); return nullptr; }
    Geo& g = p->g;
    g.ux = ux; g.uy = uy; g.uz = uz;
    g.nx = next_pow2(ux < 4 ? 4 : ux); g.ny = next_pow2(uy < 2 ? 2 : uy); g.nz = uz == 1 ? 1 : next_pow2(uz);
    g.Px = 2 * g.nx; g.Py = 2 * g.ny; g.Pz = g.nz > 1 ? 2 * g.nz : 1;
    g.lx = ilog2(g.Px); g.ly = ilog2(g.Py); g.lz = ilog2(g.Pz);
    g.nxr = g.nx + 1;
    p->hx = hx; p->hy = hy; p->hz = hz; p->device = dev;
    // columns per block: as many as fit ~128 KB (y) / ~96 KB (z) of shared memory, at most 16
    p->tc_y = 8192 / g.Py; if (p->tc_y > 16) p->tc_y = 16; if (p->tc_y < 1) p->tc_y = 1;
    p->tc_z = 2048 / g.Pz; if (p->tc_z > 16) p->tc_z = 16; if (p->tc_z < 1) p->tc_z = 1;
    p->smem_x = (size_t)g.Px * sizeof(double2);
    p->smem_y = (size_t)p->tc_y * g.Py * sizeof(double2);
    p->smem_z = (size_t)3 * p->tc_z * g.Pz * sizeof(double2);
    const int per[3] = {ux, uy, uz}, img[3] = {images_x, images_y, images_z};
    int rc = bd::build_reduced_spectrum(g.nx, g.ny, g.nz, hx, hy, hz, per, img, &p->Kred);
    if (!rc) rc = upload_tw(&p->twx, g.Px);
    if (!rc) rc = upload_tw(&p->twy, g.Py);
    if (!rc) rc = upload_tw(&p->twz, g.Pz);
    const size_t nX = (size_t)3 * g.nz * g.ny * g.nxr, nY = (size_t)3 * g.nz * g.Py * g.nxr;
    auto alloc = [&](void** ptr, size_t bytes) {
        if (rc) return;
        cudaError_t e = cudaMalloc(ptr, bytes);
        if (e != cudaSuccess) { *ptr = nullptr; rc = bd::micro_fail(e, "cudaMalloc"); if (e == cudaErrorMemoryAllocation) rc = -3; }
        else p->bytes += (long long)bytes;
    };
    alloc((void**)&p->X, nX * sizeof(double2));
    alloc((void**)&p->Y, nY * sizeof(double2));
    alloc((void**)&p->partial, (kEnergyBlocks + 1) * sizeof(double));
    if (!rc && cudaMemset(p->partial, 0, (kEnergyBlocks + 1) * sizeof(double)) != cudaSuccess) rc = bd::set_error(-2, "cudaMemset");
    auto optin = [&](const void* f, size_t smem) {
        if (rc || smem <= 48 * 1024) return;
        if (smem > kMaxSmem) { rc = bd::set_error(-1, "mesh too large for the fp64 engine's shared-memory tiles"); return; }
        if (cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); e != cudaSuccess)
            rc = bd::micro_fail(e, "cudaFuncSetAttribute");
    };
    optin((const void*)x_fwd<double>, p->smem_x);
    optin((const void*)x_inv<double>, p->smem_x);
    optin((const void*)y_pass<double, false>, p->smem_y);
    optin((const void*)y_pass<double, true>, p->smem_y);
    optin((const void*)k64_z_mul, p->smem_z);
    if (rc) { boris_demag_f64_plan_destroy(p); return nullptr; }
    return p;
}

int boris_demag_f64_apply(boris_demag_f64_plan* p, const double* M, double* H, void* stream) {
    if (!p || !M || !H) return bd::set_error(-1, "null argument");
    if (M == H) return bd::set_error(-1, "M and H must not alias");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device)
        return bd::set_error(-1, "the current CUDA device is not the one the plan was created on");
    cudaStream_t st = (cudaStream_t)stream;
    const Geo& g = p->g;
    const int rows = 3 * g.nz * g.ny;
    const int ytiles = (g.nxr + p->tc_y - 1) / p->tc_y, ztiles = (g.nxr + p->tc_z - 1) / p->tc_z;
    x_fwd<double><<<rows, kThreads, p->smem_x, st>>>(M, p->X, g, p->twx);
    y_pass<double, false><<<3 * g.nz * ytiles, kThreads, p->smem_y, st>>>(p->X, p->Y, g, p->tc_y, p->twy);
    k64_z_mul<<<g.Py * ztiles, kThreads, p->smem_z, st>>>(p->Y, p->Kred, g, p->tc_z, p->twz);
    y_pass<double, true><<<3 * g.nz * ytiles, kThreads, p->smem_y, st>>>(p->X, p->Y, g, p->tc_y, p->twy);
    x_inv<double><<<rows, kThreads, p->smem_x, st>>>(p->X, H, g, p->twx);
    if (cudaError_t e = cudaGetLastError(); e != cudaSuccess) return bd::micro_fail(e, "fp64 kernel launch");
    return 0;
}

int boris_demag_f64_energy(boris_demag_f64_plan* p, const double* M, const double* H, double* E_dev, void* stream) {
    if (!p || !M || !H || !E_dev) return bd::set_error(-1, "null argument");
    const size_t n = (size_t)3 * p->g.ux * p->g.uy * p->g.uz;
    size_t nblk = (n + 4 * kThreads - 1) / (4 * kThreads);
    nblk = nblk < 1 ? 1 : (nblk > (size_t)kEnergyBlocks ? (size_t)kEnergyBlocks : nblk);
    const double factor = -0.5 * (4e-7 * kPi64) * p->hx * p->hy * p->hz;
    energy<double><<<(unsigned)nblk, kThreads, 0, (cudaStream_t)stream>>>(M, H, n, n, 1, nullptr, p->partial,
                                                                         reinterpret_cast<unsigned*>(p->partial + kEnergyBlocks), factor, E_dev);
    if (cudaError_t e = cudaGetLastError(); e != cudaSuccess) return bd::micro_fail(e, "k64_energy");
    return 0;
}

int boris_demag_f64_plan_info(const boris_demag_f64_plan* p, long long* workspace_bytes, int padded[3], int* kernel_launches) {
    if (!p) return bd::set_error(-1, "null plan");
    if (workspace_bytes) *workspace_bytes = p->bytes;
    if (padded) { padded[0] = p->g.Px; padded[1] = p->g.Py; padded[2] = p->g.Pz; }
    if (kernel_launches) *kernel_launches = 5;
    return 0;
}

}  // extern "C"
