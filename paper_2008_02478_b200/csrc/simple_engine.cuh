// simple_engine.cuh — precision-generic transform kernels of the double-precision variant
// (boris_demag_f64.cu) and of the multi-layered convolution (boris_demag_ml.cu).
//
// "1D FFTs along the x, y, z directions ... multiplication ... z, y, x inverse 1D FFTs".  These are
// the plain kernels of that sequence, templated on the real type T (float / double): in-place radix-2 transforms in
// shared memory, decimation in frequency forward (natural -> bit-reversed order), decimation in time inverse
// (bit-reversed -> natural): nothing is reordered, a multiply looks the frequency of a position up by bit
// reversal.  Twiddles come from tables rounded once from fp64.  They are correctness-first kernels: the tuned
// fp32 path of the single mesh is the one in xt.h / yfused.h / plane.h.
#pragma once
#include <cuda_runtime.h>

namespace se {

template <class T> struct Cx;
template <> struct Cx<double> { using type = double2; };
template <> struct Cx<float> { using type = float2; };
template <class T> using C2 = typename Cx<T>::type;
template <class T> __device__ __forceinline__ C2<T> mk(T x, T y) { C2<T> r; r.x = x; r.y = y; return r; }

template <class C> __device__ __forceinline__ C c_add(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <class C> __device__ __forceinline__ C c_sub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
template <class C> __device__ __forceinline__ C c_mul(C a, C w) { C r; r.x = a.x * w.x - a.y * w.y; r.y = a.x * w.y + a.y * w.x; return r; }
template <class C> __device__ __forceinline__ C c_mulc(C a, C w) { C r; r.x = a.x * w.x + a.y * w.y; r.y = a.y * w.x - a.x * w.y; return r; }

constexpr int kThreads = 256;

template <class T>
__device__ __forceinline__ C2<T>* smem() {
    extern __shared__ __align__(16) unsigned char se_smem_raw[];
    return reinterpret_cast<C2<T>*>(se_smem_raw);
}

// `batch` pencils of L = 2^logL points, pencil b at s + b * L.  tw[k] = exp(-2 pi i k / L), k < L / 2.
template <class C>
__device__ void fft_dif(C* s, int L, int logL, int batch, const C* __restrict__ tw) {
    for (int st = 0; st < logL; ++st) {
        const int half = L >> (st + 1);
        for (int w = threadIdx.x; w < batch * (L / 2); w += blockDim.x) {
            const int b = w / (L / 2), r = w - b * (L / 2);
            const int g = r / half, j = r - g * half;
            C* p = s + (size_t)b * L + g * 2 * half + j;
            const C x0 = p[0], x1 = p[half];
            p[0] = c_add(x0, x1);
            p[half] = c_mul(c_sub(x0, x1), tw[j << st]);
        }
        __syncthreads();
    }
}
// inverse, unnormalised
template <class C>
__device__ void fft_dit_inv(C* s, int L, int logL, int batch, const C* __restrict__ tw) {
    for (int st = logL - 1; st >= 0; --st) {
        const int half = L >> (st + 1);
        for (int w = threadIdx.x; w < batch * (L / 2); w += blockDim.x) {
            const int b = w / (L / 2), r = w - b * (L / 2);
            const int g = r / half, j = r - g * half;
            C* p = s + (size_t)b * L + g * 2 * half + j;
            const C x0 = p[0], x1 = c_mulc(p[half], tw[j << st]);
            p[0] = c_add(x0, x1);
            p[half] = c_sub(x0, x1);
        }
        __syncthreads();
    }
}
__device__ __forceinline__ int bitrev(int v, int bits) { return bits == 0 ? 0 : (int)(__brev((unsigned)v) >> (32 - bits)); }

struct Geo {
    int ux, uy, uz;        // the caller's mesh (uz: layers of a stack)
    int nx, ny, nz;        // the power-of-two in-plane mesh the transforms work on; nz slabs (z cells or layers)
    int Px, Py, Pz, lx, ly, lz;   // padded lengths and their log2 (Pz = 1, lz = 0: no z transform)
    int nxr;               // nx + 1 frequencies along x
};

// S1: one block per row (c, z, y); M real [3][uz][uy][ux] -> X[3][nz][ny][nxr]
template <class T>
__global__ void __launch_bounds__(kThreads) x_fwd(const T* __restrict__ M, C2<T>* __restrict__ X, Geo g, const C2<T>* __restrict__ twx) {
    C2<T>* sm = smem<T>();
    const int row = blockIdx.x, y = row % g.ny, z = (row / g.ny) % g.nz, c = row / (g.ny * g.nz);
    C2<T>* out = X + (size_t)row * g.nxr;
    if (y >= g.uy || z >= g.uz) {                       // a row of the zero padding around the caller's mesh
        for (int k = threadIdx.x; k < g.nxr; k += blockDim.x) out[k] = mk<T>(0, 0);
        return;
    }
    const T* in = M + (((size_t)c * g.uz + z) * g.uy + y) * g.ux;
    for (int i = threadIdx.x; i < g.Px; i += blockDim.x) sm[i] = mk<T>(i < g.ux ? in[i] : T(0), T(0));
    __syncthreads();
    fft_dif(sm, g.Px, g.lx, 1, twx);
    for (int k = threadIdx.x; k < g.nxr; k += blockDim.x) out[k] = sm[bitrev(k, g.lx)];
}

// S7: Hermitian half spectrum -> real row
template <class T>
__global__ void __launch_bounds__(kThreads) x_inv(const C2<T>* __restrict__ X, T* __restrict__ H, Geo g, const C2<T>* __restrict__ twx) {
    C2<T>* sm = smem<T>();
    const int row = blockIdx.x, y = row % g.ny, z = (row / g.ny) % g.nz, c = row / (g.ny * g.nz);
    if (y >= g.uy || z >= g.uz) return;
    const C2<T>* in = X + (size_t)row * g.nxr;
    for (int k = threadIdx.x; k < g.nxr; k += blockDim.x) {
        C2<T> v = in[k];
        if (k == 0 || k == g.nx) v.y = T(0);              // DC and Nyquist of a real row are real
        sm[bitrev(k, g.lx)] = v;
        if (k > 0 && k < g.nx) sm[bitrev(g.Px - k, g.lx)] = mk<T>(v.x, -v.y);
    }
    __syncthreads();
    fft_dit_inv(sm, g.Px, g.lx, 1, twx);
    T* out = H + (((size_t)c * g.uz + z) * g.uy + y) * g.ux;
    for (int i = threadIdx.x; i < g.ux; i += blockDim.x) out[i] = sm[i].x;
}

// S2 / S6: block = tc consecutive kx of one (c, z); pencils along y (element stride nxr).
// X[3][nz][ny][nxr] <-> Y[3][nz][Py][nxr] (y in bit-reversed order)
template <class T, bool INV>
__global__ void __launch_bounds__(kThreads) y_pass(C2<T>* __restrict__ X, C2<T>* __restrict__ Y, Geo g, int tc, const C2<T>* __restrict__ twy) {
    C2<T>* sm = smem<T>();
    const int tiles = (g.nxr + tc - 1) / tc;
    const int cz = blockIdx.x / tiles, k0 = (blockIdx.x - cz * tiles) * tc;
    const int cols = min(tc, g.nxr - k0);
    C2<T>* x = X + (size_t)cz * g.ny * g.nxr + k0;
    C2<T>* yv = Y + (size_t)cz * g.Py * g.nxr + k0;
    if (!INV) {
        for (int w = threadIdx.x; w < g.Py * tc; w += blockDim.x) {
            const int e = w / tc, col = w - e * tc;
            sm[(size_t)col * g.Py + e] = (e < g.ny && col < cols) ? x[(size_t)e * g.nxr + col] : mk<T>(0, 0);
        }
        __syncthreads();
        fft_dif(sm, g.Py, g.ly, tc, twy);
        for (int w = threadIdx.x; w < g.Py * tc; w += blockDim.x) {
            const int e = w / tc, col = w - e * tc;
            if (col < cols) yv[(size_t)e * g.nxr + col] = sm[(size_t)col * g.Py + e];
        }
    } else {
        for (int w = threadIdx.x; w < g.Py * tc; w += blockDim.x) {
            const int e = w / tc, col = w - e * tc;
            sm[(size_t)col * g.Py + e] = col < cols ? yv[(size_t)e * g.nxr + col] : mk<T>(0, 0);
        }
        __syncthreads();
        fft_dit_inv(sm, g.Py, g.ly, tc, twy);
        for (int w = threadIdx.x; w < g.ny * tc; w += blockDim.x) {
            const int e = w / tc, col = w - e * tc;
            if (col < cols) x[(size_t)e * g.nxr + col] = sm[(size_t)col * g.Py + e];
        }
    }
}

// S8: fp64 sum of w[slab] M.H over [3][slabs][cells_per_slab] (w = nullptr: weight 1), two levels in one launch; the
// last block adds the partial sums in index order: bit-identical across calls
template <class T>
__global__ void __launch_bounds__(kThreads) energy(const T* __restrict__ M, const T* __restrict__ H, size_t n, size_t per_slab,
                                                   int slabs, const double* __restrict__ wslab, double* partial, unsigned* ticket,
                                                   double factor, double* E) {
    __shared__ double sh[kThreads];
    __shared__ bool last;
    double acc = 0.0;
    const size_t per = (n + gridDim.x - 1) / gridDim.x, lo = blockIdx.x * per, hi = lo + per < n ? lo + per : n;
    for (size_t i = lo + threadIdx.x; i < hi; i += blockDim.x) {
        const double w = wslab ? wslab[(i / per_slab) % slabs] : 1.0;
        acc += w * (double)M[i] * (double)H[i];
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = kThreads / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = sh[0];
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double tot = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) tot += __ldcg(&partial[i]);
    sh[threadIdx.x] = tot;
    __syncthreads();
    for (int o = kThreads / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) { *E = factor * sh[0]; *ticket = 0u; }
}

inline int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
inline int next_pow2(int n) { int p = 1; while (p < n) p <<= 1; return p; }
constexpr int kEnergyBlocks = 592;
constexpr size_t kMaxSmem = 200 * 1024;

}  // namespace se
