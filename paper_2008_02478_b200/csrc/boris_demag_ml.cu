// boris_demag_ml.cu — multi-layered convolution (include/boris_demag_ml.h; Eq. 4) for a film stack.
//
//   x_fwd        per layer and row: M [3][n][uy][ux] -> X[3][n][ny][nx+1]       (simple_engine.cuh)
//   y_pass<fwd>  X -> Y[3][n][Py][nx+1]
//   ml_mul       per (ky, kx): H^_k = sum_i K^_ki M^_i over all layer pairs — "summation of inter-mesh contributions
//                moved to the transform space" (L76) — in place on Y
//   y_pass<inv>, x_inv
//
// Kernel spectra (plan time, fp64): for every ORDERED pair (k, i) the in-plane tensor table N_c(i hx, j hy, z_k - z_i)
// of ml_math.h goes through the cosine / sine sums of plan_math.h.  At a fixed height difference xx, yy, zz are even in
// x and y, xy is odd in both (spectrum real, (-i)^2 = -1), xz is odd in x only and yz in y only (spectrum imaginary):
//     K^_xz = -i J_xz,  K^_yz = -i J_yz;   stored per pair: (xx, yy, zz, xy, J_xz, J_yz)[ky <= ny][kx <= nx], real,
// with -1/(Px Py) folded in; a mirrored ky reads the stored value with the sign of the y-odd components (xy, yz).
#include <cuda_runtime.h>

#include <cmath>
#include <new>
#include <vector>

#include "../../include/boris_demag_ml.h"
#include "ml_math.h"
#include "simple_engine.cuh"

namespace bd {
int micro_fail(cudaError_t e, const char* what);
int set_error(int code, const char* msg);
void clear_error();
}  // namespace bd

namespace {

using namespace se;
constexpr double kPiML = 3.14159265358979323846264338327950288;
constexpr int kMaxLayers = 32;

// ---- plan time (fp64)
__global__ void k_pair_tensor(double* T, int nx, int ny, double hx, double hy, double tk, double ti, double Z) {
    const long total = (long)nx * ny;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        double out[6];
        bd::pair_tensor_point((int)(idx % nx), (int)(idx / nx), Z, hx, hy, tk, ti, out);
        for (int c = 0; c < 6; ++c) T[c * total + idx] = out[c];
    }
}
// in[c][d1][d0] -> out[c][o1][o0], cosine / sine sums along dimension `dim` (n samples -> n + 1 frequencies)
__global__ void k_pair_transform(const double* in, double* out, int d0, int d1, int dim, const double2* cs) {
    const int n = dim == 0 ? d0 : d1, nk = n + 1;
    const int o0 = dim == 0 ? nk : d0, o1 = dim == 1 ? nk : d1;
    const long total = 6L * o1 * o0;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        const int a0 = (int)(idx % o0), a1 = (int)((idx / o0) % o1), c = (int)(idx / ((long)o0 * o1));
        const long base = ((long)c * d1 + (dim == 1 ? 0 : a1)) * d0 + (dim == 0 ? 0 : a0);
        out[idx] = bd::real_transform(in + base, dim == 0 ? 1 : d0, n, dim == 0 ? a0 : a1, bd::pair_comp_is_odd(c, dim), cs);
    }
}
// fold the (-i) factors and the normalisation; store in the plan's precision
template <class T>
__global__ void k_pair_store(const double* B, T* K, long per, double scale) {
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < 6 * per; idx += (long)gridDim.x * blockDim.x) {
        const int c = (int)(idx / per);
        // xy: (-i)^2 = -1.  xz, yz: one factor -i, kept as the real J with K^ = -i J
        K[idx] = (T)((c == 3 ? -scale : scale) * B[idx]);
    }
}

// ---- the multiply over layer pairs: block = tc consecutive kx at one y position; shared: m[c][layer][col]
template <class T>
__global__ void __launch_bounds__(kThreads) ml_mul(C2<T>* __restrict__ Y, const T* __restrict__ K, Geo g, int n, int tc) {
    C2<T>* sm = smem<T>();
    const int tiles = (g.nxr + tc - 1) / tc;
    const int pos_y = blockIdx.x / tiles, k0 = (blockIdx.x - pos_y * tiles) * tc;
    const int cols = min(tc, g.nxr - k0);
    const size_t lstride = (size_t)g.Py * g.nxr, cstride = lstride * g.nz;
    C2<T>* base = Y + (size_t)pos_y * g.nxr + k0;
    for (int w = threadIdx.x; w < 3 * n * tc; w += blockDim.x) {
        const int col = w % tc, l = (w / tc) % n, c = w / (tc * n);
        sm[w] = col < cols ? base[c * cstride + l * lstride + col] : mk<T>(0, 0);
    }
    __syncthreads();
    const int ky = bitrev(pos_y, g.ly);
    const bool ymir = 2 * ky > g.Py;
    const int kyr = ymir ? g.Py - ky : ky;
    const T sy = ymir ? T(-1) : T(1);
    const size_t per = (size_t)(g.ny + 1) * g.nxr;          // one component of one pair
    for (int w = threadIdx.x; w < n * tc; w += blockDim.x) {
        const int col = w % tc, k = w / tc;
        if (col >= cols) continue;
        C2<T> hx = mk<T>(0, 0), hy = mk<T>(0, 0), hz = mk<T>(0, 0);
        for (int i = 0; i < n; ++i) {
            const T* kp = K + ((size_t)(k * n + i) * 6) * per + (size_t)kyr * g.nxr + k0 + col;
            const T kxx = kp[0], kyy = kp[per], kzz = kp[2 * per], kxy = sy * kp[3 * per], jxz = kp[4 * per], jyz = sy * kp[5 * per];
            const C2<T> mx = sm[(0 * n + i) * tc + col], my = sm[(1 * n + i) * tc + col], mz = sm[(2 * n + i) * tc + col];
            // -i J (a + i b) = J b - i J a
            hx.x += kxx * mx.x + kxy * my.x + jxz * mz.y;  hx.y += kxx * mx.y + kxy * my.y - jxz * mz.x;
            hy.x += kxy * mx.x + kyy * my.x + jyz * mz.y;  hy.y += kxy * mx.y + kyy * my.y - jyz * mz.x;
            hz.x += jxz * mx.y + jyz * my.y + kzz * mz.x;  hz.y += -jxz * mx.x - jyz * my.x + kzz * mz.y;
        }
        base[0 * cstride + k * lstride + col] = hx;
        base[1 * cstride + k * lstride + col] = hy;
        base[2 * cstride + k * lstride + col] = hz;
    }
}

template <class T>
int upload_tw(C2<T>** dst, int L) {
    const int n = L > 1 ? L / 2 : 1;
    std::vector<C2<T>> h((size_t)n);
    for (int k = 0; k < n; ++k) {
        const double a = -2.0 * kPiML * (double)k / (double)L;
        double c = std::cos(a), s = std::sin(a);
        if (k == 0) { c = 1.0; s = 0.0; }
        if (4 * k == L) { c = 0.0; s = -1.0; }
        h[k].x = (T)c; h[k].y = (T)s;
    }
    cudaError_t e = cudaMalloc((void**)dst, (size_t)n * sizeof(C2<T>));
    if (e == cudaSuccess) e = cudaMemcpy(*dst, h.data(), (size_t)n * sizeof(C2<T>), cudaMemcpyHostToDevice);
    return e == cudaSuccess ? 0 : bd::micro_fail(e, "twiddle table");
}

int upload_cs(double2** dst, int P) {
    std::vector<double2> h((size_t)P);
    for (int m = 0; m < P; ++m) {
        const double a = 2.0 * kPiML * (double)m / (double)P;
        h[m].x = std::cos(a); h[m].y = std::sin(a);
        if ((4 * m) % P == 0) {
            const double cx[4] = {1, 0, -1, 0}, sy[4] = {0, 1, 0, -1};
            h[m].x = cx[(4 * m) / P % 4]; h[m].y = sy[(4 * m) / P % 4];
        }
    }
    cudaError_t e = cudaMalloc((void**)dst, (size_t)P * sizeof(double2));
    if (e == cudaSuccess) e = cudaMemcpy(*dst, h.data(), (size_t)P * sizeof(double2), cudaMemcpyHostToDevice);
    return e == cudaSuccess ? 0 : bd::micro_fail(e, "cosine table");
}

int grid_for(long total, int threads) {
    long g = (total + threads - 1) / threads;
    return (int)(g < 1 ? 1 : (g > 148L * 64 ? 148L * 64 : g));
}

}  // namespace

struct boris_demag_ml_plan {
    Geo g;
    int n, fp64, device;
    double hx, hy;
    std::vector<double> t, z;
    int tc_y, tc_m;
    size_t smem_x, smem_y, smem_m;
    void* K = nullptr;               // [n][n][6][ny+1][nx+1], T
    void *twx = nullptr, *twy = nullptr;
    void *X = nullptr, *Y = nullptr;
    double* wlayer = nullptr;        // thickness per layer (energy weights)
    double* partial = nullptr;
};

namespace {

template <class T>
int build(boris_demag_ml_plan* p) {
    const Geo& g = p->g;
    const int n = p->n;
    const long cells = (long)g.nx * g.ny, per = (long)(g.ny + 1) * g.nxr;
    double *dT = nullptr, *dA = nullptr, *dB = nullptr;
    double2 *csx = nullptr, *csy = nullptr;
    int rc = 0;
    auto fin = [&]() { cudaFree(dT); cudaFree(dA); cudaFree(dB); cudaFree(csx); cudaFree(csy); };
    auto ck = [&](cudaError_t e, const char* what) { if (!rc && e != cudaSuccess) rc = bd::micro_fail(e, what); };
    ck(cudaMalloc((void**)&dT, (size_t)6 * cells * sizeof(double)), "cudaMalloc");
    ck(cudaMalloc((void**)&dA, (size_t)6 * g.ny * g.nxr * sizeof(double)), "cudaMalloc");
    ck(cudaMalloc((void**)&dB, (size_t)6 * per * sizeof(double)), "cudaMalloc");
    ck(cudaMalloc(&p->K, (size_t)n * n * 6 * per * sizeof(T)), "cudaMalloc");
    if (!rc) rc = upload_cs(&csx, g.Px);
    if (!rc) rc = upload_cs(&csy, g.Py);
    const double scale = -1.0 / ((double)g.Px * (double)g.Py);
    for (int k = 0; k < n && !rc; ++k)
        for (int i = 0; i < n && !rc; ++i) {
            k_pair_tensor<<<grid_for(cells, 128), 128>>>(dT, g.nx, g.ny, p->hx, p->hy, p->t[k], p->t[i], p->z[k] - p->z[i]);
            k_pair_transform<<<grid_for(6L * g.ny * g.nxr, 128), 128>>>(dT, dA, g.nx, g.ny, 0, csx);
            k_pair_transform<<<grid_for(6 * per, 128), 128>>>(dA, dB, g.nxr, g.ny, 1, csy);
            k_pair_store<T><<<grid_for(6 * per, 256), 256>>>(dB, (T*)p->K + (size_t)(k * n + i) * 6 * per, per, scale);
            ck(cudaGetLastError(), "plan kernels");
        }
    ck(cudaDeviceSynchronize(), "plan kernels");
    fin();
    if (!rc) rc = upload_tw<T>((C2<T>**)&p->twx, g.Px);
    if (!rc) rc = upload_tw<T>((C2<T>**)&p->twy, g.Py);
    ck(cudaMalloc(&p->X, (size_t)3 * n * g.ny * g.nxr * sizeof(C2<T>)), "cudaMalloc");
    ck(cudaMalloc(&p->Y, (size_t)3 * n * g.Py * g.nxr * sizeof(C2<T>)), "cudaMalloc");
    auto optin = [&](const void* f, size_t smem) {
        if (rc || smem <= 48 * 1024) return;
        if (smem > kMaxSmem) { rc = bd::set_error(-1, "mesh too large for the multi-layer engine's shared-memory tiles"); return; }
        ck(cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "cudaFuncSetAttribute");
    };
    optin((const void*)x_fwd<T>, p->smem_x);
    optin((const void*)x_inv<T>, p->smem_x);
    optin((const void*)y_pass<T, false>, p->smem_y);
    optin((const void*)y_pass<T, true>, p->smem_y);
    optin((const void*)ml_mul<T>, p->smem_m);
    return rc;
}

template <class T>
int apply(boris_demag_ml_plan* p, const void* M, void* H, cudaStream_t st) {
    const Geo& g = p->g;
    const int rows = 3 * g.nz * g.ny;
    const int ytiles = (g.nxr + p->tc_y - 1) / p->tc_y, mtiles = (g.nxr + p->tc_m - 1) / p->tc_m;
    x_fwd<T><<<rows, kThreads, p->smem_x, st>>>((const T*)M, (C2<T>*)p->X, g, (const C2<T>*)p->twx);
    y_pass<T, false><<<3 * g.nz * ytiles, kThreads, p->smem_y, st>>>((C2<T>*)p->X, (C2<T>*)p->Y, g, p->tc_y, (const C2<T>*)p->twy);
    ml_mul<T><<<g.Py * mtiles, kThreads, p->smem_m, st>>>((C2<T>*)p->Y, (const T*)p->K, g, p->n, p->tc_m);
    y_pass<T, true><<<3 * g.nz * ytiles, kThreads, p->smem_y, st>>>((C2<T>*)p->X, (C2<T>*)p->Y, g, p->tc_y, (const C2<T>*)p->twy);
    x_inv<T><<<rows, kThreads, p->smem_x, st>>>((const C2<T>*)p->X, (T*)H, g, (const C2<T>*)p->twx);
    if (cudaError_t e = cudaGetLastError(); e != cudaSuccess) return bd::micro_fail(e, "multi-layer kernel launch");
    return 0;
}

}  // namespace

extern "C" {

void boris_demag_ml_plan_destroy(boris_demag_ml_plan* p) {
    if (!p) return;
    cudaFree(p->K); cudaFree(p->twx); cudaFree(p->twy); cudaFree(p->X); cudaFree(p->Y); cudaFree(p->wlayer); cudaFree(p->partial);
    delete p;
}

boris_demag_ml_plan* boris_demag_ml_plan_create(int ux, int uy, int nlayers, double hx, double hy, const double* thickness,
                                                const double* z_centre, int fp64) {
    bd::clear_error();
    if (ux < 1 || ux > 1024 || uy < 1 || uy > 1024) { bd::set_error(-1, "nx and ny must be in [1, 1024]"); return nullptr; }
    if (nlayers < 1 || nlayers > kMaxLayers) { bd::set_error(-1, "nlayers must be in [1, 32]"); return nullptr; }
    if (!(hx > 0) || !(hy > 0) || !std::isfinite(hx) || !std::isfinite(hy) || !thickness || !z_centre) {
        bd::set_error(-1, "cell sides must be positive and finite; thickness and z_centre must not be NULL");
        return nullptr;
    }
    for (int k = 0; k < nlayers; ++k) {
        if (!(thickness[k] > 0) || !std::isfinite(thickness[k]) || !std::isfinite(z_centre[k])) {
            bd::set_error(-1, "layer thickness must be positive and finite, centre heights finite");
            return nullptr;
        }
        for (int i = 0; i < k; ++i)
            if (std::fabs(z_centre[k] - z_centre[i]) < 0.5 * (thickness[k] + thickness[i]) * (1.0 - 1e-12)) {
                bd::set_error(-1, "layers overlap");
                return nullptr;
            }
    }
    int dev = 0;
    if (cudaError_t e = cudaGetDevice(&dev); e != cudaSuccess) {
        bd::micro_fail(e, "cudaGetDevice (no CUDA device: this library has no CPU fallback)");
        return nullptr;
    }
    boris_demag_ml_plan* p = new (std::nothrow) boris_demag_ml_plan();
    if (!p) { bd::set_error(-3, "out of host memory"); return nullptr; }
    p->n = nlayers; p->fp64 = fp64 ? 1 : 0; p->device = dev; p->hx = hx; p->hy = hy;
    p->t.assign(thickness, thickness + nlayers);
    p->z.assign(z_centre, z_centre + nlayers);
    Geo& g = p->g;
    g.ux = ux; g.uy = uy; g.uz = nlayers;
    g.nx = next_pow2(ux < 4 ? 4 : ux); g.ny = next_pow2(uy < 2 ? 2 : uy); g.nz = nlayers;
    g.Px = 2 * g.nx; g.Py = 2 * g.ny; g.Pz = 1;
    g.lx = ilog2(g.Px); g.ly = ilog2(g.Py); g.lz = 0;
    g.nxr = g.nx + 1;
    const size_t csz = fp64 ? sizeof(double2) : sizeof(float2);
    p->tc_y = 8192 / g.Py; if (p->tc_y > 16) p->tc_y = 16; if (p->tc_y < 1) p->tc_y = 1;
    p->tc_m = 16;
    p->smem_x = (size_t)g.Px * csz;
    p->smem_y = (size_t)p->tc_y * g.Py * csz;
    p->smem_m = (size_t)3 * nlayers * p->tc_m * csz;
    int rc = fp64 ? build<double>(p) : build<float>(p);
    if (!rc && cudaMalloc((void**)&p->wlayer, nlayers * sizeof(double)) != cudaSuccess) rc = bd::set_error(-3, "cudaMalloc");
    if (!rc && cudaMemcpy(p->wlayer, thickness, nlayers * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess) rc = bd::set_error(-2, "cudaMemcpy");
    if (!rc && cudaMalloc((void**)&p->partial, (kEnergyBlocks + 1) * sizeof(double)) != cudaSuccess) rc = bd::set_error(-3, "cudaMalloc");
    if (!rc && cudaMemset(p->partial, 0, (kEnergyBlocks + 1) * sizeof(double)) != cudaSuccess) rc = bd::set_error(-2, "cudaMemset");
    if (rc) { boris_demag_ml_plan_destroy(p); return nullptr; }
    return p;
}

int boris_demag_ml_apply(boris_demag_ml_plan* p, const void* M, void* H, void* stream) {
    if (!p || !M || !H) return bd::set_error(-1, "null argument");
    if (M == H) return bd::set_error(-1, "M and H must not alias");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device)
        return bd::set_error(-1, "the current CUDA device is not the one the plan was created on");
    return p->fp64 ? apply<double>(p, M, H, (cudaStream_t)stream) : apply<float>(p, M, H, (cudaStream_t)stream);
}

int boris_demag_ml_energy(boris_demag_ml_plan* p, const void* M, const void* H, double* E_dev, void* stream) {
    if (!p || !M || !H || !E_dev) return bd::set_error(-1, "null argument");
    const size_t per_layer = (size_t)p->g.ux * p->g.uy, n = 3 * per_layer * p->n;
    size_t nblk = (n + 4 * kThreads - 1) / (4 * kThreads);
    nblk = nblk < 1 ? 1 : (nblk > (size_t)kEnergyBlocks ? (size_t)kEnergyBlocks : nblk);
    const double factor = -0.5 * (4e-7 * kPiML) * p->hx * p->hy;
    unsigned* ticket = reinterpret_cast<unsigned*>(p->partial + kEnergyBlocks);
    if (p->fp64)
        energy<double><<<(unsigned)nblk, kThreads, 0, (cudaStream_t)stream>>>((const double*)M, (const double*)H, n, per_layer, p->n,
                                                                            p->wlayer, p->partial, ticket, factor, E_dev);
    else
        energy<float><<<(unsigned)nblk, kThreads, 0, (cudaStream_t)stream>>>((const float*)M, (const float*)H, n, per_layer, p->n,
                                                                           p->wlayer, p->partial, ticket, factor, E_dev);
    if (cudaError_t e = cudaGetLastError(); e != cudaSuccess) return bd::micro_fail(e, "energy");
    return 0;
}

int boris_demag_ml_pair_tensor_host(int nx, int ny, double hx, double hy, double tk, double ti, double Z, double* out) {
    if (!out || nx < 1 || ny < 1 || !(hx > 0) || !(hy > 0) || !(tk > 0) || !(ti > 0)) return bd::set_error(-1, "invalid argument");
    const long cells = (long)nx * ny;
    for (long idx = 0; idx < cells; ++idx) {
        double v[6];
        bd::pair_tensor_point((int)(idx % nx), (int)(idx / nx), Z, hx, hy, tk, ti, v);
        for (int c = 0; c < 6; ++c) out[c * cells + idx] = v[c];
    }
    return 0;
}

}  // extern "C"
