// boris_llg.cu — C ABI of include/boris_llg.h: the LLG evaluation around the demag path
// (SURVEY.md section 8(f), NEXT-1).  The demagnetizing field comes from boris_demag_apply; the
// kernels here are the cheap local terms of one evaluation (Eq. (1) at L33)
// and the RK4 bookkeeping.  All of them stream planar fp32 fields once: HBM-bound.
#include <cuda_runtime.h>

#include <cmath>
#include <new>
#include <string>

#include "../../include/boris_llg.h"

namespace bd { int set_error(int code, const char* msg); }   // boris_demag.cu: the library's thread-local error text

namespace {

int llg_fail(int code, const char* msg) { return bd::set_error(code, msg); }

constexpr double kMu0 = 4e-7 * 3.14159265358979323846264338327950288;

struct Dims { int nx, ny, nz; };

// Heff = Ms Hd + cx (m[x+1] - 2 m + m[x-1]) + cy (...) + cz (...) + Hext on input Hd = H_demag(m) (the demag
// operator is linear: H_demag(Ms m) = Ms H_demag(m), so the unit field goes through boris_demag_apply as it is);
// a missing neighbour contributes nothing (homogeneous Neumann condition); c* = 2A / (mu0 Ms h*^2).
// One block walks over rows (c, z, y); its threads over x.
__global__ void k_exchange_zeeman(const float* __restrict__ m, float* __restrict__ H, Dims d, float Ms, float cx, float cy,
                                  float cz, float hx, float hy, float hz) {
    const long rows = 3L * d.nz * d.ny, plane = (long)d.nx * d.ny;
    for (long row = blockIdx.x; row < rows; row += gridDim.x) {
        const int y = (int)(row % d.ny);
        const int z = (int)((row / d.ny) % d.nz);
        const int c = (int)(row / ((long)d.ny * d.nz));
        const float hext = c == 0 ? hx : (c == 1 ? hy : hz);
        const float* mr = m + row * d.nx;
        float* hr = H + row * d.nx;
        const bool yp = y + 1 < d.ny, ym = y > 0, zp = z + 1 < d.nz, zm = z > 0;
        for (int x = threadIdx.x; x < d.nx; x += blockDim.x) {
            const float v = mr[x];
            float lap = 0.f;
            if (x + 1 < d.nx) lap += cx * (mr[x + 1] - v);
            if (x > 0) lap += cx * (mr[x - 1] - v);
            if (yp) lap += cy * (mr[x + d.nx] - v);
            if (ym) lap += cy * (mr[x - d.nx] - v);
            if (zp) lap += cz * (mr[x + plane] - v);
            if (zm) lap += cz * (mr[x - plane] - v);
            hr[x] = Ms * hr[x] + lap + hext;
        }
    }
}

// One RK4 stage per cell: k = -g [u x H + alpha u x (u x H)]  (Eq. (1) solved for dm/dt, g = gamma / (1 + alpha^2));
// acc = (first ? 0 : acc) + w k;  then either the next stage state u_next = m0 + a k, or (last) the step
// m0 <- normalise(m0 + dt/6 acc) (m0 and mout may be the same array: a thread reads its cell before it writes it).
// The local field terms are gathered on the way (no separate pass over H): Hd is H_demag of the unit stage state
// u, and H_eff = Ms Hd + exchange stencil of u + H_applied is formed per cell.  u and unext must be different
// arrays (neighbours of u are read).  One block walks over rows (z, y); threads over x.
__global__ void k_rk4_stage_fused(const float* m0, const float* __restrict__ u, const float* __restrict__ Hd,
                                  float* __restrict__ acc, float* __restrict__ unext, float* mout, Dims d, float Ms, float cx,
                                  float cy, float cz, float hx, float hy, float hz, float g, float alpha, float w, float a,
                                  float dt6, int first, int last) {
    const long rows = (long)d.nz * d.ny, plane = (long)d.nx * d.ny, cells = plane * d.nz;
    for (long row = blockIdx.x; row < rows; row += gridDim.x) {
        const int y = (int)(row % d.ny), z = (int)(row / d.ny);
        const bool yp = y + 1 < d.ny, ym = y > 0, zp = z + 1 < d.nz, zm = z > 0;
        for (int x = threadIdx.x; x < d.nx; x += blockDim.x) {
            const long i = row * d.nx + x;
            float uv[3], H[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float* uc = u + c * cells + i;
                const float v = uc[0];
                float lap = 0.f;
                if (x + 1 < d.nx) lap += cx * (uc[1] - v);
                if (x > 0) lap += cx * (uc[-1] - v);
                if (yp) lap += cy * (uc[d.nx] - v);
                if (ym) lap += cy * (uc[-d.nx] - v);
                if (zp) lap += cz * (uc[plane] - v);
                if (zm) lap += cz * (uc[-plane] - v);
                uv[c] = v;
                H[c] = Ms * Hd[c * cells + i] + lap + (c == 0 ? hx : (c == 1 ? hy : hz));
            }
            const float tx = uv[1] * H[2] - uv[2] * H[1], ty = uv[2] * H[0] - uv[0] * H[2], tz = uv[0] * H[1] - uv[1] * H[0];
            const float dx = uv[1] * tz - uv[2] * ty, dy = uv[2] * tx - uv[0] * tz, dz = uv[0] * ty - uv[1] * tx;
            const float kx = -g * (tx + alpha * dx), ky = -g * (ty + alpha * dy), kz = -g * (tz + alpha * dz);
            float ax = w * kx, ay = w * ky, az = w * kz;
            if (!first) { ax += acc[i]; ay += acc[i + cells]; az += acc[i + 2 * cells]; }
            const float px = m0[i], py = m0[i + cells], pz = m0[i + 2 * cells];
            if (!last) {
                acc[i] = ax; acc[i + cells] = ay; acc[i + 2 * cells] = az;
                unext[i] = px + a * kx; unext[i + cells] = py + a * ky; unext[i + 2 * cells] = pz + a * kz;
            } else {
                const float nx = px + dt6 * ax, ny = py + dt6 * ay, nz = pz + dt6 * az;
                const float inv = rsqrtf(nx * nx + ny * ny + nz * nz);
                mout[i] = nx * inv; mout[i + cells] = ny * inv; mout[i + 2 * cells] = nz * inv;
            }
        }
    }
}

}  // namespace

struct boris_llg {
    boris_demag_plan* plan;
    Dims d;
    double hx, hy, hz, Ms, A, alpha, gamma;
    double Hext[3] = {0.0, 0.0, 0.0};
    float *H = nullptr, *u = nullptr, *u2 = nullptr, *acc = nullptr;     // [3][nz][ny][nx] each; u, u2: stage states
};

extern "C" {

void boris_llg_destroy(boris_llg* s) {
    if (!s) return;
    cudaFree(s->H); cudaFree(s->u); cudaFree(s->u2); cudaFree(s->acc);
    delete s;
}

boris_llg* boris_llg_create(boris_demag_plan* plan, int nx, int ny, int nz, double hx, double hy, double hz,
                            double Ms, double A, double alpha, double gamma) {
    if (!plan || nx < 1 || ny < 1 || nz < 1 || !(hx > 0) || !(hy > 0) || !(hz > 0) || !(Ms > 0) || !(A >= 0) ||
        !(alpha >= 0) || !(gamma > 0)) {
        llg_fail(-1, "boris_llg_create: invalid argument");
        return nullptr;
    }
    // the work arrays are sized from (nx, ny, nz) and boris_demag_apply reads and writes the plan's mesh:
    // the two must be the same mesh
    int cells[3];
    double sides[3];
    if (boris_demag_plan_mesh(plan, cells, sides)) return nullptr;
    if (cells[0] != nx || cells[1] != ny || cells[2] != nz) {
        llg_fail(-1, "boris_llg_create: (nx, ny, nz) differ from the mesh the demag plan was created for");
        return nullptr;
    }
    const double tol = 1e-12;
    if (std::fabs(sides[0] - hx) > tol * hx || std::fabs(sides[1] - hy) > tol * hy || std::fabs(sides[2] - hz) > tol * hz) {
        llg_fail(-1, "boris_llg_create: (hx, hy, hz) differ from the cell sides of the demag plan");
        return nullptr;
    }
    boris_llg* s = new (std::nothrow) boris_llg();
    if (!s) { llg_fail(-3, "boris_llg_create: out of host memory"); return nullptr; }
    s->plan = plan; s->d = Dims{nx, ny, nz};
    s->hx = hx; s->hy = hy; s->hz = hz; s->Ms = Ms; s->A = A; s->alpha = alpha; s->gamma = gamma;
    const size_t bytes = (size_t)3 * nx * ny * nz * sizeof(float);
    if (cudaMalloc((void**)&s->H, bytes) != cudaSuccess || cudaMalloc((void**)&s->u, bytes) != cudaSuccess ||
        cudaMalloc((void**)&s->u2, bytes) != cudaSuccess || cudaMalloc((void**)&s->acc, bytes) != cudaSuccess) {
        cudaGetLastError();
        boris_llg_destroy(s);
        llg_fail(-3, "boris_llg_create: out of device memory");
        return nullptr;
    }
    return s;
}

int boris_llg_set_applied_field(boris_llg* s, double Hx, double Hy, double Hz) {
    if (!s || !std::isfinite(Hx) || !std::isfinite(Hy) || !std::isfinite(Hz))
        return llg_fail(-1, "boris_llg_set_applied_field: invalid argument");
    s->Hext[0] = Hx; s->Hext[1] = Hy; s->Hext[2] = Hz;
    return 0;
}

int boris_llg_effective_field(boris_llg* s, const float* m, float* Heff, void* stream) {
    if (!s || !m || !Heff || m == Heff) return llg_fail(-1, "boris_llg_effective_field: null or aliasing argument");
    cudaStream_t st = (cudaStream_t)stream;
    if (int rc = boris_demag_apply(s->plan, m, Heff, stream)) return rc;          // H_demag of the unit field
    const double c = 2.0 * s->A / (kMu0 * s->Ms);
    const long rows = 3L * s->d.nz * s->d.ny;
    const int threads = s->d.nx >= 256 ? 256 : (s->d.nx >= 64 ? 64 : 32);
    k_exchange_zeeman<<<(unsigned)(rows < (1L << 20) ? rows : (1L << 20)), threads, 0, st>>>(
        m, Heff, s->d, (float)s->Ms, (float)(c / (s->hx * s->hx)), (float)(c / (s->hy * s->hy)), (float)(c / (s->hz * s->hz)),
        (float)s->Hext[0], (float)s->Hext[1], (float)s->Hext[2]);
    if (cudaError_t e = cudaGetLastError(); e != cudaSuccess) return llg_fail(-2, cudaGetErrorString(e));
    return 0;
}

int boris_llg_rk4(boris_llg* s, float* m, double dt, int nsteps, void* stream) {
    if (!s || !m || !(dt > 0) || nsteps < 0) return llg_fail(-1, "boris_llg_rk4: invalid argument");
    cudaStream_t st = (cudaStream_t)stream;
    const float g = (float)(s->gamma / (1.0 + s->alpha * s->alpha)), al = (float)s->alpha;
    const float w[4] = {1.f, 2.f, 2.f, 1.f};
    const float a[4] = {(float)(0.5 * dt), (float)(0.5 * dt), (float)dt, 0.f};
    const double c = 2.0 * s->A / (kMu0 * s->Ms);
    const float cx = (float)(c / (s->hx * s->hx)), cy = (float)(c / (s->hy * s->hy)), cz = (float)(c / (s->hz * s->hz));
    const long rows = (long)s->d.nz * s->d.ny;
    const int threads = s->d.nx >= 256 ? 256 : (s->d.nx >= 64 ? 64 : 32);
    const unsigned blocks = (unsigned)(rows < (1L << 20) ? rows : (1L << 20));
    for (int step = 0; step < nsteps; ++step) {
        const float* u = m;                                      // stage state: m0, then the two work arrays in turn
        for (int k = 0; k < 4; ++k) {
            float* un = (k & 1) ? s->u2 : s->u;
            if (int rc = boris_demag_apply(s->plan, u, s->H, stream)) return rc;      // H_demag of the unit stage state
            k_rk4_stage_fused<<<blocks, threads, 0, st>>>(m, u, s->H, s->acc, un, m, s->d, (float)s->Ms, cx, cy, cz,
                                                          (float)s->Hext[0], (float)s->Hext[1], (float)s->Hext[2], g, al,
                                                          w[k], a[k], (float)(dt / 6.0), k == 0, k == 3);
            if (cudaError_t e = cudaGetLastError(); e != cudaSuccess) return llg_fail(-2, cudaGetErrorString(e));
            u = un;
        }
    }
    return 0;
}

}  // extern "C"
