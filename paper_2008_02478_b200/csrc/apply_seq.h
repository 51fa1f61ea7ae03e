// apply_seq.h — launch configuration and the launch sequence of one demag evaluation,
// written against a Launcher policy so that boris_demag.cu (CUDA launches) and the
// host emulation of the CPU tests (tests/emu) step through the same code.
#pragma once
#include <cmath>
#include <vector>

#include "kernels.h"
#include "khat_layout.h"
#include "plane.h"
#include "xt.h"
#include "xz.h"
#include "yfused.h"

namespace bd {

struct LaunchCfg {
    int rb;        // rows per block of XFwd / XInv
    int nb_y;      // rows per block of YFwd / YInv
    int cs;        // kx slots per chunk of the 3-D path
    int ty;        // y positions per block of ZFused
    int tiled;     // 1: tiled path (xt.h / yfused.h), 0: the kernels of kernels.h
    int cols;      // kx columns per tile
    int rbt;       // rows per block of XFwdT / XInvT
    int pf_y;      // L2 prefetch distance of YFused in blocks, 0: off (set by the plan)
    int pf_xz;     // ... of XZFwd
    PlaneGeom plane;   // plane path (plane.h): thin slabs, takes precedence over the tiled path
};

// kx columns per tile of the tiled path: 3 * L * cols complex = 96 KB of shared memory
// per block at L >= 512 (two blocks per SM)
BD_HD constexpr int cols_for(int Ly) { return Ly >= 2048 ? 2 : (Ly >= 1024 ? 4 : 8); }
// 3-D: same rule.  (8-column tiles at Ly = 1024 were measured: the x/z kernels gain 7 % from
// the 64-byte pieces, YFused loses 17 % with one 512-thread block per SM; profiles/r01_tiled.md)
BD_HD constexpr int cols_for3d(int Ly) { return cols_for(Ly); }
constexpr long kMaxDynSmem = 227L * 1024;
// the 3-D tiled path keeps the nz rows of one (component, y) in shared memory and each
// z column (2 nz points) in registers
inline bool tiled_supported(int nx, int ny, int nz) {
    if (nz == 1) return true;
    return nz <= 256 && ((long)nz * ((prow(nx, nx) + 1) | 1) + (nz > 32 ? 2 * nz : 0)) * (long)sizeof(float2) <= kMaxDynSmem;
}

inline LaunchCfg make_launch_cfg(int nx, int ny, int nz) {
    LaunchCfg c;
    const int Py = 2 * ny, Pz = nz > 1 ? 2 * nz : 1;
    c.rb = nx <= 512 ? 16 : 8;
    while (c.rb > ny) c.rb >>= 1;
    c.nb_y = Py >= 1024 ? 2 : 2048 / Py;
    c.ty = Pz <= 128 ? 16 : (Pz <= 256 ? 8 : (Pz <= 512 ? 4 : 2));
    while (c.ty > Py) c.ty >>= 1;
    if (nz == 1) c.ty = 1;
    // kx slots per chunk: the scratch T (~32 MB) stays in the 126 MB L2 between YFwd,
    // ZFused and YInv, so the y-padded spectrum never reaches HBM
    const long slot_bytes = 3L * nz * Py * (long)sizeof(float2);
    long cs = (32L << 20) / slot_bytes;
    c.cs = (int)(cs < 1 ? 1 : (cs > nx + 1 ? nx + 1 : cs));
    c.tiled = tiled_supported(nx, ny, nz) ? 1 : 0;
    c.cols = nz == 1 ? cols_for(Py) : cols_for3d(Py);
    // narrow 2-D meshes: narrower tiles, so that YFused's (nx + 1) / cols blocks reach at least half of the SMs
    if (nz == 1) while (c.cols > 2 && (nx + c.cols) / c.cols < 74) c.cols >>= 1;
    // rows per block of the tiled 2-D x kernels: about 384 blocks (one wave at 3 blocks per SM) where the mesh has the rows for
    // it, at most 32 KB of rows, at least 8 rows up to nx = 256 and 2 from nx = 512 (measured: profiles/r02_plane.md)
    {
        int hi = nx >= 512 ? 8 : 4096 / nx;
        while (hi > ny) hi >>= 1;
        int lo = nx >= 512 ? 2 : (nx <= 32 ? 32 : 8);
        if (lo > hi) lo = hi;
        int r = 1;
        while (2 * r <= 3 * ny / 384) r <<= 1;
        c.rbt = r < lo ? lo : (r > hi ? hi : r);
    }
    c.pf_y = 0; c.pf_xz = 0;       // set by the plan from the SM count
    c.plane = plane_geom(nx, ny, nz);
    // 64-cell slabs: where the nz rows of a (c, y) slab fit one SM the tiled kernels are as fast (measured: 256 x 256 x 64
    // 0.493 against 0.515 ms, 128 x 128 x 64 0.134 against 0.138 ms) unless the mesh is narrow (64 x 64 x 64 60 against 46 us,
    // 256 x 64 x 64 155 against 128 us, 64 x 256 x 64 173 against 153 us); the plane path also takes the slabs they cannot
    // hold (nx >= 512), instead of the chunked kernels
    if (nz == 64 && c.tiled && nx > 64 && ny > 64) c.plane.on = 0;
    return c;
}

// h[k] = exp(-2 pi i k / denom), k < count, rounded once from fp64; exact at quarter turns
inline void fill_twiddles(float2* h, int count, int denom) {
    const double pi = 3.14159265358979323846264338327950288;
    for (int k = 0; k < count; ++k) {
        if ((4L * k) % denom == 0) {
            const int quarter = (int)((4L * k) / denom % 4);
            const float cx[4] = {1.f, 0.f, -1.f, 0.f}, sy[4] = {0.f, -1.f, 0.f, 1.f};
            h[k].x = cx[quarter]; h[k].y = sy[quarter];
        } else {
            const double a = -2.0 * pi * (double)k / (double)denom;
            h[k].x = (float)std::cos(a);
            h[k].y = (float)std::sin(a);
        }
    }
}

struct PlanView {
    int nx, ny, nz;
    LaunchCfg cfg;
    const float* Kst;
    const float2 *tw_x, *tw_xpost, *tw_y, *tw_z;
    float2 *W, *T;
    const float2 *ptw_x = nullptr, *ptw_y = nullptr;   // per-pass twiddles (tiled path)
    float2* V = nullptr;                               // tiled spectrum (tiled path)
    const float4* xpost = nullptr;                     // fill_xpost table (tiled path)
    EnergyArgs en = {nullptr, nullptr, nullptr, nullptr, 0.0};   // energy fused into the last kernel (tiled path)
    // plane path (plane.h)
    float2 *X = nullptr, *P = nullptr;
    const float* KP = nullptr;
    const int* kidx = nullptr;
    const float2 *pl_tw = nullptr, *pl_zt = nullptr;
};

template <int L> struct IC { static constexpr int value = L; };
template <class F>
int dispatch_len(int L, F&& f) {
    switch (L) {
        case 4: return f(IC<4>{});
        case 8: return f(IC<8>{});
        case 16: return f(IC<16>{});
        case 32: return f(IC<32>{});
        case 64: return f(IC<64>{});
        case 128: return f(IC<128>{});
        case 256: return f(IC<256>{});
        case 512: return f(IC<512>{});
        case 1024: return f(IC<1024>{});
        case 2048: return f(IC<2048>{});
        default: return -1;
    }
}

struct Grid { unsigned x, y; };

inline int apply_launch_count(int nx, int nz, const LaunchCfg& c) {
    const int NS = nx + 1;
    if (c.plane.on || c.tiled) return 3;
    return nz == 1 ? 3 : 2 + 3 * ((NS + c.cs - 1) / c.cs);
}

// tiled path, nz = 1: XFwdT -> YFused -> XInvT
template <int COLS, class Launcher>
int enqueue_tiled_2d(Launcher& run, const PlanView& p, const float* M, float* H) {
    const int nx = p.nx, ny = p.ny, Py = 2 * ny;
    const int ntl = (nx + 1 + COLS - 1) / COLS;
    XTArgs xa{M, H, p.V, p.ptw_x, p.xpost, ny, ntl, p.cfg.rbt, ilog2c(p.cfg.rbt), p.en};
    const Grid gx{(unsigned)(3L * ny / p.cfg.rbt), 1};
    int rc = dispatch_len(nx, [&](auto ic) { return run.template run<XFwdT<decltype(ic)::value, COLS>>(gx, xa); });
    if (rc) return rc;
    YFArgs ya{p.V, p.Kst, p.ptw_y, ntl, 1, p.cfg.pf_y};
    const Grid gy{(unsigned)ntl, 1};
    rc = dispatch_len(Py, [&](auto ic) {
        constexpr int L = decltype(ic)::value;
        if constexpr (COLS <= cols_for(L)) return run.template run<YFused<L, 4, COLS>>(gy, ya);
        else return -1;
    });
    if (rc) return rc;
    return dispatch_len(nx, [&](auto ic) { return run.template run<XInvT<decltype(ic)::value, COLS>>(gx, xa); });
}

template <class Launcher>
int dispatch_tiled_2d(Launcher& run, const PlanView& p, const float* M, float* H) {
    switch (p.cfg.cols) {
        case 2: return enqueue_tiled_2d<2>(run, p, M, H);
        case 4: return enqueue_tiled_2d<4>(run, p, M, H);
        case 8: return enqueue_tiled_2d<8>(run, p, M, H);
        default: return -1;
    }
}

// tiled path, nz = 2..256: XZFwd -> YFused -> ZXInv.  The pieces are separate templates so
// that the CUDA build can put them into translation units of their own (launcher.cuh).
// x + z transforms of the meshes with NZLO <= nz <= NZHI
template <int NZLO, int NZHI, class Launcher>
int enqueue_xz(Launcher& run, const PlanView& p, const float* M, float* H, bool fwd) {
    const int nx = p.nx, ny = p.ny, nz = p.nz, cols = p.cfg.cols;
    const int ntl = (nx + 1 + cols - 1) / cols;
    XZArgs xa{M, H, p.V, p.ptw_x, p.xpost, ny, ntl, ilog2c(cols), p.tw_z, p.cfg.pf_xz, p.en};
    const Grid gx{(unsigned)(3 * ny), 1};
    return dispatch_len(nx, [&](auto ic) {
        constexpr int LX = decltype(ic)::value;
        auto go = [&](auto nzc) {
            constexpr int NZ = decltype(nzc)::value;
            if constexpr (NZ >= NZLO && NZ <= NZHI && LX <= 1024 &&
                          (long)NZ * SRows<LX>::PITCH * (long)sizeof(float2) <= kMaxDynSmem) {
                if (fwd) return run.template run<XZFwd<LX, NZ>>(gx, xa);
                return run.template run<ZXInv<LX, NZ>>(gx, xa);
            } else {
                return -1;
            }
        };
        switch (nz) {
            case 2: return go(IC<2>{});
            case 4: return go(IC<4>{});
            case 8: return go(IC<8>{});
            case 16: return go(IC<16>{});
            case 32: return go(IC<32>{});
            case 64: return go(IC<64>{});
            case 128: return go(IC<128>{});
            case 256: return go(IC<256>{});
            default: return -1;
        }
    });
}

template <class Launcher>
int enqueue_yfused3(Launcher& run, const PlanView& p) {
    const int cols = p.cfg.cols, ntl = (p.nx + 1 + cols - 1) / cols, Py = 2 * p.ny, Pz = 2 * p.nz;
    YFArgs ya{p.V, p.Kst, p.ptw_y, ntl, Pz, p.cfg.pf_y};
    const Grid gy{(unsigned)(ntl * Pz), 1};
    return dispatch_len(Py, [&](auto ic) {
        constexpr int L = decltype(ic)::value;
        return run.template run<YFused<L, 6, cols_for3d(L)>>(gy, ya);
    });
}

// plane path (plane.h), nz = 32: XFwdT<LX,1> -> YZFused -> XInvP
template <class Launcher>
int enqueue_plane_x(Launcher& run, const PlanView& p, const float* M, float* H, bool fwd) {
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const PlaneGeom& g = p.cfg.plane;
    if (fwd) {
        XTArgs xa{M, H, p.X, p.ptw_x, p.xpost, ny, nx + 1, 16, 4, p.en};
        const Grid gx{(unsigned)(3L * nz * ny / 16), 1};
        return dispatch_len(nx, [&](auto ic) { return run.template run<XFwdT<decltype(ic)::value, 1>>(gx, xa); });
    }
    XPArgs ia{p.P, H, p.ptw_x, p.xpost, ny, nx + 1, g.lsp, 3L * nz * (nx + 1) * g.lsp, p.en};
    const Grid gi{(unsigned)(3L * nz * ny / 16), 1};
    return dispatch_len(nx, [&](auto ic) {
        constexpr int LX = decltype(ic)::value;
        switch (g.nq) {
            case 1: return run.template run<XInvP<LX, 1>>(gi, ia);
            case 2: return run.template run<XInvP<LX, 2>>(gi, ia);
            case 4: return run.template run<XInvP<LX, 4>>(gi, ia);
            case 8: return run.template run<XInvP<LX, 8>>(gi, ia);
            default: return -1;
        }
    });
}
// the fused y/z kernel of slabs of NZ cells (separate templates: one translation unit per thickness)
template <int NZ, class Launcher>
int enqueue_plane_yz_nz(Launcher& run, const PlanView& p) {
    const PlaneGeom& g = p.cfg.plane;
    YZArgs ya{p.X, p.P, p.KP, p.kidx, p.pl_tw, p.pl_zt, p.nx + 1, p.ny};
    const Grid gy{(unsigned)((p.nx + 1) * g.nq), 1};
    auto go = [&](auto lsc) {
        constexpr int LS = decltype(lsc)::value;
        switch (g.nq) {
            case 1: return run.template run<YZFused<LS, 1, NZ>>(gy, ya);
            case 2: return run.template run<YZFused<LS, 2, NZ>>(gy, ya);
            case 4: return run.template run<YZFused<LS, 4, NZ>>(gy, ya);
            case 8: return run.template run<YZFused<LS, 8, NZ>>(gy, ya);
            default: return -1;
        }
    };
    switch (g.ls) {
        case 64: return go(IC<64>{});
        case 128: return go(IC<128>{});
        case 256: return go(IC<256>{});
        default: return -1;
    }
}
template <class Launcher>
int enqueue_plane_yz(Launcher& run, const PlanView& p) {
    switch (p.nz) {
        case 64: return enqueue_plane_yz_nz<64>(run, p);
        case 32: return enqueue_plane_yz_nz<32>(run, p);
        case 16: return enqueue_plane_yz_nz<16>(run, p);
        case 8: return enqueue_plane_yz_nz<8>(run, p);
        case 4: return enqueue_plane_yz_nz<4>(run, p);
        case 2: return enqueue_plane_yz_nz<2>(run, p);
        default: return -1;
    }
}

// Launcher::run<K>(Grid, const K::Args&) -> 0 on success; Launcher::tiled_2d / xz / yfused3
// forward to dispatch_tiled_2d / enqueue_xz / enqueue_yfused3.
template <class Launcher>
int enqueue_apply(Launcher& run, const PlanView& p, const float* M, float* H) {
    if (p.cfg.plane.on) {
        int rc = run.plane_x(p, M, H, true);
        if (!rc) rc = run.plane_yz(p);
        if (!rc) rc = run.plane_x(p, M, H, false);
        return rc;
    }
    if (p.cfg.tiled) {
        if (p.nz == 1) return run.tiled_2d(p, M, H);
        int rc = run.xz(p, M, H, true);
        if (!rc) rc = run.yfused3(p);
        if (!rc) rc = run.xz(p, M, H, false);
        return rc;
    }
    const int nx = p.nx, ny = p.ny, nz = p.nz, NS = nx + 1, Py = 2 * ny, Pz = 2 * nz;
    const LaunchCfg& c = p.cfg;
    XArgs xa{M, H, p.W, p.tw_x, p.tw_xpost, ny, nz, c.rb};
    const Grid gx{(unsigned)(3L * nz * ny / c.rb), 1};
    int rc = dispatch_len(nx, [&](auto ic) { return run.template run<XFwd<decltype(ic)::value>>(gx, xa); });
    if (rc) return rc;
    if (nz == 1) {
        return -1;               // 2-D meshes always take the tiled path
    } else {
        const long w_cstride = (long)NS * nz * ny;
        for (int s0 = 0; s0 < NS; s0 += c.cs) {
            const int cs = (NS - s0 < c.cs) ? NS - s0 : c.cs;
            const int rows = cs * nz;
            const long t_cstride = (long)cs * nz * Py;
            YArgs yf{p.W + (long)s0 * nz * ny, p.T, ny, Py, w_cstride, t_cstride, rows, c.nb_y, p.tw_y};
            const Grid gy{(unsigned)((rows + c.nb_y - 1) / c.nb_y), 3};
            rc = dispatch_len(Py, [&](auto ic) { return run.template run<YPass<decltype(ic)::value, false>>(gy, yf); });
            if (rc) return rc;
            FusedArgs fa{p.T, p.Kst, p.tw_z, 0, 0, Py, cs, s0, c.ty};
            const Grid gz{(unsigned)(Py / c.ty), (unsigned)cs};
            rc = dispatch_len(Pz, [&](auto ic) { return run.template run<ZFused<decltype(ic)::value>>(gz, fa); });
            if (rc) return rc;
            YArgs yi{p.T, p.W + (long)s0 * nz * ny, Py, ny, t_cstride, w_cstride, rows, c.nb_y, p.tw_y};
            rc = dispatch_len(Py, [&](auto ic) { return run.template run<YPass<decltype(ic)::value, true>>(gy, yi); });
            if (rc) return rc;
        }
    }
    return dispatch_len(nx, [&](auto ic) { return run.template run<XInv<decltype(ic)::value>>(gx, xa); });
}

}  // namespace bd
