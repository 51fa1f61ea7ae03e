// yfused.h — the pipelined step of the tiled path: y FFT, per-frequency symmetric
// tensor multiply and inverse y FFT in one launch, all 3 vector components together
// ("(inverse)FFTs and point-by-point multiplications are done using a
// single CUDA kernel launch, simultaneously for all 3 vector components"; here the
// fused dimension is y — reading in DESIGN.md §7).
//
// Data: the spectrum after the x (and z) transforms, tiled by kx so that a block's
// pencils are one contiguous piece of memory:
//     V[c (3)][kz (Pz)][tile (NTL)][y (ny)][col (COLS)]   complex64,  kx = tile*COLS + col
// One block = one (kz, tile): 3*COLS pencils of ny -> L = 2 ny points, held in shared
// memory as S[c][swz(e)][col].  The pencil index e after the forward passes is in the
// digit-reversed order of fft_core.h; the kernel spectrum is stored in the order the
// multiply meets it (KTile below), real and symmetry-reduced in y and z (pin P12).
#pragma once
#include <cmath>

#include "fft_core.h"
#include "pk.h"

namespace bd {

// slots of boris_demag_apply_timed: x forward = 0, fused multiply = 1, x inverse = 5
constexpr int kKindYFused = 1, kKindXFwdT = 0, kKindXInvT = 5, kKindXZFwd = 0, kKindZXInv = 5;

// ------------------------------------------------------------------ per-pass twiddle tables
// pass p < NP-1 of a length-L transform: T_p[(q-1)*S_p + j] = exp(-2 pi i j q / L_p),
// j < S_p = L_p / R_p, q = 1..R_p-1 (consecutive butterflies read consecutive entries).
BD_HD constexpr int ptw_off(int L, int p) {
    return p == 0 ? 0 : (dec_r(L, 0) - 1) * (L / dec_r(L, 0));
}
BD_HD constexpr int ptw_total(int L) {
    return dec_np(L) == 1 ? 1
         : dec_np(L) == 2 ? (dec_r(L, 0) - 1) * (L / dec_r(L, 0))
                          : ptw_off(L, 1) + (dec_r(L, 1) - 1) * (dec_sublen(L, 1) / dec_r(L, 1));
}
inline void fill_pass_twiddles(float2* h, int L) {
    const double pi = 3.14159265358979323846264338327950288;
    h[0] = bd_f2(1.f, 0.f);
    for (int p = 0; p + 1 < dec_np(L); ++p) {
        const int R = dec_r(L, p), Lp = dec_sublen(L, p), S = Lp / R;
        for (int q = 1; q < R; ++q)
            for (int j = 0; j < S; ++j) {
                const long m = ((long)j * q) % Lp;
                float2 w;
                if ((4 * m) % Lp == 0) {
                    const float cx[4] = {1.f, 0.f, -1.f, 0.f}, sy[4] = {0.f, -1.f, 0.f, 1.f};
                    w = bd_f2(cx[(4 * m) / Lp], sy[(4 * m) / Lp]);
                } else {
                    const double a = -2.0 * pi * (double)m / (double)Lp;
                    w = bd_f2((float)std::cos(a), (float)std::sin(a));
                }
                h[ptw_off(L, p) + (q - 1) * S + j] = w;
            }
    }
}

// ------------------------------------------------------------------ shared-memory order
BD_HD constexpr int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }
// XOR swizzle of the pencil index: a half warp touches 16/COLS different e per access;
// they must differ in their low bits.  Plain passes give consecutive e; the last pass
// gives e = 8 i + q with consecutive i; the multiply gives i = (f % R0) R1 + f / R0
// with consecutive f.
template <int L, int COLS>
BD_HD int swz(int e) {
    constexpr int SW = 16 / COLS;
    if constexpr (dec_np(L) == 1 || SW <= 1) {
        return e;
    } else if constexpr (dec_np(L) == 2) {
        return e ^ ((e >> 3) & (SW - 1));
    } else {
        constexpr int SH = 3 + ilog2c(dec_r(L, 1));
        return e ^ (((e >> 3) ^ (e >> SH)) & (SW - 1));
    }
}

template <int L, int COLS>
struct STile {                 // shared: S[c][swz(e)][col]
    float2* p;                 // already offset by col
    BD_HD float2 get(int c, int e) const { return p[(c * L + swz<L, COLS>(e)) * COLS]; }
    BD_HD void put(int c, int e, float2 v) const { p[(c * L + swz<L, COLS>(e)) * COLS] = v; }
};
template <int COLS>
struct GTile {                 // global: V tile [y][col], component stride cstride
    float2* p; long cstride;   // already offset by col
    BD_HD float2 get(int c, int e) const { return p[c * cstride + (long)e * COLS]; }
    BD_HD void put(int c, int e, float2 v) const { p[c * cstride + (long)e * COLS] = v; }
};

// ------------------------------------------------------------------ passes, 3 components per thread
// pencils c = c0, c0 + cstep, ... < cend share the butterfly index `it` and its twiddles
template <int L, int P, class In, class Out>
BD_HD void fwd_passM(int it, int c0, int cstep, int cend, const In& in, const Out& out, const float2* __restrict__ ptw) {
    constexpr int NP = dec_np(L), R = dec_r(L, P), Lp = dec_sublen(L, P), S = Lp / R;
    const int blk = it / S, j = it - blk * S, base = blk * Lp + j;
    Tw tw[R];
    if constexpr (P < NP - 1) {
        BD_UNROLL
        for (int q = 1; q < R; ++q) tw[q] = make_tw(BD_LDG(&ptw[ptw_off(L, P) + (q - 1) * S + j]));
    }
    for (int c = c0; c < cend; c += cstep) {
        float2 v[R];
        if constexpr (P == 0) {
            BD_UNROLL
            for (int r = 0; r < R / 2; ++r) v[r] = in.get(c, base + r * S);
            PkDftPruned<R, -1>::run(v);
        } else {
            BD_UNROLL
            for (int r = 0; r < R; ++r) v[r] = in.get(c, base + r * S);
            PkDft<R, -1>::run(v);
        }
        if constexpr (P < NP - 1) {
            BD_UNROLL
            for (int q = 1; q < R; ++q) v[q] = pk_cmul(v[q], tw[q]);
        }
        BD_UNROLL
        for (int q = 0; q < R; ++q) out.put(c, base + q * S, v[q]);
    }
}

template <int L, int P, class In, class Out>
BD_HD void inv_passM(int it, int c0, int cstep, int cend, const In& in, const Out& out, const float2* __restrict__ ptw) {
    constexpr int NP = dec_np(L), R = dec_r(L, P), Lp = dec_sublen(L, P), S = Lp / R;
    const int blk = it / S, j = it - blk * S, base = blk * Lp + j;
    Tw tw[R];
    if constexpr (P < NP - 1) {
        BD_UNROLL
        for (int q = 1; q < R; ++q) tw[q] = make_tw(BD_LDG(&ptw[ptw_off(L, P) + (q - 1) * S + j]));
    }
    for (int c = c0; c < cend; c += cstep) {
        float2 v[R];
        BD_UNROLL
        for (int q = 0; q < R; ++q) v[q] = in.get(c, base + q * S);
        if constexpr (P < NP - 1) {
            BD_UNROLL
            for (int q = 1; q < R; ++q) v[q] = pk_cmulc(v[q], tw[q]);
        }
        if constexpr (P == 0) {
            PkDftTrunc<R, +1>::run(v);
            BD_UNROLL
            for (int r = 0; r < R / 2; ++r) out.put(c, base + r * S, v[r]);
        } else {
            PkDft<R, +1>::run(v);
            BD_UNROLL
            for (int r = 0; r < R; ++r) out.put(c, base + r * S, v[r]);
        }
    }
}

template <int L, int P, class In, class Out>
BD_HD void fwd_pass3(int it, const In& in, const Out& out, const float2* __restrict__ ptw) {
    fwd_passM<L, P>(it, 0, 1, 3, in, out, ptw);
}
template <int L, int P, class In, class Out>
BD_HD void inv_pass3(int it, const In& in, const Out& out, const float2* __restrict__ ptw) {
    inv_passM<L, P>(it, 0, 1, 3, in, out, ptw);
}

// ------------------------------------------------------------------ kernel-spectrum tile
// K[kzr (Pz/2+1)][tile][row (F/2+1)][col][c (NC)][q (RL)], fp32.  Row r, entry q holds the
// natural spectrum at ky = r + F q folded to [0, L/2] with the sign of the components
// odd in y applied (F = L / RL items of the last pass).  Item f <= F/2 reads row f
// as stored; item f > F/2 reads row F - f with q reversed and the y-odd components
// negated (its frequencies are the mirrors L - k of that row).  Rows 0 and F/2 are
// their own mirrors.  A block at kz > Pz/2 reads the tile of Pz - kz and negates the
// z-odd components.
template <int L>
struct KTile {
    static constexpr int RL = dec_rlast(L), F = L / RL, NR = F / 2 + 1;
};

// last forward pass + multiply + first inverse pass of item i (frequency offset f)
template <int L, int NC, bool REV, class In, class Out>
BD_HD void mid3(int i, const float* __restrict__ krow, float sz, const In& in, const Out& out) {
    constexpr int NP = dec_np(L), RL = dec_rlast(L);
    float2 v[3][RL];
    BD_UNROLL
    for (int c = 0; c < 3; ++c) {
        if constexpr (NP == 1) {
            BD_UNROLL
            for (int q = 0; q < RL / 2; ++q) v[c][q] = in.get(c, i * RL + q);
            PkDftPruned<RL, -1>::run(v[c]);
        } else {
            BD_UNROLL
            for (int q = 0; q < RL; ++q) v[c][q] = in.get(c, i * RL + q);
            PkDft<RL, -1>::run(v[c]);
        }
    }
    float k[NC][RL];
    BD_UNROLL
    for (int c = 0; c < NC; ++c) {
        if constexpr (RL % 4 == 0) {
            BD_UNROLL
            for (int q4 = 0; q4 < RL / 4; ++q4) {
                const float4 t = BD_LDG(reinterpret_cast<const float4*>(krow + c * RL) + q4);
                k[c][4 * q4] = t.x; k[c][4 * q4 + 1] = t.y; k[c][4 * q4 + 2] = t.z; k[c][4 * q4 + 3] = t.w;
            }
        } else {
            BD_UNROLL
            for (int q = 0; q < RL; ++q) k[c][q] = BD_LDG(krow + c * RL + q);
        }
    }
    // odd-component signs moved onto the data: with my' = sy my, mz' = sz mz the products
    // use the stored values and Hy = sy Hy', Hz = sz Hz'  (sy = -1 for REV, else +1)
    BD_UNROLL
    for (int q = 0; q < RL; ++q) {
        const int qq = REV ? RL - 1 - q : q;
        const float2 mx = v[0][q];
        const float2 my = REV ? pk_neg(v[1][q]) : v[1][q];
        const float2 kxx = pk_bc(k[0][qq]), kyy = pk_bc(k[1][qq]), kzz = pk_bc(k[2][qq]), kxy = pk_bc(k[3][qq]);
        if constexpr (NC == 4) {
            // 2-D mode (reading R7): Nxz = Nyz = 0, Hz = -Nzz * Mz alone
            const float2 hx = pk_fma(kxy, my, pk_mul(kxx, mx));
            const float2 hy = pk_fma(kyy, my, pk_mul(kxy, mx));
            v[0][q] = hx;
            v[1][q] = REV ? pk_neg(hy) : hy;
            v[2][q] = pk_mul(kzz, v[2][q]);
        } else {
            const float2 mz = pk_mul(pk_bc(sz), v[2][q]);
            const float2 kxz = pk_bc(k[4][qq]), kyz = pk_bc(k[5][qq]);
            const float2 hx = pk_fma(kxz, mz, pk_fma(kxy, my, pk_mul(kxx, mx)));
            const float2 hy = pk_fma(kyz, mz, pk_fma(kyy, my, pk_mul(kxy, mx)));
            const float2 hz = pk_fma(kzz, mz, pk_fma(kyz, my, pk_mul(kxz, mx)));
            v[0][q] = hx;
            v[1][q] = REV ? pk_neg(hy) : hy;
            v[2][q] = pk_mul(pk_bc(sz), hz);
        }
    }
    BD_UNROLL
    for (int c = 0; c < 3; ++c) {
        if constexpr (NP == 1) {
            PkDftTrunc<RL, +1>::run(v[c]);
            BD_UNROLL
            for (int q = 0; q < RL / 2; ++q) out.put(c, i * RL + q, v[c][q]);
        } else {
            PkDft<RL, +1>::run(v[c]);
            BD_UNROLL
            for (int q = 0; q < RL; ++q) out.put(c, i * RL + q, v[c][q]);
        }
    }
}

// item of the last pass whose frequency offset is f (inverse of item_partial_freq)
BD_HD int item_of_partial_freq(int L, int f) {
    const int np = dec_np(L);
    if (np == 1) return 0;
    if (np == 2) return f;
    const int r0 = dec_r(L, 0), r1 = dec_r(L, 1);
    return (f % r0) * r1 + f / r0;
}

// ------------------------------------------------------------------ YFused (S2+S4+S6)
struct YFArgs {
    float2* V;            // [3][Pz][ntl][ny][COLS]
    const float* K;       // [Pz/2+1][ntl][NR][COLS][NC][RL]
    const float2* ptw;    // per-pass twiddles of length L
    int ntl;              // kx tiles
    int pz;               // padded z length (1 in 2-D mode)
};

// blockIdx.x = o + pz * tile; o enumerates kz so that a plane and its mirror Pz - kz,
// which read the same kernel tile, run next to each other (the second read hits L2)
BD_HD int kz_of_order(int o, int pz) {
    if (pz == 1) return 0;
    if (o < 2) return o * (pz / 2);
    return (o & 1) ? pz - (o >> 1) : (o >> 1);
}

template <int L, int NC, int COLS>
struct YFused {
    using Args = YFArgs;
    static constexpr int KIND = kKindYFused;
    static constexpr int NT = 256;
    static constexpr int NP = dec_np(L);
    static constexpr int NPHASES = 2 * NP - 1;
    static constexpr int RL = dec_rlast(L), F = L / RL, NR = F / 2 + 1;
    static constexpr int NY = L / 2;
    static BD_HD long smem_elems(const Args&) { return NP == 1 ? 0 : 3L * L * COLS; }

    struct Blk { int tile, kz, kzr; float sz; };
    static BD_HD Blk decode(int bx, const Args& a) {
        Blk b;
        const int o = bx % a.pz;
        b.tile = bx / a.pz;
        b.kz = kz_of_order(o, a.pz);
        const bool zrev = 2 * b.kz > a.pz;
        b.kzr = zrev ? a.pz - b.kz : b.kz;
        b.sz = zrev ? -1.f : 1.f;
        return b;
    }
    static BD_HD GTile<COLS> gtile(const Blk& b, int col, const Args& a) {
        const long cstride = (long)a.pz * a.ntl * NY * COLS;
        return GTile<COLS>{a.V + ((long)b.kz * a.ntl + b.tile) * NY * COLS + col, cstride};
    }

    template <int P, bool INV>
    static BD_HD void pass(int tid, int bx, const Args& a, float2* sm) {
        constexpr int ITEMS = (L / dec_r(L, P)) * COLS;
        const Blk b = decode(bx, a);
        for (int w = tid; w < ITEMS; w += NT) {
            const int col = w % COLS, it = w / COLS;
            STile<L, COLS> s{sm + col};
            if constexpr (P == 0) {
                GTile<COLS> g = gtile(b, col, a);
                if constexpr (!INV) fwd_pass3<L, 0>(it, g, s, a.ptw);
                else inv_pass3<L, 0>(it, s, g, a.ptw);
            } else if constexpr (!INV) fwd_pass3<L, P>(it, s, s, a.ptw);
            else inv_pass3<L, P>(it, s, s, a.ptw);
        }
    }

    static BD_HD void mid(int tid, int bx, const Args& a, float2* sm) {
        constexpr int ITEMS = F * COLS;
        const Blk b = decode(bx, a);
        const float* kt = a.K + ((long)b.kzr * a.ntl + b.tile) * ((long)NR * COLS * NC * RL);
        for (int w = tid; w < ITEMS; w += NT) {
            const int col = w % COLS, u = w / COLS;
            // units u < F/2: items f = u as stored; u >= F/2: f = F/2 (u = F/2, its own
            // mirror) then the mirrored items f = F - (u - F/2)
            int f = u, row = u;
            bool rev = false;
            if (F >= 2 && u >= F / 2) {
                const int up = u - F / 2;
                if (up == 0) { f = F / 2; row = F / 2; }
                else { f = F - up; row = up; rev = true; }
            }
            const int i = item_of_partial_freq(L, f);
            const float* krow = kt + ((long)row * COLS + col) * (NC * RL);
            if constexpr (NP == 1) {
                GTile<COLS> g = gtile(b, col, a);
                mid3<L, NC, false>(i, krow, b.sz, g, g);
            } else {
                STile<L, COLS> s{sm + col};
                if (rev) mid3<L, NC, true>(i, krow, b.sz, s, s);
                else mid3<L, NC, false>(i, krow, b.sz, s, s);
            }
        }
    }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        if constexpr (PH < NP - 1) pass<PH, false>(tid, bx, a, sm);
        else if constexpr (PH == NP - 1) mid(tid, bx, a, sm);
        else pass<2 * NP - 2 - PH, true>(tid, bx, a, sm);
    }
};

}  // namespace bd
