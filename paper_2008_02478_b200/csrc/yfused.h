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
// memory as S[c][p(e)][col] (p: padding, below).  The pencil index e after the forward passes is in the
// digit-reversed order of fft_core.h; the kernel spectrum is stored in the order the
// multiply meets it (kernel-spectrum tile below), real and symmetry-reduced in y and z (pin P12).
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

// ------------------------------------------------------------------ accessors
// Shared pencils are padded by one element per 8: physical index p(e) = e + (e >> 3).
// Every pass reads e = base + r S with S = 1 (base a multiple of 8) or S >= 8 (a power
// of two, r S bit-disjoint from base), so p(base + r S) = p(base) + r * pstep(S):
// addresses are one base plus compile-time offsets.  Half warps touch 16/COLS
// consecutive base indices, or items 8 apart in the last pass (stride 9): no bank
// conflicts beyond one 2-way overlap per 16 consecutive elements.
BD_HD constexpr int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }
BD_HD constexpr int padlen8(int L) { return L + (L >> 3); }
BD_HD int pidx(int e) { return e + (e >> 3); }
BD_HD constexpr int pstep(int S) { return S >= 8 ? S + (S >> 3) : S; }

// An accessor gives ptr(c, e) -> address of element e of pencil c, off(S, r) -> distance
// (in elements of the pointer) between e and e + r S, and ld() to read.
template <int L, int COLS>
struct STile {                 // shared: S[c][p(e)][col]
    float2* p;                 // already offset by col
    static constexpr int CP = padlen8(L) * COLS;
    static BD_HD constexpr int off(int S, int r) { return r * pstep(S) * COLS; }
    BD_HD float2* ptr(int c, int e) const { return p + c * CP + pidx(e) * COLS; }
    static BD_HD float2 ld(const float2* q) { return *q; }
    BD_HD void st(float2* q, float2 v) const { BD_STS(q, v); }
    BD_HD void pre(const float2*, int) const {}
    BD_HD void stq(float2* q, float2 v, int) const { BD_STS(q, v); }
};
template <int COLS>
struct GTile {                 // global: V tile [y][col], component stride cstride
    float2* p; long cstride;   // already offset by col
    static BD_HD constexpr int off(int S, int r) { return r * S * COLS; }
    BD_HD float2* ptr(int c, int e) const { return p + c * cstride + (long)e * COLS; }
    static BD_HD float2 ld(const float2* q) { return BD_LDCG(q); }     // streamed once: keep it out of L1
    BD_HD void st(float2* q, float2 v) const { *q = v; }
    BD_HD void pre(const float2*, int) const {}
    BD_HD void stq(float2* q, float2 v, int) const { *q = v; }
};

// ------------------------------------------------------------------ passes
// pencils c = c0, c0 + cstep, ... < cend share the butterfly index `it` and its twiddles
template <int L, int P, int NCT = 0, class In, class Out>
BD_HD void fwd_passM(int it, int c0, int cstep, int cend, const In& in, const Out& out, const float2* __restrict__ ptw) {
    constexpr int NP = dec_np(L), R = dec_r(L, P), Lp = dec_sublen(L, P), S = Lp / R;
    if (c0 >= cend) return;      // more row groups than rows: nothing to do (and nothing to read)
    const int blk = it / S, j = it - blk * S, base = blk * Lp + j;
    Tw tw[R];
    if constexpr (P < NP - 1) {
        BD_UNROLL
        for (int q = 1; q < R; ++q) tw[q] = make_tw(BD_LDG(&ptw[ptw_off(L, P) + (q - 1) * S + j]));
    }
    // the inputs of the next pencil are loaded before the current one is transformed
    constexpr int NIN = P == 0 ? R / 2 : R;
    float2 nxt[NIN];
    {
        const auto* pi = in.ptr(c0, base);
        BD_UNROLL
        for (int r = 0; r < NIN; ++r) nxt[r] = In::ld(pi + In::off(S, r));
    }
    // NCT > 0: the pencil count is known, the loop is unrolled and the copies below vanish
    BD_UNROLL_N(NCT > 0 ? NCT : 1)
    for (int c = c0; c < cend; c += cstep) {
        float2 v[R];
        BD_UNROLL
        for (int r = 0; r < NIN; ++r) v[r] = nxt[r];
        if (c + cstep < cend) {
            const auto* pi = in.ptr(c + cstep, base);
            BD_UNROLL
            for (int r = 0; r < NIN; ++r) nxt[r] = In::ld(pi + In::off(S, r));
        }
        if constexpr (P == 0) PkDftPruned<R, -1>::run(v);
        else PkDft<R, -1>::run(v);
        if constexpr (P < NP - 1) {
            BD_UNROLL
            for (int q = 1; q < R; ++q) v[q] = pk_cmul(v[q], tw[q]);
        }
        float2* po = out.ptr(c, base);
        BD_UNROLL
        for (int q = 0; q < R; ++q) out.st(po + Out::off(S, q), v[q]);
    }
}

template <int L, int P, int NCT = 0, class In, class Out>
BD_HD void inv_passM(int it, int c0, int cstep, int cend, const In& in, const Out& out, const float2* __restrict__ ptw) {
    constexpr int NP = dec_np(L), R = dec_r(L, P), Lp = dec_sublen(L, P), S = Lp / R;
    if (c0 >= cend) return;
    const int blk = it / S, j = it - blk * S, base = blk * Lp + j;
    Tw tw[R];
    if constexpr (P < NP - 1) {
        BD_UNROLL
        for (int q = 1; q < R; ++q) tw[q] = make_tw(BD_LDG(&ptw[ptw_off(L, P) + (q - 1) * S + j]));
    }
    float2 nxt[R];
    {
        const auto* pi = in.ptr(c0, base);
        BD_UNROLL
        for (int q = 0; q < R; ++q) nxt[q] = In::ld(pi + In::off(S, q));
    }
    BD_UNROLL_N(NCT > 0 ? NCT : 1)
    for (int c = c0; c < cend; c += cstep) {
        float2 v[R];
        BD_UNROLL
        for (int q = 0; q < R; ++q) v[q] = nxt[q];
        if (c + cstep < cend) {
            const auto* pi = in.ptr(c + cstep, base);
            BD_UNROLL
            for (int q = 0; q < R; ++q) nxt[q] = In::ld(pi + In::off(S, q));
        }
        if constexpr (P < NP - 1) {
            BD_UNROLL
            for (int q = 1; q < R; ++q) v[q] = pk_cmulc(v[q], tw[q]);
        }
        float2* po = out.ptr(c, base);
        if constexpr (P == 0) {
            // an accessor that needs something from memory per output (the fused energy) asks for it now
            BD_UNROLL
            for (int r = 0; r < R / 2; ++r) out.pre(po + Out::off(S, r), r);
            PkDftTrunc<R, +1>::run(v);
            BD_UNROLL
            for (int r = 0; r < R / 2; ++r) out.stq(po + Out::off(S, r), v[r], r);
        } else {
            PkDft<R, +1>::run(v);
            BD_UNROLL
            for (int r = 0; r < R; ++r) out.st(po + Out::off(S, r), v[r]);
        }
    }
}

template <int L, int P, class In, class Out>
BD_HD void fwd_pass3(int it, const In& in, const Out& out, const float2* __restrict__ ptw) {
    fwd_passM<L, P, 3>(it, 0, 1, 3, in, out, ptw);
}
template <int L, int P, class In, class Out>
BD_HD void inv_pass3(int it, const In& in, const Out& out, const float2* __restrict__ ptw) {
    inv_passM<L, P, 3>(it, 0, 1, 3, in, out, ptw);
}

// ------------------------------------------------------------------ kernel-spectrum tile
// K[kzr (Pz/2+1)][tile][c (NC)][chunk (RL/CH)][slot (F/2+1)][col][CH], fp32, CH = 4 floats
// (one 16-byte load; CH = RL when RL < 4).  F = L / RL items of the last pass.  Slot s
// stands for the item with frequency offset f = slot_to_f(s) <= F/2; its entry q holds
// the natural spectrum at ky = f + F q folded to [0, L/2] with the sign of the components
// odd in y applied.  Item f <= F/2 reads its slot as stored; item f > F/2 reads the slot
// of F - f with q reversed and the y-odd components negated (its frequencies are the
// mirrors L - k of that slot).  f = 0 and f = F/2 are their own mirrors.  Slots are
// numbered in the thread order of the multiply, so a warp reads consecutive 16-byte
// pieces.  A block at kz > Pz/2 reads the tile of Pz - kz and negates the z-odd components.
BD_HD constexpr int k_chunk(int L) { return dec_rlast(L) % 4 == 0 ? 4 : dec_rlast(L); }
BD_HD int slot_to_f(int L, int slot) {
    const int RL = dec_rlast(L), F = L / RL;
    if (dec_np(L) <= 2 || 2 * slot == F) return slot;
    const int R0 = dec_r(L, 0), HA = dec_r(L, 1) / 2;
    return slot / HA + R0 * (slot % HA);
}
BD_HD int f_to_slot(int L, int f) {       // f <= F/2
    const int RL = dec_rlast(L), F = L / RL;
    if (dec_np(L) <= 2 || 2 * f == F) return f;
    const int R0 = dec_r(L, 0), HA = dec_r(L, 1) / 2;
    return f / R0 + HA * (f % R0);
}

// last forward pass + multiply + first inverse pass of item i (frequency offset f)
template <int L, int NC, bool REV, bool ZREV, class In, class Out>
BD_HD void mid3(int i, const float* __restrict__ kslot, int cstride, const In& in, const Out& out) {
    constexpr int NP = dec_np(L), RL = dec_rlast(L);
    // kslot points at chunk 0 of component 0 for this thread's (slot, col); consecutive
    // chunks are cstride floats apart
    constexpr int CH = k_chunk(L), NCH = RL / CH;
    float k[NC][RL];
    BD_UNROLL
    for (int c = 0; c < NC; ++c) {
        BD_UNROLL
        for (int ch = 0; ch < NCH; ++ch) {
            const float* kp = kslot + (long)(c * NCH + ch) * cstride;
            if constexpr (CH == 4) {
                const float4 t = BD_LDCG(reinterpret_cast<const float4*>(kp));
                k[c][4 * ch] = t.x; k[c][4 * ch + 1] = t.y; k[c][4 * ch + 2] = t.z; k[c][4 * ch + 3] = t.w;
            } else {
                BD_UNROLL
                for (int q = 0; q < CH; ++q) k[c][ch * CH + q] = BD_LDG(kp + q);
            }
        }
    }
    float2 v[3][RL];
    BD_UNROLL
    for (int c = 0; c < 3; ++c) {
        if constexpr (NP == 1) {
            BD_UNROLL
            for (int q = 0; q < RL / 2; ++q) v[c][q] = In::ld(in.ptr(c, i * RL) + In::off(1, q));
            PkDftPruned<RL, -1>::run(v[c]);
        } else {
            BD_UNROLL
            for (int q = 0; q < RL; ++q) v[c][q] = In::ld(in.ptr(c, i * RL) + In::off(1, q));
            PkDft<RL, -1>::run(v[c]);
        }
    }
    // odd-component signs moved onto the data: with my' = sy my, mz' = sz mz the products
    // use the stored values and Hy = sy Hy', Hz = sz Hz'  (sy = -1 for REV, sz = -1 for ZREV)
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
            const float2 mz = ZREV ? pk_neg(v[2][q]) : v[2][q];
            const float2 kxz = pk_bc(k[4][qq]), kyz = pk_bc(k[5][qq]);
            const float2 hx = pk_fma(kxz, mz, pk_fma(kxy, my, pk_mul(kxx, mx)));
            const float2 hy = pk_fma(kyz, mz, pk_fma(kyy, my, pk_mul(kxy, mx)));
            const float2 hz = pk_fma(kzz, mz, pk_fma(kyz, my, pk_mul(kxz, mx)));
            v[0][q] = hx;
            v[1][q] = REV ? pk_neg(hy) : hy;
            v[2][q] = ZREV ? pk_neg(hz) : hz;
        }
    }
    BD_UNROLL
    for (int c = 0; c < 3; ++c) {
        if constexpr (NP == 1) {
            PkDftTrunc<RL, +1>::run(v[c]);
            BD_UNROLL
            for (int q = 0; q < RL / 2; ++q) out.ptr(c, i * RL)[Out::off(1, q)] = v[c][q];
        } else {
            PkDft<RL, +1>::run(v[c]);
            BD_UNROLL
            for (int q = 0; q < RL; ++q) out.ptr(c, i * RL)[Out::off(1, q)] = v[c][q];
        }
    }
}

// ------------------------------------------------------------------ YFused (S2+S4+S6)
struct YFArgs {
    float2* V;            // [3][Pz][ntl][ny][COLS]
    const float* K;       // [Pz/2+1][ntl][NC][RL/CH][F/2+1][COLS][CH]
    const float2* ptw;    // per-pass twiddles of length L
    int ntl;              // kx tiles
    int pz;               // padded z length (1 in 2-D mode)
    int pf;               // blocks ahead whose input tile is started towards L2 (0: none)
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
    // two 256-thread blocks per SM while two tiles fit in shared memory, else one of 512
    static constexpr bool BIG = 3L * padlen8(L) * COLS * (long)sizeof(float2) > 113L * 1024;
    static constexpr int NT = BIG ? 512 : 256;
    static constexpr int MINB = BIG ? 1 : 2;
    static constexpr int NP = dec_np(L);
    static constexpr int NPHASES = 2 * NP - 1;
    static constexpr int RL = dec_rlast(L), F = L / RL, NR = F / 2 + 1;
    static constexpr int NY = L / 2;
    static BD_HD long smem_elems(const Args&) { return NP == 1 ? 0 : 3L * padlen8(L) * COLS; }

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

    // before the predecessor kernel has finished (launcher.cuh): the block's kernel-spectrum tile starts on its way to L2
    static BD_HD void prologue(int tid, int bx, const Args& a) {
        const Blk b = decode(bx, a);
        constexpr long KB = (long)NR * COLS * NC * RL * sizeof(float);
        const char* kt = reinterpret_cast<const char*>(a.K) + ((long)b.kzr * a.ntl + b.tile) * KB;
        for (long o = (long)tid * 128; o < KB; o += NT * 128) bd_prefetch_l2(kt + o);
    }

    template <int P, bool INV>
    static BD_HD void pass(int tid, int bx, const Args& a, float2* sm) {
        constexpr int ITEMS = (L / dec_r(L, P)) * COLS;
        const Blk b = decode(bx, a);
        if constexpr (P == 0 && !INV) {
            // ... and the input tile of the block that will follow this one on the SM
            const int nb = bx + a.pf;
            if (a.pf > 0 && nb < a.ntl * a.pz) {
                const Blk n = decode(nb, a);
                const GTile<COLS> g = gtile(n, 0, a);
                constexpr long TB = (long)NY * COLS * sizeof(float2);
                for (long o = (long)tid * 128; o < 3 * TB; o += NT * 128) {
                    const long c = o / TB;
                    bd_prefetch_l2(reinterpret_cast<const char*>(g.p + c * g.cstride) + (o - c * TB));
                }
            }
        }
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
            // thread order of the multiply: first the items whose frequencies are stored as
            // they are, then their mirrors, so that a warp takes one branch; inside each
            // half the item index i = a + R1 b runs over a first (shared-memory stride 9)
            int i, f;
            if constexpr (NP <= 2) {
                i = u; f = u;
            } else {
                constexpr int R0 = dec_r(L, 0), R1 = dec_r(L, 1), HA = R1 / 2;
                const int h = u / (F / 2), t = u - h * (F / 2);
                const int av = t % HA + h * HA, bv = t / HA;
                i = av + R1 * bv; f = bv + R0 * av;
            }
            const bool rev = 2 * f > F;
            const int row = rev ? F - f : f;
            constexpr int CH = k_chunk(L), KCS = NR * COLS * CH;
            const float* krow = kt + ((long)f_to_slot(L, row) * COLS + col) * CH;
            if constexpr (NP == 1) {
                GTile<COLS> g = gtile(b, col, a);
                if (b.sz < 0.f) mid3<L, NC, false, true>(i, krow, KCS, g, g);
                else mid3<L, NC, false, false>(i, krow, KCS, g, g);
            } else {
                STile<L, COLS> s{sm + col};
                if (b.sz < 0.f) {
                    if (rev) mid3<L, NC, true, true>(i, krow, KCS, s, s);
                    else mid3<L, NC, false, true>(i, krow, KCS, s, s);
                } else {
                    if (rev) mid3<L, NC, true, false>(i, krow, KCS, s, s);
                    else mid3<L, NC, false, false>(i, krow, KCS, s, s);
                }
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
