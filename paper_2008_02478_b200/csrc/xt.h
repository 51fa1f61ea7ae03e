// xt.h — x transforms of the tiled 2-D path (nz = 1): S1 and S7 of SURVEY.md §8(a)
// ("1D FFTs along the x ... direction"; zero padding PAPER.md:L283).
//
//   XFwdT  rows of nx reals, zero-padded to Px = 2 nx -> half spectrum kx = 0..nx,
//          written into the kx-tiled array V[c][0][tile][y][col] that YFused reads
//   XInvT  the mirror: V -> rows of H, first nx outputs kept
//
// The real row is transformed as a complex row of half the padded length
// (z[m] = x[2m] + i x[2m+1], LX = nx points of which the first nx/2 are non-zero):
//   2 X[k]      = A + w_k (-i B),   A = Z[k] + conj Z[LX-k],  B = Z[k] - conj Z[LX-k]
//   2 X[LX-k]   = conj(A - w_k (-i B)),                       w_k = exp(-2 pi i k / Px)
// and back:
//   Z[k]    = E' + i O',  E' = Y[k] + conj Y[LX-k],  O' = conj(w_k) (Y[k] - conj Y[LX-k])
//   Z[LX-k] = conj(E') + i conj(O')
// The factors 2 are folded into the kernel spectrum (reading R12).
#pragma once
#include <cstring>

#include "yfused.h"

namespace bd {

// Shared rows (one pencil per row, threads of a half warp on 16 consecutive elements, on
// items 8 apart, or — the z columns of xz.h — on consecutive kx, whose positions are L/R0
// apart): padded by one element per 16 and crow(L) per 128, which keeps those patterns on
// different banks (at most 2-way conflicts) and still gives p(base + r S) = p(base) + p(r S).
BD_HD constexpr int crow(int L) { return L == 256 ? 2 : 1; }
BD_HD constexpr int prow(int L, int e) { return e + (e >> 4) + crow(L) * (e >> 7); }
template <int L>
struct SRows {
    float2* p;
    static constexpr int PITCH = (prow(L, L) + 1) | 1;        // one spare slot after the row (xz.h)
    static BD_HD constexpr int off(int S, int r) { return prow(L, r * S); }
    BD_HD float2* ptr(int row, int e) const { return p + row * PITCH + prow(L, e); }
    static BD_HD float2 ld(const float2* q) { return *q; }
    BD_HD void st(float2* q, float2 v) const { BD_STS(q, v); }
    BD_HD void pre(const float2*, int) const {}
    BD_HD void stq(float2* q, float2 v, int) const { BD_STS(q, v); }
};
struct GRowsIn {               // rows of a real array read as (x[2m], x[2m+1]) pairs
    const float* p; long pitch;
    static BD_HD constexpr int off(int S, int r) { return r * S; }
    BD_HD const float2* ptr(int row, int e) const { return reinterpret_cast<const float2*>(p + row * pitch) + e; }
    static BD_HD float2 ld(const float2* q) { return BD_LDCG(q); }
};
struct GRowsOut {
    float* p; long pitch;
    static BD_HD constexpr int off(int S, int r) { return r * S; }
    BD_HD float2* ptr(int row, int e) const { return reinterpret_cast<float2*>(p + row * pitch) + e; }
    BD_HD void st(float2* q, float2 v) const { *q = v; }
    BD_HD void pre(const float2*, int) const {}
    BD_HD void stq(float2* q, float2 v, int) const { *q = v; }
};
// H rows written, and sum M.H gathered on the way (S8 fused into S7): M has H's layout, so
// the matching M pair sits at a fixed byte distance from the H pair
struct GRowsOutE {
    float* p; long pitch; long m_minus_h; double* acc;
    static BD_HD constexpr int off(int S, int r) { return r * S; }
    BD_HD float2* ptr(int row, int e) const { return reinterpret_cast<float2*>(p + row * pitch) + e; }
    mutable float2 mbuf[8];        // M pairs of the outputs of one butterfly, loaded before it is computed
    BD_HD void pre(const float2* q, int r) const {
        mbuf[r] = BD_LDCG(reinterpret_cast<const float2*>(reinterpret_cast<const char*>(q) + m_minus_h));
    }
    BD_HD void stq(float2* q, float2 v, int r) const {
        *q = v;
        *acc += (double)mbuf[r].x * v.x + (double)mbuf[r].y * v.y;
    }
    BD_HD void st(float2* q, float2 v) const { *q = v; }
};

// H += the field instead of H = it (BORIS_DEMAG_ACCUMULATE, the additive effective field of PAPER.md:L36): the old
// pairs are loaded before the last butterfly is computed
struct GRowsOutA {
    float* p; long pitch;
    static BD_HD constexpr int off(int S, int r) { return r * S; }
    BD_HD float2* ptr(int row, int e) const { return reinterpret_cast<float2*>(p + row * pitch) + e; }
    mutable float2 hbuf[8];
    BD_HD void pre(const float2* q, int r) const { hbuf[r] = BD_LDCG(q); }
    BD_HD void stq(float2* q, float2 v, int r) const { *q = bd_f2(hbuf[r].x + v.x, hbuf[r].y + v.y); }
    BD_HD void st(float2* q, float2 v) const { *q = v; }
};

// Energy fused into the last kernel of an evaluation (boris_demag_apply_energy): every block
// leaves sum M.H of its rows in partial[block]; the block that finishes last adds them in
// index order (the ticket decides who adds, not what: E is bit-identical across calls).
struct EnergyArgs {
    const float* M;        // nullptr: no energy
    double* partial;       // one slot per block
    unsigned* ticket;
    double* E;             // device scalar
    double factor;         // -(mu0/2) hx hy hz
    int accumulate;        // 1: the last kernel adds the field to H instead of overwriting it (no energy then)
};
BD_HD void energy_finish(double acc, const EnergyArgs& en) {
#if defined(__CUDA_ARCH__)
    __shared__ double sh[32];
    __shared__ bool last;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) sh[wid] = acc;
    __syncthreads();
    if (wid == 0) {
        double v = lane < nw ? sh[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) {
            en.partial[blockIdx.x] = v;
            __threadfence();
            last = atomicAdd(en.ticket, 1u) == gridDim.x - 1;
        }
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double tot = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) tot += __ldcg(&en.partial[i]);
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    __syncthreads();
    if (lane == 0) sh[wid] = tot;
    __syncthreads();
    if (wid == 0) {
        double v = lane < nw ? sh[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) { *en.E = en.factor * v; *en.ticket = 0u; }
    }
#else
    (void)acc; (void)en;       // the host emulation checks H only
#endif
}

struct XTArgs {
    const float* M;        // [3][ny][nx]
    float* H;              // [3][ny][nx]            (XInvT)
    float2* V;             // [3][1][ntl][ny][COLS]
    const float2* ptw;     // per-pass twiddles of length LX
    const float4* xpost;   // per kp <= LX/2: (cos, sin) of exp(-2 pi i kp / Px) and, as int bits, the padded
                           // shared positions of Z[kp] and Z[LX-kp] (fill_xpost)
    int ny;
    int ntl;
    int rb;                // rows (consecutive y of one component) per block; a power of two dividing ny
    int rbs;               // log2(rb)
    EnergyArgs en;         // XInvT: energy gathered while H is written (en.M == nullptr: off)
};

BD_HD int bd_float_as_int(float f) {
#if defined(__CUDA_ARCH__)
    return __float_as_int(f);
#else
    int i; std::memcpy(&i, &f, sizeof i); return i;
#endif
}
inline void fill_xpost(float4* h, int LX) {
    const double pi = 3.14159265358979323846264338327950288;
    for (int kp = 0; kp <= LX / 2; ++kp) {
        const double a = -2.0 * pi * (double)kp / (double)(2 * LX);
        float2 w = bd_f2((float)std::cos(a), (float)std::sin(a));
        if (kp == 0) w = bd_f2(1.f, 0.f);
        if (2 * kp == LX) w = bd_f2(0.f, -1.f);
        const int pk = prow(LX, pos_of_freq(LX, kp)), pm = prow(LX, pos_of_freq(LX, (LX - kp) & (LX - 1)));
        float fk, fm;
        std::memcpy(&fk, &pk, sizeof fk); std::memcpy(&fm, &pm, sizeof fm);
        h[kp].x = w.x; h[kp].y = w.y; h[kp].z = fk; h[kp].w = fm;
    }
}

constexpr int XB = 4;     // independent items per trip of the post / pre loops

// all rows of a block through pass P; a thread keeps its butterfly index (and twiddles)
// and walks over rows
template <int LX, int P, bool INV, int NT, class In, class Out>
BD_HD void x_rows_pass(int tid, int nrows, const In& in, const Out& out, const float2* ptw) {
    constexpr int IPR = LX / dec_r(LX, P);                 // butterflies per row
    constexpr int S = dec_sublen(LX, P) / dec_r(LX, P);    // stride of the pass
    if constexpr (P >= 1 && S == 8 && 2 * IPR <= NT && NT % 16 == 0) {
        // The middle pass of a three-pass length works on runs of 8 consecutive points (16 banks): the two runs of a
        // half-warp are 64 points = 68 padded slots apart and overlap in 8 banks.  Rows 8 apart are 16 banks apart (the
        // pitch is odd), so lanes 8..15 take the same run eight rows further down: no conflicts.
        if ((nrows & 15) == 0) {
            constexpr int G2 = NT / (2 * IPR);             // threads per butterfly and half of 8 rows
            const int j = tid & 7, rh = (tid >> 3) & 1, rest = tid >> 4;
            const int it = (rest % (IPR / 8)) * 8 + j, rl = rest / (IPR / 8);
            for (int r16 = 0; r16 < nrows; r16 += 16) {
                if constexpr (!INV) fwd_passM<LX, P>(it, r16 + 8 * rh + rl, G2, r16 + 8 * rh + 8, in, out, ptw);
                else inv_passM<LX, P>(it, r16 + 8 * rh + rl, G2, r16 + 8 * rh + 8, in, out, ptw);
            }
            return;
        }
    }
    if constexpr (IPR <= NT) {
        constexpr int G = NT / IPR;
        const int it = tid % IPR, rg = tid / IPR;
        if (rg >= G) return;
        if constexpr (!INV) fwd_passM<LX, P>(it, rg, G, nrows, in, out, ptw);
        else inv_passM<LX, P>(it, rg, G, nrows, in, out, ptw);
    } else {
        for (int it = tid; it < IPR; it += NT) {
            if constexpr (!INV) fwd_passM<LX, P>(it, 0, 1, nrows, in, out, ptw);
            else inv_passM<LX, P>(it, 0, 1, nrows, in, out, ptw);
        }
    }
}

template <int LX, int COLS>
struct XFwdT {
    using Args = XTArgs;
    static constexpr int KIND = kKindXFwdT;
    static constexpr int NT = 256;
    static constexpr int MINB = 3;
    static constexpr int NP = dec_np(LX);
    static constexpr int NPHASES = NP + 1;
    static BD_HD long smem_elems(const Args& a) { return (long)a.rb * SRows<LX>::PITCH; }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        const long g0 = (long)bx * a.rb;                   // first global row (c, y0)
        SRows<LX> s{sm};
        if constexpr (PH == 0) {
            GRowsIn in{a.M + g0 * LX, LX};
            x_rows_pass<LX, 0, false, NT>(tid, a.rb, in, s, a.ptw);
        } else if constexpr (PH < NP) {
            x_rows_pass<LX, PH, false, NT>(tid, a.rb, s, s, a.ptw);
        } else {
            const int c = (int)(g0 / a.ny), y0 = (int)(g0 - (long)c * a.ny);
            const int items = (LX / 2 + 1) * a.rb;
            float2* vc = a.V + (long)c * a.ntl * a.ny * COLS;
            // XB independent items per trip: loads first, then arithmetic and stores
            for (int w0 = tid; w0 < items; w0 += XB * NT) {
                float2 Zk[XB], Zm[XB], tw[XB];
                BD_UNROLL
                for (int u = 0; u < XB; ++u) {
                    const int w = w0 + u * NT;
                    if (w < items) {
                        const int kp = w >> a.rbs, row = w & (a.rb - 1);
                        const float4 xp = BD_LDG(&a.xpost[kp]);
                        const float2* zr = sm + row * SRows<LX>::PITCH;
                        Zk[u] = zr[bd_float_as_int(xp.z)];
                        Zm[u] = zr[bd_float_as_int(xp.w)];
                        tw[u] = bd_f2(xp.x, xp.y);
                    }
                }
                BD_UNROLL
                for (int u = 0; u < XB; ++u) {
                    const int w = w0 + u * NT;
                    if (w < items) {
                        const int kp = w >> a.rbs, row = w & (a.rb - 1);
                        const int km = LX - kp;
                        const float2 A = bd_f2(Zk[u].x + Zm[u].x, Zk[u].y - Zm[u].y);
                        const float2 B = bd_f2(Zk[u].x - Zm[u].x, Zk[u].y + Zm[u].y);
                        const float2 T = pk_cmul(bd_f2(B.y, -B.x), make_tw(tw[u]));
                        const float2 Xk = pk_add(A, T), Xm = bd_f2(A.x - T.x, T.y - A.y);
                        const int y = y0 + row;
                        BD_STCG(&vc[((kp / COLS) * a.ny + y) * COLS + kp % COLS], Xk);
                        if (2 * kp != LX) BD_STCG(&vc[((km / COLS) * a.ny + y) * COLS + km % COLS], Xm);
                    }
                }
            }
        }
    }
};

template <int LX, int COLS>
struct XInvT {
    using Args = XTArgs;
    static constexpr int KIND = kKindXInvT;
    static constexpr int NT = 256;
    static constexpr int MINB = 3;
    static constexpr int NP = dec_np(LX);
    static constexpr int NPHASES = NP + 1;
    static BD_HD long smem_elems(const Args& a) { return (long)a.rb * SRows<LX>::PITCH; }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        const long g0 = (long)bx * a.rb;
        SRows<LX> s{sm};
        if constexpr (PH == 0) {
            const int c = (int)(g0 / a.ny), y0 = (int)(g0 - (long)c * a.ny);
            const int items = (LX / 2 + 1) * a.rb;
            const float2* vc = a.V + (long)c * a.ntl * a.ny * COLS;
            for (int w0 = tid; w0 < items; w0 += XB * NT) {
                float2 Yk[XB], Ym[XB];
                float4 xp[XB];
                BD_UNROLL
                for (int u = 0; u < XB; ++u) {
                    const int w = w0 + u * NT;
                    if (w < items) {
                        const int kp = w >> a.rbs, row = w & (a.rb - 1);
                        const int km = LX - kp, y = y0 + row;
                        Yk[u] = BD_LDCG(&vc[((kp / COLS) * a.ny + y) * COLS + kp % COLS]);
                        Ym[u] = BD_LDCG(&vc[((km / COLS) * a.ny + y) * COLS + km % COLS]);
                        xp[u] = BD_LDG(&a.xpost[kp]);
                    }
                }
                BD_UNROLL
                for (int u = 0; u < XB; ++u) {
                    const int w = w0 + u * NT;
                    if (w < items) {
                        const int kp = w >> a.rbs, row = w & (a.rb - 1);
                        if (kp == 0) { Yk[u].y = 0.f; Ym[u].y = 0.f; }    // DC and Nyquist of a real row are real
                        const float2 E = bd_f2(Yk[u].x + Ym[u].x, Yk[u].y - Ym[u].y);
                        const float2 D = bd_f2(Yk[u].x - Ym[u].x, Yk[u].y + Ym[u].y);
                        const float2 O = pk_cmulc(D, make_tw(bd_f2(xp[u].x, xp[u].y)));
                        float2* zr = sm + row * SRows<LX>::PITCH;
                        BD_STS(zr + bd_float_as_int(xp[u].z), bd_f2(E.x - O.y, E.y + O.x));
                        if (kp != 0 && 2 * kp != LX) BD_STS(zr + bd_float_as_int(xp[u].w), bd_f2(E.x + O.y, O.x - E.y));
                    }
                }
            }
        } else if constexpr (PH < NP) {
            x_rows_pass<LX, NP - PH, true, NT>(tid, a.rb, s, s, a.ptw);
        } else {
            if (a.en.M) {
                double acc = 0.0;
                GRowsOutE out{a.H + g0 * LX, LX, (long)((const char*)a.en.M - (const char*)a.H), &acc};
                x_rows_pass<LX, 0, true, NT>(tid, a.rb, s, out, a.ptw);
                energy_finish(acc, a.en);
            } else if (a.en.accumulate) {
                GRowsOutA out{a.H + g0 * LX, LX};
                x_rows_pass<LX, 0, true, NT>(tid, a.rb, s, out, a.ptw);
            } else {
                GRowsOut out{a.H + g0 * LX, LX};
                x_rows_pass<LX, 0, true, NT>(tid, a.rb, s, out, a.ptw);
            }
        }
    }
};

}  // namespace bd
