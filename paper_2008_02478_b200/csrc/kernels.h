// kernels.h — the chunked FALLBACK kernels of boris_demag_apply (3-D meshes the tiled
// path of xt.h / xz.h / yfused.h does not cover: DESIGN.md section 8), as sequences of
// barrier-separated phases.  Each kernel is a struct K with
//     K::NT                       threads per block
//     K::NPHASES                  phases; a __syncthreads() separates consecutive phases
//     K::smem_elems(args)         float2 elements of dynamic shared memory
//     K::phase<PH>(tid, bx, by, args, smem)
// All state that crosses a phase boundary lives in shared or global memory, so the
// same code runs as a CUDA kernel (boris_demag.cu: run_phases) and, thread by thread,
// in the host emulation of the CPU tests (tests/emu).
//
// Path:            workspace W[3][NS][nz][ny] complex
//   XFwd   S1  x: zero-pad + real->complex FFT (pruned, half-length complex trick),
//              written transposed (y fastest) so that y pencils are contiguous
//   YFwd   S2  (nz > 1) y FFT of a slab of kx slots into the L2-resident scratch T
//   ZFused S3+S4+S5: z FFT, tensor multiply, inverse z FFT in one launch (the paper's
//              pipelined kernel), in place on T
//   YInv   S6  inverse y FFT, T -> W
//   XInv   S7  complex->real inverse x FFT, W -> H
#pragma once
#include "fft_core.h"

namespace bd {

// K::KIND numbers the kernels for the per-kernel timing of boris_demag_apply_timed
constexpr int kNumKinds = 6;   // timing slots: x forward, fused y (tiled path), YFwd, ZFused, YInv, x inverse

// ------------------------------------------------------------------ accessors
struct SmemPencil {            // contiguous padded pencils, one buffer per component
    float2* base; int cpitch;
    BD_HD float2 get(int c, int e) const { return base[c * cpitch + padidx(e)]; }
    BD_HD void put(int c, int e, float2 v) const { base[c * cpitch + padidx(e)] = v; }
};
struct SmemInterleaved {       // TY pencils interleaved: element e of pencil t at e*TY + t
    float2* base; int cpitch; int ty;
    BD_HD float2 get(int c, int e) const { return base[c * cpitch + e * ty]; }
    BD_HD void put(int c, int e, float2 v) const { base[c * cpitch + e * ty] = v; }
};
struct GlobalPencil {          // element e of component c at p[c*cstride + e*estride]
    float2* p; long cstride; long estride;
    BD_HD float2 get(int c, int e) const { return p[c * cstride + e * estride]; }
    BD_HD void put(int c, int e, float2 v) const { p[c * cstride + e * estride] = v; }
};
struct GlobalConstPencil {
    const float2* p; long cstride; long estride;
    BD_HD float2 get(int c, int e) const { return BD_LDG(&p[c * cstride + e * estride]); }
};

// ------------------------------------------------------------------ XFwd (S1)
struct XArgs {
    const float* M;        // [3][nz][ny][nx]
    float* H;              // [3][nz][ny][nx]   (XInv)
    float2* W;             // [3][NS][nz][ny]
    const float2* tw;      // exp(-2 pi i k / LX), k < LX
    const float2* twx;     // exp(-2 pi i k / Px), k <= LX/2
    int ny, nz;
    int rb;                // rows (consecutive y, same c and z) per block; power of two dividing ny
};

// Row of nx = LX reals, zero-padded to Px = 2 LX.  z[m] = x[2m] + i x[2m+1] (m < LX/2
// non-zero), Z = FFT_LX(z); then, with E, O the transforms of the even/odd samples,
//   2 X[k]      = A + w_k (-i B),   A = Z[k] + conj Z[LX-k],  B = Z[k] - conj Z[LX-k]
//   2 X[LX-k]   = conj(A - w_k (-i B)),                       w_k = exp(-2 pi i k / Px)
// The factor 2 is folded into the kernel spectrum.
template <int LX>
struct XFwd {
    using Args = XArgs;
    static constexpr int KIND = 0;
    static constexpr int NT = 256;
    static constexpr int NP = dec_np(LX);
    static constexpr int NPHASES = NP + 1;
    static constexpr int PITCH = padlen(LX) | 1;     // odd: rows land in different banks
    static constexpr int NS = LX + 1;
    static BD_HD long smem_elems(const Args& a) { return (long)a.rb * PITCH; }

    template <int P>
    static BD_HD void pass(int tid, long g0, const Args& a, float2* sm) {
        constexpr int IPR = LX / dec_r(LX, P);       // butterflies per row
        const int items = a.rb * IPR;
        for (int w = tid; w < items; w += NT) {
            const int row = w / IPR, it = w - row * IPR;
            SmemPencil s{sm + row * PITCH, 0};
            if constexpr (P == 0) {
                GlobalConstPencil in{reinterpret_cast<const float2*>(a.M + (g0 + row) * (long)LX), 0, 1};
                fwd_pass<LX, 0>(0, it, in, s, a.tw);
            } else {
                fwd_pass<LX, P>(0, it, s, s, a.tw);
            }
        }
    }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        const long g0 = (long)bx * a.rb;             // first global row (c, z, y0)
        if constexpr (PH < NP) {
            pass<PH>(tid, g0, a, sm);
        } else {
            const int c = (int)(g0 / ((long)a.nz * a.ny));
            const int rem = (int)(g0 - (long)c * a.nz * a.ny);
            const int z = rem / a.ny, y0 = rem - z * a.ny;
            const int items = (LX / 2 + 1) * a.rb;
            for (int w = tid; w < items; w += NT) {
                const int kp = w / a.rb, row = w - kp * a.rb;
                const float2* zb = sm + row * PITCH;
                const int m = (LX - kp) & (LX - 1);
                const float2 Zk = zb[padidx(pos_of_freq(LX, kp))];
                const float2 Zm = zb[padidx(pos_of_freq(LX, m))];
                const float2 A = bd_f2(Zk.x + Zm.x, Zk.y - Zm.y);
                const float2 B = bd_f2(Zk.x - Zm.x, Zk.y + Zm.y);
                const float2 T = cmul(BD_LDG(&a.twx[kp]), bd_f2(B.y, -B.x));
                float2* out = a.W + ((long)c * NS * a.nz + z) * a.ny + y0 + row;
                const long sstride = (long)a.nz * a.ny;
                const float2 Xk = cadd(A, T), Xm = cconj(csub(A, T));
                if (kp == 0) {
                    out[0] = Xk;
                    out[(long)LX * sstride] = Xm;
                } else {
                    out[(long)kp * sstride] = Xk;
                    if (2 * kp != LX) out[(long)(LX - kp) * sstride] = Xm;
                }
            }
        }
    }
};

// ------------------------------------------------------------------ XInv (S7)
// Hermitian half spectrum Y[k], k = 0..LX, of a real row of length Px = 2 LX:
//   Z[k]    = E' + i O',  E' = Y[k] + conj Y[LX-k],  O' = conj(w_k) (Y[k] - conj Y[LX-k])
//   Z[LX-k] = conj(E') + i conj(O')
// z = IFFT_LX(Z) (unnormalised) = (x[2m], x[2m+1]); only m < LX/2 is kept.
template <int LX>
struct XInv {
    using Args = XArgs;
    static constexpr int KIND = 5;
    static constexpr int NT = 256;
    static constexpr int NP = dec_np(LX);
    static constexpr int NPHASES = NP + 1;
    static constexpr int PITCH = padlen(LX) | 1;
    static constexpr int NS = LX + 1;
    static BD_HD long smem_elems(const Args& a) { return (long)a.rb * PITCH; }

    template <int P>
    static BD_HD void pass(int tid, long g0, const Args& a, float2* sm) {
        constexpr int IPR = LX / dec_r(LX, P);
        const int items = a.rb * IPR;
        for (int w = tid; w < items; w += NT) {
            const int row = w / IPR, it = w - row * IPR;
            SmemPencil s{sm + row * PITCH, 0};
            if constexpr (P == 0) {
                GlobalPencil out{reinterpret_cast<float2*>(a.H + (g0 + row) * (long)LX), 0, 1};
                inv_pass<LX, 0>(0, it, s, out, a.tw);
            } else {
                inv_pass<LX, P>(0, it, s, s, a.tw);
            }
        }
    }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        const long g0 = (long)bx * a.rb;
        if constexpr (PH == 0) {
            const int c = (int)(g0 / ((long)a.nz * a.ny));
            const int rem = (int)(g0 - (long)c * a.nz * a.ny);
            const int z = rem / a.ny, y0 = rem - z * a.ny;
            const int items = (LX / 2 + 1) * a.rb;
            for (int w = tid; w < items; w += NT) {
                const int kp = w / a.rb, row = w - kp * a.rb;
                float2* zb = sm + row * PITCH;
                const float2* in = a.W + ((long)c * NS * a.nz + z) * a.ny + y0 + row;
                const long sstride = (long)a.nz * a.ny;
                float2 Yk = in[(long)kp * sstride];
                float2 Ym = in[(long)(LX - kp) * sstride];
                if (kp == 0) { Yk.y = 0.f; Ym.y = 0.f; }          // DC and Nyquist of a real row are real
                const float2 E = bd_f2(Yk.x + Ym.x, Yk.y - Ym.y);
                const float2 D = bd_f2(Yk.x - Ym.x, Yk.y + Ym.y);
                const float2 O = cmulc(D, BD_LDG(&a.twx[kp]));
                zb[padidx(pos_of_freq(LX, kp))] = bd_f2(E.x - O.y, E.y + O.x);
                if (kp != 0 && 2 * kp != LX)
                    zb[padidx(pos_of_freq(LX, LX - kp))] = bd_f2(E.x + O.y, O.x - E.y);
            }
        } else {
            // phases 1..NP run inverse passes NP-1..0
            pass<NP - PH>(tid, g0, a, sm);
        }
    }
};

// ------------------------------------------------------------------ fused kernels (S2+S4+S6 / S3+S4+S5)
struct KAcc3D {                 // K[slot][ytile][c(6)][q(RL)][row][t]
    const float* p; int nrows; int rl; int ty;
    BD_HD float get(int c, int q, int row) const { return BD_LDG(&p[(((long)c * rl + q) * nrows + row) * ty]); }
};

struct FusedArgs {
    float2* D;             // T [3][CS][nz][Py]
    const float* K;        // kernel spectrum in fused-pass order
    const float2* tw;      // exp(-2 pi i k / L)
    int npencils;          // unused
    int nb;                // unused
    int py;                // ZFused: padded y length (pencil stride)
    int cs, s0;            // ZFused: slots in this chunk, first global slot
    int ty;                // ZFused: pencils per block (power of two, divides py)
};

// nz > 1: one block = ty adjacent y positions x 3 components of one kx slot; pencils
// along z have stride py.  T holds nz planes per (component, slot): z stays unpadded
// in memory, the padded z spectrum exists only in shared memory.
template <int L>
struct ZFused {
    using Args = FusedArgs;
    static constexpr int KIND = 3;
    static constexpr int NT = 128;
    static constexpr int NP = dec_np(L);
    static constexpr int NPHASES = 2 * NP - 1;
    static constexpr int RL = dec_rlast(L);
    static BD_HD long smem_elems(const Args& a) { return NP == 1 ? 0 : (long)3 * L * a.ty; }

    static BD_HD GlobalPencil gacc(int bx, int by, int t, const Args& a) {
        const long cstride = (long)a.cs * (L / 2) * a.py;
        return GlobalPencil{a.D + ((long)by * (L / 2)) * a.py + (long)bx * a.ty + t, cstride, (long)a.py};
    }

    template <int P, bool INV>
    static BD_HD void pass(int tid, int bx, int by, const Args& a, float2* sm) {
        constexpr int IPP = L / dec_r(L, P);
        const int items = 3 * IPP * a.ty;
        for (int w = tid; w < items; w += NT) {
            const int t = w & (a.ty - 1), rest = w / a.ty;
            const int c = rest / IPP, it = rest - c * IPP;
            SmemInterleaved s{sm + t, L * a.ty, a.ty};
            if constexpr (P == 0) {
                GlobalPencil g = gacc(bx, by, t, a);
                if constexpr (!INV) fwd_pass<L, 0>(c, it, g, s, a.tw);
                else inv_pass<L, 0>(c, it, s, g, a.tw);
            } else if constexpr (!INV) fwd_pass<L, P>(c, it, s, s, a.tw);
            else inv_pass<L, P>(c, it, s, s, a.tw);
        }
    }

    static BD_HD void mid(int tid, int bx, int by, const Args& a, float2* sm) {
        constexpr int F = dec_items(L);
        const int items = F * a.ty;
        const int nrows = khat_rows(L);
        const int ntiles = a.py / a.ty;
        for (int w = tid; w < items; w += NT) {
            const int t = w & (a.ty - 1), i = w / a.ty;
            const long blk = ((long)(a.s0 + by) * ntiles + bx) * 6 * RL * nrows * a.ty;
            KAcc3D K{a.K + blk + t, nrows, RL, a.ty};
            if constexpr (NP == 1) {
                GlobalPencil g = gacc(bx, by, t, a);
                fused_mid<L, 6>(i, g, g, K);
            } else {
                SmemInterleaved s{sm + t, L * a.ty, a.ty};
                fused_mid<L, 6>(i, s, s, K);
            }
        }
    }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        if constexpr (PH < NP - 1) pass<PH, false>(tid, bx, by, a, sm);
        else if constexpr (PH == NP - 1) mid(tid, bx, by, a, sm);
        else pass<2 * NP - 2 - PH, true>(tid, bx, by, a, sm);
    }
};

// ------------------------------------------------------------------ YFwd / YInv (S2, S6; nz > 1)
struct YArgs {
    const float2* src; float2* dst;
    long src_pitch, dst_pitch;       // elements between consecutive rows
    long src_cstride, dst_cstride;   // elements between components (blockIdx.y = component)
    int rows;                        // rows per component
    int nb;                          // rows per block
    const float2* tw;
};

template <int L, bool INV>
struct YPass {
    using Args = YArgs;
    static constexpr int KIND = INV ? 4 : 2;
    static constexpr int NT = 128;
    static constexpr int NP = dec_np(L);
    static constexpr int NPHASES = NP;
    static constexpr int PL = padlen(L);
    static BD_HD long smem_elems(const Args& a) { return NP == 1 ? 0 : (long)a.nb * PL; }

    // forward: phases 0..NP-1 = passes 0..NP-1; inverse: phases 0..NP-1 = passes NP-1..0
    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        constexpr int P = INV ? NP - 1 - PH : PH;
        constexpr int IPP = L / dec_r(L, P);
        constexpr bool FIRST = PH == 0, LAST = PH == NP - 1;
        const int items = a.nb * IPP;
        for (int w = tid; w < items; w += NT) {
            const int pb = w / IPP, it = w - pb * IPP;
            const int row = bx * a.nb + pb;
            if (row >= a.rows) continue;
            SmemPencil s{sm + (long)pb * PL, 0};
            GlobalConstPencil gi{a.src + by * a.src_cstride + row * a.src_pitch, 0, 1};
            GlobalPencil go{a.dst + by * a.dst_cstride + row * a.dst_pitch, 0, 1};
            if constexpr (!INV) {
                if constexpr (FIRST && LAST) fwd_pass<L, P>(0, it, gi, go, a.tw);
                else if constexpr (FIRST) fwd_pass<L, P>(0, it, gi, s, a.tw);
                else if constexpr (LAST) fwd_pass<L, P>(0, it, s, go, a.tw);
                else fwd_pass<L, P>(0, it, s, s, a.tw);
            } else {
                if constexpr (FIRST && LAST) inv_pass<L, P>(0, it, gi, go, a.tw);
                else if constexpr (FIRST) inv_pass<L, P>(0, it, gi, s, a.tw);
                else if constexpr (LAST) inv_pass<L, P>(0, it, s, go, a.tw);
                else inv_pass<L, P>(0, it, s, s, a.tw);
            }
        }
    }
};

}  // namespace bd
