// xz.h — x and z transforms of the tiled 3-D path (nz = 2..32): S1+S3 and S5+S7 of
// SURVEY.md §8(a) ("1D FFTs along the x, y, z directions"; zero padding L283).
//
//   XZFwd  one block per (component, y): the nz rows M[c][:][y][:] are transformed along
//          x in shared memory (real rows as half-length complex rows, xt.h), then every
//          kx column is transformed along z in registers (nz -> Pz = 2 nz, pruned) and
//          written to the kx-tiled spectrum V[c][kz][tile][y][col] that YFused reads.
//   ZXInv  the mirror: V -> inverse z (first nz outputs kept) -> inverse x -> H rows.
//
// The kx = 0 and kx = nx (Nyquist) columns of a real row are real; they travel through
// the z transform as the one complex column P = X[0] + i X[nx] and are separated after it
// (X0^[kz] = (P^[kz] + conj P^[Pz-kz]) / 2, XN^[kz] = (P^[kz] - conj P^[Pz-kz]) / 2i), so
// a block has exactly nx columns of work.
#pragma once
#include "xt.h"

namespace bd {

// cos(2 pi m / 64): the first quarter turn rounded once from fp64, the rest by symmetry (m is known after unrolling)
BD_HD constexpr float cos64(int m) {
    constexpr float q[17] = {
        1.000000000e+00f, 9.951847267e-01f, 9.807852804e-01f, 9.569403357e-01f, 9.238795325e-01f, 8.819212643e-01f,
        8.314696123e-01f, 7.730104534e-01f, 7.071067812e-01f, 6.343932842e-01f, 5.555702330e-01f, 4.713967368e-01f,
        3.826834324e-01f, 2.902846773e-01f, 1.950903220e-01f, 9.801714033e-02f, 0.000000000e+00f
    };
    m &= 63;
    return m <= 16 ? q[m] : (m <= 32 ? -q[32 - m] : (m <= 48 ? -q[m - 32] : q[64 - m]));
}
BD_HD constexpr float sin64(int m) { return cos64(m - 16); }

// z * exp(DIR 2 pi i m / 64), m known after unrolling
template <int DIR>
BD_HD float2 pk_mul_w64(float2 z, int m) {
    m &= 63;
    if (m == 0) return z;
    if (m == 32) return pk_neg(z);
    if (m == 16) return pk_ib<DIR>(z);
    if (m == 48) return pk_ib<-DIR>(z);
    const float c = cos64(m), s = (float)DIR * sin64(m);
    return pk_fma(pk_swap(z), bd_f2(-s, s), pk_mul(z, pk_bc(c)));
}

// Column transforms in registers, one half of the padded spectrum at a time (a column of
// PZ = 2 NZ points would not fit the register budget of a 512-thread block):
//   fwd_half<PAR>: x[0..NZ) (zero-padded to PZ) -> v[k] = X[2k + PAR]
//                  X[2k + PAR] = sum_z (x[z] W_PZ^(PAR z)) W_NZ^(k z)
//   inv_half<PAR>: v[k] = Y[2k + PAR] -> the part of x[z], z < NZ, carried by those
//                  frequencies: W_PZ^(-PAR z) sum_k Y[2k + PAR] W_NZ^(-k z)   (unnormalised)
template <int PZ>
struct ZCol {
    static constexpr int NZ = PZ / 2;
    template <int PAR>
    static BD_HD void fwd_half(float2* v) {
        if constexpr (PAR == 1) {
            BD_UNROLL
            for (int z = 0; z < NZ; ++z) v[z] = pk_mul_w64<-1>(v[z], z * (64 / PZ));
        }
        PkDft<NZ, -1>::run(v);
    }
    template <int PAR>
    static BD_HD void inv_half(float2* v) {
        PkDft<NZ, +1>::run(v);
        if constexpr (PAR == 1) {
            BD_UNROLL
            for (int z = 0; z < NZ; ++z) v[z] = pk_mul_w64<+1>(v[z], z * (64 / PZ));
        }
    }
};

struct XZArgs {
    const float* M;        // [3][nz][ny][nx]
    float* H;              // [3][nz][ny][nx]            (ZXInv)
    float2* V;             // [3][Pz][ntl][ny][cols]
    const float2* ptw;     // per-pass twiddles of length LX
    const float4* xpost;   // fill_xpost table
    int ny;
    int ntl;
    int cs;                // log2(cols)
    const float2* ztw;     // exp(-2 pi i n / Pz), n < Pz   (columns longer than 64 points)
    int pf;                // blocks ahead whose input rows are started towards L2 (0: none; XZFwd)
    EnergyArgs en;         // ZXInv: energy gathered while H is written (en.M == nullptr: off)
};

// Columns of more than 64 points (nz > 32) go through the registers in SP = Pz / 32 passes
// of 32-point transforms:
//   forward, pass p:  X[SP k + p] = sum_{z' < 32} W_32^(k z') [ W_Pz^(p z') sum_{m < SP/2} x[z' + 32 m] W_SP^(p m) ]
//   inverse, pass p:  x[z' + 32 m] += W_SP^(-p m) W_Pz^(-p z') sum_k Y[SP k + p] W_32^(-k z')      (m < SP/2)
// with the unit roots read from the table ztw (W_SP^(p m) = W_Pz^(32 p m)).  The DC and
// Nyquist columns of x are then kept as two separate columns (the Nyquist one in the
// spare slot after each row), because a pass does not hold both members of a mirror pair.
template <int NZ>
struct ZSplit {
    static constexpr bool ON = NZ > 32;
    static constexpr int SUB = ON ? 32 : NZ, PZ = 2 * NZ, SP = PZ / SUB;
};
BD_HD float2 pk_cmul2(float2 a, float2 w) { return pk_cmul(a, make_tw(w)); }
BD_HD float2 pk_cmulc2(float2 a, float2 w) { return pk_cmulc(a, make_tw(w)); }

// body(kp, row, xp) for kp = 0..LX/2 and row < nrows: a thread keeps kp (and its xpost entry)
// and walks over rows; kp = LX/2, its own mirror, is taken by one thread per row at the end
template <int LX, int NT, class Body>
BD_HD void for_kp_rows(int tid, int nrows, const float4* __restrict__ xpost, Body&& body) {
    constexpr int HK = LX / 2;
    if constexpr (HK <= NT) {
        constexpr int G = NT / HK;
        const int kp = tid % HK, rg = tid / HK;
        if (rg < G) {
            const float4 xp = BD_LDG(&xpost[kp]);
            for (int row = rg; row < nrows; row += G) body(kp, row, xp);
        }
    } else {
        for (int kp = tid; kp < HK; kp += NT) {
            const float4 xp = BD_LDG(&xpost[kp]);
            for (int row = 0; row < nrows; ++row) body(kp, row, xp);
        }
    }
    const float4 xh = BD_LDG(&xpost[HK]);
    for (int row = tid; row < nrows; row += NT) body(HK, row, xh);
}

// shared position of X[kx] (kx < LX) inside a row, from the xpost table
BD_HD int xz_pos(const float4* __restrict__ xpost, int LX, int kx) {
    return 2 * kx <= LX ? bd_float_as_int(BD_LDG(&xpost[kx]).z) : bd_float_as_int(BD_LDG(&xpost[LX - kx]).w);
}

template <int LX, int NZ>
struct XZFwd {
    using Args = XZArgs;
    static constexpr int KIND = kKindXZFwd;
    static constexpr int NT = 512;
    static constexpr int MINB = 1;
    static constexpr int NP = dec_np(LX);
    static constexpr int NPHASES = NP + 2;
    static constexpr int PZ = 2 * NZ;
    static constexpr int PITCH = SRows<LX>::PITCH;
    // nz > 32: behind the rows, the twiddles of the z passes in the order the lanes read them, stw[z SP + p] = W_PZ^(p z)
    // (neighbouring lanes = neighbouring passes of a column: one wavefront per load, and no global load in the z stage)
    static BD_HD long smem_elems(const Args&) { return (long)NZ * PITCH + (ZSplit<NZ>::ON ? PZ : 0); }

    // pass p of one column (nz > 32, ZSplit): frequencies kz = SP k + p
    static BD_HD void zpass(const float2* col, float2* out, long kzs, int p, const float2* __restrict__ ztw, const float2* stw) {
        constexpr int SUB = ZSplit<NZ>::SUB, SP = ZSplit<NZ>::SP;
        float2 v[SUB];
        BD_UNROLL
        for (int z = 0; z < SUB; ++z) v[z] = col[z * PITCH];
        for (int m = 1; m < SP / 2; ++m) {
            const Tw w = make_tw(BD_LDG(&ztw[(p * m * SUB) & (PZ - 1)]));
            BD_UNROLL
            for (int z = 0; z < SUB; ++z) v[z] = pk_add(v[z], pk_cmul(col[(z + SUB * m) * PITCH], w));
        }
        if (p != 0) {
            BD_UNROLL
            for (int z = 1; z < SUB; ++z) v[z] = pk_cmul2(v[z], stw[z * SP + p]);
        }
        PkDft<SUB, -1>::run(v);
        out += p * kzs;
        BD_UNROLL
        for (int k = 0; k < SUB; ++k) { BD_STCG(out, v[k]); out += SP * kzs; }
    }

    // frequencies kz = 2k + PAR of one column; column 0 carries P = X[0] + i X[LX]
    template <int PAR>
    static BD_HD void zhalf(const float2* col, float2* out, float2* outn, long kzs, int kx) {
        float2 v[NZ];
        BD_UNROLL
        for (int z = 0; z < NZ; ++z) v[z] = col[z * PITCH];
        ZCol<PZ>::template fwd_half<PAR>(v);
        out += PAR * kzs; outn += PAR * kzs;
        if (kx != 0) {
            BD_UNROLL
            for (int k = 0; k < NZ; ++k) { BD_STCG(out, v[k]); out += 2 * kzs; }
        } else {
            BD_UNROLL
            for (int k = 0; k < NZ; ++k) {
                // mirror frequency PZ - (2k + PAR) sits in the same half at index km
                const int km = PAR ? NZ - 1 - k : (NZ - k) % NZ;
                const float2 p = v[k], m = v[km];
                BD_STCG(out, bd_f2(0.5f * (p.x + m.x), 0.5f * (p.y - m.y)));
                BD_STCG(outn, bd_f2(0.5f * (p.y + m.y), 0.5f * (m.x - p.x)));
                out += 2 * kzs; outn += 2 * kzs;
            }
        }
    }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        const int c = bx / a.ny, y = bx - c * a.ny;
        SRows<LX> s{sm};
        if constexpr (PH == 0) {
            GRowsIn in{a.M + ((long)c * NZ * a.ny + y) * LX, (long)a.ny * LX};
            const int nb = bx + a.pf;                      // rows of the block that follows this one on the SM
            if (a.pf > 0 && nb < 3 * a.ny) {
                const int cn = nb / a.ny, yn = nb - cn * a.ny;
                const char* mn = reinterpret_cast<const char*>(a.M + ((long)cn * NZ * a.ny + yn) * LX);
                constexpr int LPR = LX * 4 / 128 > 0 ? LX * 4 / 128 : 1;         // 128-byte lines per row
                for (int o = tid; o < NZ * LPR; o += NT)
                    bd_prefetch_l2(mn + (long)(o / LPR) * a.ny * LX * 4 + (o % LPR) * 128);
            }
            if constexpr (ZSplit<NZ>::ON) {
                constexpr int SP = ZSplit<NZ>::SP;
                for (int i = tid; i < PZ; i += NT) sm[NZ * PITCH + i] = BD_LDG(&a.ztw[((i % SP) * (i / SP)) & (PZ - 1)]);
            }
            x_rows_pass<LX, 0, false, NT>(tid, NZ, in, s, a.ptw);
        } else if constexpr (PH < NP) {
            x_rows_pass<LX, PH, false, NT>(tid, NZ, s, s, a.ptw);
        } else if constexpr (PH == NP) {
            // untangle in place: Z[kp], Z[LX-kp] -> X[kp], X[LX-kp]; kp = 0 -> P = (X[0], X[LX])
            for_kp_rows<LX, NT>(tid, NZ, a.xpost, [&](int kp, int row, const float4& xp) {
                float2* zr = sm + row * PITCH;
                const int pk = bd_float_as_int(xp.z), pm = bd_float_as_int(xp.w);
                const float2 Zk = zr[pk], Zm = zr[pm];
                const float2 A = bd_f2(Zk.x + Zm.x, Zk.y - Zm.y);
                const float2 B = bd_f2(Zk.x - Zm.x, Zk.y + Zm.y);
                const float2 T = pk_cmul(bd_f2(B.y, -B.x), make_tw(bd_f2(xp.x, xp.y)));
                const float2 Xk = pk_add(A, T), Xm = bd_f2(A.x - T.x, T.y - A.y);
                if (kp == 0) {
                    if constexpr (ZSplit<NZ>::ON) {
                        zr[pk] = Xk;
                        zr[prow(LX, LX)] = Xm;
                    } else {
                        zr[pk] = bd_f2(Xk.x, Xm.x);
                    }
                } else {
                    zr[pk] = Xk;
                    if (2 * kp != LX) zr[pm] = Xm;
                }
            });
        } else {
            const int cols = 1 << a.cs;
            const long kzs = (long)a.ntl * a.ny * cols;                 // elements between kz planes
            float2* vc = a.V + (long)c * PZ * kzs;
            if constexpr (ZSplit<NZ>::ON) {
                constexpr int SP = ZSplit<NZ>::SP;
                for (int w = tid; w < (LX + 1) * SP; w += NT) {       // one (column, pass) per trip
                    const int kx = w / SP, p = w - kx * SP;
                    const float2* col = sm + (kx == LX ? prow(LX, LX) : xz_pos(a.xpost, LX, kx));
                    float2* out = vc + ((long)((kx >> a.cs) * a.ny + y) << a.cs) + (kx & (cols - 1));
                    zpass(col, out, kzs, p, a.ztw, sm + NZ * PITCH);
                }
            } else {
                for (int kx = tid; kx < LX; kx += NT) {
                    const float2* col = sm + xz_pos(a.xpost, LX, kx);
                    float2* out = vc + ((long)((kx >> a.cs) * a.ny + y) << a.cs) + (kx & (cols - 1));
                    float2* outn = vc + ((long)((LX >> a.cs) * a.ny + y) << a.cs) + (LX & (cols - 1));
                    zhalf<0>(col, out, outn, kzs, kx);
                    zhalf<1>(col, out, outn, kzs, kx);
                }
            }
        }
    }
};

template <int LX, int NZ>
struct ZXInv {
    using Args = XZArgs;
    static constexpr int KIND = kKindZXInv;
    static constexpr int NT = 512;
    static constexpr int MINB = 1;
    static constexpr int NP = dec_np(LX);
    static constexpr int NPHASES = NP + 2;
    static constexpr int PZ = 2 * NZ;
    static constexpr int PITCH = SRows<LX>::PITCH;
    static BD_HD long smem_elems(const Args&) { return (long)NZ * PITCH + (ZSplit<NZ>::ON ? PZ : 0); }     // + the twiddle table of XZFwd

    // all passes of one column (nz > 32, ZSplit)
    static BD_HD void zcolumn(const float2* in, float2* col, long kzs, const float2* __restrict__ ztw) {
        constexpr int SUB = ZSplit<NZ>::SUB, SP = ZSplit<NZ>::SP;
        for (int p = 0; p < SP; ++p) {
            float2 v[SUB];
            const float2* ip = in + p * kzs;
            for (int k = 0; k < SUB; ++k) { v[k] = BD_LDCG(ip); ip += SP * kzs; }
            PkDft<SUB, +1>::run(v);
            if (p != 0) {
                BD_UNROLL
                for (int z = 1; z < SUB; ++z) v[z] = pk_cmulc2(v[z], BD_LDG(&ztw[p * z]));
            }
            if (p == 0) {
                for (int m = 0; m < SP / 2; ++m) {
                    BD_UNROLL
                    for (int z = 0; z < SUB; ++z) BD_STS(col + (z + SUB * m) * PITCH, v[z]);
                }
            } else {
                for (int m = 0; m < SP / 2; ++m) {
                    const Tw w = make_tw(BD_LDG(&ztw[(p * m * SUB) & (PZ - 1)]));
                    BD_UNROLL
                    for (int z = 0; z < SUB; ++z) {
                        float2* q = col + (z + SUB * m) * PITCH;
                        BD_STS(q, pk_add(*q, pk_cmulc(v[z], w)));
                    }
                }
            }
        }
    }

#if defined(__CUDA_ARCH__)
    // The same column by SP lanes of one warp, lane p = its pass: u_p[z] = W_PZ^(-p z) (32-point inverse transform of the
    // inputs p + SP k), then x[z + 32 m] = sum_p u_p[z] w^(p m), w = exp(2 pi i / SP), m < SP / 2, across the lanes: a
    // radix-2 inverse transform over p truncated to its first half, one stage per lane distance D = T / 2 (T = SP, SP / 2, ..):
    //   even m = 2 m':  sum_(p < D) (u_p + u_(p+D)) w_D^(p m'),      odd m = 2 m' + 1:  sum_(p < D) (u_p - u_(p+D)) w_T^p w_D^(p m')
    // - two problems of half the size.  Lane p < D keeps the lower half of the z range of both, lane p + D the upper half: a lane
    // always holds 32 values (2^s vectors of 32 / 2^s points) and ends with the SP / 2 outputs m of the 32 / SP points z from
    // z = p 32 / SP on.  (The last stage, T = 2, has only m' = 0.)  Every lane of the warp must call (full-mask shuffles).
    template <int T, int NV>
    static __device__ __forceinline__ void lanes_stage(float2 (&a)[32], int p, const float2* __restrict__ ztw) {
        constexpr int D = T / 2, LEN = 32 / NV, HL = LEN / 2;
        const bool hi = (p & D) != 0;
        const float sg = hi ? -1.f : 1.f;
        float2 b[32];
        Tw w;
        if constexpr (T > 2) w = make_tw(BD_LDG(&ztw[(p & (D - 1)) * (PZ / T)]));
        BD_UNROLL
        for (int v = 0; v < NV; ++v) {
            BD_UNROLL
            for (int z = 0; z < HL; ++z) {
                const float2 lo = a[v * LEN + z], up = a[v * LEN + HL + z];
                const float2 mine = hi ? up : lo, send = hi ? lo : up;
                float2 oth;
                oth.x = __shfl_xor_sync(0xffffffffu, send.x, D);
                oth.y = __shfl_xor_sync(0xffffffffu, send.y, D);
                if constexpr (T > 2) {
                    b[(2 * v) * HL + z] = pk_add(mine, oth);
                    b[(2 * v + 1) * HL + z] = pk_cmulc(pk_mul(pk_sub(mine, oth), pk_bc(sg)), w);
                } else {
                    b[v * HL + z] = pk_add(mine, oth);
                }
            }
        }
        BD_UNROLL
        for (int i = 0; i < (T > 2 ? 32 : 16); ++i) a[i] = b[i];
        if constexpr (T > 2) lanes_stage<T / 2, 2 * NV>(a, p, ztw);
    }
    // inn / coln (column 0 only, else null): the Nyquist column kx = LX rides along as the imaginary part, P^ = Y0^ + i YN^ —
    // both are spectra of real columns, so the transform of P^ has x0 in its real and xN in its imaginary part; column 0
    // keeps the pair (the x pre-pass reads its real part only), the Nyquist slot gets (xN, 0)
    static __device__ __forceinline__ void zcolumn_lanes(const float2* in, const float2* inn, float2* col, float2* coln, long kzs, int p,
                                                         bool active, const float2* __restrict__ ztw, const float2* stw) {
        constexpr int SUB = ZSplit<NZ>::SUB, SP = ZSplit<NZ>::SP;
        static_assert(SUB == 32 && (SP == 4 || SP == 8 || SP == 16), "32-point passes on 4, 8 or 16 lanes");
        float2 v[32];
        if (active) {
            const float2* ip = in + p * kzs;
            BD_UNROLL
            for (int k = 0; k < SUB; ++k) { v[k] = BD_LDCG(ip); ip += SP * kzs; }
            if (inn) {
                const float2* np = inn + p * kzs;
                BD_UNROLL
                for (int k = 0; k < SUB; ++k) { const float2 n = BD_LDCG(np); np += SP * kzs; v[k] = bd_f2(v[k].x - n.y, v[k].y + n.x); }
            }
        } else {
            BD_UNROLL
            for (int k = 0; k < SUB; ++k) v[k] = bd_f2(0.f, 0.f);
        }
        PkDft<SUB, +1>::run(v);
        BD_UNROLL
        for (int z = 1; z < SUB; ++z) v[z] = pk_cmulc2(v[z], stw[z * SP + p]);
        lanes_stage<SP, 1>(v, p, ztw);
        if (!active) return;
        // vector i of the result is output m = bit-reversed i (the first stage's parity is the top bit of i)
        constexpr int NVF = SP / 2, ZL = 32 / SP, LB = SP == 4 ? 1 : (SP == 8 ? 2 : 3);
        BD_UNROLL
        for (int i = 0; i < NVF; ++i) {
            int m = 0;
            BD_UNROLL
            for (int bit = 0; bit < LB; ++bit) m |= ((i >> bit) & 1) << (LB - 1 - bit);
            BD_UNROLL
            for (int z = 0; z < ZL; ++z) {
                BD_STS(col + (p * ZL + z + SUB * m) * PITCH, v[i * ZL + z]);
                if (coln) BD_STS(coln + (p * ZL + z + SUB * m) * PITCH, bd_f2(v[i * ZL + z].y, 0.f));
            }
        }
    }
#endif

    // frequencies kz = 2k + PAR of one column -> their part of x[z]; the odd half adds to
    // what the even half left in shared memory.  Column 0 carries P^ = Y0^ + i YN^.
    // nq: the Nyquist column, spread over the lanes of warp 0 (lane l holds kz = l and l + 32); only
    // that warp's first trip (kx = lane) carries column 0 and calls with WARP0 = true
    static constexpr int NQ = (PZ + 31) / 32;
    static constexpr bool COOP = LX >= 32;                  // all 32 lanes of warp 0 are in the first trip
    template <int PAR, bool WARP0>
    static BD_HD void zhalf(const float2* in, const float2* inn, const float2* nq, float2* col, long kzs, int kx) {
        float2 v[NZ];
        in += PAR * kzs;
        BD_UNROLL
        for (int k = 0; k < NZ; ++k) { v[k] = BD_LDCG(in); in += 2 * kzs; }
#if defined(__CUDA_ARCH__)
        if constexpr (WARP0 && COOP) {
            // every lane hands its share of the Nyquist column to lane 0 (kx = 0)
            BD_UNROLL
            for (int k = 0; k < NZ; ++k) {
                const int kz = 2 * k + PAR;
                float2 n;
                n.x = __shfl_sync(0xffffffffu, nq[kz >> 5].x, kz & 31);
                n.y = __shfl_sync(0xffffffffu, nq[kz >> 5].y, kz & 31);
                if (kx == 0) v[k] = bd_f2(v[k].x - n.y, v[k].y + n.x);
            }
        } else
#endif
        if (kx == 0) {
            (void)nq;
            inn += PAR * kzs;
            BD_UNROLL
            for (int k = 0; k < NZ; ++k) {
                const float2 n = BD_LDCG(inn);
                inn += 2 * kzs;
                v[k] = bd_f2(v[k].x - n.y, v[k].y + n.x);
            }
        }
        ZCol<PZ>::template inv_half<PAR>(v);
        if constexpr (PAR == 0) {
            BD_UNROLL
            for (int z = 0; z < NZ; ++z) BD_STS(col + z * PITCH, v[z]);
        } else {
            BD_UNROLL
            for (int z = 0; z < NZ; ++z) BD_STS(col + z * PITCH, pk_add(col[z * PITCH], v[z]));
        }
    }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        const int c = bx / a.ny, y = bx - c * a.ny;
        SRows<LX> s{sm};
        if constexpr (PH == 0) {
            const int cols = 1 << a.cs;
            const long kzs = (long)a.ntl * a.ny * cols;
            const float2* vc = a.V + (long)c * PZ * kzs;
            if constexpr (ZSplit<NZ>::ON) {
#if defined(__CUDA_ARCH__)
                // one (column, pass) per lane, the SP passes of a column on neighbouring lanes (whole warps make the trips)
                constexpr int SP = ZSplit<NZ>::SP;
                const float2* inn = vc + ((long)((LX >> a.cs) * a.ny + y) << a.cs) + (LX & (cols - 1));
                for (int i = tid; i < PZ; i += NT) sm[NZ * PITCH + i] = BD_LDG(&a.ztw[((i % SP) * (i / SP)) & (PZ - 1)]);
                __syncthreads();
                for (int w = tid; (w & ~31) < LX * SP; w += NT) {
                    const bool active = w < LX * SP;
                    const int kx = active ? w / SP : 1, p = w % SP;
                    const float2* in = vc + ((long)((kx >> a.cs) * a.ny + y) << a.cs) + (kx & (cols - 1));
                    float2* col = sm + xz_pos(a.xpost, LX, kx);
                    zcolumn_lanes(in, kx == 0 ? inn : nullptr, col, kx == 0 ? sm + prow(LX, LX) : nullptr, kzs, p, active, a.ztw, sm + NZ * PITCH);
                }
#else
                for (int kx = tid; kx <= LX; kx += NT) {
                    const float2* in = vc + ((long)((kx >> a.cs) * a.ny + y) << a.cs) + (kx & (cols - 1));
                    float2* col = sm + (kx == LX ? prow(LX, LX) : xz_pos(a.xpost, LX, kx));
                    zcolumn(in, col, kzs, a.ztw);
                }
#endif
            } else {
                const float2* inn = vc + ((long)((LX >> a.cs) * a.ny + y) << a.cs) + (LX & (cols - 1));
                float2 nq[NQ];
                BD_UNROLL
                for (int q = 0; q < NQ; ++q) nq[q] = bd_f2(0.f, 0.f);
#if defined(__CUDA_ARCH__)
                if (COOP && tid < 32) {
                    // the Nyquist column (column 0 needs it: P^ = Y0^ + i YN^) is fetched by the 32 lanes of
                    // warp 0 together, in flight with their own columns, instead of by lane 0 alone afterwards
                    BD_UNROLL
                    for (int q = 0; q < NQ; ++q)
                        if (tid + 32 * q < PZ) nq[q] = BD_LDCG(inn + (long)(tid + 32 * q) * kzs);
                }
#endif
                for (int kx = tid; kx < LX; kx += NT) {
                    const float2* in = vc + ((long)((kx >> a.cs) * a.ny + y) << a.cs) + (kx & (cols - 1));
                    float2* col = sm + xz_pos(a.xpost, LX, kx);
                    if (kx < 32) {                 // warp 0, first trip
                        zhalf<0, true>(in, inn, nq, col, kzs, kx);
                        zhalf<1, true>(in, inn, nq, col, kzs, kx);
                    } else {
                        zhalf<0, false>(in, inn, nq, col, kzs, kx);
                        zhalf<1, false>(in, inn, nq, col, kzs, kx);
                    }
                }
            }
        } else if constexpr (PH == 1) {
            for_kp_rows<LX, NT>(tid, NZ, a.xpost, [&](int kp, int row, const float4& xp) {
                float2* zr = sm + row * PITCH;
                const int pk = bd_float_as_int(xp.z), pm = bd_float_as_int(xp.w);
                float2 Yk = zr[pk], Ym = zr[pm];
                if (kp == 0) {
                    if constexpr (ZSplit<NZ>::ON) {               // Y[0], Y[LX] separate, both real
                        Ym = bd_f2(zr[prow(LX, LX)].x, 0.f);
                        Yk.y = 0.f;
                    } else {                                      // P = (Y[0], Y[LX]), both real
                        Ym = bd_f2(Yk.y, 0.f);
                        Yk.y = 0.f;
                    }
                }
                const float2 E = bd_f2(Yk.x + Ym.x, Yk.y - Ym.y);
                const float2 D = bd_f2(Yk.x - Ym.x, Yk.y + Ym.y);
                const float2 O = pk_cmulc(D, make_tw(bd_f2(xp.x, xp.y)));
                zr[pk] = bd_f2(E.x - O.y, E.y + O.x);
                if (kp != 0 && 2 * kp != LX) zr[pm] = bd_f2(E.x + O.y, O.x - E.y);
            });
        } else if constexpr (PH <= NP) {
            // phases 2..NP run inverse passes NP-1..1
            x_rows_pass<LX, NP + 1 - PH, true, NT>(tid, NZ, s, s, a.ptw);
        } else {
            if (a.en.M) {
                double acc = 0.0;
                GRowsOutE out{a.H + ((long)c * NZ * a.ny + y) * LX, (long)a.ny * LX,
                              (long)((const char*)a.en.M - (const char*)a.H), &acc};
                x_rows_pass<LX, 0, true, NT>(tid, NZ, s, out, a.ptw);
                energy_finish(acc, a.en);
            } else if (a.en.accumulate) {
                GRowsOutA out{a.H + ((long)c * NZ * a.ny + y) * LX, (long)a.ny * LX};
                x_rows_pass<LX, 0, true, NT>(tid, NZ, s, out, a.ptw);
            } else {
                GRowsOut out{a.H + ((long)c * NZ * a.ny + y) * LX, (long)a.ny * LX};
                x_rows_pass<LX, 0, true, NT>(tid, NZ, s, out, a.ptw);
            }
        }
    }
};

}  // namespace bd
