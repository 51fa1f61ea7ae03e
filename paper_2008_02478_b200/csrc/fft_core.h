// fft_core.h — register butterflies, pass geometry and index maps of the in-place
// mixed-radix FFTs used by every transform of the demag convolution
// ("1D FFTs along the x, y, z directions ... multiplication ...
// z, y, x inverse 1D FFTs"; "manually coding the FFT algorithm").
//
// Scheme.  An L-point transform (L = 2..2048, power of two) is NP <= 3 passes of
// radix R0, R1, R2 (dec_r).  Forward = decimation in frequency, in place:
//   pass p works on sub-blocks of length Lp (L0 = L, L1 = L/R0, L2 = L1/R1);
//   butterfly j of a block reads e_r = blk*Lp + j + r*(Lp/Rp), r = 0..Rp-1,
//   takes an Rp-point DFT over r -> q, multiplies by W_Lp^(j q) (not in the last
//   pass) and writes q back to e_q.
// After the last pass position p = q0*L1 + q1*L2 + q2 holds frequency
// k = q0 + R0*(q1 + R1*q2): digit-reversed order.  The inverse is the exact mirror
// (decimation in time): conjugate twiddle first, inverse butterfly, passes in
// reverse order; it takes digit-reversed input to natural-order output.  Nothing is
// ever reordered: the kernel spectrum is stored in the order the fused multiply
// meets it (khat_* below), fixed at plan time.
//
// Zero padding makes the upper half of every forward input zero
// and the upper half of every inverse output unwanted: pass 0 uses a pruned
// butterfly forward (DftPruned) and a truncated one inverse (DftTrunc).
//
// No normalisation anywhere: the factor is folded into the kernel spectrum
// (reading R12).
#pragma once
#include "hd.h"

namespace bd {

// ------------------------------------------------------------------ complex helpers
BD_HD float2 cadd(float2 a, float2 b) { return bd_f2(a.x + b.x, a.y + b.y); }
BD_HD float2 csub(float2 a, float2 b) { return bd_f2(a.x - b.x, a.y - b.y); }
BD_HD float2 cmul(float2 a, float2 b) { return bd_f2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * conj(b)
BD_HD float2 cmulc(float2 a, float2 b) { return bd_f2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
BD_HD float2 cscale(float s, float2 a) { return bd_f2(s * a.x, s * a.y); }
BD_HD float2 cconj(float2 a) { return bd_f2(a.x, -a.y); }

// z * exp(DIR * 2 pi i * m / 32), m = 0..15, m known after unrolling (the switch folds).
template <int DIR>
BD_HD float2 mul_w32(float2 z, int m) {
    constexpr float C1 = 0.98078528040323044913f, C2 = 0.92387953251128675613f,
                    C3 = 0.83146961230254523708f, C4 = 0.70710678118654752440f,
                    C5 = 0.55557023301960222474f, C6 = 0.38268343236508977173f,
                    C7 = 0.19509032201612826785f;
    constexpr float D = (float)DIR;
    float c, s;
    switch (m) {
        case 0: return z;
        case 8: return bd_f2(-D * z.y, D * z.x);
        case 4: return bd_f2((z.x - D * z.y) * C4, (z.y + D * z.x) * C4);
        case 12: return bd_f2((-z.x - D * z.y) * C4, (-z.y + D * z.x) * C4);
        case 1: c = C1; s = C7; break;
        case 2: c = C2; s = C6; break;
        case 3: c = C3; s = C5; break;
        case 5: c = C5; s = C3; break;
        case 6: c = C6; s = C2; break;
        case 7: c = C7; s = C1; break;
        case 9: c = -C7; s = C1; break;
        case 10: c = -C6; s = C2; break;
        case 11: c = -C5; s = C3; break;
        case 13: c = -C3; s = C5; break;
        case 14: c = -C2; s = C6; break;
        default: c = -C1; s = C7; break;   // 15
    }
    s *= D;
    return bd_f2(c * z.x - s * z.y, c * z.y + s * z.x);
}
// z * W_R^r with W_R = exp(DIR 2 pi i / R), r in [0, R/2)
template <int R, int DIR>
BD_HD float2 mul_w(float2 z, int r) { return mul_w32<DIR>(z, r * (32 / R)); }

// ------------------------------------------------------------------ register DFTs
// In place, natural order in and out: v[q] <- sum_r v[r] exp(DIR 2 pi i q r / R).
template <int R, int DIR>
struct Dft {
    static BD_HD void run(float2* v) {
        float2 a[R / 2], b[R / 2];
        BD_UNROLL
        for (int r = 0; r < R / 2; ++r) {
            a[r] = cadd(v[r], v[r + R / 2]);
            b[r] = mul_w<R, DIR>(csub(v[r], v[r + R / 2]), r);
        }
        Dft<R / 2, DIR>::run(a);
        Dft<R / 2, DIR>::run(b);
        BD_UNROLL
        for (int q = 0; q < R / 2; ++q) { v[2 * q] = a[q]; v[2 * q + 1] = b[q]; }
    }
};
template <int DIR>
struct Dft<1, DIR> { static BD_HD void run(float2*) {} };

// Inputs v[r] = 0 for r >= R/2 (zero padding): only v[0..R/2) is read.
template <int R, int DIR>
struct DftPruned {
    static BD_HD void run(float2* v) {
        float2 a[R / 2], b[R / 2];
        BD_UNROLL
        for (int r = 0; r < R / 2; ++r) { a[r] = v[r]; b[r] = mul_w<R, DIR>(v[r], r); }
        Dft<R / 2, DIR>::run(a);
        Dft<R / 2, DIR>::run(b);
        BD_UNROLL
        for (int q = 0; q < R / 2; ++q) { v[2 * q] = a[q]; v[2 * q + 1] = b[q]; }
    }
};

// Only outputs q < R/2 are produced (in v[0..R/2)); the rest of v is garbage.
template <int R, int DIR>
struct DftTrunc {
    static BD_HD void run(float2* v) {
        float2 e[R / 2], o[R / 2];
        BD_UNROLL
        for (int r = 0; r < R / 2; ++r) { e[r] = v[2 * r]; o[r] = v[2 * r + 1]; }
        Dft<R / 2, DIR>::run(e);
        Dft<R / 2, DIR>::run(o);
        BD_UNROLL
        for (int q = 0; q < R / 2; ++q) v[q] = cadd(e[q], mul_w<R, DIR>(o[q], q));
    }
};

// ------------------------------------------------------------------ decomposition
constexpr int kMaxFft = 2048;

BD_HD constexpr int dec_np(int L) { return L <= 8 ? 1 : (L <= 128 ? 2 : 3); }
// radix of pass p (1 if the pass does not exist)
BD_HD constexpr int dec_r(int L, int p) {
    return L == 2    ? (p == 0 ? 2 : 1)
         : L == 4    ? (p == 0 ? 4 : 1)
         : L == 8    ? (p == 0 ? 8 : 1)
         : L == 16   ? (p == 0 ? 2 : p == 1 ? 8 : 1)
         : L == 32   ? (p == 0 ? 4 : p == 1 ? 8 : 1)
         : L == 64   ? (p == 0 ? 8 : p == 1 ? 8 : 1)
         : L == 128  ? (p == 0 ? 16 : p == 1 ? 8 : 1)
         : L == 256  ? (p == 0 ? 4 : 8)
         : L == 512  ? 8
         : L == 1024 ? (p == 0 ? 16 : 8)
         : L == 2048 ? (p <= 1 ? 16 : 8)
         : 0;
}
BD_HD constexpr bool dec_supported(int L) { return L >= 2 && L <= kMaxFft && (L & (L - 1)) == 0; }
// length of the sub-blocks pass p works on
BD_HD constexpr int dec_sublen(int L, int p) { return p == 0 ? L : (p == 1 ? L / dec_r(L, 0) : L / (dec_r(L, 0) * dec_r(L, 1))); }
BD_HD constexpr int dec_rlast(int L) { return dec_r(L, dec_np(L) - 1); }
// number of last-pass butterflies ("items") = spacing of the frequencies inside one item
BD_HD constexpr int dec_items(int L) { return L / dec_rlast(L); }

// position (after the forward transform) that holds frequency k, and back
BD_HD int pos_of_freq(int L, int k) {
    const int np = dec_np(L), r0 = dec_r(L, 0), r1 = dec_r(L, 1);
    if (np == 1) return k;
    if (np == 2) return (k % r0) * r1 + k / r0;
    const int r2 = dec_r(L, 2);
    return (k % r0) * (L / r0) + ((k / r0) % r1) * r2 + k / (r0 * r1);
}
BD_HD int freq_of_pos(int L, int p) {
    const int np = dec_np(L), r0 = dec_r(L, 0), r1 = dec_r(L, 1);
    if (np == 1) return p;
    if (np == 2) return p / r1 + r0 * (p % r1);
    const int r2 = dec_r(L, 2), l1 = L / r0;
    return p / l1 + r0 * ((p % l1) / r2 + r1 * (p % r2));
}
// Item i of the last pass holds frequencies f(i) + F*q, q = 0..RL-1, F = dec_items(L).
BD_HD int item_partial_freq(int L, int i) {
    const int np = dec_np(L);
    if (np == 1) return 0;
    if (np == 2) return i;
    const int r0 = dec_r(L, 0), r1 = dec_r(L, 1);
    return i / r1 + r0 * (i % r1);
}

// Kernel-spectrum rows along the fused dimension (symmetry-reduced storage, pin P12).
// The mirror of item f is item F - f with q reversed (f != 0), so only the
// canonical items f' = min(f, F - f) in [0, F/2] are stored: F/2 + 1 rows of RL
// entries (L/2 + RL values instead of L/2 + 1; rows 0 and F/2 are self-mirrored and
// hold their own mirror images with the sign already applied).  Rows are numbered
// so that consecutive items of a warp read consecutive rows.
BD_HD int khat_rows(int L) { const int F = dec_items(L); return F >= 2 ? F / 2 + 1 : 1; }
BD_HD int khat_row_of_f(int L, int fc) {
    const int np = dec_np(L);
    if (np <= 2) return fc;
    const int r0 = dec_r(L, 0), r1 = dec_r(L, 1), F = r0 * r1;
    const int q0 = fc % r0, q1 = fc / r0;
    return q1 < r1 / 2 ? q0 * (r1 / 2) + q1 : F / 2;
}
BD_HD int khat_f_of_row(int L, int row) {
    const int np = dec_np(L);
    if (np <= 2) return row;
    const int r0 = dec_r(L, 0), r1 = dec_r(L, 1), F = r0 * r1;
    if (row == F / 2) return F / 2;
    return row / (r1 / 2) + r0 * (row % (r1 / 2));
}

// shared-memory padding of a contiguous pencil: one float2 of slack per 16
BD_HD constexpr int padlen(int L) { return L + (L >> 4); }
BD_HD int padidx(int e) { return e + (e >> 4); }

// ------------------------------------------------------------------ passes
// Accessors: In::get(c, e) -> float2, Out::put(c, e, v).  c = vector component.
// tw[k] = exp(-2 pi i k / L), k in [0, L).
template <int L, int P, class In, class Out>
BD_HD void fwd_pass(int c, int w, const In& in, const Out& out, const float2* __restrict__ tw) {
    constexpr int NP = dec_np(L), R = dec_r(L, P), Lp = dec_sublen(L, P), S = Lp / R, TWS = L / Lp;
    const int blk = w / S, j = w - blk * S, base = blk * Lp + j;
    float2 v[R];
    if constexpr (P == 0) {
        BD_UNROLL
        for (int r = 0; r < R / 2; ++r) v[r] = in.get(c, base + r * S);
        DftPruned<R, -1>::run(v);
    } else {
        BD_UNROLL
        for (int r = 0; r < R; ++r) v[r] = in.get(c, base + r * S);
        Dft<R, -1>::run(v);
    }
    if constexpr (P < NP - 1) {
        BD_UNROLL
        for (int q = 1; q < R; ++q) v[q] = cmul(v[q], BD_LDG(&tw[TWS * j * q]));
    }
    BD_UNROLL
    for (int q = 0; q < R; ++q) out.put(c, base + q * S, v[q]);
}

template <int L, int P, class In, class Out>
BD_HD void inv_pass(int c, int w, const In& in, const Out& out, const float2* __restrict__ tw) {
    constexpr int NP = dec_np(L), R = dec_r(L, P), Lp = dec_sublen(L, P), S = Lp / R, TWS = L / Lp;
    const int blk = w / S, j = w - blk * S, base = blk * Lp + j;
    float2 v[R];
    BD_UNROLL
    for (int q = 0; q < R; ++q) v[q] = in.get(c, base + q * S);
    if constexpr (P < NP - 1) {
        BD_UNROLL
        for (int q = 1; q < R; ++q) v[q] = cmulc(v[q], BD_LDG(&tw[TWS * j * q]));
    }
    if constexpr (P == 0) {
        DftTrunc<R, +1>::run(v);
        BD_UNROLL
        for (int r = 0; r < R / 2; ++r) out.put(c, base + r * S, v[r]);
    } else {
        Dft<R, +1>::run(v);
        BD_UNROLL
        for (int r = 0; r < R; ++r) out.put(c, base + r * S, v[r]);
    }
}

// The pipelined step (innermost FFT, "point-by-point multiplications"
// and innermost inverse FFT in one kernel, "simultaneously for all 3 vector
// components"): last forward pass, H^ = K^ M^ with the real symmetric tensor, first
// inverse pass, all in registers.  NC = 4: 2-D mode, fused dimension y, components
// (xx, yy, zz, xy), Nxz = Nyz = 0 (reading R7).  NC = 6: fused dimension z,
// components (xx, yy, zz, xy, xz, yz).  K.get(comp, q, row) reads the stored row.
template <int L, int NC, class In, class Out, class KAcc>
BD_HD void fused_mid(int i, const In& in, const Out& out, const KAcc& K) {
    constexpr int NP = dec_np(L), RL = dec_rlast(L), F = dec_items(L);
    float2 v[3][RL];
    BD_UNROLL
    for (int c = 0; c < 3; ++c) {
        if constexpr (NP == 1) {
            BD_UNROLL
            for (int q = 0; q < RL / 2; ++q) v[c][q] = in.get(c, i * RL + q);
            DftPruned<RL, -1>::run(v[c]);
        } else {
            BD_UNROLL
            for (int q = 0; q < RL; ++q) v[c][q] = in.get(c, i * RL + q);
            Dft<RL, -1>::run(v[c]);
        }
    }
    const int f = item_partial_freq(L, i);
    const bool rev = 2 * f > F;
    const int row = khat_row_of_f(L, rev ? F - f : f);
    const float s = rev ? -1.f : 1.f;   // sign of the components odd in the fused dimension
    BD_UNROLL
    for (int q = 0; q < RL; ++q) {
        const int qq = rev ? RL - 1 - q : q;
        const float2 mx = v[0][q], my = v[1][q], mz = v[2][q];
        const float kxx = K.get(0, qq, row), kyy = K.get(1, qq, row), kzz = K.get(2, qq, row);
        if constexpr (NC == 4) {
            const float kxy = s * K.get(3, qq, row);
            v[0][q] = bd_f2(kxx * mx.x + kxy * my.x, kxx * mx.y + kxy * my.y);
            v[1][q] = bd_f2(kxy * mx.x + kyy * my.x, kxy * mx.y + kyy * my.y);
            v[2][q] = bd_f2(kzz * mz.x, kzz * mz.y);
        } else {
            const float kxy = K.get(3, qq, row), kxz = s * K.get(4, qq, row), kyz = s * K.get(5, qq, row);
            v[0][q] = bd_f2(kxx * mx.x + kxy * my.x + kxz * mz.x, kxx * mx.y + kxy * my.y + kxz * mz.y);
            v[1][q] = bd_f2(kxy * mx.x + kyy * my.x + kyz * mz.x, kxy * mx.y + kyy * my.y + kyz * mz.y);
            v[2][q] = bd_f2(kxz * mx.x + kyz * my.x + kzz * mz.x, kxz * mx.y + kyz * my.y + kzz * mz.y);
        }
    }
    BD_UNROLL
    for (int c = 0; c < 3; ++c) {
        if constexpr (NP == 1) {
            DftTrunc<RL, +1>::run(v[c]);
            BD_UNROLL
            for (int q = 0; q < RL / 2; ++q) out.put(c, i * RL + q, v[c][q]);
        } else {
            Dft<RL, +1>::run(v[c]);
            BD_UNROLL
            for (int q = 0; q < RL; ++q) out.put(c, i * RL + q, v[c][q]);
        }
    }
}

}  // namespace bd
