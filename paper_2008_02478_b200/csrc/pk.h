// pk.h — packed (f32x2) complex arithmetic and register DFTs built on it.
//
// sm_100a executes add/mul/fma on a pair of floats in one issue slot
// (FADD2/FMUL2/FFMA2); a complex number is such a pair, so a complex add is one
// instruction, a complex x real-pair product one, and a complex x complex
// product two (profiles/r01_microbench.md: same lane rate as scalar, half the
// issue slots).  On the host (tests/emu) the same functions are plain scalar code.
//
// Used by the transforms of the demag convolution ("manually
// coding the FFT algorithm").
#pragma once
#include "hd.h"

#if !defined(__CUDA_ARCH__)
#include <cmath>
#endif

namespace bd {

#if defined(__CUDA_ARCH__)
BD_HD float2 pk_add(float2 a, float2 b) { return __fadd2_rn(a, b); }
BD_HD float2 pk_mul(float2 a, float2 b) { return __fmul2_rn(a, b); }
BD_HD float2 pk_fma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
#else
BD_HD float2 pk_add(float2 a, float2 b) { return bd_f2(a.x + b.x, a.y + b.y); }
BD_HD float2 pk_mul(float2 a, float2 b) { return bd_f2(a.x * b.x, a.y * b.y); }
BD_HD float2 pk_fma(float2 a, float2 b, float2 c) { return bd_f2(std::fma(a.x, b.x, c.x), std::fma(a.y, b.y, c.y)); }
#endif
BD_HD float2 pk_neg(float2 a) { return bd_f2(-a.x, -a.y); }
BD_HD float2 pk_sub(float2 a, float2 b) { return pk_add(a, pk_neg(b)); }
BD_HD float2 pk_swap(float2 a) { return bd_f2(a.y, a.x); }
BD_HD float2 pk_bc(float s) { return bd_f2(s, s); }

// a + DIR*i*b        (DIR = -1: a - i b, DIR = +1: a + i b)
template <int DIR>
BD_HD float2 pk_add_ib(float2 a, float2 b) { return pk_fma(pk_swap(b), bd_f2(-(float)DIR, (float)DIR), a); }
// DIR*i*b
template <int DIR>
BD_HD float2 pk_ib(float2 b) { return pk_mul(pk_swap(b), bd_f2(-(float)DIR, (float)DIR)); }

// twiddle w = c + i s held as c and the pair (-s, s)
struct Tw { float c; float2 ns; };
BD_HD Tw make_tw(float2 w) { Tw t; t.c = w.x; t.ns = bd_f2(-w.y, w.y); return t; }
// a * w
BD_HD float2 pk_cmul(float2 a, const Tw& w) { return pk_fma(pk_swap(a), w.ns, pk_mul(a, pk_bc(w.c))); }
// a * conj(w)
BD_HD float2 pk_cmulc(float2 a, const Tw& w) { return pk_fma(pk_swap(a), pk_neg(w.ns), pk_mul(a, pk_bc(w.c))); }

// z * exp(DIR 2 pi i m / 32), m = 0..15 known after unrolling
template <int DIR>
BD_HD float2 pk_mul_w32(float2 z, int m) {
    constexpr float C1 = 0.98078528040323044913f, C2 = 0.92387953251128675613f,
                    C3 = 0.83146961230254523708f, C4 = 0.70710678118654752440f,
                    C5 = 0.55557023301960222474f, C6 = 0.38268343236508977173f,
                    C7 = 0.19509032201612826785f;
    constexpr float D = (float)DIR;
    float c, s;
    switch (m) {
        case 0: return z;
        case 8: return pk_ib<DIR>(z);
        case 4: return pk_mul(pk_add_ib<DIR>(z, z), pk_bc(C4));                  // (1 + D i) z / sqrt2
        case 12: return pk_mul(pk_add_ib<DIR>(pk_neg(z), z), pk_bc(C4));         // (-1 + D i) z / sqrt2
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
    return pk_fma(pk_swap(z), bd_f2(-s, s), pk_mul(z, pk_bc(c)));
}
template <int R, int DIR>
BD_HD float2 pk_mul_w(float2 z, int r) { return pk_mul_w32<DIR>(z, r * (32 / R)); }

// In place, natural order in and out: v[q] <- sum_r v[r] exp(DIR 2 pi i q r / R).
template <int R, int DIR>
struct PkDft {
    static BD_HD void run(float2* v) {
        float2 a[R / 2], b[R / 2];
        BD_UNROLL
        for (int r = 0; r < R / 2; ++r) {
            a[r] = pk_add(v[r], v[r + R / 2]);
            if (4 * r == R) b[r] = pk_add_ib<-DIR>(pk_ib<DIR>(v[r]), v[r + R / 2]);  // DIR i (v[r] - v[r+R/2])
            else b[r] = pk_mul_w<R, DIR>(pk_sub(v[r], v[r + R / 2]), r);
        }
        PkDft<R / 2, DIR>::run(a);
        PkDft<R / 2, DIR>::run(b);
        BD_UNROLL
        for (int q = 0; q < R / 2; ++q) { v[2 * q] = a[q]; v[2 * q + 1] = b[q]; }
    }
};
template <int DIR>
struct PkDft<1, DIR> { static BD_HD void run(float2*) {} };

// Inputs v[r] = 0 for r >= R/2 (zero padding): only v[0..R/2) is read.
template <int R, int DIR>
struct PkDftPruned {
    static BD_HD void run(float2* v) {
        float2 a[R / 2], b[R / 2];
        BD_UNROLL
        for (int r = 0; r < R / 2; ++r) { a[r] = v[r]; b[r] = pk_mul_w<R, DIR>(v[r], r); }
        PkDft<R / 2, DIR>::run(a);
        PkDft<R / 2, DIR>::run(b);
        BD_UNROLL
        for (int q = 0; q < R / 2; ++q) { v[2 * q] = a[q]; v[2 * q + 1] = b[q]; }
    }
};

// Only outputs q < R/2 are produced (in v[0..R/2)).
template <int R, int DIR>
struct PkDftTrunc {
    static BD_HD void run(float2* v) {
        float2 e[R / 2], o[R / 2];
        BD_UNROLL
        for (int r = 0; r < R / 2; ++r) { e[r] = v[2 * r]; o[r] = v[2 * r + 1]; }
        PkDft<R / 2, DIR>::run(e);
        PkDft<R / 2, DIR>::run(o);
        BD_UNROLL
        for (int q = 0; q < R / 2; ++q) v[q] = pk_add(e[q], pk_mul_w<R, DIR>(o[q], q));
    }
};

}  // namespace bd
