// plan_math.h — plan-time arithmetic (fp64): the demagnetizing tensor and its real,
// symmetry-reduced spectrum.  BD_HD so that the device kernels of plan_create and the
// host-only test entry points (boris_demag_tensor_host / _spectrum_host) compile
// the same source.
//
// Tensor ("N computed using formulas in Ref. [50]"; the method here
// is deliberately NOT the oracle's, so that the two cross-check — DESIGN.md R3):
//   near  |R| <= kNearCells * max(h):  Newell's closed form (f, g and the 27-point
//         stencil) in plain fp64, where its cancellation error is <= ~3e-13;
//   far   the cell-averaged tensor is the point-dipole tensor
//             D_ab(R) = (1/4pi) (delta_ab / R^3 - 3 R_a R_b / R^5)
//         averaged over the separation u = r - r' of a point r in the target cell
//         and r' in the source cell.  Each u_a is the difference of two uniform
//         variables on a cell side, i.e. triangular on [-h_a, h_a], so
//             N_ab(R) = V * sum_ijk w_i w_j w_k D_ab(R + (t_i hx, t_j hy, t_k hz))
//         with the 4-point Gauss rule of the weight (1 - |t|) on [-1, 1]
//         (exact through degree 7).  Measured against the extended-precision closed form the
//         quadrature is good to 3e-13 beyond 10 cells and 1e-15 beyond 16, while the fp64
//         closed form degrades from 1e-14 at 4 cells to 1e-12 at 16: the seam sits at 10.
//
// Spectrum ("the demagnetizing kernel in the transform space").  The
// padded tensor is even or odd in every coordinate (pin P4), so its DFT is real up
// to a factor (-i) per odd coordinate and separates into 1-D cosine / sine sums over
// the non-negative displacements:
//   even:  E(k) = v[0] + 2 sum_{i=1}^{n-1} v[i] cos(2 pi i k / P)
//   odd:   S(k) =        2 sum_{i=1}^{n-1} v[i] sin(2 pi i k / P)        (times -i)
// for k = 0..P/2, P = 2n (displacement n itself is never used: reading R5).  Every
// off-diagonal component is odd in exactly two coordinates: (-i)^2 = -1.
#pragma once
#include <math.h>

#include "hd.h"

namespace bd {

constexpr double kNearCells = 10.0;
constexpr double kPi = 3.14159265358979323846264338327950288;

// ------------------------------------------------------------------ Newell closed form
BD_HD double nw_asinh_ratio(double num, double den2) { return den2 > 0.0 ? asinh(num / sqrt(den2)) : 0.0; }
BD_HD double nw_atan_ratio(double num, double den) { return den != 0.0 ? atan(num / den) : 0.0; }

BD_HD double newell_f(double x, double y, double z) {
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = sqrt(x2 + y2 + z2);
    return 0.5 * y * (z2 - x2) * nw_asinh_ratio(y, x2 + z2) + 0.5 * z * (y2 - x2) * nw_asinh_ratio(z, x2 + y2)
         - x * y * z * nw_atan_ratio(y * z, x * R) + (2.0 * x2 - y2 - z2) * R / 6.0;
}
BD_HD double newell_g(double x, double y, double z) {
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = sqrt(x2 + y2 + z2);
    return x * y * z * nw_asinh_ratio(z, x2 + y2) + y * (3.0 * z2 - y2) * nw_asinh_ratio(x, y2 + z2) / 6.0
         + x * (3.0 * z2 - x2) * nw_asinh_ratio(y, x2 + z2) / 6.0 - z2 * z * nw_atan_ratio(x * y, z * R) / 6.0
         - 0.5 * z * y2 * nw_atan_ratio(x * z, y * R) - 0.5 * z * x2 * nw_atan_ratio(y * z, x * R) - x * y * R / 3.0;
}

// component c = xx, yy, zz, xy, xz, yz of Newell's generating function at (x, y, z)
BD_HD double newell_gen(int c, double x, double y, double z) {
    switch (c) {
        case 0: return newell_f(x, y, z);
        case 1: return newell_f(y, x, z);
        case 2: return newell_f(z, y, x);
        case 3: return newell_g(x, y, z);
        case 4: return newell_g(x, z, y);
        default: return newell_g(y, z, x);
    }
}

BD_HD double tensor_near(int c, double X, double Y, double Z, double hx, double hy, double hz) {
    double acc = 0.0;
    for (int a = -1; a <= 1; ++a)
        for (int b = -1; b <= 1; ++b)
            for (int d = -1; d <= 1; ++d) {
                const int m = (a != 0) + (b != 0) + (d != 0);
                const double w = m == 0 ? 8.0 : (m == 1 ? -4.0 : (m == 2 ? 2.0 : -1.0));
                acc += w * newell_gen(c, X + a * hx, Y + b * hy, Z + d * hz);
            }
    return acc / (4.0 * kPi * hx * hy * hz);
}

// 4-point Gauss rule for the weight (1 - |t|) on [-1, 1] (total weight 1).  In s = t^2
// the nodes are the roots of s^2 - (31/49) s + 19/490 (orthogonal to 1 and s under the
// even moments 1, 1/6, 1/15, 1/28).
BD_HD void tri_gauss4(double t[4], double w[4]) {
    const double p = 31.0 / 49.0, q = 19.0 / 490.0, disc = sqrt(p * p - 4.0 * q);
    const double s1 = 0.5 * (p + disc), s2 = 0.5 * (p - disc);
    const double W1 = (1.0 / 6.0 - s2) / (s1 - s2), W2 = 1.0 - W1;   // weight of the +- pair
    t[0] = -sqrt(s1); t[1] = -sqrt(s2); t[2] = sqrt(s2); t[3] = sqrt(s1);
    w[0] = 0.5 * W1; w[1] = 0.5 * W2; w[2] = 0.5 * W2; w[3] = 0.5 * W1;
}

BD_HD void tensor_far(double X, double Y, double Z, double hx, double hy, double hz, double out[6]) {
    double t[4], w[4];
    tri_gauss4(t, w);
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j)
            for (int k = 0; k < 4; ++k) {
                const double x = X + t[i] * hx, y = Y + t[j] * hy, z = Z + t[k] * hz;
                const double r2 = x * x + y * y + z * z, r = sqrt(r2), ir5 = 1.0 / (r2 * r2 * r);
                const double ww = w[i] * w[j] * w[k] * ir5;
                acc[0] += ww * (r2 - 3.0 * x * x);
                acc[1] += ww * (r2 - 3.0 * y * y);
                acc[2] += ww * (r2 - 3.0 * z * z);
                acc[3] += ww * (-3.0 * x * y);
                acc[4] += ww * (-3.0 * x * z);
                acc[5] += ww * (-3.0 * y * z);
            }
    const double s = hx * hy * hz / (4.0 * kPi);
    for (int c = 0; c < 6; ++c) out[c] = s * acc[c];
}

// N_c at displacement (i hx, j hy, k hz), i, j, k >= 0, all six components.
BD_HD void tensor_point(int i, int j, int k, double hx, double hy, double hz, double out[6]) {
    const double X = i * hx, Y = j * hy, Z = k * hz;
    const double hmax = fmax(hx, fmax(hy, hz)), rn = kNearCells * hmax;
    if (X * X + Y * Y + Z * Z <= rn * rn) {
        for (int c = 0; c < 6; ++c) out[c] = tensor_near(c, X, Y, Z, hx, hy, hz);
    } else {
        tensor_far(X, Y, Z, hx, hy, hz, out);
    }
    // odd components vanish exactly on their nodal planes (pin P4)
    if (i == 0) { out[3] = 0.0; out[4] = 0.0; }
    if (j == 0) { out[3] = 0.0; out[5] = 0.0; }
    if (k == 0) { out[4] = 0.0; out[5] = 0.0; }
}

// Periodic boundary conditions by the multiple-images method (Ref. [51]; reading R15):
// the tensor of a mesh repeated `img[d]` times on each side along dimension d with period per[d] cells,
//     N^img_c(i, j, k) = sum_{|a| <= img[0]} sum_{|b| <= img[1]} sum_{|e| <= img[2]} N_c(i + a per[0], j + b per[1], k + e per[2]),
// negative displacements by the parity of the component.  img = (0, 0, 0) is tensor_point itself.
BD_HD void tensor_point_images(int i, int j, int k, const int per[3], const int img[3], double hx, double hy, double hz,
                               double out[6]) {
    if (img[0] == 0 && img[1] == 0 && img[2] == 0) { tensor_point(i, j, k, hx, hy, hz, out); return; }
    double acc[6] = {0, 0, 0, 0, 0, 0};
    // far copies first: the small terms are added before the large ones
    for (int e = img[2]; e >= -img[2]; e = (e > 0 ? -e : -e - 1)) {
        for (int b = img[1]; b >= -img[1]; b = (b > 0 ? -b : -b - 1)) {
            for (int a = img[0]; a >= -img[0]; a = (a > 0 ? -a : -a - 1)) {
                const int ii = i + a * per[0], jj = j + b * per[1], kk = k + e * per[2];
                const double sx = ii < 0 ? -1.0 : 1.0, sy = jj < 0 ? -1.0 : 1.0, sz = kk < 0 ? -1.0 : 1.0;
                double t[6];
                tensor_point(ii < 0 ? -ii : ii, jj < 0 ? -jj : jj, kk < 0 ? -kk : kk, hx, hy, hz, t);
                acc[0] += t[0]; acc[1] += t[1]; acc[2] += t[2];
                acc[3] += sx * sy * t[3]; acc[4] += sx * sz * t[4]; acc[5] += sy * sz * t[5];
                if (a == 0) break;
            }
            if (b == 0) break;
        }
        if (e == 0) break;
    }
    for (int c = 0; c < 6; ++c) out[c] = acc[c];
    // the symmetric block of copies keeps every component's parity: exact zeros on the nodal planes
    if (i == 0) { out[3] = 0.0; out[4] = 0.0; }
    if (j == 0) { out[3] = 0.0; out[5] = 0.0; }
    if (k == 0) { out[4] = 0.0; out[5] = 0.0; }
}

// parity of component c along dimension d (0 = x, 1 = y, 2 = z): true = odd
BD_HD bool comp_is_odd(int c, int d) {
    return (c == 3 && (d == 0 || d == 1)) || (c == 4 && (d == 0 || d == 2)) || (c == 5 && (d == 1 || d == 2));
}

// ------------------------------------------------------------------ 1-D real transforms
// One output of the cosine (odd = false) or sine (odd = true) sum over n samples
// v[i * stride]; cs[m] = (cos, sin)(2 pi m / P), m < P = 2n.  n == 1 is the flat
// dimension (P = 1): the only frequency is k = 0 and the transform is the identity
// (the sine sum of an odd component is then 0: reading R7).
BD_HD double real_transform(const double* v, long stride, int n, int k, bool odd, const double2* cs) {
    if (n == 1) return odd ? 0.0 : v[0];
    const int P = 2 * n;
    double acc = 0.0;
    if (!odd) {
        for (int i = n - 1; i >= 1; --i) acc += v[i * stride] * cs[(i * k) & (P - 1)].x;
        return v[0] + 2.0 * acc;
    }
    for (int i = n - 1; i >= 1; --i) acc += v[i * stride] * cs[(i * k) & (P - 1)].y;
    return 2.0 * acc;
}

}  // namespace bd
