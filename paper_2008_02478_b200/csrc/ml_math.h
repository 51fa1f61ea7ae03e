// ml_math.h — plan-time tensor of the multi-layered convolution (boris_demag_ml.cu; Eq. 4):
// N(R, h_k, h_i) between a source cuboid (hx, hy, ti) and a target cuboid (hx, hy, tk) whose centres are
// R = (i hx, j hy, Z) apart, averaged over the target cell (reading R17).  As for the single mesh
// (plan_math.h) the method is deliberately not the oracle's:
//   near  Newell's closed form in fp64, the z part of the 27-point stencil replaced by the 4-point second
//         difference that two unequal heights leave:
//             -F(Z + (tk+ti)/2) + F(Z + (tk-ti)/2) + F(Z - (tk-ti)/2) - F(Z - (tk+ti)/2),  normalised by hx hy tk;
//   far   the point-dipole tensor averaged over the separation of a point of the target and a point of the
//         source cell: 4-point Gauss rule of the triangular density in x and y (equal sides), 3 x 3 Gauss-Legendre
//         points over the two heights.
#pragma once
#include "plan_math.h"

namespace bd {

BD_HD double pair_near(int c, double X, double Y, double Z, double hx, double hy, double tk, double ti) {
    const double zo[4] = {0.5 * (tk + ti), 0.5 * (tk - ti), -0.5 * (tk - ti), -0.5 * (tk + ti)};
    const double zw[4] = {-1.0, 1.0, 1.0, -1.0};
    double acc = 0.0;
    for (int a = -1; a <= 1; ++a)
        for (int b = -1; b <= 1; ++b) {
            const double wxy = (a == 0 ? 2.0 : -1.0) * (b == 0 ? 2.0 : -1.0);
            for (int d = 0; d < 4; ++d) acc += wxy * zw[d] * newell_gen(c, X + a * hx, Y + b * hy, Z + zo[d]);
        }
    return acc / (4.0 * kPi * hx * hy * tk);
}

BD_HD void pair_far(double X, double Y, double Z, double hx, double hy, double tk, double ti, double out[6]) {
    double t[4], w[4];
    tri_gauss4(t, w);
    const double g3 = 0.38729833462074168852, gl[3] = {-g3, 0.0, g3}, gw[3] = {5.0 / 18.0, 8.0 / 18.0, 5.0 / 18.0};   // on [-1/2, 1/2]
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j)
            for (int p = 0; p < 3; ++p)
                for (int q = 0; q < 3; ++q) {
                    const double x = X + t[i] * hx, y = Y + t[j] * hy, z = Z + gl[p] * tk - gl[q] * ti;
                    const double r2 = x * x + y * y + z * z, r = sqrt(r2), ir5 = 1.0 / (r2 * r2 * r);
                    const double ww = w[i] * w[j] * gw[p] * gw[q] * ir5;
                    acc[0] += ww * (r2 - 3.0 * x * x);
                    acc[1] += ww * (r2 - 3.0 * y * y);
                    acc[2] += ww * (r2 - 3.0 * z * z);
                    acc[3] += ww * (-3.0 * x * y);
                    acc[4] += ww * (-3.0 * x * z);
                    acc[5] += ww * (-3.0 * y * z);
                }
    const double s = hx * hy * ti / (4.0 * kPi);          // source volume: N = V_s <D>
    for (int c = 0; c < 6; ++c) out[c] = s * acc[c];
}

// all six components at in-plane displacement (i hx, j hy), i, j >= 0, height difference Z (any sign)
BD_HD void pair_tensor_point(int i, int j, double Z, double hx, double hy, double tk, double ti, double out[6]) {
    const double X = i * hx, Y = j * hy;
    const double hmax = fmax(fmax(hx, hy), fmax(tk, ti)), rn = kNearCells * hmax;
    if (X * X + Y * Y + Z * Z <= rn * rn) {
        for (int c = 0; c < 6; ++c) out[c] = pair_near(c, X, Y, Z, hx, hy, tk, ti);
    } else {
        pair_far(X, Y, Z, hx, hy, tk, ti, out);
    }
    if (i == 0) { out[3] = 0.0; out[4] = 0.0; }       // odd in x
    if (j == 0) { out[3] = 0.0; out[5] = 0.0; }       // odd in y
    if (Z == 0.0) { out[4] = 0.0; out[5] = 0.0; }     // odd in z: centres at the same height
}

// parity of component c along in-plane dimension d (0 = x, 1 = y) at fixed Z: true = odd
BD_HD bool pair_comp_is_odd(int c, int d) { return (c == 3) || (c == 4 && d == 0) || (c == 5 && d == 1); }

}  // namespace bd
