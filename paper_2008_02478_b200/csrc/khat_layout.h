// khat_layout.h — where the fused multiply finds the kernel spectrum.
//
// Natural, symmetry-reduced spectrum (pin P12):
//     Kred[c][kz <= Pz/2][ky <= Py/2][kx <= Px/2]      (fp64 at plan time)
// with the value at a mirrored frequency Py - ky (Pz - kz) equal to the stored one
// times -1 for the components odd in y (z).  kx needs no mirror (real -> complex in x).
//
// Device storage (fp32), in the order the fused kernels meet it:
//   tiled path (YFused, fused dimension y; yfused.h "kernel-spectrum tile"):
//       K[kzr][tile][c][chunk][slot][col][CH]
//   chunked fallback, nz > 1 (ZFused, fused dimension z, fft_core.h khat_*; y is a plain
//            tile coordinate and keeps all Py
//            positions of the in-place y FFT, in its digit-reversed order):
//       K[slot = kx][ytile][c (6)][q (RL)][row][t]             py = ytile*ty + t
// The entry (q, row) of the fused dimension holds frequency k = f'(row) + F*q; if
// k > L/2 it is read from the natural array at L - k with the odd-component sign.
#pragma once
#include "fft_core.h"
#include "plan_math.h"
#include "yfused.h"

namespace bd {

struct KLayout {
    int nx, ny, nz;        // cells
    int Px, Py, Pz;        // padded (Pz = 1 when nz = 1)
    int ncomp;             // 4 (nz = 1) or 6
    int Lf;                // fused FFT length: Py (nz = 1) or Pz
    int RL, nrows;         // last radix and canonical rows of the fused dimension
    int ty, ntiles;        // y tile of ZFused (ty = ntiles = 1... for nz = 1: ty = 1, ntiles = 1)
    // tiled path (yfused.h): K[kzr][tile][c][chunk][slot (NRy)][col][CH], fused dimension y
    int tiled;             // 1: tiled layout below, 0: the layouts above
    int cols, ntl;         // kx columns per tile, tiles
    int RLy, Fy, NRy;      // last radix of the y transform, its items, stored rows Fy/2 + 1
    BD_HD int nxr() const { return nx + 1; }
    BD_HD int nyr() const { return ny + 1; }
    BD_HD int nzr() const { return nz > 1 ? nz + 1 : 1; }
    BD_HD long reduced_elems() const { return (long)ncomp * nzr() * nyr() * nxr(); }
    BD_HD long storage_elems() const {
        if (tiled) return (long)nzr() * ntl * NRy * cols * ncomp * RLy;
        return nz == 1 ? (long)nxr() * 4 * RL * nrows : (long)nxr() * ntiles * 6 * RL * nrows * ty;
    }
    BD_HD long reduced_index(int c, int kz, int ky, int kx) const {
        return (((long)c * nzr() + kz) * nyr() + ky) * nxr() + kx;
    }
};

BD_HD KLayout make_klayout(int nx, int ny, int nz, int ty) {
    KLayout k;
    k.nx = nx; k.ny = ny; k.nz = nz;
    k.Px = 2 * nx; k.Py = 2 * ny; k.Pz = nz > 1 ? 2 * nz : 1;
    k.ncomp = nz > 1 ? 6 : 4;
    k.Lf = nz > 1 ? k.Pz : k.Py;
    k.RL = dec_rlast(k.Lf);
    k.nrows = khat_rows(k.Lf);
    k.ty = nz > 1 ? ty : 1;
    k.ntiles = nz > 1 ? k.Py / ty : 1;
    k.tiled = 0; k.cols = 1; k.ntl = nx + 1;
    k.RLy = dec_rlast(k.Py); k.Fy = k.Py / k.RLy; k.NRy = k.Fy / 2 + 1;
    return k;
}
BD_HD KLayout make_klayout_tiled(int nx, int ny, int nz, int cols) {
    KLayout k = make_klayout(nx, ny, nz, 1);
    k.tiled = 1; k.cols = cols; k.ntl = (nx + 1 + cols - 1) / cols;
    return k;
}

// fold a full frequency k of a length-L dimension to the stored half: returns the
// reduced index and flips `sign` for components odd in that dimension
BD_HD int fold_freq(int L, int k, bool odd, double& sign) {
    if (2 * k > L) { if (odd) sign = -sign; return L - k; }
    return k;
}

// value of storage element idx, read from the natural reduced array
BD_HD double storage_value(const KLayout& kl, long idx, const double* Kred) {
    double sign = 1.0;
    if (kl.tiled) {
        const int CH = k_chunk(kl.Py), NCH = kl.RLy / CH;
        const int qi = (int)(idx % CH); idx /= CH;
        const int col = (int)(idx % kl.cols); idx /= kl.cols;
        const int slot = (int)(idx % kl.NRy); idx /= kl.NRy;
        const int ch = (int)(idx % NCH); idx /= NCH;
        const int c = (int)(idx % kl.ncomp); idx /= kl.ncomp;
        const int tile = (int)(idx % kl.ntl); const int kzr = (int)(idx / kl.ntl);
        const int kx = tile * kl.cols + col, q = ch * CH + qi;
        if (kx > kl.nx) return 0.0;                      // padding columns of the last tile
        const int kyr = fold_freq(kl.Py, slot_to_f(kl.Py, slot) + kl.Fy * q, comp_is_odd(c, 1), sign);
        return sign * Kred[kl.reduced_index(c, kzr, kyr, kx)];
    }
    const int t = (int)(idx % kl.ty); idx /= kl.ty;
    const int row = (int)(idx % kl.nrows); idx /= kl.nrows;
    const int q = (int)(idx % kl.RL); idx /= kl.RL;
    const int c = (int)(idx % 6); idx /= 6;
    const int tile = (int)(idx % kl.ntiles); const int slot = (int)(idx / kl.ntiles);
    const int ky = freq_of_pos(kl.Py, tile * kl.ty + t);
    const int kyr = fold_freq(kl.Py, ky, comp_is_odd(c, 1), sign);
    const int kz = khat_f_of_row(kl.Pz, row) + dec_items(kl.Pz) * q;
    const int kzr = fold_freq(kl.Pz, kz, comp_is_odd(c, 2), sign);
    return sign * Kred[kl.reduced_index(c, kzr, kyr, slot)];
}

// storage index and sign that hold the natural reduced entry (c, kz, ky, kx)
BD_HD long storage_index_of(const KLayout& kl, int c, int kz, int ky, int kx, float& sign) {
    sign = 1.f;
    if (kl.tiled) {
        int f = ky % kl.Fy, q = ky / kl.Fy;
        if (2 * f > kl.Fy) {        // stored in the row of its mirror item, q reversed
            f = kl.Fy - f; q = kl.RLy - 1 - q;
            if (comp_is_odd(c, 1)) sign = -1.f;
        }
        const int CH = k_chunk(kl.Py), NCH = kl.RLy / CH;
        return ((((((long)kz * kl.ntl + kx / kl.cols) * kl.ncomp + c) * NCH + q / CH) * kl.NRy + f_to_slot(kl.Py, f)) * kl.cols
                + kx % kl.cols) * CH + q % CH;
    }
    const int L = kl.Lf, F = dec_items(L), kf = kl.nz == 1 ? ky : kz;
    int f = kf % F, q = kf / F;
    if (2 * f > F) {            // stored under its mirror item, q reversed
        f = F - f; q = kl.RL - 1 - q;
        if (comp_is_odd(c, kl.nz == 1 ? 1 : 2)) sign = -1.f;
    }
    const int row = khat_row_of_f(L, f);
    if (kl.nz == 1) return (((long)kx * 4 + c) * kl.RL + q) * kl.nrows + row;
    const int py = pos_of_freq(kl.Py, ky), tile = py / kl.ty, t = py % kl.ty;
    return (((((long)kx * kl.ntiles + tile) * 6 + c) * kl.RL + q) * kl.nrows + row) * kl.ty + t;
}

}  // namespace bd
