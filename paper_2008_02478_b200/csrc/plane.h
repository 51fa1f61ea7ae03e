// plane.h — the plane path of slabs (nz = 2, 4, 8, 16, 32 and, on wide meshes, 64, the paper's
// pipelined regime of few cells along z): the x spectrum stays y- and z-UNPADDED in HBM and the whole padded
// (y, z) plane of one kx is transformed, multiplied by the kernel spectrum and transformed back
// on chip (S2..S6 of SURVEY.md §8(a) in one launch, all 3 components).
//
//   XFwdT<LX,1>   S1          M -> X[cz = c nz + z][kx (nx+1)][y (ny)]          (xt.h, y fastest)
//   YZFused       S2..S6      X -> P[q (NQ)][cz][kx][n (LSP)]                   (this file)
//   XInvP         S7 (+S8)    P -> H, summing the NQ partial planes            (this file)
//
// The padded plane of one kx (3 x nz x Py complex) does not fit one SM, so the y transform is
// split by the residue q of ky modulo NQ = 1, 2, 4 or 8 (decimation in frequency, first stage done on load):
//     X^[q + NQ k] = sum_{n < LS} W_LS^(n k) a_q[n],   LS = Py / NQ <= 256 (128 at nz = 64),
//     a_q[n] = W_Py^(n q) sum_r x[n + LS r] W_NQ^(q r)            (x = 0 beyond ny: r < NQ/2)
// Block (kx, q) holds its 3 x nz pencils of LS points in shared memory (3 x 32 x 256 complex =
// 204 KB with padding at nz = 32; slabs of 16 / 8 cells take half / a quarter of that and of the threads, 2 / 4 blocks per
// SM), runs the z transform, the multiply and the inverse z transform in registers per ky column — ZS = nz / 8 lanes per
// column, lane p taking the 16 frequencies kz = ZS m + p (one lane with all 2 nz frequencies below 8 cells) — transforms back along y and writes its PARTIAL result
//     P_q[n] = W_Py^(-n q) sum_k H^[q + NQ k] W_LS^(-n k),        n < LS,
// of which the inverse x kernel forms  h[n + LS r] = sum_q W_NQ^(-q r) P_q[n]  (r < NQ/2 kept).
// HBM per evaluation at 512x512x32: 0.10 + 0.20 | 0.20 + 0.25 + 0.40 | 0.40 + 0.10 GB = 1.66 GB
// (the tiled path: 2.04 GB), all of it in pieces of at least 64 contiguous bytes (32 at NQ = 8).
#pragma once
#include "xt.h"
#include "xz.h"

namespace bd {

#ifndef BD_YZ_NT
#define BD_YZ_NT 384
#endif
constexpr int kKindYZFused = 1;          // timing slot of the fused kernel (as YFused)
constexpr int kPlaneNZ = 32;             // the slab the plane path was built for (4 lanes per ky column); 64, 16 and 8 cells: 8, 2, 1 lanes

BD_HD constexpr int pl_pe(int e) { return e + (e >> 4); }            // shared pencil padding: 1 per 16
// odd: the four lanes of a ky column store rows 4 apart (zstage), which then fall into different banks
BD_HD constexpr int pl_pitch(int LS) { return (LS + (LS >> 4)) | 1; }
// sub-transform of LS = R0 x 16 points, two passes: position e = q0 16 + q1 holds k = q0 + R0 q1
BD_HD int pl_freq_of_pos(int LS, int e) { return e / 16 + (LS / 16) * (e % 16); }
BD_HD int pl_pos_of_freq(int LS, int k) { return (k % (LS / 16)) * 16 + k / (LS / 16); }

struct PlaneGeom {
    int on;        // 1: the mesh takes the plane path
    int nq;        // residues of ky (1, 2, 4 or 8)
    int ls;        // points of the sub-transform, Py / nq  (64, 128 or 256)
    int lsp;       // stored points of a partial plane: min(ls, ny)
    int zs;        // lanes per ky column, Pz / 16 (1 for slabs of fewer than 8 cells)
    int nsl;       // kernel-spectrum slots per residue, ls / 2 + 1
};
// nq_force > 0: take that many residues if the geometry allows it (tests)
inline PlaneGeom plane_geom(int nx, int ny, int nz, int nq_force = 0) {
    PlaneGeom g{0, 1, 0, 0, 0, 0};
    if ((nz != 64 && nz != 32 && nz != 16 && nz != 8 && nz != 4 && nz != 2) || nx < 4 || ny < 32 || ny > 1024) return g;
    const int Py = 2 * ny;
    const int lsmax = nz > 32 ? 128 : 256;           // 3 nz pencils of LS points in 227 KB
    int nq = 1;
    while (Py / nq > lsmax) nq *= 2;
    // narrow meshes: more residues while the (nx + 1) nq blocks of YZFused still fit the SMs at once (measured on 148 SMs:
    // 64 x 64 x 32 31.6 -> 25.6 us, 128 x 128 x 8 31.7 -> 23.5 us, 32 x 128 x 32 48 -> 30 us; profiles/r02_plane.md)
    const int per_sm = nz >= 32 ? 1 : (nz >= 8 ? 32 / nz : 4);
    while (nq < 8 && Py / (2 * nq) >= 64 && (long)(nx + 1) * nq * 2 <= 148L * per_sm) nq *= 2;
    if (nq_force > 0) nq = nq_force;
    if (nq != 1 && nq != 2 && nq != 4 && nq != 8) return g;
    const int ls = Py / nq;
    if (ls < 64 || ls > lsmax) return g;
    g.on = 1; g.nq = nq; g.ls = ls; g.lsp = ls < ny ? ls : ny; g.zs = nz >= 8 ? 2 * nz / 16 : 1; g.nsl = ls / 2 + 1;
    return g;
}

// ------------------------------------------------------------------ kernel spectrum, plane order
// KP[kx][qs (NQ)][c (6)][pr (ZS+1)][h (2)][slot (NSL)][4]   fp32
// Slot s of residue qs stands for one ky = qs + NQ k <= Py/2 (the direct frequencies of block qs, in the
// order of their positions e); entry (pr, h, i) holds kz = ZS (4 h + i) + pr for pr < ZS — the direct
// frequencies kz <= Pz/2 of lane pr — and kz = ZS (4 h + i + 1) for pr = ZS (lane 0's mirror list, which
// ends in the Nyquist plane).  A column at ky > Py/2 reads the slot of Py - ky (residue (NQ - q) % NQ) and
// negates the y-odd components; a lane's mirrored frequencies kz = ZS m + p, m >= 8, read entry 15 - m of
// residue (ZS - p) % ZS (pr = ZS for p = 0) and negate the z-odd components.
// kidx[q LS + e] = slot | qs << 12 | (ky > Py/2) << 15
struct PlaneK {
    int nx, ny, nz, nq, ls, zs, nsl;
    // a lane's lists hold hb = min(8, nz) frequencies each (8: a lane has 16 frequencies; slabs of 4 / 2 cells have 8 / 4
    // frequencies in all), stored as nh = 2 or 1 groups of four
    BD_HD int hb() const { return nz >= 8 ? 8 : nz; }
    BD_HD int nh() const { return nz >= 8 ? 2 : 1; }
    BD_HD long per_kx() const { return (long)nq * 6 * (zs + 1) * nh() * nsl * 4; }
    BD_HD long storage_elems() const { return (long)(nx + 1) * per_kx(); }
    BD_HD long index(int kx, int qs, int c, int pr, int h, int slot, int i) const {
        return ((((((long)kx * nq + qs) * 6 + c) * (zs + 1) + pr) * nh() + h) * nsl + slot) * 4 + i;
    }
};
inline PlaneK make_plane_k(int nx, int ny, int nz, const PlaneGeom& g) {
    return PlaneK{nx, ny, nz, g.nq, g.ls, g.zs, g.nsl};
}
// host tables: kidx as above, slot_ky[qs nsl + slot] = ky of the slot (-1: unused)
inline void plane_fill_tables(int ny, const PlaneGeom& g, int* kidx, int* slot_ky) {
    const int Py = 2 * ny, LS = g.ls, NQ = g.nq, NSL = g.nsl;
    for (int i = 0; i < NQ * NSL; ++i) slot_ky[i] = -1;
    for (int qs = 0; qs < NQ; ++qs) {
        int n = 0;
        for (int e = 0; e < LS; ++e) {
            const int ky = qs + NQ * pl_freq_of_pos(LS, e);
            if (2 * ky <= Py) { kidx[qs * LS + e] = n | (qs << 12); slot_ky[qs * NSL + n] = ky; ++n; }
        }
    }
    for (int q = 0; q < NQ; ++q)
        for (int e = 0; e < LS; ++e) {
            const int ky = q + NQ * pl_freq_of_pos(LS, e);
            if (2 * ky <= Py) continue;
            const int km = Py - ky, qs = km % NQ, em = pl_pos_of_freq(LS, (km - qs) / NQ);
            kidx[q * LS + e] = (kidx[qs * LS + em] & 0xfff) | (qs << 12) | (1 << 15);
        }
}
// value of storage element idx from the natural reduced spectrum Kred[c][kz <= nz][ky <= ny][kx <= nx]
BD_HD double plane_storage_value(const PlaneK& k, long idx, const int* slot_ky, const double* Kred) {
    const int i = (int)(idx % 4); idx /= 4;
    const int slot = (int)(idx % k.nsl); idx /= k.nsl;
    const int h = (int)(idx % k.nh()); idx /= k.nh();
    const int pr = (int)(idx % (k.zs + 1)); idx /= (k.zs + 1);
    const int c = (int)(idx % 6); idx /= 6;
    const int qs = (int)(idx % k.nq); const int kx = (int)(idx / k.nq);
    const int ky = slot_ky[qs * k.nsl + slot];
    if (ky < 0 || 4 * h + i >= k.hb()) return 0.0;
    const int kz = pr < k.zs ? k.zs * (4 * h + i) + pr : k.zs * (4 * h + i + 1);
    return Kred[(((long)c * (k.nz + 1) + kz) * (k.ny + 1) + ky) * (k.nx + 1) + kx];
}
// storage index that holds the natural reduced entry (c, kz, ky, kx)
BD_HD long plane_storage_index_of(const PlaneK& k, const int* kidx, int c, int kz, int ky, int kx) {
    const int qs = ky % k.nq, e = pl_pos_of_freq(k.ls, ky / k.nq);
    const int slot = kidx[qs * k.ls + e] & 0xfff;
    int pr = kz % k.zs, m = kz / k.zs;
    if (m >= k.hb()) { pr = k.zs; m = k.hb() - 1; }          // the Nyquist plane kz = Pz/2 = ZS hb
    return k.index(kx, qs, c, pr, m / 4, slot, m % 4);
}

// tw[(q R0 + q0) 16 + j] = W_Py^(j (NQ q0 + q)): output twiddle of the first pass (j < 16, q0 < R0) with the
// common factor W_Py^(j q) of the residue's input twiddle folded in
inline void plane_fill_tw(float2* h, int ny, const PlaneGeom& g) {
    const double pi = 3.14159265358979323846264338327950288;
    const int Py = 2 * ny, R0 = g.ls / 16;
    for (int q = 0; q < g.nq; ++q)
        for (int q0 = 0; q0 < R0; ++q0)
            for (int j = 0; j < 16; ++j) {
                const long m = ((long)j * (g.nq * q0 + q)) % Py;
                float2 w;
                if ((4 * m) % Py == 0) {
                    const float cx[4] = {1.f, 0.f, -1.f, 0.f}, sy[4] = {0.f, -1.f, 0.f, 1.f};
                    w = bd_f2(cx[(4 * m) / Py], sy[(4 * m) / Py]);
                } else {
                    const double a = -2.0 * pi * (double)m / (double)Py;
                    w = bd_f2((float)std::cos(a), (float)std::sin(a));
                }
                h[(q * R0 + q0) * 16 + j] = w;
            }
}
// Slot j of lane p of a 4- or 2-lane z stage holds cell (and inverse-transform output) pl_zrot(ZS, p, j): the lane's 16
// values rotated by its own block of 16 / ZS, which puts the block the lane keeps in slots [0, 16 / ZS) and the block
// lane p + r needs in slots [16 - r 16 / ZS, ...) for EVERY lane: the exchange of the partial inverse transforms needs
// no per-lane selection of registers.  (Rotating the inputs of the 16-point transform by s modulates its outputs by
// W_16^(-s m); the multiplication by the real K^ keeps that factor, and the inverse transform turns it back into the
// same rotation of the outputs.)  The 8-lane stage of nz = 64 is not rotated.
BD_HD constexpr int pl_zrot(int zs, int p, int j) { return (zs == 4 || zs == 2) ? ((j + (16 / zs) * p) & 15) : j; }
// zt[p 16 + j] = W_Pz^(j' p), j' = pl_zrot(ZS, p, j), p < ZS, j < 16
inline void plane_fill_zt(float2* h, int nz, const PlaneGeom& g) {
    const double pi = 3.14159265358979323846264338327950288;
    const int Pz = 2 * nz;
    for (int p = 0; p < g.zs; ++p)
        for (int j = 0; j < 16; ++j) {
            const int m = (pl_zrot(g.zs, p, j) * p) % Pz;
            float2 w;
            if ((4 * m) % Pz == 0) {
                const float cx[4] = {1.f, 0.f, -1.f, 0.f}, sy[4] = {0.f, -1.f, 0.f, 1.f};
                w = bd_f2(cx[(4 * m) / Pz], sy[(4 * m) / Pz]);
            } else {
                const double a = -2.0 * pi * (double)m / (double)Pz;
                w = bd_f2((float)std::cos(a), (float)std::sin(a));
            }
            h[p * 16 + j] = w;
        }
}

// ------------------------------------------------------------------ YZFused (S2..S6)
struct YZArgs {
    const float2* X;       // [3 NZ][nkx][ny]
    float2* P;             // [NQ][3 NZ][nkx][LSP]
    const float* KP;       // kernel spectrum, plane order
    const int* kidx;       // [NQ][LS]
    const float2* tw;      // plane_fill_tw
    const float2* zt;      // plane_fill_zt
    int nkx;               // nx + 1
    int ny;
};

// (-i)^Q b + a
template <int Q>
BD_HD float2 pl_add_rot(float2 a, float2 b) {
    if constexpr (Q == 0) return pk_add(a, b);
    else if constexpr (Q == 1) return pk_add_ib<-1>(a, b);
    else if constexpr (Q == 2) return pk_sub(a, b);
    else return pk_add_ib<+1>(a, b);
}

// H^ = K^ M^ at one frequency: k = (xx, yy, zz, xy, xz, yz), real
BD_HD void pl_mul3(float kxx, float kyy, float kzz, float kxy, float kxz, float kyz, float2& mx, float2& my, float2& mz) {
    const float2 hx = pk_fma(pk_bc(kxz), mz, pk_fma(pk_bc(kxy), my, pk_mul(pk_bc(kxx), mx)));
    const float2 hy = pk_fma(pk_bc(kyz), mz, pk_fma(pk_bc(kyy), my, pk_mul(pk_bc(kxy), mx)));
    const float2 hz = pk_fma(pk_bc(kzz), mz, pk_fma(pk_bc(kyz), my, pk_mul(pk_bc(kxz), mx)));
    mx = hx; my = hy; mz = hz;
}

BD_HD float pl_f4(const float4& v, int i) { return i == 0 ? v.x : (i == 1 ? v.y : (i == 2 ? v.z : v.w)); }

// One lane of a ky column: frequencies kz = ZS m + p, m < 16, of the 2 NZ-point z transform of the NZ cells
// (ZS = NZ / 8 lanes per column: 4, 2 or 1); returns its part y_p[c][j] of the inverse transform: for NZ = 32
//     out[j] = sum_p y_p[j],   out[j + 16] = sum_p i^p y_p[j]          (j < 16),
// for NZ = 16 out[j] = y_0[j] + y_1[j], for NZ = 8 out[j] = y[j], j < 8.  For NZ = 32 and 16 the lane works on rotated
// slots (pl_zrot): v[c][j] = y_p[c][pl_zrot(ZS, p, j)].
// col: the column in shared memory (element z of component c at col[(c NZ + z) pitch]);
// k: the lane's direct and mirror lists (pl_load_k: kA / kB point at h = 0 of component 0, kcs / khs are the float4
// strides between components and halves); sy = -1 for a column at ky > Py/2.
template <int NH> struct PlK { float4 d[NH][6]; const float4* kB; };     // a lane's direct list [h][c]; its mirror list is read when needed
template <int NH>
BD_HD void pl_load_k(const float4* __restrict__ kA, const float4* __restrict__ kB, long kcs, long khs, PlK<NH>& k) {
    BD_UNROLL
    for (int h = 0; h < NH; ++h) {
        BD_UNROLL
        for (int c = 0; c < 6; ++c) {
            k.d[h][c] = BD_LDG(kA + c * kcs + h * khs);
        }
    }
    k.kB = kB;
}
// exp(-2 pi i m / 8), m at run time (a lane's constant)
BD_HD float2 pl_w8(int m) {
    constexpr float C = 0.70710678118654752440f;
    switch (m & 7) {
        case 0: return bd_f2(1.f, 0.f);
        case 1: return bd_f2(C, -C);
        case 2: return bd_f2(0.f, -1.f);
        case 3: return bd_f2(-C, -C);
        case 4: return bd_f2(-1.f, 0.f);
        case 5: return bd_f2(-C, C);
        case 6: return bd_f2(0.f, 1.f);
        default: return bd_f2(C, C);
    }
}

// zt: the block's copy of the z twiddles in shared memory, zt[j ZS + p] = (plane_fill_zt)[p 16 + j] (the lanes of a column are
// neighbours: one wavefront per load)
template <int NZ>
BD_HD void pl_zlane(int p, float sy, const float2* col, int pitch, const PlK<(NZ >= 8 ? 2 : 1)>& k, long kcs, long khs,
                    const float2* zt, float2 (&v)[3][16]) {
    constexpr int ZSL = NZ >= 8 ? 2 * NZ / 16 : 1;
    // first stage of the 2 NZ-point transform of the NZ cells, split by the residue p of kz modulo ZS = NZ / 8 and pruned to
    // its non-zero inputs:  a_p[j] = W_Pz^(j p) sum_{r < ZS/2} x[j + 16 r] W_ZS^(r p)
    if constexpr (NZ == 64) {
        // eight lanes: x[j] + W_8^p x[j + 16] + (-i)^p x[j + 32] + W_8^(3p) x[j + 48]
        const int p4 = p & 3;
        Tw rot;
        rot.c = p4 == 0 ? 1.f : (p4 == 2 ? -1.f : 0.f);
        { const float s = p4 == 1 ? -1.f : (p4 == 3 ? 1.f : 0.f); rot.ns = bd_f2(-s, s); }
        const Tw w1 = make_tw(pl_w8(p)), w3 = make_tw(pl_w8(3 * p));
        BD_UNROLL
        for (int c = 0; c < 3; ++c) {
            BD_UNROLL
            for (int j = 0; j < 16; ++j) {
                const Tw t = make_tw(zt[j * ZSL + p]);
                const float2 x0 = col[(c * 64 + j) * pitch], x1 = col[(c * 64 + j + 16) * pitch];
                const float2 x2 = col[(c * 64 + j + 32) * pitch], x3 = col[(c * 64 + j + 48) * pitch];
                float2 a = pk_fma(pk_swap(x2), rot.ns, pk_fma(x2, pk_bc(rot.c), x0));
                a = pk_add(a, pk_add(pk_cmul(x1, w1), pk_cmul(x3, w3)));
                v[c][j] = pk_cmul(a, t);
            }
            PkDft<16, -1>::run(v[c]);
        }
    } else if constexpr (NZ == 32) {
        // (-i)^p as the pair (c, (-s, s)) of a twiddle
        Tw rot;
        rot.c = p == 0 ? 1.f : (p == 2 ? -1.f : 0.f);
        { const float s = p == 1 ? -1.f : (p == 3 ? 1.f : 0.f); rot.ns = bd_f2(-s, s); }
        // slot j = 4 a + b reads cell pl_zrot(4, p, j) = 4 ((a + p) & 3) + b
        const float2* cr[4];
        BD_UNROLL
        for (int a = 0; a < 4; ++a) cr[a] = col + 4 * ((a + p) & 3) * pitch;
        BD_UNROLL
        for (int c = 0; c < 3; ++c) {
            BD_UNROLL
            for (int j = 0; j < 16; ++j) {
                const Tw t = make_tw(zt[j * ZSL + p]);
                const float2 x0 = cr[j >> 2][(c * 32 + (j & 3)) * pitch], x1 = cr[j >> 2][(c * 32 + (j & 3) + 16) * pitch];
                const float2 a = pk_fma(pk_swap(x1), rot.ns, pk_fma(x1, pk_bc(rot.c), x0));
                v[c][j] = pk_cmul(a, t);
            }
            PkDft<16, -1>::run(v[c]);
        }
    } else if constexpr (NZ == 16) {
        // slot j = 8 a + b reads cell pl_zrot(2, p, j) = 8 ((a + p) & 1) + b
        const float2* cr[2] = {col + 8 * (p & 1) * pitch, col + 8 * ((p + 1) & 1) * pitch};
        BD_UNROLL
        for (int c = 0; c < 3; ++c) {
            BD_UNROLL
            for (int j = 0; j < 16; ++j)
                v[c][j] = pk_cmul(cr[j >> 3][(c * 16 + (j & 7)) * pitch], make_tw(zt[j * ZSL + p]));
            PkDft<16, -1>::run(v[c]);
        }
    } else {
        // one lane, all 2 NZ frequencies, NZ <= 8 cells: the zero padding prunes the transform itself
        BD_UNROLL
        for (int c = 0; c < 3; ++c) {
            BD_UNROLL
            for (int j = 0; j < NZ; ++j) v[c][j] = col[(c * NZ + j) * pitch];
            PkDftPruned<2 * NZ, -1>::run(v[c]);
        }
    }
    constexpr int NH = NZ >= 8 ? 2 : 1, HB = NZ >= 8 ? 8 : NZ, FPL = 2 * HB;     // list groups, list entries, the lane's frequencies
    // direct frequencies m = 0..HB-1, then the mirrored ones m = FPL - 1 - i
    BD_UNROLL
    for (int h = 0; h < NH; ++h) {
        BD_UNROLL
        for (int i = 0; i < (HB < 4 ? HB : 4); ++i) {
            const int m = 4 * h + i;
            pl_mul3(pl_f4(k.d[h][0], i), pl_f4(k.d[h][1], i), pl_f4(k.d[h][2], i), sy * pl_f4(k.d[h][3], i), pl_f4(k.d[h][4], i),
                    sy * pl_f4(k.d[h][5], i), v[0][m], v[1][m], v[2][m]);
        }
    }
    // the mirror list is the direct list of the partner lane (same warp, same iteration): mostly still in L1
    BD_UNROLL
    for (int h = 0; h < NH; ++h) {
        float4 km[6];
        BD_UNROLL
        for (int c = 0; c < 6; ++c) km[c] = BD_LDG(k.kB + c * kcs + h * khs);
        BD_UNROLL
        for (int i = 0; i < (HB < 4 ? HB : 4); ++i) {
            const int m = FPL - 1 - (4 * h + i);
            pl_mul3(pl_f4(km[0], i), pl_f4(km[1], i), pl_f4(km[2], i), sy * pl_f4(km[3], i), -pl_f4(km[4], i),
                    -sy * pl_f4(km[5], i), v[0][m], v[1][m], v[2][m]);
        }
    }
    if constexpr (NZ <= 8) {
        BD_UNROLL
        for (int c = 0; c < 3; ++c) PkDftTrunc<2 * NZ, +1>::run(v[c]);   // the NZ cells: v[c][0..NZ)
    } else {
        BD_UNROLL
        for (int c = 0; c < 3; ++c) PkDft<16, +1>::run(v[c]);
        BD_UNROLL
        for (int j = 0; j < 16; ++j) {
            const Tw t = make_tw(zt[j * ZSL + p]);
            BD_UNROLL
            for (int c = 0; c < 3; ++c) v[c][j] = pk_cmulc(v[c][j], t);
        }
    }
}

#if defined(__CUDA_ARCH__)
// Four lanes q = 2 hi + lo (xor distances 2 and 1) each hold C_q[c][0..NJ); afterwards the lane holds, for the NJ / 4
// values j = jb + i (jb = hi NJ/2 + lo NJ/4),  o0[c][i] = sum_q C_q[c][j]  and  o1[c][i] = sum_q i^q C_q[c][j]
// (the two exchange rounds of the 4-lane z stage, for any NJ).
template <int NJ>
__device__ __forceinline__ void pl_exchange4(const float2 (&C)[3][NJ], bool hi, bool lo, float2 (&o0)[3][NJ / 4], float2 (&o1)[3][NJ / 4]) {
    const float sg = hi ? -1.f : 1.f;
    float2 S[3][NJ / 2], D[3][NJ / 2];
    BD_UNROLL
    for (int c = 0; c < 3; ++c) {
        BD_UNROLL
        for (int i = 0; i < NJ / 2; ++i) {
            const float2 send = hi ? C[c][i] : C[c][NJ / 2 + i], mine = hi ? C[c][NJ / 2 + i] : C[c][i];
            float2 oth;
            oth.x = __shfl_xor_sync(0xffffffffu, send.x, 2);
            oth.y = __shfl_xor_sync(0xffffffffu, send.y, 2);
            S[c][i] = pk_add(mine, oth);
            D[c][i] = pk_mul(pk_sub(mine, oth), pk_bc(sg));
        }
    }
    BD_UNROLL
    for (int c = 0; c < 3; ++c) {
        BD_UNROLL
        for (int i = 0; i < NJ / 4; ++i) {
            const float2 sS = lo ? S[c][i] : S[c][NJ / 4 + i], sD = lo ? D[c][i] : D[c][NJ / 4 + i];
            const float2 kS = lo ? S[c][NJ / 4 + i] : S[c][i], kD = lo ? D[c][NJ / 4 + i] : D[c][i];
            float2 rS, rD;
            rS.x = __shfl_xor_sync(0xffffffffu, sS.x, 1);
            rS.y = __shfl_xor_sync(0xffffffffu, sS.y, 1);
            rD.x = __shfl_xor_sync(0xffffffffu, sD.x, 1);
            rD.y = __shfl_xor_sync(0xffffffffu, sD.y, 1);
            const float2 ev = lo ? rD : kD, od = lo ? kD : rD;
            o0[c][i] = pk_add(kS, rS);
            o1[c][i] = pk_add_ib<+1>(ev, od);
        }
    }
}
#endif

// cos(2 pi m / 128): quarter-wave table as cos64 (xz.h); the residue twiddles of NQ = 8 are 128th roots
BD_HD constexpr float cos128(int m) {
    constexpr float q[33] = {
        1.000000000e+00f, 9.987954562e-01f, 9.951847267e-01f, 9.891765100e-01f, 9.807852804e-01f, 9.700312532e-01f,
        9.569403357e-01f, 9.415440652e-01f, 9.238795325e-01f, 9.039892931e-01f, 8.819212643e-01f, 8.577286100e-01f,
        8.314696123e-01f, 8.032075315e-01f, 7.730104534e-01f, 7.409511254e-01f, 7.071067812e-01f, 6.715589548e-01f,
        6.343932842e-01f, 5.956993045e-01f, 5.555702330e-01f, 5.141027442e-01f, 4.713967368e-01f, 4.275550934e-01f,
        3.826834324e-01f, 3.368898534e-01f, 2.902846773e-01f, 2.429801799e-01f, 1.950903220e-01f, 1.467304745e-01f,
        9.801714033e-02f, 4.906767433e-02f, 0.000000000e+00f
    };
    m &= 127;
    return m <= 32 ? q[m] : (m <= 64 ? -q[64 - m] : (m <= 96 ? -q[m - 64] : q[128 - m]));
}
// z * exp(DIR 2 pi i m / 128), m known after unrolling
template <int DIR>
BD_HD float2 pk_mul_w128(float2 z, int m) {
    m &= 127;
    if ((m & 1) == 0) return pk_mul_w64<DIR>(z, m >> 1);
    const float c = cos128(m), s = (float)DIR * cos128(m - 32);
    return pk_fma(pk_swap(z), bd_f2(-s, s), pk_mul(z, pk_bc(c)));
}
// z * exp(DIR 2 pi i m / 8)
template <int DIR>
BD_HD float2 pk_mul_w8(float2 z, int m) { return pk_mul_w64<DIR>(z, 8 * (m & 7)); }

template <int LS, int NQ, int NZ_ = kPlaneNZ>
struct YZFused {
    using Args = YZArgs;
    static constexpr int KIND = kKindYZFused;
    static constexpr int NZ = NZ_, NPEN = 3 * NZ, ZS = NZ >= 8 ? 2 * NZ / 16 : 1, NH = NZ >= 8 ? 2 : 1;
    // thinner slabs: smaller blocks (at least 96 threads), 32 / NZ (at most 4) of them per SM
    static constexpr int NT = NZ >= kPlaneNZ ? BD_YZ_NT : (NZ >= 8 ? BD_YZ_NT * NZ / kPlaneNZ : BD_YZ_NT / 4);
    static constexpr int MINB = NZ >= kPlaneNZ ? 1 : (NZ >= 8 ? kPlaneNZ / NZ : 4);
    static constexpr int NPHASES = 5;
    static constexpr int R0 = LS / 16;                   // first-pass radix; the second pass is radix 16
    static constexpr int PITCH = pl_pitch(LS);
    static constexpr int NSL = LS / 2 + 1;
    static constexpr int LSP = NQ == 1 ? LS / 2 : LS;    // stored points of a partial plane
    static constexpr int NIN = NQ == 1 ? R0 / 2 : R0;    // first-pass inputs that are not zero padding
    static_assert(NT % 16 == 0 && NT % R0 == 0 && NT % 4 == 0, "thread mapping");
    static BD_HD long smem_elems(const Args&) { return (long)NPEN * PITCH + ZS * 16; }      // pencils, then the z twiddles
    // With R0 = 16 the 16 threads that run a pencil's first pass (phase 0) also run its radix-16 pass (phase 1), and
    // likewise phases 3 and 4: those phases meet at a warp barrier, so the warps of a block drift apart and the global
    // loads and stores of phases 0 and 4 overlap the arithmetic of phases 1 and 3 of other warps
    static BD_HD constexpr bool warp_local_after(int ph) { return R0 == 16 && NT % 32 == 0 && (ph == 0 || ph == 3); }

    // blockIdx.x = kx NQ + o; residues q and NQ - q (which read each other's kernel-spectrum slots) are neighbours
    static BD_HD int q_of_order(int o) {
        if (NQ == 4) return (o >> 1) | ((o & 1) << 1);                       // 0, 2, 1, 3
        if (NQ == 8) return o == 0 ? 0 : (o == 1 ? 4 : ((o & 1) ? 8 - (o >> 1) : (o >> 1)));   // 0, 4, 1, 7, 2, 6, 3, 5
        return o;
    }

    // constant input twiddle of the residue: z * W_(NQ R0)^(DIR r Q)
    template <int DIR, int Q>
    static BD_HD float2 in_tw(float2 z, int r) {
        if constexpr (Q == 0) return z;
        else if constexpr (NQ * R0 <= 64) return pk_mul_w64<DIR>(z, r * Q * (64 / (NQ * R0)));
        else return pk_mul_w128<DIR>(z, r * Q * (128 / (NQ * R0)));
    }

    // phase 0: load, residue stage and first pass (radix R0, stride 16) of every pencil
    template <int Q>
    static BD_HD void load_pass(int tid, int kx, const Args& a, float2* sm) {
        constexpr int PG = NT / 16;
        const int j = tid % 16, pg = tid / 16;
        Tw tw[R0];
        BD_UNROLL
        for (int q0 = 0; q0 < R0; ++q0) tw[q0] = make_tw(BD_LDG(&a.tw[(Q * R0 + q0) * 16 + j]));
        if constexpr (NQ == 8) {
            // four non-zero quarters x[n + LS r'], r' < 4: a_q[n] = sum_r' W_8^(q r') x[n + LS r'], two quarters at a time
            for (int pc = pg; pc < NPEN; pc += PG) {
                const float2* xp = a.X + ((long)pc * a.nkx + kx) * a.ny + j;
                float2 v[R0], b0[R0], b1[R0];
                BD_UNROLL
                for (int r = 0; r < R0; ++r) { b0[r] = BD_LDCG(xp + 16 * r); b1[r] = BD_LDCG(xp + 16 * r + LS); }
                BD_UNROLL
                for (int r = 0; r < R0; ++r) v[r] = pk_add(b0[r], pk_mul_w8<-1>(b1[r], Q));
                BD_UNROLL
                for (int r = 0; r < R0; ++r) { b0[r] = BD_LDCG(xp + 16 * r + 2 * LS); b1[r] = BD_LDCG(xp + 16 * r + 3 * LS); }
                BD_UNROLL
                for (int r = 0; r < R0; ++r)
                    v[r] = in_tw<-1, Q>(pk_add(v[r], pk_add(pk_mul_w8<-1>(b0[r], 2 * Q), pk_mul_w8<-1>(b1[r], 3 * Q))), r);
                PkDft<R0, -1>::run(v);
                float2* po = sm + pc * PITCH + j;
                BD_UNROLL
                for (int q0 = 0; q0 < R0; ++q0) {
                    if (Q == 0 && q0 == 0) BD_STS(po + 0, v[0]);
                    else BD_STS(po + 17 * q0, pk_cmul(v[q0], tw[q0]));
                }
            }
            return;
        }
        constexpr int NLD = NQ == 4 ? 2 * R0 : NIN;
        float2 nxt[NLD];
        auto issue = [&](int pc) {
            const float2* xp = a.X + ((long)pc * a.nkx + kx) * a.ny + j;
            BD_UNROLL
            for (int r = 0; r < NIN; ++r) nxt[r] = BD_LDCG(xp + 16 * r);
            if constexpr (NQ == 4) {
                BD_UNROLL
                for (int r = 0; r < R0; ++r) nxt[R0 + r] = BD_LDCG(xp + 16 * r + LS);
            }
        };
        if (pg < NPEN) issue(pg);
        for (int pc = pg; pc < NPEN; pc += PG) {
            float2 v[R0];
            BD_UNROLL
            for (int r = 0; r < NIN; ++r) {
                if constexpr (NQ == 4) v[r] = in_tw<-1, Q>(pl_add_rot<Q>(nxt[r], nxt[R0 + r]), r);
                else v[r] = in_tw<-1, Q>(nxt[r], r);
            }
            if (pc + PG < NPEN) issue(pc + PG);
            if constexpr (NQ == 1) PkDftPruned<R0, -1>::run(v);
            else PkDft<R0, -1>::run(v);
            float2* po = sm + pc * PITCH + j;
            BD_UNROLL
            for (int q0 = 0; q0 < R0; ++q0) {
                if (Q == 0 && q0 == 0) BD_STS(po + 0, v[0]);
                else BD_STS(po + 17 * q0, pk_cmul(v[q0], tw[q0]));
            }
        }
    }

    // phases 1 and 3: second pass (radix 16 on 16 contiguous points), forward / inverse
    template <int DIR>
    static BD_HD void pass16(int tid, float2* sm) {
        constexpr int PG = NT / R0;
        const int q0 = tid % R0, pg = tid / R0;
        // the next pencil's points are read before this one's transform: their latency runs under the arithmetic
        float2 nxt[16];
        if (pg < NPEN) {
            BD_UNROLL
            for (int i = 0; i < 16; ++i) nxt[i] = sm[pg * PITCH + 17 * q0 + i];
        }
        for (int pc = pg; pc < NPEN; pc += PG) {
            float2* ps = sm + pc * PITCH + 17 * q0;
            float2 v[16];
            BD_UNROLL
            for (int i = 0; i < 16; ++i) v[i] = nxt[i];
            if (pc + PG < NPEN) {
                BD_UNROLL
                for (int i = 0; i < 16; ++i) nxt[i] = ps[PG * PITCH + i];
            }
            PkDft<16, DIR>::run(v);
            BD_UNROLL
            for (int i = 0; i < 16; ++i) BD_STS(ps + i, v[i]);
        }
    }

    // phase 4: inverse first pass, residue stage, store of the partial plane
    template <int Q>
    static BD_HD void pass_store(int tid, int kx, const Args& a, float2* sm) {
        constexpr int PG = NT / 16;
        const int j = tid % 16, pg = tid / 16;
        Tw tw[R0];
        BD_UNROLL
        for (int q0 = 0; q0 < R0; ++q0) tw[q0] = make_tw(BD_LDG(&a.tw[(Q * R0 + q0) * 16 + j]));
        for (int pc = pg; pc < NPEN; pc += PG) {
            const float2* pi = sm + pc * PITCH + j;
            float2 v[R0];
            BD_UNROLL
            for (int q0 = 0; q0 < R0; ++q0) {
                if (Q == 0 && q0 == 0) v[0] = pi[0];
                else v[q0] = pk_cmulc(pi[17 * q0], tw[q0]);
            }
            if constexpr (NQ == 1) PkDftTrunc<R0, +1>::run(v);
            else PkDft<R0, +1>::run(v);
            float2* po = a.P + (((long)Q * NPEN + pc) * a.nkx + kx) * LSP + j;
            BD_UNROLL
            for (int r = 0; r < NIN; ++r) { const float2 o = in_tw<+1, Q>(v[r], r); BD_STCG(po + 16 * r, o); }
        }
    }

    // phase 2: z transform, multiply, inverse z transform of every ky column; 4 lanes per column
    static BD_HD void zstage(int tid, int kx, int q, const Args& a, float2* sm) {
        const float4* kbase = reinterpret_cast<const float4*>(a.KP) + (long)kx * (NQ * 6L * (ZS + 1) * NH * NSL);
        constexpr long KCS = (long)(ZS + 1) * NH * NSL, KHS = NSL;
        // item w = (column e, lane p): its kernel-spectrum lists and the sign of the y-odd components
        auto lists = [&](int w, PlK<NH>& k) {
            const int p = w & (ZS - 1), e = w / ZS;
            const int ki = BD_LDG(&a.kidx[q * LS + e]);
            const float4* kq = kbase + (long)((ki >> 12) & 7) * 6 * KCS + (ki & 0xfff);
            pl_load_k<NH>(kq + (long)p * NH * NSL, kq + (long)(p ? ZS - p : ZS) * NH * NSL, KCS, KHS, k);
            return (ki >> 15) ? -1.f : 1.f;
        };
        for (int w = tid; w < LS * ZS; w += NT) {
            const int p = w & (ZS - 1), e = w / ZS;
            float2* col = sm + pl_pe(e);
#if defined(__CUDA_ARCH__)
            PlK<NH> kc;
            const float sy = lists(w, kc);
            float2 y[3][16];
            pl_zlane<NZ>(p, sy, col, PITCH, kc, KCS, KHS, sm + NPEN * PITCH, y);
            if constexpr (ZS == 4) {
                // out[j] = sum_p y_p[j], out[j + 16] = sum_p i^p y_p[j].  The lane keeps j = 4 p + i, i < 4: its own values
                // sit in slots i, those of lane p + r (mod 4) in that lane's slots 16 - 4 r + i (pl_zrot): three rounds, the
                // same registers sent by every lane.  sum_s i^s y_s = i^p (t_0 + i t_1 - t_2 - i t_3), t_r from lane p + r
                Tw ip;
                ip.c = p == 0 ? 1.f : (p == 2 ? -1.f : 0.f);
                { const float sn = p == 1 ? 1.f : (p == 3 ? -1.f : 0.f); ip.ns = bd_f2(-sn, sn); }
                BD_UNROLL
                for (int c = 0; c < 3; ++c) {
                    BD_UNROLL
                    for (int i = 0; i < 4; ++i) {
                        float2 t[4];
                        t[0] = y[c][i];
                        BD_UNROLL
                        for (int r = 1; r < 4; ++r) {
                            t[r].x = __shfl_sync(0xffffffffu, y[c][16 - 4 * r + i].x, (p + r) & 3, 4);
                            t[r].y = __shfl_sync(0xffffffffu, y[c][16 - 4 * r + i].y, (p + r) & 3, 4);
                        }
                        BD_STS(col + (c * NZ + 4 * p + i) * PITCH, pk_add(pk_add(t[0], t[2]), pk_add(t[1], t[3])));
                        BD_STS(col + (c * NZ + 16 + 4 * p + i) * PITCH,
                               pk_cmul(pk_add_ib<+1>(pk_sub(t[0], t[2]), pk_sub(t[1], t[3])), ip));
                    }
                }
            } else if constexpr (ZS == 8) {
                // out[j + 16 r] = sum_p W_8^(-r p) y_p[j], r < 4.  Lanes p and p + 4 first: A = y_q + y_(q+4) feeds r = 0, 2,
                // B = y_q - y_(q+4) feeds r = 1, 3; then the four lanes q of a half combine A and W_8^(-q) B as the 4-lane stage does
                const bool top = (p & 4) != 0, hi = (p & 2) != 0, lo = (p & 1) != 0;
                const float st = top ? -1.f : 1.f;
                const Tw wq = make_tw(pl_w8(p & 3));            // W_8^(-q) = conj(W_8^q)
                float2 A[3][8], B[3][8];
                BD_UNROLL
                for (int c = 0; c < 3; ++c) {
                    BD_UNROLL
                    for (int i = 0; i < 8; ++i) {
                        const float2 send = top ? y[c][i] : y[c][8 + i], mine = top ? y[c][8 + i] : y[c][i];
                        float2 oth;
                        oth.x = __shfl_xor_sync(0xffffffffu, send.x, 4);
                        oth.y = __shfl_xor_sync(0xffffffffu, send.y, 4);
                        A[c][i] = pk_add(mine, oth);
                        B[c][i] = pk_cmulc(pk_mul(pk_sub(mine, oth), pk_bc(st)), wq);
                    }
                }
                float2 r0[3][2], r2[3][2], r1[3][2], r3[3][2];
                pl_exchange4<8>(A, hi, lo, r0, r2);
                pl_exchange4<8>(B, hi, lo, r1, r3);
                const int jb = (top ? 8 : 0) + (hi ? 4 : 0) + (lo ? 2 : 0);
                BD_UNROLL
                for (int c = 0; c < 3; ++c) {
                    BD_UNROLL
                    for (int i = 0; i < 2; ++i) {
                        BD_STS(col + (c * NZ + jb + i) * PITCH, r0[c][i]);
                        BD_STS(col + (c * NZ + 16 + jb + i) * PITCH, r1[c][i]);
                        BD_STS(col + (c * NZ + 32 + jb + i) * PITCH, r2[c][i]);
                        BD_STS(col + (c * NZ + 48 + jb + i) * PITCH, r3[c][i]);
                    }
                }
            } else if constexpr (ZS == 2) {
                // out[j] = y_0[j] + y_1[j]: the lane keeps j = 8 p + i (its slots i) and sends its slots 8 + i (pl_zrot)
                BD_UNROLL
                for (int c = 0; c < 3; ++c) {
                    BD_UNROLL
                    for (int i = 0; i < 8; ++i) {
                        float2 oth;
                        oth.x = __shfl_xor_sync(0xffffffffu, y[c][8 + i].x, 1);
                        oth.y = __shfl_xor_sync(0xffffffffu, y[c][8 + i].y, 1);
                        BD_STS(col + (c * NZ + 8 * p + i) * PITCH, pk_add(y[c][i], oth));
                    }
                }
            } else {
                BD_UNROLL
                for (int c = 0; c < 3; ++c) {
                    BD_UNROLL
                    for (int j = 0; j < NZ; ++j) BD_STS(col + (c * NZ + j) * PITCH, y[c][j]);
                }
            }
#else
            // host emulation (tests/emu): lane 0 of a column runs the four lanes in turn, same arithmetic
            if (p != 0) continue;
            float2 y[ZS][3][16];
            for (int pp = 0; pp < ZS; ++pp) {
                PlK<NH> k;
                const float sy = lists(w + pp, k);
                pl_zlane<NZ>(pp, sy, col, PITCH, k, KCS, KHS, sm + NPEN * PITCH, y[pp]);
            }
            for (int c = 0; c < 3; ++c)
                for (int j = 0; j < 16; ++j) {
                    if constexpr (ZS == 8) {
                        for (int r = 0; r < 4; ++r) {
                            float2 acc = bd_f2(0.f, 0.f);
                            for (int pp = 0; pp < 8; ++pp) acc = pk_add(acc, pk_cmulc(y[pp][c][j], make_tw(pl_w8(r * pp))));
                            col[(c * NZ + 16 * r + j) * PITCH] = acc;
                        }
                    } else if constexpr (ZS == 4) {
                        // y_p[j] sits in lane p's slot (j - 4 p) & 15 (pl_zrot); lane pk = j / 4 combines, starting with its own
                        const int pk = j >> 2;
                        float2 t[4];
                        for (int r = 0; r < 4; ++r) t[r] = y[(pk + r) & 3][c][(j - 4 * ((pk + r) & 3)) & 15];
                        Tw ip;
                        ip.c = pk == 0 ? 1.f : (pk == 2 ? -1.f : 0.f);
                        { const float sn = pk == 1 ? 1.f : (pk == 3 ? -1.f : 0.f); ip.ns = bd_f2(-sn, sn); }
                        col[(c * NZ + j) * PITCH] = pk_add(pk_add(t[0], t[2]), pk_add(t[1], t[3]));
                        col[(c * NZ + 16 + j) * PITCH] = pk_cmul(pk_add_ib<+1>(pk_sub(t[0], t[2]), pk_sub(t[1], t[3])), ip);
                    } else if constexpr (ZS == 2) {
                        const int pk = j >> 3;
                        col[(c * NZ + j) * PITCH] = pk_add(y[pk][c][j & 7], y[pk ^ 1][c][8 + (j & 7)]);
                    } else {
                        if (j < NZ) col[(c * NZ + j) * PITCH] = y[0][c][j];
                    }
                }
#endif
        }
    }

    // before the predecessor kernel has finished (launcher.cuh): the kernel-spectrum slots of this residue start towards
    // L2 (the blocks of one kx run side by side: between them they fetch all of its slots)
    static BD_HD void prologue(int tid, int bx, const Args& a) {
        const int kx = bx / NQ, q = q_of_order(bx % NQ);
        constexpr long KB = 6L * (ZS + 1) * NH * NSL * 4 * (long)sizeof(float);
        const char* kq = reinterpret_cast<const char*>(a.KP) + ((long)kx * NQ + q) * KB;
        for (long o = (long)tid * 128; o < KB; o += NT * 128) bd_prefetch_l2(kq + o);
    }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        const int kx = bx / NQ, q = q_of_order(bx % NQ);
        if constexpr (PH == 0) {
            for (int i = tid; i < ZS * 16; i += NT) sm[NPEN * PITCH + i] = BD_LDG(&a.zt[(i % ZS) * 16 + i / ZS]);
            if (q == 0) load_pass<0>(tid, kx, a, sm);
            if constexpr (NQ >= 2) { if (q == 1) load_pass<1>(tid, kx, a, sm); }
            if constexpr (NQ >= 4) { if (q == 2) load_pass<2>(tid, kx, a, sm); else if (q == 3) load_pass<3>(tid, kx, a, sm); }
            if constexpr (NQ == 8) {
                if (q == 4) load_pass<4>(tid, kx, a, sm); else if (q == 5) load_pass<5>(tid, kx, a, sm);
                else if (q == 6) load_pass<6>(tid, kx, a, sm); else if (q == 7) load_pass<7>(tid, kx, a, sm);
            }
        } else if constexpr (PH == 1) {
            pass16<-1>(tid, sm);
        } else if constexpr (PH == 2) {
            zstage(tid, kx, q, a, sm);
        } else if constexpr (PH == 3) {
            pass16<+1>(tid, sm);
        } else {
            if (q == 0) pass_store<0>(tid, kx, a, sm);
            if constexpr (NQ >= 2) { if (q == 1) pass_store<1>(tid, kx, a, sm); }
            if constexpr (NQ >= 4) { if (q == 2) pass_store<2>(tid, kx, a, sm); else if (q == 3) pass_store<3>(tid, kx, a, sm); }
            if constexpr (NQ == 8) {
                if (q == 4) pass_store<4>(tid, kx, a, sm); else if (q == 5) pass_store<5>(tid, kx, a, sm);
                else if (q == 6) pass_store<6>(tid, kx, a, sm); else if (q == 7) pass_store<7>(tid, kx, a, sm);
            }
        }
    }
};

// ------------------------------------------------------------------ XInvP (S7, S8 on the way)
struct XPArgs {
    const float2* P;       // [NQ][3 nz][nkx][LSP]
    float* H;              // [3][nz][ny][nx]
    const float2* ptw;     // per-pass twiddles of length LX
    const float4* xpost;   // fill_xpost table
    int ny;
    int nkx;               // nx + 1
    int lsp;               // stored points of a partial plane
    long qstride;          // elements between partial planes
    EnergyArgs en;         // energy gathered while H is written (en.M == nullptr: off)
};

// rows of H that are not consecutive: row = hi JB + lo sits at y0 + lo + hi (hi_pitch / pitch)
struct GRowsOutMap {
    float* p; long pitch; long hi_pitch; int jbs;
    static BD_HD constexpr int off(int S, int r) { return r * S; }
    BD_HD float2* ptr(int row, int e) const {
        return reinterpret_cast<float2*>(p + (row & ((1 << jbs) - 1)) * pitch + (row >> jbs) * hi_pitch) + e;
    }
    BD_HD void st(float2* q, float2 v) const { *q = v; }
    BD_HD void pre(const float2*, int) const {}
    BD_HD void stq(float2* q, float2 v, int) const { *q = v; }
};
struct GRowsOutMapA {          // H += the field (xt.h GRowsOutA)
    float* p; long pitch; long hi_pitch; int jbs;
    static BD_HD constexpr int off(int S, int r) { return r * S; }
    BD_HD float2* ptr(int row, int e) const {
        return reinterpret_cast<float2*>(p + (row & ((1 << jbs) - 1)) * pitch + (row >> jbs) * hi_pitch) + e;
    }
    mutable float2 hbuf[8];
    BD_HD void pre(const float2* q, int r) const { hbuf[r] = BD_LDCG(q); }
    BD_HD void stq(float2* q, float2 v, int r) const { *q = bd_f2(hbuf[r].x + v.x, hbuf[r].y + v.y); }
    BD_HD void st(float2* q, float2 v) const { *q = v; }
};
struct GRowsOutMapE {
    float* p; long pitch; long hi_pitch; int jbs; long m_minus_h; double* acc;
    static BD_HD constexpr int off(int S, int r) { return r * S; }
    BD_HD float2* ptr(int row, int e) const {
        return reinterpret_cast<float2*>(p + (row & ((1 << jbs) - 1)) * pitch + (row >> jbs) * hi_pitch) + e;
    }
    mutable float2 mbuf[8];
    BD_HD void pre(const float2* q, int r) const {
        mbuf[r] = BD_LDCG(reinterpret_cast<const float2*>(reinterpret_cast<const char*>(q) + m_minus_h));
    }
    BD_HD void stq(float2* q, float2 v, int r) const {
        *q = v;
        *acc += (double)mbuf[r].x * v.x + (double)mbuf[r].y * v.y;
    }
    BD_HD void st(float2* q, float2 v) const { *q = v; }
};

// Z[kp], Z[LX - kp] of the half-length complex row from the spectrum pair Y[kp], Y[LX - kp] (xt.h header)
BD_HD void xinv_pre(int LX, int kp, float2 Yk, float2 Ym, const float4& xp, float2* zr) {
    if (kp == 0) { Yk.y = 0.f; Ym.y = 0.f; }            // DC and Nyquist of a real row are real
    const float2 E = bd_f2(Yk.x + Ym.x, Yk.y - Ym.y);
    const float2 D = bd_f2(Yk.x - Ym.x, Yk.y + Ym.y);
    const float2 O = pk_cmulc(D, make_tw(bd_f2(xp.x, xp.y)));
    zr[bd_float_as_int(xp.z)] = bd_f2(E.x - O.y, E.y + O.x);
    if (kp != 0 && 2 * kp != LX) zr[bd_float_as_int(xp.w)] = bd_f2(E.x + O.y, O.x - E.y);
}

template <int LX, int NQ>
struct XInvP {
    using Args = XPArgs;
    static constexpr int KIND = kKindXInvT;
    static constexpr int NT = 256;
    static constexpr int MINB = LX >= 1024 ? 1 : 3;
    static constexpr int NP = dec_np(LX);
    static constexpr int NPHASES = NP + 1;
    static constexpr int RB = 16;                        // rows of H per block
    static constexpr int JB = NQ == 8 ? 4 : (NQ == 4 ? 8 : 16), JBS = NQ == 8 ? 2 : (NQ == 4 ? 3 : 4);   // points of a partial plane per block
    static BD_HD long smem_elems(const Args&) { return (long)RB * SRows<LX>::PITCH; }

    // h[n + LS r] = sum_q W_8^(-q r) P_q[n], r < 4: the first half of an inverse 8-point transform
    static BD_HD void quarter8(const float2 (&p)[NQ], float2 (&y)[4]) {
        const float2 e0 = pk_add(p[0], p[4 % NQ]), e1 = pk_sub(p[0], p[4 % NQ]), e2 = pk_add(p[2 % NQ], p[6 % NQ]), e3 = pk_sub(p[2 % NQ], p[6 % NQ]);
        const float2 o0 = pk_add(p[1 % NQ], p[5 % NQ]), o1 = pk_sub(p[1 % NQ], p[5 % NQ]), o2 = pk_add(p[3 % NQ], p[7 % NQ]), o3 = pk_sub(p[3 % NQ], p[7 % NQ]);
        const float2 ev[4] = {pk_add(e0, e2), pk_add_ib<+1>(e1, e3), pk_sub(e0, e2), pk_add_ib<-1>(e1, e3)};
        const float2 od[4] = {pk_add(o0, o2), pk_add_ib<+1>(o1, o3), pk_sub(o0, o2), pk_add_ib<-1>(o1, o3)};
        y[0] = pk_add(ev[0], od[0]);
        y[1] = pk_add(ev[1], pk_mul_w8<+1>(od[1], 1));
        y[2] = pk_add_ib<+1>(ev[2], od[2]);
        y[3] = pk_add(ev[3], pk_mul_w8<+1>(od[3], 3));
    }

    template <int PH>
    static BD_HD void phase(int tid, int bx, int by, const Args& a, float2* sm) {
        const int bpc = a.lsp / JB;                        // blocks per (c, z)
        const int cz = bx / bpc, j0 = (bx - cz * bpc) * JB;
        SRows<LX> s{sm};
        if constexpr (PH == 0) {
            // two neighbouring points of the partial planes per item: 16-byte loads, NQ x 2 of them in flight per thread
            constexpr int items = (LX / 2 + 1) * (JB / 2);
            auto emit = [&](int kp, int jj, const float4& xp, const float2 (&ak)[NQ], const float2 (&am)[NQ]) {
                if constexpr (NQ == 4) {
                    // h[n] = P0 + P1 + P2 + P3,  h[n + LS] = P0 + i P1 - P2 - i P3
                    const float2 Yk0 = pk_add(pk_add(ak[0], ak[2]), pk_add(ak[1], ak[3]));
                    const float2 Ym0 = pk_add(pk_add(am[0], am[2]), pk_add(am[1], am[3]));
                    const float2 Yk1 = pk_add_ib<+1>(pk_sub(ak[0], ak[2]), pk_sub(ak[1], ak[3]));
                    const float2 Ym1 = pk_add_ib<+1>(pk_sub(am[0], am[2]), pk_sub(am[1], am[3]));
                    xinv_pre(LX, kp, Yk0, Ym0, xp, sm + jj * SRows<LX>::PITCH);
                    xinv_pre(LX, kp, Yk1, Ym1, xp, sm + (JB + jj) * SRows<LX>::PITCH);
                } else if constexpr (NQ == 8) {
                    float2 Yk[4], Ym[4];
                    quarter8(ak, Yk);
                    quarter8(am, Ym);
                    BD_UNROLL
                    for (int r = 0; r < 4; ++r) xinv_pre(LX, kp, Yk[r], Ym[r], xp, sm + (r * JB + jj) * SRows<LX>::PITCH);
                } else if constexpr (NQ == 2) {
                    xinv_pre(LX, kp, pk_add(ak[0], ak[1]), pk_add(am[0], am[1]), xp, sm + jj * SRows<LX>::PITCH);
                } else {
                    xinv_pre(LX, kp, ak[0], am[0], xp, sm + jj * SRows<LX>::PITCH);
                }
            };
            for (int w = tid; w < items; w += NT) {
                const int kp = w >> (JBS - 1), jj = 2 * (w & (JB / 2 - 1)), km = LX - kp;
                const float4 xp = BD_LDG(&a.xpost[kp]);
                const float4* pk = reinterpret_cast<const float4*>(a.P + ((long)cz * a.nkx + kp) * a.lsp + j0 + jj);
                const float4* pm = reinterpret_cast<const float4*>(a.P + ((long)cz * a.nkx + km) * a.lsp + j0 + jj);
                float4 bk[NQ], bm[NQ];
                BD_UNROLL
                for (int q = 0; q < NQ; ++q) { bk[q] = BD_LDCG(pk + q * (a.qstride / 2)); bm[q] = BD_LDCG(pm + q * (a.qstride / 2)); }
                float2 ak[NQ], am[NQ];
                BD_UNROLL
                for (int q = 0; q < NQ; ++q) { ak[q] = bd_f2(bk[q].x, bk[q].y); am[q] = bd_f2(bm[q].x, bm[q].y); }
                emit(kp, jj, xp, ak, am);
                BD_UNROLL
                for (int q = 0; q < NQ; ++q) { ak[q] = bd_f2(bk[q].z, bk[q].w); am[q] = bd_f2(bm[q].z, bm[q].w); }
                emit(kp, jj + 1, xp, ak, am);
            }
        } else if constexpr (PH < NP) {
            x_rows_pass<LX, NP - PH, true, NT>(tid, RB, s, s, a.ptw);
        } else {
            // row = hi JB + lo  ->  y = j0 + lo + hi lsp   (hi > 0 only for NQ = 4 and 8, where lsp = ny / 2 and ny / 4)
            float* h0 = a.H + ((long)cz * a.ny + j0) * LX;
            if (a.en.M) {
                double acc = 0.0;
                GRowsOutMapE out{h0, LX, (long)a.lsp * LX, JBS, (long)((const char*)a.en.M - (const char*)a.H), &acc};
                x_rows_pass<LX, 0, true, NT>(tid, RB, s, out, a.ptw);
                energy_finish(acc, a.en);
            } else if (a.en.accumulate) {
                GRowsOutMapA out{h0, LX, (long)a.lsp * LX, JBS};
                x_rows_pass<LX, 0, true, NT>(tid, RB, s, out, a.ptw);
            } else {
                GRowsOutMap out{h0, LX, (long)a.lsp * LX, JBS};
                x_rows_pass<LX, 0, true, NT>(tid, RB, s, out, a.ptw);
            }
        }
    }
};

}  // namespace bd
