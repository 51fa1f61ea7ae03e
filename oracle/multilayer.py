"""Multi-layered demagnetizing field (oracle, test infrastructure).

PAPER.md:L71-L76, Eq. (4): for a collection of meshes V_k (k = 1..n)

    H(r'_kl) = - sum_{i = 1..n} sum_{r_ij in V_i}  N(r'_kl - r_ij, h_k, h_i) M(r_ij),      r'_kl in V_k,

"N are inter and intra-mesh demagnetizing tensors generalized from the Newell et al. formulas [50] in Ref. [23]", and
"with multiple input meshes ... summation of inter-mesh contributions moved to the transform space".

Ref. [23] is not in the container.  What is restated here is the case its generalization reduces to when the meshes
are LAYERS of one film stack (the paper's use: the CoFe/Ru multilayer of L76, the Co/Pt/SiO2 stack of L209) —
DESIGN.md reading R17:

  * every layer k is one cell thick, nx x ny cells of the SAME in-plane size (hx, hy) on the same in-plane grid,
    with its OWN thickness t_k and centre height z_k (arbitrary spacers, no common z grid);
  * N(R, h_k, h_i) is the tensor between a source cuboid (hx, hy, t_i) and a target cuboid (hx, hy, t_k) whose centres
    are R apart, averaged over the TARGET cell.  For equal in-plane sizes only the z part of Newell's 27-point
    stencil changes.  Newell's per-direction weights (-1, 2, -1) at offsets (-h, 0, +h) are the second difference
    that  int_0^h dz int_0^h dz' phi''(Z + z - z')  leaves; with unequal heights the same double integral leaves

        - phi(Z + (t_k+t_i)/2) + phi(Z + (t_k-t_i)/2) + phi(Z - (t_k-t_i)/2) - phi(Z - (t_k+t_i)/2)

    (Z the centre-to-centre height difference), normalised by the TARGET volume hx hy t_k.  t_k = t_i = hz gives
    back oracle.newell exactly.

Functions: ``pair_tensor_point`` (one displacement), ``pair_tensor_table`` (in-plane octant for one layer pair),
``multilayer_direct`` (Eq. 4 written out), ``multilayer_fft`` (Eq. 4 through the convolution theorem, in-plane
zero padding as in oracle.demag_fft, inter-layer terms summed in the transform space).  Pinned in
tests/test_oracle_multilayer.py: brute-force 6-D quadrature of the dipolar kernel between unequal cuboids,
additivity over a split source / target cell, reciprocity, the single-mesh oracle on a stack that does sit on a
common z grid, direct sum vs FFT route.

Arrays: M, H are [3][n][ny][nx] (the layer index where a 3-D mesh has z); fp64; tensor in x87 extended precision.
"""
import itertools

import numpy as np
import scipy.fft

from .demag_fft import _wrap_kernel
from .newell import LD, SYM_INDEX, _GENERATORS

# parity of each component under x -> -x and y -> -y at FIXED height difference Z (z is not mirrored here)
PARITY_XY = np.array([[+1, +1], [+1, +1], [+1, +1], [-1, -1], [-1, +1], [+1, -1]])


def _z_offsets(tk, ti):
    """Offsets and weights of the z part of the stencil (module docstring)."""
    tk, ti = LD(tk), LD(ti)
    return ((tk + ti) / 2, (tk - ti) / 2, -(tk - ti) / 2, -(tk + ti) / 2), (-1, 1, 1, -1)


def pair_tensor_table(nx, ny, hx, hy, tk, ti, Z, components=range(6)):
    """N_c((i hx, j hy, Z), target thickness tk, source thickness ti) for 0 <= i < nx, 0 <= j < ny: fp64 [6][ny][nx]."""
    hx, hy = LD(hx), LD(hy)
    x = (np.arange(-1, nx + 1, dtype=LD) * hx)[None, :]
    y = (np.arange(-1, ny + 1, dtype=LD) * hy)[:, None]
    zo, zw = _z_offsets(tk, ti)
    out = np.zeros((6, ny, nx), np.float64)
    for c in components:
        acc = np.zeros((ny, nx), LD)
        for dz, wz in zip(zo, zw):
            F = np.broadcast_to(_GENERATORS[c](x, y, LD(Z) + dz), (ny + 2, nx + 2))
            for a, b in itertools.product((-1, 0, 1), repeat=2):
                w = (2 if a == 0 else -1) * (2 if b == 0 else -1) * wz
                acc += LD(w) * F[1 + b:1 + b + ny, 1 + a:1 + a + nx]
        out[c] = (acc / (4 * LD(np.pi) * hx * hy * LD(tk))).astype(np.float64)
        px, py = PARITY_XY[c]
        if px < 0:
            out[c][:, 0] = 0.0          # odd in x: exact zero on the nodal line
        if py < 0:
            out[c][0, :] = 0.0
    return out


def pair_tensor_point(c, X, Y, Z, hx, hy, tk, ti):
    """One entry at an arbitrary (signed) in-plane displacement."""
    hx, hy = LD(hx), LD(hy)
    x = (LD(X) + np.array([-1, 0, 1], LD) * hx)[None, :]
    y = (LD(Y) + np.array([-1, 0, 1], LD) * hy)[:, None]
    zo, zw = _z_offsets(tk, ti)
    acc = LD(0)
    for dz, wz in zip(zo, zw):
        F = np.broadcast_to(_GENERATORS[c](x, y, LD(Z) + dz), (3, 3))
        for a, b in itertools.product((-1, 0, 1), repeat=2):
            acc += LD((2 if a == 0 else -1) * (2 if b == 0 else -1) * wz) * F[1 + b, 1 + a]
    return float(acc / (4 * LD(np.pi) * hx * hy * LD(tk)))


def _signed(table_c, parity_xy, dj, di):
    W = table_c[np.ix_(np.abs(dj), np.abs(di))]
    if parity_xy[0] < 0:
        W = W * np.sign(di)[None, :]
    if parity_xy[1] < 0:
        W = W * np.sign(dj)[:, None]
    return W


def multilayer_direct(M, hx, hy, t, z):
    """Eq. (4) as it stands: for every target layer k and cell, the sum over every source layer i and cell.
    t[k], z[k]: thickness and centre height of layer k.  O(n^2 N^2): small stacks only."""
    M = np.asarray(M, np.float64)
    _, n, ny, nx = M.shape
    js, is_ = np.arange(ny), np.arange(nx)
    H = np.zeros_like(M)
    for k in range(n):
        for i in range(n):
            tab = pair_tensor_table(nx, ny, hx, hy, t[k], t[i], z[k] - z[i])
            for jt, it in itertools.product(range(ny), range(nx)):
                dj, di = jt - js, it - is_                       # target - source
                Nc = [_signed(tab[c], PARITY_XY[c], dj, di) for c in range(6)]
                for a in range(3):
                    for b in range(3):
                        H[a, k, jt, it] -= np.sum(Nc[SYM_INDEX[a, b]] * M[b, i])
    return H


def pair_spectra(nx, ny, hx, hy, t, z):
    """Khat[k][i][c]: rfft2 of the wrapped, zero-padded in-plane kernel of every ordered layer pair (complex128)."""
    n = len(t)
    workers = scipy.fft.get_workers()
    out = [[None] * n for _ in range(n)]
    for k in range(n):
        for i in range(n):
            tab = pair_tensor_table(nx, ny, hx, hy, t[k], t[i], z[k] - z[i])
            out[k][i] = [scipy.fft.rfftn(_wrap_kernel(tab[c][None], (PARITY_XY[c][0], PARITY_XY[c][1], +1),
                                                      (1, 2 * ny, 2 * nx))[0], workers=workers) for c in range(6)]
    return out


def multilayer_fft(M, hx, hy, t, z, Khat=None):
    """Eq. (4) by the convolution theorem: per layer a zero-padded 2-D transform, the inter-layer contributions
    summed in the transform space, per layer an inverse transform."""
    M = np.asarray(M, np.float64)
    _, n, ny, nx = M.shape
    if Khat is None:
        Khat = pair_spectra(nx, ny, hx, hy, t, z)
    Mhat = np.empty((3, n, 2 * ny, nx + 1), np.complex128)
    for b in range(3):
        for i in range(n):
            pad = np.zeros((2 * ny, 2 * nx))
            pad[:ny, :nx] = M[b, i]
            Mhat[b, i] = scipy.fft.rfftn(pad)
    H = np.empty_like(M)
    for a in range(3):
        for k in range(n):
            Hhat = np.zeros((2 * ny, nx + 1), np.complex128)
            for i in range(n):
                for b in range(3):
                    Hhat -= Khat[k][i][SYM_INDEX[a, b]] * Mhat[b, i]
            H[a, k] = scipy.fft.irfftn(Hhat, s=(2 * ny, 2 * nx))[:ny, :nx]
    return H


def multilayer_energy(M, H, hx, hy, t):
    """E = -(mu0/2) sum_k hx hy t_k sum_cells M_k . H_k  (oracle.energy with per-layer cell volumes)."""
    M = np.asarray(M, np.float64)
    H = np.asarray(H, np.float64)
    mu0 = 4e-7 * np.pi
    return -0.5 * mu0 * sum(float(hx) * float(hy) * float(t[k]) * float(np.sum(M[:, k] * H[:, k])) for k in range(M.shape[1]))
