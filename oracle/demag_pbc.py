"""Demagnetizing field with periodic boundary conditions by the multiple-images method
(oracle, test infrastructure).

PAPER.md:L76 (section 3, after Eq. 4): "we extend this algorithm to use periodic boundary conditions
based on the multiple images method [51]" (Ref. [51]: Fangohr et al., "the
macrogeometry"; used by the paper's workloads at L89 and L209).  The magnetization of the mesh is
repeated at the lattice translations n o L, L = (nx hx, ny hy, nz hz), and the field in the mesh is
the sum of the fields of a FINITE block of copies:

    H_a(t) = - sum_{|nx'| <= Ix} sum_{|ny'| <= Iy} sum_{|nz'| <= Iz}  sum_{s in mesh}  sum_b
                 N_ab(r_t - r_s - n o L) M_b(s)                                                (1)

with `images = (Ix, Iy, Iz)` copies on each side along x, y, z (0: that direction is not periodic;
all 0 is PAPER.md:L323).  N is the plain Newell tensor of ``oracle.newell``.  The paper prints
neither the number of images nor a far-field correction: reading R15 of DESIGN.md takes the plain
finite sum (1), symmetric in +-n so that every component keeps its parity.

Because the copies carry the same M, (1) is a convolution of the mesh's own M with the image-summed
tensor

    N^img_ab(R) = sum_n N_ab(R - n o L),      R = r_t - r_s,  |R_x| < nx hx, ...              (2)

which ``image_tensor_table`` tabulates on the octant of non-negative R; ``demag_pbc_fft`` then runs
the zero-padded convolution of ``oracle.demag_fft`` with that table (a periodic direction could drop
its padding — an optimisation, not part of the definition).  ``demag_pbc_direct`` is (1) written out,
copy by copy, from the plain tensor over the whole macro-geometry; tests/test_oracle_pbc.py checks the
two against each other and against what the mathematics fixes (the non-periodic double sum over the
tiled macro-geometry, the trace of (2), the infinite-film limit).

Arrays as in ``oracle.demag_direct``: M, H are [3][nz][ny][nx], fp64 arithmetic.
"""
import itertools

import numpy as np

from .demag_direct import _components_needed
from .demag_fft import demag_fft, kernel_spectrum
from .newell import PARITY, SYM_INDEX, newell_tensor_octant


def _check_images(images):
    ix, iy, iz = (int(v) for v in images)
    if min(ix, iy, iz) < 0:
        raise ValueError("images must be >= 0")
    return ix, iy, iz


def macro_table(shape, h, images):
    """Plain Newell octant table [6][(Iz+1) nz][(Iy+1) ny][(Ix+1) nx]: every |displacement| that
    occurs between a cell of the mesh and a cell of any of its copies."""
    nz, ny, nx = shape
    ix, iy, iz = _check_images(images)
    comps = (0, 1, 2, 3, 4, 5) if (nz > 1 or iz > 0) else _components_needed(nz)
    return newell_tensor_octant((ix + 1) * nx, (iy + 1) * ny, (iz + 1) * nz, h[0], h[1], h[2], components=comps)


def _signed_lookup(table_c, parity, dk, dj, di):
    """table_c at the signed displacements dk x dj x di (1-D integer arrays), by parity."""
    W = table_c[np.ix_(np.abs(dk), np.abs(dj), np.abs(di))]
    px, py, pz = parity
    if px < 0:
        W = W * np.sign(di)[None, None, :]
    if py < 0:
        W = W * np.sign(dj)[None, :, None]
    if pz < 0:
        W = W * np.sign(dk)[:, None, None]
    return W


def demag_pbc_direct(M, h, images, table=None):
    """Eq. (1) as it stands: for every target cell, copy by copy, the plain sum over the source cells
    of that copy.  O(N^2 (2Ix+1)(2Iy+1)(2Iz+1)): small meshes only."""
    M = np.asarray(M, np.float64)
    _, nz, ny, nx = M.shape
    ix, iy, iz = _check_images(images)
    if table is None:
        table = macro_table((nz, ny, nx), h, images)
    ks, js, is_ = np.arange(nz), np.arange(ny), np.arange(nx)
    H = np.zeros((3, nz, ny, nx), np.float64)
    for kt, jt, it in itertools.product(range(nz), range(ny), range(nx)):
        acc = np.zeros(3, np.float64)
        for c_, b_, a_ in itertools.product(range(-iz, iz + 1), range(-iy, iy + 1), range(-ix, ix + 1)):
            # target - (source + n o L), in cells
            dk, dj, di = kt - ks - c_ * nz, jt - js - b_ * ny, it - is_ - a_ * nx
            Nc = [_signed_lookup(table[c], PARITY[c], dk, dj, di) for c in range(6)]
            for a in range(3):
                for b in range(3):
                    acc[a] += np.sum(Nc[SYM_INDEX[a, b]] * M[b])
        H[:, kt, jt, it] = -acc
    return H


def image_tensor_table(shape, h, images, table=None):
    """Eq. (2) on the octant 0 <= R < mesh: fp64 array [6][nz][ny][nx]."""
    nz, ny, nx = shape
    ix, iy, iz = _check_images(images)
    if table is None:
        table = macro_table(shape, h, images)
    ks, js, is_ = np.arange(nz), np.arange(ny), np.arange(nx)
    out = np.zeros((6, nz, ny, nx), np.float64)
    for c_, b_, a_ in itertools.product(range(-iz, iz + 1), range(-iy, iy + 1), range(-ix, ix + 1)):
        dk, dj, di = ks - c_ * nz, js - b_ * ny, is_ - a_ * nx
        for c in range(6):
            out[c] += _signed_lookup(table[c], PARITY[c], dk, dj, di)
    # an odd component of the symmetric sum vanishes on its nodal plane: replace the rounding residue by 0
    for c in range(6):
        px, py, pz = PARITY[c]
        if px < 0:
            out[c][:, :, 0] = 0.0
        if py < 0:
            out[c][:, 0, :] = 0.0
        if pz < 0:
            out[c][0, :, :] = 0.0
    if nz == 1:
        out[4] = 0.0        # Nxz, Nyz: odd in z, every displacement of a single layer and its copies pairs up
        out[5] = 0.0
    return out


def pbc_kernel_spectrum(shape, h, images):
    """Spectrum of the wrapped, zero-padded image-summed tensor (steps 1-2 of oracle.demag_fft)."""
    return kernel_spectrum(shape, h, table=image_tensor_table(shape, h, images))


def demag_pbc_fft(M, h, images, Khat=None):
    """Eq. (1) through the convolution theorem: oracle.demag_fft with the kernel of Eq. (2)."""
    M = np.asarray(M, np.float64)
    if Khat is None:
        Khat = pbc_kernel_spectrum(M.shape[1:], h, images)
    return demag_fft(M, h, Khat=Khat)
