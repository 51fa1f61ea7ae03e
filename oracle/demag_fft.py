"""Zero-padded FFT convolution H = -N * M in fp64 (oracle, test infrastructure).

Follows PAPER.md:L275 step by step, with no pruning, fusion or symmetry trick:
"a (2)3D fast Fourier transform (FFT) algorithm is used on the input
magnetization; this is then multiplied with the demagnetizing kernel in the
transform space, and an inverse (2)3D FFT algorithm is used to obtain the
output demagnetizing field", and PAPER.md:L283: "the circular convolution
theorem requires doubling the input data size by zero padding when not using
periodic boundary conditions".

  1. Kpad_ab[k mod Pz][j mod Py][i mod Px] = N_ab(i hx, j hy, k hz) for
     |i| < nx, |j| < ny, |k| < nz;  the slots at displacement exactly +-n are 0
     (reading R5);  P = 2n per padded dimension, Pz = 1 when nz = 1 (R6).
  2. Khat_ab = rfftn(Kpad_ab)                (library FFT: scipy pocketfft, fp64)
  3. Mpad = M in the corner [0,nz) x [0,ny) x [0,nx), zeros elsewhere;  Mhat = rfftn(Mpad)
  4. Hhat_a = - sum_b Khat_ab Mhat_b
  5. H = irfftn(Hhat)[:nz, :ny, :nx]

The plain definition this reaches (up to rounding) is ``oracle.demag_direct``;
``tests/test_oracle_demag.py`` checks the two against each other.
"""
import os

import numpy as np
import scipy.fft

from .newell import PARITY, SYM_INDEX
from .demag_direct import tensor_table

_WORKERS = os.cpu_count() or 1


def padded_shape(shape):
    nz, ny, nx = shape
    return (1 if nz == 1 else 2 * nz, 2 * ny, 2 * nx)


def _wrap_kernel(oct_c, parity, pshape):
    """Step 1 for one component: octant table -> wrapped padded array."""
    nz, ny, nx = oct_c.shape
    Pz, Py, Px = pshape
    K = np.zeros(pshape, np.float64)
    px, py, pz = parity
    for sz in ((+1,) if nz == 1 else (+1, -1)):
        for sy in (+1, -1):
            for sx in (+1, -1):
                # displacement (sx*i, sy*j, sz*k); i = 0 belongs to the + branch only
                i0 = 0 if sx > 0 else 1
                j0 = 0 if sy > 0 else 1
                k0 = 0 if sz > 0 else 1
                if i0 >= nx or j0 >= ny or k0 >= nz:
                    continue
                sign = (px if sx < 0 else 1) * (py if sy < 0 else 1) * (pz if sz < 0 else 1)
                src = oct_c[k0:, j0:, i0:]
                ii = (sx * np.arange(i0, nx)) % Px
                jj = (sy * np.arange(j0, ny)) % Py
                kk = (sz * np.arange(k0, nz)) % Pz
                K[np.ix_(kk, jj, ii)] = sign * src
    return K


def kernel_spectrum(shape, h, table=None):
    """Steps 1-2: list of six complex128 arrays Khat_c[Pz][Py][Px/2+1] (None if unused)."""
    if table is None:
        table = tensor_table(shape, h)
    pshape = padded_shape(shape)
    comps = (0, 1, 2, 3) if shape[0] == 1 else range(6)
    Khat = [None] * 6
    for c in comps:
        Khat[c] = scipy.fft.rfftn(_wrap_kernel(table[c], PARITY[c], pshape), workers=_WORKERS)
    return Khat


def demag_fft(M, h, Khat=None, table=None):
    """Steps 3-5: H [3][nz][ny][nx] in fp64 from M [3][nz][ny][nx]."""
    M = np.asarray(M, np.float64)
    _, nz, ny, nx = M.shape
    shape = (nz, ny, nx)
    pshape = padded_shape(shape)
    if Khat is None:
        Khat = kernel_spectrum(shape, h, table=table)
    Mhat = []
    for b in range(3):
        Mpad = np.zeros(pshape, np.float64)
        Mpad[:nz, :ny, :nx] = M[b]
        Mhat.append(scipy.fft.rfftn(Mpad, workers=_WORKERS))
    H = np.empty((3, nz, ny, nx), np.float64)
    for a in range(3):
        Hhat = np.zeros_like(Mhat[0])
        for b in range(3):
            Kab = Khat[SYM_INDEX[a, b]]
            if Kab is not None:
                Hhat -= Kab * Mhat[b]
        H[a] = scipy.fft.irfftn(Hhat, s=pshape, workers=_WORKERS)[:nz, :ny, :nx]
    return H
