"""Newell demagnetizing tensor for two equal cuboid cells (oracle, test infrastructure).

PAPER.md:L323-L324 (Table 1): "H(r0) = - sum_r N(r - r0) M(r);  N computed
using formulas in Ref. [50]" (Newell, Williams, Dunlop, J. Geophys. Res. 98,
9551 (1993)).  The paper does not print the formulas; they are
restated here in the notation of SURVEY.md Appendix A.  With
R = sqrt(x^2 + y^2 + z^2):

    f(x,y,z) =  (y/2)(z^2 - x^2) asinh( y / sqrt(x^2 + z^2) )
              + (z/2)(y^2 - x^2) asinh( z / sqrt(x^2 + y^2) )
              -  x y z           atan ( y z / (x R) )
              + (1/6)(2x^2 - y^2 - z^2) R

    g(x,y,z) =  x y z            asinh( z / sqrt(x^2 + y^2) )
              + (y/6)(3z^2 - y^2) asinh( x / sqrt(y^2 + z^2) )
              + (x/6)(3z^2 - x^2) asinh( y / sqrt(x^2 + z^2) )
              - (z^3/6)          atan ( x y / (z R) )
              - (z y^2/2)        atan ( x z / (y R) )
              - (z x^2/2)        atan ( y z / (x R) )
              -  x y R / 3

A term whose asinh/atan argument has a zero denominator is 0: its prefactor
vanishes faster (reading R4).

27-point stencil, weight by the number m of non-zero offsets,
w(0) = 8, w(1) = -4, w(2) = 2, w(3) = -1:

    S[F](X,Y,Z) = 1/(4 pi hx hy hz) * sum_{a,b,c in {-1,0,1}} w(|a|+|b|+|c|)
                                       F(X + a hx, Y + b hy, Z + c hz)

    Nxx = S[(x,y,z) -> f(x,y,z)]   Nyy = S[(x,y,z) -> f(y,x,z)]   Nzz = S[(x,y,z) -> f(z,y,x)]
    Nxy = S[(x,y,z) -> g(x,y,z)]   Nxz = S[(x,y,z) -> g(x,z,y)]   Nyz = S[(x,y,z) -> g(y,z,x)]

Precision (reading R3): f and g are sums of terms of size ~R^3 whose
27-point combination is ~R^-3, so fp64 loses ~6 log10(R/h) digits.  Everything
up to and including the stencil sum is therefore evaluated in numpy.longdouble
(x87 80-bit, eps 1.08e-19) and rounded to fp64 once at the end.

Component order everywhere in the oracle: (xx, yy, zz, xy, xz, yz) = 0..5.
"""
import itertools

import numpy as np

LD = np.longdouble
COMPONENTS = ("xx", "yy", "zz", "xy", "xz", "yz")

if not np.finfo(LD).eps < 2e-19:  # pragma: no cover - x86-64 always passes
    raise RuntimeError(
        "oracle/newell.py needs an extended-precision numpy.longdouble "
        "(x87 80-bit); this platform's longdouble is plain double")


def _asinh_ratio(num, den2):
    """asinh(num / sqrt(den2)), defined as 0 where den2 == 0 (reading R4)."""
    ok = den2 > 0
    safe = np.where(ok, den2, LD(1))
    return np.where(ok, np.arcsinh(num / np.sqrt(safe)), LD(0))


def _atan_ratio(num, den):
    """atan(num / den), defined as 0 where den == 0 (reading R4)."""
    ok = den != 0
    safe = np.where(ok, den, LD(1))
    return np.where(ok, np.arctan(num / safe), LD(0))


def newell_f(x, y, z):
    """Newell's f (docstring of this module), elementwise, in longdouble."""
    x = np.asarray(x, LD)
    y = np.asarray(y, LD)
    z = np.asarray(z, LD)
    x2, y2, z2 = x * x, y * y, z * z
    R = np.sqrt(x2 + y2 + z2)
    out = (y / 2) * (z2 - x2) * _asinh_ratio(y, x2 + z2)
    out = out + (z / 2) * (y2 - x2) * _asinh_ratio(z, x2 + y2)
    out = out - x * y * z * _atan_ratio(y * z, x * R)
    out = out + (2 * x2 - y2 - z2) * R / 6
    return out


def newell_g(x, y, z):
    """Newell's g (docstring of this module), elementwise, in longdouble."""
    x = np.asarray(x, LD)
    y = np.asarray(y, LD)
    z = np.asarray(z, LD)
    x2, y2, z2 = x * x, y * y, z * z
    R = np.sqrt(x2 + y2 + z2)
    out = x * y * z * _asinh_ratio(z, x2 + y2)
    out = out + (y / 6) * (3 * z2 - y2) * _asinh_ratio(x, y2 + z2)
    out = out + (x / 6) * (3 * z2 - x2) * _asinh_ratio(y, x2 + z2)
    out = out - (z2 * z / 6) * _atan_ratio(x * y, z * R)
    out = out - (z * y2 / 2) * _atan_ratio(x * z, y * R)
    out = out - (z * x2 / 2) * _atan_ratio(y * z, x * R)
    out = out - x * y * R / 3
    return out


# F(x,y,z) of each component, in COMPONENTS order (module docstring).
_GENERATORS = (
    lambda x, y, z: newell_f(x, y, z),
    lambda x, y, z: newell_f(y, x, z),
    lambda x, y, z: newell_f(z, y, x),
    lambda x, y, z: newell_g(x, y, z),
    lambda x, y, z: newell_g(x, z, y),
    lambda x, y, z: newell_g(y, z, x),
)

_WEIGHT = {0: 8, 1: -4, 2: 2, 3: -1}


def _stencil(F, hx, hy, hz):
    """27-point stencil over an array F[k+1+c][j+1+b][i+1+a] (one-cell halo)."""
    nz, ny, nx = (s - 2 for s in F.shape)
    acc = np.zeros((nz, ny, nx), LD)
    for a, b, c in itertools.product((-1, 0, 1), repeat=3):
        w = _WEIGHT[abs(a) + abs(b) + abs(c)]
        acc += LD(w) * F[1 + c:1 + c + nz, 1 + b:1 + b + ny, 1 + a:1 + a + nx]
    return acc / (4 * LD(np.pi) * LD(hx) * LD(hy) * LD(hz))


def newell_tensor_octant(nx, ny, nz, hx, hy, hz, components=range(6)):
    """N_ab at displacements (i hx, j hy, k hz), 0 <= i < nx, 0 <= j < ny, 0 <= k < nz.

    Returns fp64 array [6][nz][ny][nx] (rows of components not requested are 0).
    Negative displacements follow from parity (``parity_signs``).
    """
    hx, hy, hz = LD(hx), LD(hy), LD(hz)
    x = (np.arange(-1, nx + 1, dtype=LD) * hx)[None, None, :]
    y = (np.arange(-1, ny + 1, dtype=LD) * hy)[None, :, None]
    z = (np.arange(-1, nz + 1, dtype=LD) * hz)[:, None, None]
    out = np.zeros((6, nz, ny, nx), np.float64)
    for c in components:
        F = np.broadcast_to(_GENERATORS[c](x, y, z), (nz + 2, ny + 2, nx + 2))
        out[c] = _stencil(F, hx, hy, hz).astype(np.float64)
        # an odd function vanishes on its nodal plane (pin P4); the stencil sum
        # leaves ~1e-19 of rounding there, which is replaced by the exact 0.
        px, py, pz = PARITY[c]
        if px < 0:
            out[c][:, :, 0] = 0.0
        if py < 0:
            out[c][:, 0, :] = 0.0
        if pz < 0:
            out[c][0, :, :] = 0.0
    return out


def newell_point(c, X, Y, Z, hx, hy, hz):
    """N_ab of component index c at one displacement (X, Y, Z) (any sign), fp64."""
    hx, hy, hz = LD(hx), LD(hy), LD(hz)
    x = (LD(X) + np.array([-1, 0, 1], LD) * hx)[None, None, :]
    y = (LD(Y) + np.array([-1, 0, 1], LD) * hy)[None, :, None]
    z = (LD(Z) + np.array([-1, 0, 1], LD) * hz)[:, None, None]
    F = np.broadcast_to(_GENERATORS[c](x, y, z), (3, 3, 3))
    return float(_stencil(F, hx, hy, hz)[0, 0, 0])


# Parity of each component under x -> -x, y -> -y, z -> -z (pin P4): the
# diagonal components are even in every coordinate, N_ab (a != b) is odd in a
# and in b and even in the third coordinate.
PARITY = np.array([
    # x   y   z
    [+1, +1, +1],   # xx
    [+1, +1, +1],   # yy
    [+1, +1, +1],   # zz
    [-1, -1, +1],   # xy
    [-1, +1, -1],   # xz
    [+1, -1, -1],   # yz
])

# (row, col) -> component index of the symmetric 3x3 tensor.
SYM_INDEX = np.array([[0, 3, 4],
                      [3, 1, 5],
                      [4, 5, 2]])
