"""Pins for oracle/newell.py against things other than itself (CPU only).

PAPER.md:L324 only cites the tensor formulas (Ref. [50]); the pins below are
what the mathematics fixes.  Pin numbers refer to SURVEY.md §8(c) / DESIGN.md.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import newell

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "newell_self_terms.txt")
CELLS = [(5.0, 5.0, 3.0), (2.0, 2.0, 1.0), (4.0, 4.0, 4.0), (3.0, 7.0, 2.0), (1e-9, 2.5e-9, 4e-9)]


def aharoni_Dz(A, B, C):
    """Demagnetizing factor along z of a uniformly magnetized A x B x C prism.

    Aharoni, J. Appl. Phys. 83, 3432 (1998), Eq. (1), retyped with a, b, c the
    half-sides.  An independent closed form: it does not involve Newell's f, g.
    """
    a, b, c = A / 2, B / 2, C / 2
    r = np.sqrt(a * a + b * b + c * c)
    rab, rbc, rac = np.hypot(a, b), np.hypot(b, c), np.hypot(a, c)
    t = (b * b - c * c) / (2 * b * c) * np.log((r - a) / (r + a))
    t += (a * a - c * c) / (2 * a * c) * np.log((r - b) / (r + b))
    t += b / (2 * c) * np.log((rab + a) / (rab - a))
    t += a / (2 * c) * np.log((rab + b) / (rab - b))
    t += c / (2 * a) * np.log((rbc - b) / (rbc + b))
    t += c / (2 * b) * np.log((rac - a) / (rac + a))
    t += 2 * np.arctan(a * b / (c * r))
    t += (a ** 3 + b ** 3 - 2 * c ** 3) / (3 * a * b * c)
    t += (a * a + b * b - 2 * c * c) / (3 * a * b * c) * r
    t += c / (a * b) * (rac + rbc)
    t -= (rab ** 3 + rbc ** 3 + rac ** 3) / (3 * a * b * c)
    return t / np.pi


def aharoni_factors(L):
    """(Nxx, Nyy, Nzz) of a prism with sides L = (Lx, Ly, Lz) by cyclic permutation."""
    Lx, Ly, Lz = L
    return aharoni_Dz(Ly, Lz, Lx), aharoni_Dz(Lz, Lx, Ly), aharoni_Dz(Lx, Ly, Lz)


@pytest.mark.parametrize("h", CELLS)
def test_self_term_equals_aharoni_closed_form(h):
    T = newell.newell_tensor_octant(1, 1, 1, *h)[:, 0, 0, 0]
    np.testing.assert_allclose(T[:3], aharoni_factors(h), rtol=0, atol=2e-13)
    np.testing.assert_allclose(T[3:], 0, atol=1e-15)


def test_self_terms_match_survey_golden_values():
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    assert len(rows) == 6
    for Lx, Ly, Lz, nxx, nzz, _tag in rows:
        L = (float(Lx), float(Ly), float(Lz))
        T = newell.newell_tensor_octant(1, 1, 1, *L)[:, 0, 0, 0]
        assert abs(T[0] - float(nxx)) < 1e-11 and abs(T[1] - float(nxx)) < 1e-11
        assert abs(T[2] - float(nzz)) < 1e-11
        # and the independent closed form agrees with the stored digits too
        assert abs(aharoni_factors(L)[2] - float(nzz)) < 1e-11


@pytest.mark.parametrize("h", CELLS[:4])
def test_P1_trace_is_one_at_origin_and_zero_elsewhere(h):
    T = newell.newell_tensor_octant(12, 9, 5, *h)
    tr = T[0] + T[1] + T[2]
    assert abs(tr[0, 0, 0] - 1) < 1e-13
    tr[0, 0, 0] = 0
    assert np.abs(tr).max() < 1e-13


def test_P1_trace_far(capsys=None):
    # far displacements (hundreds of cells): trace still 0 to 1e-10 in extended precision
    for X, Y, Z in [(300, 200, 0), (1000, 3, 0), (700, 700, 20)]:
        tr = sum(newell.newell_point(c, 2.0 * X, 2.0 * Y, 1.0 * Z, 2.0, 2.0, 1.0) for c in range(3))
        assert abs(tr) < 1e-10


def test_P2_cube_self_term_is_one_third():
    T = newell.newell_tensor_octant(1, 1, 1, 2.0, 2.0, 2.0)[:, 0, 0, 0]
    np.testing.assert_allclose(T[:3], 1 / 3, atol=1e-14)
    np.testing.assert_allclose(T[3:], 0, atol=1e-15)


def test_P4_parity_of_every_component():
    h = (5.0, 4.0, 3.0)
    T = newell.newell_tensor_octant(4, 4, 4, *h)
    for c in range(6):
        for (i, j, k) in [(1, 2, 3), (3, 1, 2), (2, 3, 1)]:
            for sx, sy, sz in itertools.product((1, -1), repeat=3):
                v = newell.newell_point(c, sx * i * h[0], sy * j * h[1], sz * k * h[2], *h)
                sign = ((newell.PARITY[c][0] if sx < 0 else 1) * (newell.PARITY[c][1] if sy < 0 else 1)
                        * (newell.PARITY[c][2] if sz < 0 else 1))
                assert abs(v - sign * T[c, k, j, i]) < 1e-15
    # odd components vanish on their nodal planes
    assert np.abs(T[3][:, 0, :]).max() == 0 and np.abs(T[3][:, :, 0]).max() == 0
    assert np.abs(T[4][0]).max() == 0 and np.abs(T[4][:, :, 0]).max() == 0
    assert np.abs(T[5][0]).max() == 0 and np.abs(T[5][:, 0, :]).max() == 0


def test_P5_components_are_axis_permutations_of_each_other():
    h = (5.0, 4.0, 3.0)
    X, Y, Z = 2 * h[0], 3 * h[1], 1 * h[2]
    p = newell.newell_point
    assert abs(p(1, X, Y, Z, *h) - p(0, Y, X, Z, h[1], h[0], h[2])) < 1e-16      # Nyy
    assert abs(p(2, X, Y, Z, *h) - p(0, Z, Y, X, h[2], h[1], h[0])) < 1e-16      # Nzz
    assert abs(p(4, X, Y, Z, *h) - p(3, X, Z, Y, h[0], h[2], h[1])) < 1e-16      # Nxz
    assert abs(p(5, X, Y, Z, *h) - p(3, Y, Z, X, h[1], h[2], h[0])) < 1e-16      # Nyz


def test_scale_invariance_nm_vs_metres():
    a = newell.newell_tensor_octant(6, 5, 4, 5.0, 4.0, 3.0)
    b = newell.newell_tensor_octant(6, 5, 4, 5e-9, 4e-9, 3e-9)
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-15)


def dipole_tensor(R):
    """Point-dipole limit D_ab = (1/4pi)(delta_ab/R^3 - 3 R_a R_b / R^5), as [3][3]."""
    R = np.asarray(R, float)
    r = np.linalg.norm(R)
    return (np.eye(3) / r ** 3 - 3 * np.outer(R, R) / r ** 5) / (4 * np.pi)


def test_P6_point_dipole_limit_with_sign():
    h = (5.0, 5.0, 3.0)
    V = h[0] * h[1] * h[2]
    cells = (40, 25, 12)
    R = [cells[0] * h[0], cells[1] * h[1], cells[2] * h[2]]
    D = V * dipole_tensor(R)
    for c in range(6):
        a, b = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)][c]
        v = newell.newell_point(c, *R, *h)
        assert abs(v - D[a, b]) < 5e-4 * abs(D[a, b])
    # cubic cells converge as (h/R)^4
    hc = (2.0, 2.0, 2.0)
    Rc = [40.0, 26.0, 14.0]
    Dc = 8.0 * dipole_tensor(Rc)
    for c in range(6):
        a, b = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)][c]
        assert abs(newell.newell_point(c, *Rc, *hc) - Dc[a, b]) < 2e-5 * np.abs(Dc).max()


@pytest.mark.parametrize("disp", [(2, 1, 1), (1, 2, 0), (0, 0, 2), (3, 0, 1)])
def test_brute_force_quadrature_of_the_dipolar_kernel(disp):
    """N_ab(R) = (1/V) int_cell d3r int_cell' d3r' D_ab(R + r - r')  by 6-D Gauss-Legendre.

    First-principles definition of the cell-averaged tensor (two uniformly
    magnetized cuboids, PAPER.md:L323 via Ref. [50]); no f, g involved.  The
    cells are separated by at least one cell so the integrand is analytic.
    """
    h = np.array([5.0, 4.0, 3.0])
    R = np.array(disp) * h
    n = 8
    t, w = np.polynomial.legendre.leggauss(n)
    t, w = t / 2, w / 2                       # unit interval [-1/2, 1/2], weights sum to 1
    # separation u = r - r' per axis: all n*n pairs, weight w_i w_j
    du = (t[:, None] - t[None, :]).ravel()
    wu = (w[:, None] * w[None, :]).ravel()
    ux = R[0] + h[0] * du[:, None, None]
    uy = R[1] + h[1] * du[None, :, None]
    uz = R[2] + h[2] * du[None, None, :]
    W = wu[:, None, None] * wu[None, :, None] * wu[None, None, :]
    r2 = ux * ux + uy * uy + uz * uz
    r5 = r2 ** 2.5
    V = h.prod()
    comps = {
        0: (r2 - 3 * ux * ux), 1: (r2 - 3 * uy * uy), 2: (r2 - 3 * uz * uz),
        3: (-3 * ux * uy), 4: (-3 * ux * uz), 5: (-3 * uy * uz),
    }
    for c, num in comps.items():
        brute = V * np.sum(W * num / r5) / (4 * np.pi)
        got = newell.newell_point(c, *R, *h)
        assert abs(got - brute) < 2e-9, (c, got, brute)


def test_golden_file_is_what_its_generator_writes():
    """tests/golden/make_self_terms.py (Aharoni's closed form, 50-digit mpmath, no oracle, no product code)."""
    import subprocess
    import sys
    pytest.importorskip("mpmath")
    gen = os.path.join(os.path.dirname(GOLDEN), "make_self_terms.py")
    assert subprocess.run([sys.executable, gen, "--check"], capture_output=True).returncode == 0
