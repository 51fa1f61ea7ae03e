"""Pins of oracle/multilayer.py (multi-layered convolution, Eq. 4; reading R17), none of
which re-calls the function under test:

  * the tensor between UNEQUAL cuboids against its first-principles definition, a 6-D Gauss-Legendre quadrature of
    the dipolar kernel over the two cells (no f, g, no stencil);
  * additivity: a source (target) cell split into two stacked cells gives the sum (volume-weighted mean) of the parts;
  * reciprocity V_t N(R; t <- s) = V_s N(-R; s <- t);
  * a stack whose layers DO sit on a common z grid (equal thickness, integer levels, gaps allowed) is a single 3-D
    mesh with empty layers: Eq. 4 must reproduce the single-mesh double sum of oracle.demag_direct (itself pinned);
  * the direct sum against the FFT route with the inter-layer terms summed in the transform space.
"""
import numpy as np
import pytest

from oracle import multilayer as ML
from oracle.demag_direct import demag_direct
from oracle.newell import newell_point
from paper_2008_02478_b200 import workloads as W

COMP = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]


@pytest.mark.parametrize("disp,tk,ti", [((2, 1, 2.5), 3.0, 1.0), ((1, 2, -1.7), 0.6, 4.9), ((0, 0, 9.0), 2.9, 0.6),
                                        ((3, 0, 0.4), 1.0, 2.0), ((0, 2, 0.0), 2.0, 0.5)])
def test_unequal_cuboids_against_brute_force_quadrature(disp, tk, ti):
    """N_ab = (1 / V_t) int_target d3r int_source d3r' D_ab(R + r - r') / (4 pi), cells at least a cell apart in-plane
    or fully separated in height, so the integrand is analytic."""
    hx, hy = 5.0, 4.0
    R = np.array([disp[0] * hx, disp[1] * hy, disp[2]])
    n = 10
    t, w = np.polynomial.legendre.leggauss(n)
    t, w = t / 2, w / 2
    du = (t[:, None] - t[None, :]).ravel()                       # equal sides: r - r' per axis
    wu = (w[:, None] * w[None, :]).ravel()
    dz = (tk * t[:, None] - ti * t[None, :]).ravel()             # unequal heights
    ux = R[0] + hx * du[:, None, None]
    uy = R[1] + hy * du[None, :, None]
    uz = R[2] + dz[None, None, :]
    Wt = wu[:, None, None] * wu[None, :, None] * wu[None, None, :]
    r2 = ux * ux + uy * uy + uz * uz
    r5 = r2 ** 2.5
    Vs = hx * hy * ti
    num = {0: r2 - 3 * ux * ux, 1: r2 - 3 * uy * uy, 2: r2 - 3 * uz * uz, 3: -3 * ux * uy, 4: -3 * ux * uz, 5: -3 * uy * uz}
    for c in range(6):
        brute = Vs * np.sum(Wt * num[c] / r5) / (4 * np.pi)
        got = ML.pair_tensor_point(c, *R, hx, hy, tk, ti)
        assert abs(got - brute) < 3e-9, (c, got, brute)


def test_equal_cells_give_back_newell():
    hx, hy, hz = 3.0, 2.0, 1.5
    for X, Y, Z in [(0, 0, 0), (3.0, 0, 1.5), (6.0, 4.0, -3.0), (0.0, 2.0, 0.7)]:
        for c in range(6):
            assert ML.pair_tensor_point(c, X, Y, Z, hx, hy, hz, hz) == pytest.approx(newell_point(c, X, Y, Z, hx, hy, hz), abs=1e-15)
    tab = ML.pair_tensor_table(4, 3, hx, hy, hz, hz, 0.0)
    assert tab[0][0, 0] + tab[1][0, 0] + tab[2][0, 0] == pytest.approx(1.0, abs=1e-13)       # self term, trace 1


@pytest.mark.parametrize("X,Y,Z", [(0.0, 0.0, 0.0), (4.0, 0.0, 1.3), (8.0, 3.0, -2.2), (0.0, 6.0, 5.0)])
def test_additivity_over_a_split_cell_and_reciprocity(X, Y, Z):
    hx, hy, a, tk = 4.0, 3.0, 1.1, 2.7
    for c in range(6):
        big = ML.pair_tensor_point(c, X, Y, Z, hx, hy, tk, 2 * a)                 # source of thickness 2a centred at 0
        parts = ML.pair_tensor_point(c, X, Y, Z - a / 2, hx, hy, tk, a) + ML.pair_tensor_point(c, X, Y, Z + a / 2, hx, hy, tk, a)
        assert big == pytest.approx(parts, abs=2e-14)
        bigt = ML.pair_tensor_point(c, X, Y, Z, hx, hy, 2 * a, tk)                # target of thickness 2a
        partt = 0.5 * (ML.pair_tensor_point(c, X, Y, Z + a / 2, hx, hy, a, tk) + ML.pair_tensor_point(c, X, Y, Z - a / 2, hx, hy, a, tk))
        assert bigt == pytest.approx(partt, abs=2e-14)
        # reciprocity: V_t N(R; t <- s) = V_s N(-R; s <- t)
        assert tk * ML.pair_tensor_point(c, X, Y, Z, hx, hy, tk, a) == pytest.approx(
            a * ML.pair_tensor_point(c, -X, -Y, -Z, hx, hy, a, tk), abs=2e-14)


@pytest.mark.parametrize("levels", [(0,), (0, 1), (0, 2, 3), (1, 4)])
def test_a_stack_on_a_common_grid_is_a_single_mesh_with_empty_layers(levels):
    ny, nx, h = 3, 4, (3e-9, 2e-9, 1e-9)
    n = len(levels)
    M = W.make_texture("random", (n, ny, nx), 8e5, seed=101).astype(np.float64)
    nz = max(levels) + 1
    M3 = np.zeros((3, nz, ny, nx))
    M3[:, list(levels)] = M
    want = demag_direct(M3, h)[:, list(levels)]                 # PAPER.md:L323 on the 3-D mesh
    t = [h[2]] * n
    z = [lv * h[2] for lv in levels]
    got = ML.multilayer_direct(M, h[0], h[1], t, z)
    assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()
    assert np.abs(ML.multilayer_fft(M, h[0], h[1], t, z) - want).max() <= 1e-12 * np.abs(want).max()


def test_unequal_stack_direct_sum_against_the_transform_space_sum():
    """The paper's kind of stack (L76): magnetic layers of different thickness separated by thin spacers."""
    ny, nx, hx, hy = 4, 5, 5e-9, 5e-9
    t = [4.9e-9, 2.9e-9, 4.9e-9]
    z = [2.45e-9, 6.95e-9, 11.45e-9]                             # 0.6 nm spacers
    M = W.make_texture("random", (3, ny, nx), 1.4e6, seed=102).astype(np.float64)
    Hd = ML.multilayer_direct(M, hx, hy, t, z)
    Hf = ML.multilayer_fft(M, hx, hy, t, z)
    assert np.abs(Hd - Hf).max() <= 1e-12 * np.abs(Hd).max()
    # the layers do interact: switching the other layers off changes the field of layer 0
    M0 = M.copy()
    M0[:, 1:] = 0
    assert np.abs(ML.multilayer_direct(M0, hx, hy, t, z)[:, 0] - Hd[:, 0]).max() >= 1e-3 * np.abs(Hd).max()
    # energy: positive for any state (the magnetostatic self-energy of the whole stack)
    assert ML.multilayer_energy(M, Hd, hx, hy, t) > 0


def test_uniform_out_of_plane_stack_field_is_the_sum_of_its_layers_fields():
    """Linearity over layers, and the thin-film limit per layer: a wide single layer magnetized along z feels Hz ~ -Mz."""
    ny, nx, hx, hy = 16, 16, 8e-9, 8e-9
    t, z, Ms = [1e-9], [0.5e-9], 6e5
    M = np.zeros((3, 1, ny, nx))
    M[2] = Ms
    H = ML.multilayer_fft(M, hx, hy, t, z)
    assert -1.0 < H[2, 0, 8, 8] / Ms < -0.97
