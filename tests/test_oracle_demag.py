"""Pins for oracle/demag_direct.py, demag_fft.py, energy.py (CPU only).

Pin numbers refer to SURVEY.md §8(c) / DESIGN.md.  The field definition is
PAPER.md:L323; the FFT route is PAPER.md:L275 with the padding of L283.
"""
import numpy as np
import pytest

from oracle import newell
from oracle.demag_direct import demag_at, demag_direct, tensor_table
from oracle.demag_fft import demag_fft, kernel_spectrum, padded_shape
from oracle.energy import MU0, demag_energy
from paper_2008_02478_b200 import workloads as W
from test_oracle_newell import aharoni_factors, dipole_tensor

SMALL = [((3, 5, 6), (5.0, 4.0, 3.0)), ((1, 6, 7), (5.0, 5.0, 3.0)), ((4, 4, 8), (2.0, 2.0, 1.0))]


@pytest.mark.parametrize("shape,h", SMALL)
def test_P10_fft_route_equals_the_plain_double_sum(shape, h):
    Ms = 8e5
    M = W.make_texture("random", shape, Ms, seed=7)
    Hd = demag_direct(M, h)
    Hf = demag_fft(M, h)
    assert np.abs(Hd - Hf).max() < 1e-13 * Ms


@pytest.mark.parametrize("shape,h", SMALL + [((1, 32, 32), (5.0, 5.0, 3.0))])
def test_P7_uniform_body_identity_against_aharoni(shape, h):
    """M uniform  =>  mean_t H(t) = -N_self(Lx, Ly, Lz) M, N_self from Aharoni's closed form."""
    nz, ny, nx = shape
    L = (nx * h[0], ny * h[1], nz * h[2])
    Nbody = aharoni_factors(L)
    Ms = 8e5
    for a in range(3):
        M = np.zeros((3,) + shape, np.float32)
        M[a] = Ms
        H = demag_fft(M, h) if nx * ny * nz > 200 else demag_direct(M, h)
        mean = H.reshape(3, -1).mean(axis=1)
        expect = np.zeros(3)
        expect[a] = -Nbody[a] * Ms
        np.testing.assert_allclose(mean, expect, rtol=0, atol=1e-10 * Ms)


def test_thin_film_out_of_plane_field_is_close_to_minus_Mz():
    # north_star: "Hz ~ -Mz for uniform out-of-plane thin films"
    shape, h, Ms = (1, 64, 64), (5.0, 5.0, 1.0), 8e5
    M = np.zeros((3,) + shape, np.float32)
    M[2] = Ms
    H = demag_fft(M, h)
    assert -1.0 < H[2, 0, 32, 32] / Ms < -0.97
    assert abs(H[0]).max() < 1e-9 * Ms and abs(H[1]).max() < 1e-9 * Ms   # no in-plane field by symmetry of Nxz, Nyz = 0


def test_P9_delta_readout_reads_the_signed_tensor():
    """One magnetized cell s: H_a(t) = -Ms N_ab(t - s), N evaluated at the signed displacement."""
    shape, h, Ms = (3, 4, 5), (5.0, 4.0, 3.0), 1.0
    nz, ny, nx = shape
    comp_of = newell.SYM_INDEX
    for s, b in [((0, 0, 0), 0), ((2, 3, 4), 1), ((1, 2, 1), 2)]:
        M = np.zeros((3,) + shape, np.float32)
        M[b][s] = Ms
        Hd = demag_direct(M, h)
        Hf = demag_fft(M, h)
        for t in [(0, 0, 0), (2, 3, 4), (1, 0, 3), (0, 3, 0), (2, 1, 2)]:
            d = (t[2] - s[2]) * h[0], (t[1] - s[1]) * h[1], (t[0] - s[0]) * h[2]
            for a in range(3):
                expect = -Ms * newell.newell_point(comp_of[a, b], *d, *h)
                assert abs(Hd[a][t] - expect) < 1e-15
                assert abs(Hf[a][t] - expect) < 1e-14


def test_far_field_of_one_cell_is_the_textbook_dipole_field():
    """H = (1/4pi)(3 (m.r) r / r^5 - m / r^3), m = M V: fixes the overall sign of H = -N M."""
    shape, h, Ms = (1, 1, 41), (2.0, 2.0, 2.0), 1.0
    M = np.zeros((3,) + shape, np.float32)
    M[2][0, 0, 0] = Ms                      # dipole along z at cell 0
    H = demag_direct(M, h)
    r = 40 * h[0]
    m = Ms * 8.0
    # on the equator (r along x): H_z = -m / (4 pi r^3)
    assert abs(H[2][0, 0, 40] - (-m / (4 * np.pi * r ** 3))) < 1e-5 * m / (4 * np.pi * r ** 3)
    M[:] = 0
    M[0][0, 0, 0] = Ms                      # dipole along x, observed on its axis: H_x = +2m/(4 pi r^3)
    H = demag_direct(M, h)
    assert abs(H[0][0, 0, 40] - (2 * m / (4 * np.pi * r ** 3))) < 1e-5 * 2 * m / (4 * np.pi * r ** 3)
    # and the generic direction through the dipole tensor
    D = dipole_tensor([40 * 2.0, 0, 0])
    assert abs(H[0][0, 0, 40] + m * D[0, 0]) < 1e-5 * abs(m * D[0, 0])


def test_P13_linearity_reciprocity_translation():
    shape, h, Ms = (2, 6, 8), (2.0, 2.0, 1.0), 8e5
    M1 = W.make_texture("random", shape, Ms, seed=1).astype(np.float64)
    M2 = W.make_texture("helix", shape, Ms, seed=2).astype(np.float64)
    tab = tensor_table(shape, h)
    H1, H2 = demag_direct(M1, h, tab), demag_direct(M2, h, tab)
    H12 = demag_direct(2.0 * M1 - 0.5 * M2, h, tab)
    assert np.abs(H12 - (2.0 * H1 - 0.5 * H2)).max() < 1e-12 * Ms
    assert abs(np.sum(M1 * H2) - np.sum(M2 * H1)) < 1e-12 * abs(np.sum(M1 * H2))
    # translation of a sub-pattern inside a zero-filled mesh
    big = (2, 10, 12)
    A = np.zeros((3,) + big)
    B = np.zeros((3,) + big)
    A[:, :, 1:5, 2:7] = M1[:, :, :4, :5]
    B[:, :, 4:8, 5:10] = M1[:, :, :4, :5]
    HA, HB = demag_direct(A, h), demag_direct(B, h)
    assert np.abs(HA[:, :, 1:5, 2:7] - HB[:, :, 4:8, 5:10]).max() < 1e-12 * Ms


def test_P8_energy_closed_form_and_positivity():
    shape, h, Ms = (2, 6, 5), (5e-9, 4e-9, 3e-9), 8e5
    nz, ny, nx = shape
    L = (nx * h[0], ny * h[1], nz * h[2])
    M = np.zeros((3,) + shape, np.float32)
    M[2] = Ms
    E = demag_energy(M, demag_direct(M, h), h)
    expect = 0.5 * MU0 * Ms ** 2 * np.prod(L) * aharoni_factors(L)[2]
    assert abs(E - expect) < 1e-10 * expect
    for seed in range(3):
        Mr = W.make_texture("random", shape, Ms, seed=seed)
        assert demag_energy(Mr, demag_fft(Mr, h), h) > 0


@pytest.mark.parametrize("shape,h", [((4, 6, 8), (5.0, 4.0, 3.0)), ((1, 8, 16), (2.0, 2.0, 1.0))])
def test_P11_P12_kernel_spectrum_is_real_has_unit_trace_and_mirrors(shape, h):
    Khat = kernel_spectrum(shape, h)
    Pz, Py, Px = padded_shape(shape)
    tr = Khat[0] + Khat[1] + Khat[2]
    assert np.abs(tr - 1).max() < 1e-13
    for c, K in enumerate(Khat):
        if K is None:
            assert shape[0] == 1 and c in (4, 5)
            continue
        assert np.abs(K.imag).max() < 1e-15
        # P12: value at mirrored ky (kz) = value at Py-ky (Pz-kz) times the y (z) parity
        ky = np.arange(1, Py)
        np.testing.assert_allclose(K[:, Py - ky, :].real, newell.PARITY[c][1] * K[:, ky, :].real, atol=1e-15)
        if Pz > 1:
            kz = np.arange(1, Pz)
            np.testing.assert_allclose(K[Pz - kz].real, newell.PARITY[c][2] * K[kz].real, atol=1e-15)


def test_P14_sampled_direct_sum_agrees_with_fft_on_a_mid_size_mesh():
    shape, h, Ms = (4, 48, 64), (2.0, 2.0, 1.0), 1.1e6
    M = W.make_texture("helix", shape, Ms, seed=5)
    tab = tensor_table(shape, h)
    Hf = demag_fft(M, h, table=tab)
    targets = W.sample_targets(shape, 40, seed=3)
    Hs = demag_at(M, h, targets, table=tab)
    for n, t in enumerate(targets):
        assert np.abs(Hs[n] - Hf[(slice(None),) + t]).max() < 1e-9 * Ms


def test_workload_generators_are_seeded_unit_norm_float32():
    for name in ("C1", "C2"):
        cfg = W.CONFIGS[name]
        A, B = W.make_input(cfg), W.make_input(name)
        assert A.dtype == np.float32 and A.shape == (3,) + cfg.shape
        assert np.array_equal(A, B)
        norm = np.sqrt((A.astype(np.float64) ** 2).sum(axis=0))
        np.testing.assert_allclose(norm, cfg.Ms, rtol=2e-7)
    for tex in ("domains", "helix"):
        M = W.make_texture(tex, (2, 32, 64), 1.0, seed=4)
        np.testing.assert_allclose(np.sqrt((M.astype(np.float64) ** 2).sum(axis=0)), 1.0, rtol=2e-7)
