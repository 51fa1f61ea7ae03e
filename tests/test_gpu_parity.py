"""GPU parity: boris_demag_apply / boris_demag_energy (through the C ABI) vs the fp64 oracle.

Acceptance (BASELINE.json north_star): max|dH| <= 1e-5 Ms and relative L2 <= 2e-6.
Small meshes: every element against the plain double sum.  Configs
C2-C5: every element against the fp64 FFT oracle, which is itself
checked here against the sampled plain sum (pin P14), plus sampled outputs directly.
"""
import ctypes

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import newell
from oracle.demag_direct import demag_at, demag_direct, tensor_table
from oracle.demag_fft import demag_fft, kernel_spectrum, padded_shape
from oracle.energy import demag_energy
from paper_2008_02478_b200 import binding, build, workloads as W

pytestmark = pytest.mark.gpu

TOL_MAX = 1e-5      # x Ms            (north_star)
TOL_L2 = 2e-6       # relative L2     (north_star)
TOL_E = 1e-5        # relative, energy (not fixed by BASELINE.json)


@pytest.fixture(scope="module", autouse=True)
def cuda_library():
    build.build()
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(0)
    binding.lib()


def gpu_apply(plan, M_host, want_energy=False):
    M = torch.from_numpy(M_host).cuda()
    H = torch.full_like(M, float("nan"))
    plan.apply(M, H)
    E = plan.energy(M, H) if want_energy else None
    torch.cuda.synchronize()
    Hh = H.cpu().numpy()
    return (Hh, float(E.item())) if want_energy else Hh


def errors(H, H_ref, Ms):
    err = np.abs(H.astype(np.float64) - H_ref)
    return err.max() / Ms, np.sqrt((err ** 2).sum() / (H_ref ** 2).sum())


def assert_parity(H, H_ref, Ms):
    assert np.isfinite(H).all()
    emax, el2 = errors(H, H_ref, Ms)
    assert emax <= TOL_MAX, f"max|dH|/Ms = {emax:.3e}"
    assert el2 <= TOL_L2, f"rel L2 = {el2:.3e}"
    return emax, el2


# ----------------------------------------------------------------- small meshes, plain double sum
SMALL = [
    # (nz, ny, nx), h, texture
    ((1, 2, 4), (5e-9, 5e-9, 3e-9), "random"),        # smallest supported mesh
    ((1, 32, 32), (5e-9, 5e-9, 3e-9), "random"),      # C1
    ((1, 8, 64), (5e-9, 4e-9, 3e-9), "vortex"),       # ragged: fewer rows than a block holds
    ((1, 64, 4), (2e-9, 3e-9, 1e-9), "helix"),
    ((2, 2, 4), (2e-9, 2e-9, 1e-9), "random"),        # smallest 3-D mesh
    ((2, 8, 16), (5e-9, 4e-9, 3e-9), "random"),
    ((4, 16, 8), (2e-9, 2e-9, 1e-9), "helix"),
    ((8, 4, 32), (2e-9, 3e-9, 4e-9), "random"),
    ((16, 8, 8), (2e-9, 2e-9, 2e-9), "random"),
]


@pytest.mark.parametrize("shape,h,texture", SMALL)
def test_small_meshes_match_the_plain_double_sum(shape, h, texture):
    nz, ny, nx = shape
    Ms = 8e5
    M = W.make_texture(texture, shape, Ms, seed=21)
    plan = binding.DemagPlan(nx, ny, nz, *h)
    H, E = gpu_apply(plan, M, want_energy=True)
    H_ref = demag_direct(M, h)
    assert_parity(H, H_ref, Ms)
    E_ref = demag_energy(M, H_ref, h)
    assert abs(E - E_ref) <= TOL_E * abs(E_ref)
    assert E > 0                                             # pin P8: N is positive semi-definite
    plan.close()


# ----------------------------------------------------------------- medium meshes (several tiles / chunks), FFT oracle
MEDIUM = [
    ((1, 128, 512), (2e-9, 2e-9, 1e-9), "domains"),
    ((1, 1024, 16), (2e-9, 2e-9, 1e-9), "random"),        # Py = 2048: three passes
    ((1, 16, 1024), (4e-9, 4e-9, 4e-9), "helix"),         # LX = 1024
    ((1, 512, 64), (4e-9, 4e-9, 4e-9), "vortex"),
    ((32, 64, 16), (2e-9, 2e-9, 1e-9), "helix"),
    ((64, 16, 64), (2e-9, 2e-9, 2e-9), "random"),
    ((128, 8, 8), (2e-9, 2e-9, 2e-9), "random"),          # Pz = 256 as in C4
    ((512, 2, 4), (2e-9, 2e-9, 2e-9), "random"),          # Pz = 1024: largest fused z
    ((2, 256, 128), (5e-9, 5e-9, 3e-9), "vortex"),
    ((8, 512, 32), (2e-9, 2e-9, 1e-9), "helix"),          # Py = 1024 as in C5
    ((256, 4, 16), (2e-9, 2e-9, 2e-9), "random"),         # z columns in 16 passes of 32 points
    ((32, 16, 1024), (2e-9, 2e-9, 1e-9), "helix"),        # nz rows of nx = 1024 exceed shared memory: chunked fallback
    ((32, 16, 16), (2e-9, 2e-9, 1e-9), "random"),         # nz = 32 but too few rows for the plane path: tiled 3-D
    # plane path (csrc/plane.h): nz = 32, ny = 32..512
    ((32, 32, 8), (2e-9, 3e-9, 1e-9), "random"),          # sub-transform of 64 points, one ky residue
    ((32, 128, 64), (2e-9, 2e-9, 1e-9), "random"),        # 256 points, one residue
    ((32, 256, 16), (5e-9, 4e-9, 3e-9), "vortex"),        # two residues
    ((32, 512, 8), (2e-9, 2e-9, 1e-9), "helix"),          # four residues: C5's y and z
    ((32, 64, 1024), (2e-9, 2e-9, 1e-9), "helix"),        # LX = 1024 rows on the plane path
]


@pytest.mark.parametrize("shape,h,texture", MEDIUM)
def test_medium_meshes_match_the_fft_oracle(shape, h, texture):
    nz, ny, nx = shape
    Ms = 1.1e6
    M = W.make_texture(texture, shape, Ms, seed=22)
    plan = binding.DemagPlan(nx, ny, nz, *h)
    H, E = gpu_apply(plan, M, want_energy=True)
    tab = tensor_table(shape, h)
    H_ref = demag_fft(M, h, table=tab)
    assert_parity(H, H_ref, Ms)
    # sampled outputs by the plain sum, independent of any FFT
    tg = W.sample_targets(shape, 12, seed=3)
    Hs = demag_at(M, h, tg, table=tab)
    for n, p in enumerate(tg):
        assert np.abs(H[(slice(None),) + p] - Hs[n]).max() <= TOL_MAX * Ms
    E_ref = demag_energy(M, H_ref, h)
    assert abs(E - E_ref) <= TOL_E * abs(E_ref)
    plan.close()


@pytest.mark.parametrize("shape", [(1, 64, 128), (1, 1024, 16), (8, 32, 64), (64, 16, 32), (512, 2, 4)])
def test_fused_apply_energy_matches_the_two_calls_and_is_reproducible(shape):
    nz, ny, nx = shape
    h = (2e-9, 3e-9, 1e-9)
    M_host = W.make_texture("random", shape, 8e5, seed=31)
    plan = binding.DemagPlan(nx, ny, nz, *h)
    M = torch.from_numpy(M_host).cuda()
    H1, H2 = torch.empty_like(M), torch.full_like(M, float("nan"))
    plan.apply(M, H1)
    E1 = plan.energy(M, H1)
    E2 = plan.apply_energy(M, H2)
    E3 = plan.apply_energy(M, H2).clone()
    torch.cuda.synchronize()
    assert torch.equal(H1, H2)                                   # same kernels, same bits
    assert E2.item() == E3.item()                                # fixed summation order
    assert abs(E2.item() - E1.item()) <= 1e-12 * abs(E1.item())  # both fp64 sums of the same products
    E_ref = demag_energy(M_host, demag_fft(M_host, h), h)
    assert abs(E2.item() - E_ref) <= TOL_E * abs(E_ref)
    plan.close()


@pytest.mark.parametrize("shape", [(1, 1, 1), (1, 7, 9), (3, 5, 6), (1, 100, 60), (5, 33, 17), (2, 1, 3), (40, 3, 2)])
def test_meshes_that_are_not_powers_of_two_match_the_plain_double_sum(shape):
    """Any mesh is the corner of the next power-of-two mesh with M = 0 elsewhere (include/boris_demag.h)."""
    nz, ny, nx = shape
    h = (3e-9, 2e-9, 4e-9)
    Ms = 8e5
    M_host = W.make_texture("random", shape, Ms, seed=41)
    plan = binding.DemagPlan(nx, ny, nz, *h)
    H, E = gpu_apply(plan, M_host, want_energy=True)
    H_ref = demag_direct(M_host, h)
    assert_parity(H, H_ref, Ms)
    E_ref = demag_energy(M_host, H_ref, h)
    assert abs(E - E_ref) <= TOL_E * abs(E_ref)
    M = torch.from_numpy(M_host).cuda()
    H2 = torch.full_like(M, float("nan"))
    E2 = plan.apply_energy(M, H2)
    torch.cuda.synchronize()
    assert np.array_equal(H2.cpu().numpy(), H)
    assert abs(E2.item() - E_ref) <= TOL_E * abs(E_ref)
    H3 = np.empty_like(M_host)
    E3 = plan.apply_host(M_host, H3)
    assert np.array_equal(H3, H) and E3 == E2.item()
    info = plan.info()
    assert info["kernel_launches"] >= 5 and info["compulsory_bytes"] >= 24 * nx * ny * nz
    plan.close()
    with pytest.raises(binding.DemagError):
        binding.DemagPlan(1025, 4, 1, *h)
    with pytest.raises(binding.DemagError):
        binding.DemagPlan(4, 4, 0, *h)


@pytest.mark.parametrize("shape", [(1, 64, 32), (8, 16, 32), (3, 10, 6), (32, 64, 32)])
def test_float3_layout_and_accumulate_variants_match_the_oracle(shape):
    nz, ny, nx = shape
    h = (2e-9, 2e-9, 1e-9)
    M_host = W.make_texture("random", shape, 8e5, seed=51)
    H_ref = demag_fft(M_host, h)                                # fp64 oracle
    plan = binding.DemagPlan(nx, ny, nz, *h)
    M = torch.from_numpy(M_host).cuda()
    M3 = M.permute(1, 2, 3, 0).contiguous()                    # [nz][ny][nx][3]
    H3 = torch.full_like(M3, float("nan"))
    plan.apply_ex(M3, H3, plan.AOS)
    assert_parity(H3.permute(3, 0, 1, 2).cpu().numpy(), H_ref, 8e5)
    H0_host = (np.random.default_rng(52).standard_normal(M_host.shape) * 1e4).astype(np.float32)
    Hacc = torch.from_numpy(H0_host).cuda()
    plan.apply_ex(M, Hacc, plan.ACCUMULATE)
    # H0 + H rounded once more to fp32 at |H0 + H| <~ 1e6: half an ulp of 2^-4 on top of the parity tolerance
    got = Hacc.cpu().numpy().astype(np.float64) - H0_host
    assert np.abs(got - H_ref).max() <= TOL_MAX * 8e5 + 2.0 ** -4
    H0a = torch.from_numpy(H0_host).cuda().permute(1, 2, 3, 0).contiguous()
    plan.apply_ex(M3, H0a, plan.AOS | plan.ACCUMULATE)
    got = H0a.permute(3, 0, 1, 2).cpu().numpy().astype(np.float64) - H0_host
    assert np.abs(got - H_ref).max() <= TOL_MAX * 8e5 + 2.0 ** -4
    H = torch.empty_like(M)
    assert binding.lib().boris_demag_apply_ex(plan._h, M.data_ptr(), H.data_ptr(), 8, None) == -1
    plan.close()


def test_kernel_path_chosen_per_mesh():
    expect = {(1, 32, 32): 2, (1, 1024, 1024): 2, (128, 128, 128): 3, (32, 512, 512): 4, (32, 256, 16): 4, (32, 1024, 64): 4, (32, 64, 1024): 4, (16, 512, 512): 4, (8, 64, 64): 4, (16, 16, 64): 3, (4, 64, 64): 4, (2, 32, 32): 4, (4, 16, 64): 3, (64, 64, 512): 4, (64, 64, 256): 4, (64, 128, 128): 3, (64, 256, 256): 3,
              (32, 16, 1024): 0, (512, 2, 4): 0}
    for (nz, ny, nx), path in expect.items():
        plan = binding.DemagPlan(nx, ny, nz, 2e-9, 2e-9, 1e-9)
        assert plan.layout()["path"] == path
        assert plan.info()["kernel_launches"] == (3 if path else plan.info()["kernel_launches"])
        plan.close()


# ----------------------------------------------------------------- the five configs at full size
@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
def test_config_at_full_size(name):
    cfg = W.CONFIGS[name]
    M = W.make_input(cfg)
    plan = binding.DemagPlan(cfg.nx, cfg.ny, cfg.nz, *cfg.h)
    H, E = gpu_apply(plan, M, want_energy=True)
    tab = tensor_table(cfg.shape, cfg.h)
    if name == "C1":
        H_ref = demag_direct(M, cfg.h, table=tab)
    else:
        Khat = kernel_spectrum(cfg.shape, cfg.h, table=tab)
        H_ref = demag_fft(M, cfg.h, Khat=Khat)
        del Khat
    # pin P14: the FFT oracle agrees with the sampled plain sum before it is trusted
    tg = W.sample_targets(cfg.shape, 64 if cfg.cells <= 2 ** 21 else 32, seed=5)
    Hs = demag_at(M, cfg.h, tg, table=tab)
    for n, p in enumerate(tg):
        assert np.abs(H_ref[(slice(None),) + p] - Hs[n]).max() <= 1e-9 * cfg.Ms
        assert np.abs(H[(slice(None),) + p] - Hs[n]).max() <= TOL_MAX * cfg.Ms
    emax, el2 = assert_parity(H, H_ref, cfg.Ms)
    E_ref = demag_energy(M, H_ref, cfg.h)
    assert abs(E - E_ref) <= TOL_E * abs(E_ref)
    print(f"{name}: max|dH|/Ms = {emax:.3e}, rel L2 = {el2:.3e}, E = {E:.6e} J (oracle {E_ref:.6e})")
    # the host-buffer entry point gives the same bits
    H2 = np.empty_like(M)
    E2 = plan.apply_host(M, H2)
    assert np.array_equal(H2, H)
    # apply_host gathers E inside the last kernel (boris_demag_apply_energy): another fp64 summation order
    assert abs(E2 - E) <= 1e-12 * abs(E)
    assert plan.apply_host(M, H2) == E2
    plan.close()


# ----------------------------------------------------------------- properties and edge cases
def test_P9_delta_readout_reads_the_whole_signed_tensor():
    """M = Ms e_b at a corner cell: H_a(t) = -Ms N_ab(t - s) over the whole displacement range."""
    shape, h, Ms = (4, 16, 32), (5e-9, 4e-9, 3e-9), 8e5
    nz, ny, nx = shape
    plan = binding.DemagPlan(nx, ny, nz, *h)
    tab = tensor_table(shape, h)
    for s, b in [((0, 0, 0), 0), ((nz - 1, ny - 1, nx - 1), 1), ((0, ny - 1, 0), 2)]:
        M = np.zeros((3,) + shape, np.float32)
        M[b][s] = Ms
        H = gpu_apply(plan, M)
        ks, js, is_ = np.arange(nz) - s[0], np.arange(ny) - s[1], np.arange(nx) - s[2]
        for a in range(3):
            c = newell.SYM_INDEX[a, b]
            px, py, pz = newell.PARITY[c]
            ref = tab[c][np.ix_(np.abs(ks), np.abs(js), np.abs(is_))].copy()
            if px < 0:
                ref *= np.sign(is_)[None, None, :]
            if py < 0:
                ref *= np.sign(js)[None, :, None]
            if pz < 0:
                ref *= np.sign(ks)[:, None, None]
            assert np.abs(H[a] + np.float32(Ms).astype(np.float64) * ref).max() <= TOL_MAX * Ms
    plan.close()


def test_P13_linearity_reciprocity_and_zero_input():
    shape, h, Ms = (8, 32, 64), (2e-9, 2e-9, 1e-9), 8e5
    nz, ny, nx = shape
    plan = binding.DemagPlan(nx, ny, nz, *h)
    M1 = W.make_texture("random", shape, Ms, seed=1)
    M2 = W.make_texture("helix", shape, Ms, seed=2)
    H1, H2 = gpu_apply(plan, M1), gpu_apply(plan, M2)
    H12 = gpu_apply(plan, (2.0 * M1 - 0.5 * M2).astype(np.float32))
    assert np.abs(H12 - (2.0 * H1.astype(np.float64) - 0.5 * H2)).max() <= 3 * TOL_MAX * Ms
    r12, r21 = np.sum(M1.astype(np.float64) * H2), np.sum(M2.astype(np.float64) * H1)
    assert abs(r12 - r21) <= 1e-5 * np.sum(np.abs(M1.astype(np.float64) * H2))
    Z = gpu_apply(plan, np.zeros_like(M1))
    assert np.array_equal(Z, np.zeros_like(Z))                      # empty space is legal input
    plan.close()


def test_P7_uniform_thin_film_hz_close_to_minus_mz():
    cfg = W.CONFIGS["C2"]
    plan = binding.DemagPlan(cfg.nx, cfg.ny, cfg.nz, *cfg.h)
    M = np.zeros((3,) + cfg.shape, np.float32)
    M[2] = cfg.Ms
    H = gpu_apply(plan, M)
    # SURVEY.md pin P7 body factor of C2's film [1024, 1024, 4] nm (golden/newell_self_terms.txt)
    assert abs(H[2].astype(np.float64).mean() / cfg.Ms + 0.984401655301) < 1e-6
    assert np.abs(H[:2]).max() <= TOL_MAX * cfg.Ms
    plan.close()


def test_apply_is_bit_identical_across_calls_and_streams():
    cfg = W.CONFIGS["C2"]
    M_host = W.make_input(cfg)
    plan = binding.DemagPlan(cfg.nx, cfg.ny, cfg.nz, *cfg.h)
    M = torch.from_numpy(M_host).cuda()
    H1, H2 = torch.empty_like(M), torch.empty_like(M)
    plan.apply(M, H1)
    E1 = plan.energy(M, H1)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        plan.apply(M, H2, stream=s)
        E2 = plan.energy(M, H2, stream=s)
    s.synchronize()
    assert torch.equal(H1, H2) and torch.equal(E1, E2)
    plan.close()


def test_P11_uploaded_spectrum_trace_and_oracle_spectrum():
    """The fp32 spectrum the kernels read: trace == folded factor at every frequency; equals the oracle's rfftn."""
    for shape, h in [((1, 64, 128), (2e-9, 2e-9, 1e-9)), ((16, 32, 16), (5e-9, 4e-9, 3e-9))]:
        nz, ny, nx = shape
        plan = binding.DemagPlan(nx, ny, nz, *h)
        K = plan.kernel_spectrum().astype(np.float64)
        Pz, Py, Px = padded_shape(shape)
        scale = -1.0 / (2.0 * Px * Py * Pz)
        assert np.abs((K[0] + K[1] + K[2]) / scale - 1).max() < 1e-6
        Ko = kernel_spectrum(shape, h)
        for c in range(K.shape[0]):
            ref = Ko[c][:K.shape[1], :ny + 1, :nx + 1]
            assert np.abs(ref.imag).max() < 1e-12
            assert np.abs(K[c] / scale - ref.real).max() < 2e-7 * max(1.0, np.abs(ref.real).max())
        info = plan.info()
        assert info["padded"] == (Px, Py, Pz)
        ncomp = 4 if nz == 1 else 6
        assert info["compulsory_bytes"] == 24 * nx * ny * nz + 4 * ncomp * (nx + 1) * (ny + 1) * (nz + 1 if nz > 1 else 1)
        plan.close()


def test_error_codes_on_bad_arguments():
    plan = binding.DemagPlan(32, 32, 1, 5e-9, 5e-9, 3e-9)
    M = torch.zeros(3, 1, 32, 32, device="cuda")
    L = binding.lib()
    assert L.boris_demag_apply(plan._h, M.data_ptr(), M.data_ptr(), None) == -1          # aliasing
    assert "alias" in binding.last_error()
    buf = torch.zeros(3 * 32 * 32 + 4, device="cuda")
    assert L.boris_demag_apply(plan._h, M.data_ptr(), buf.data_ptr() + 4, None) == -1    # misaligned
    with pytest.raises(binding.DemagError):
        plan.apply(M.double(), M)
    with pytest.raises(binding.DemagError):
        plan.apply(M[:, :, :16], M)
    plan.close()


def test_device_probes_report_sane_rates():
    """include/boris_micro.h: the two probes `bench.py --micro` tabulates (profiles/*_microbench.md)."""
    ffma, ffma2 = binding.micro_fp32_rate(1), binding.micro_fp32_rate(3)
    assert 1e13 < ffma < 6e13 and 1e13 < ffma2 < 6e13          # 148 SMs x 128 lanes x ~1.9 GHz = 3.6e13 at most
    r128, r32 = binding.micro_segment_bw(128, False), binding.micro_segment_bw(32, False)
    assert 1500 < r128 < 9000 and 300 < r32 <= 1.05 * r128
    with pytest.raises(binding.DemagError):
        binding.micro_segment_bw(48, False)


# ----------------------------------------------------------------- periodic boundary conditions
PBC_CASES = [
    # shape (nz, ny, nx), h, images (ix, iy, iz), texture
    ((1, 64, 64), (4e-9, 4e-9, 2e-9), (4, 4, 0), "vortex"),        # film, periodic in x and y
    ((8, 16, 32), (3e-9, 3e-9, 2e-9), (3, 0, 0), "random"),        # 3-D, periodic in x
    ((3, 10, 6), (4e-9, 5e-9, 3e-9), (2, 1, 0), "random"),         # not a power of two: the period is the caller's mesh
    ((32, 32, 16), (2e-9, 2e-9, 1e-9), (0, 2, 1), "helix"),        # plane path, periodic in y and z
    ((1, 256, 256), (4e-9, 4e-9, 4e-9), (5, 5, 0), "vortex"),      # C2's mesh, 11 x 11 copies
]


@pytest.mark.parametrize("shape,h,images,texture", PBC_CASES)
def test_periodic_boundary_conditions_match_the_oracle(shape, h, images, texture):
    from oracle.demag_pbc import demag_pbc_fft
    nz, ny, nx = shape
    Ms = 8e5
    M_host = W.make_texture(texture, shape, Ms, seed=81)
    H_ref = demag_pbc_fft(M_host, h, images)
    plan = binding.DemagPlan(nx, ny, nz, *h, images=images)
    H, E = gpu_apply(plan, M_host, want_energy=True)
    assert_parity(H, H_ref, Ms)
    E_ref = demag_energy(M_host, H_ref, h)
    assert abs(E - E_ref) <= TOL_E * abs(E_ref)
    # the open-boundary plan of the same mesh gives a different field: the copies are really there
    open_plan = binding.DemagPlan(nx, ny, nz, *h)
    H_open = gpu_apply(open_plan, M_host)
    assert np.abs(H_open - H).max() >= 1e-3 * Ms
    open_plan.close()
    plan.close()


def test_periodic_tiny_mesh_against_the_copy_by_copy_sum():
    from oracle.demag_pbc import demag_pbc_direct
    shape, h, images = (2, 4, 8), (3e-9, 2e-9, 1e-9), (2, 1, 0)
    M_host = W.make_texture("random", shape, 8e5, seed=82)
    plan = binding.DemagPlan(8, 4, 2, *h, images=images)
    assert_parity(gpu_apply(plan, M_host), demag_pbc_direct(M_host, h, images), 8e5)
    plan.close()
    with pytest.raises(binding.DemagError, match="images"):
        binding.DemagPlan(8, 4, 2, *h, images=(0, -1, 0))


# ----------------------------------------------------------------- plane path beyond C5: ny = 1024 (eight ky residues), nx = 1024
@pytest.mark.parametrize("shape", [(32, 1024, 64), (32, 64, 1024)])
def test_plane_path_with_1024_cells_along_y_or_x(shape):
    nz, ny, nx = shape
    h, Ms = (2e-9, 2e-9, 1e-9), 1.1e6
    M_host = W.make_texture("helix", shape, Ms, seed=121)
    plan = binding.DemagPlan(nx, ny, nz, *h)
    assert plan.layout()["path"] == 4
    H, E = gpu_apply(plan, M_host, want_energy=True)
    H_ref = demag_fft(M_host, h)
    assert_parity(H, H_ref, Ms)
    assert abs(E - demag_energy(M_host, H_ref, h)) <= TOL_E * abs(E)
    plan.close()


def test_1024x1024x32_film_sampled_against_the_written_out_sum():
    """The next size up from C5 (33.5 M cells; plane path, eight residues, 1024-point x rows).  The oracle cannot hold its
    padded spectra, so M is a handful of magnetized cells in an empty mesh and sampled outputs are compared with the
    written-out sum of PAPER.md:L323 over those cells, N from oracle.newell one displacement at a time."""
    nz, ny, nx = 32, 1024, 1024
    h, Ms = (2e-9, 2e-9, 1e-9), 8e5
    rng = np.random.default_rng(122)
    src = [(int(rng.integers(nz)), int(rng.integers(ny)), int(rng.integers(nx))) for _ in range(6)] + [(0, 0, 0), (31, 1023, 1023)]
    vec = rng.standard_normal((len(src), 3))
    vec *= Ms / np.linalg.norm(vec, axis=1)[:, None]
    plan = binding.DemagPlan(nx, ny, nz, *h)
    assert plan.layout()["path"] == 4
    M = torch.zeros(3, nz, ny, nx, device="cuda")
    for (k, j, i), v in zip(src, vec):
        M[:, k, j, i] = torch.tensor(v, dtype=torch.float32)
    H = torch.full_like(M, float("nan"))
    plan.apply(M, H)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(H).all())
    targets = src + [(int(rng.integers(nz)), int(rng.integers(ny)), int(rng.integers(nx))) for _ in range(24)]
    targets += [(k, min(j + 1, ny - 1), i) for (k, j, i) in src[:4]] + [(min(k + 1, nz - 1), j, i) for (k, j, i) in src[:4]]
    Mv = np.array([M[:, k, j, i].cpu().numpy().astype(np.float64) for (k, j, i) in src])
    sym = [[0, 3, 4], [3, 1, 5], [4, 5, 2]]
    worst = 0.0
    for (kt, jt, it) in targets:
        want = np.zeros(3)
        for (ks, js, is_), m in zip(src, Mv):
            N = [newell.newell_point(c, (it - is_) * h[0], (jt - js) * h[1], (kt - ks) * h[2], *h) for c in range(6)]
            for a in range(3):
                want[a] -= sum(N[sym[a][b]] * m[b] for b in range(3))
        got = H[:, kt, jt, it].cpu().numpy().astype(np.float64)
        worst = max(worst, np.abs(got - want).max() / Ms)
    assert worst <= TOL_MAX, worst
    plan.close()


# ----------------------------------------------------------------- plane path on 16- and 8-cell slabs (the paper's pipelined regime, L283)
@pytest.mark.parametrize("shape,texture", [((16, 64, 128), "helix"), ((8, 256, 64), "random"), ((16, 1024, 16), "random"),
                                           ((8, 32, 32), "vortex"), ((8, 40, 100), "random"), ((16, 512, 512), "helix"),
                                           ((64, 32, 512), "random"), ((64, 256, 512), "helix"), ((64, 48, 1000), "random"),
                                           ((4, 256, 64), "random"), ((2, 512, 128), "helix"), ((4, 40, 20), "random"),
                                           ((2, 1024, 16), "random"), ((4, 1024, 1024), "helix")])
def test_plane_path_on_thin_slabs(shape, texture):
    nz, ny, nx = shape
    h, Ms = (2e-9, 3e-9, 1e-9), 8e5
    M_host = W.make_texture(texture, shape, Ms, seed=131)
    plan = binding.DemagPlan(nx, ny, nz, *h)
    assert plan.layout()["path"] == 4
    H, E = gpu_apply(plan, M_host, want_energy=True)
    H_ref = demag_fft(M_host, h)
    assert_parity(H, H_ref, Ms)
    assert abs(E - demag_energy(M_host, H_ref, h)) <= TOL_E * abs(E)
    M = torch.from_numpy(M_host).cuda()
    H0 = torch.from_numpy(H).cuda()
    if (nx & (nx - 1)) == 0 and (ny & (ny - 1)) == 0:           # fused accumulate on the plane path
        Hacc = H0.clone()
        plan.apply_ex(M, Hacc, plan.ACCUMULATE)
        assert torch.equal(Hacc, H0 + H0)
    plan.close()


@pytest.mark.parametrize("shape", [(16, 64, 128), (8, 256, 64), (32, 64, 32), (4, 128, 64), (2, 64, 256)])
def test_tiled_3d_kernels_stay_reachable_on_slabs_the_plane_path_takes(shape, monkeypatch):
    """BORIS_DEMAG_NO_PLANE=1 at plan creation selects XZFwd / YFused / ZXInv (the A/B switch of profiles/r02_plane.md)."""
    nz, ny, nx = shape
    h, Ms = (2e-9, 3e-9, 1e-9), 8e5
    M_host = W.make_texture("random", shape, Ms, seed=132)
    monkeypatch.setenv("BORIS_DEMAG_NO_PLANE", "1")
    plan = binding.DemagPlan(nx, ny, nz, *h)
    monkeypatch.delenv("BORIS_DEMAG_NO_PLANE")
    assert plan.layout()["path"] == 3
    assert_parity(gpu_apply(plan, M_host), demag_fft(M_host, h), Ms)
    plan.close()


# ----------------------------------------------------------------- narrow meshes: launch geometry chosen for the SM count
@pytest.mark.parametrize("shape,path", [((1, 64, 64), 2), ((1, 128, 512), 2), ((1, 256, 1024), 2), ((1, 1024, 128), 2), ((1, 512, 512), 2),
                                        ((32, 64, 64), 4), ((32, 128, 32), 4), ((8, 128, 128), 4), ((16, 64, 64), 4),
                                        ((64, 64, 64), 4), ((64, 32, 128), 4), ((64, 128, 128), 3),
                                        ((256, 4, 32), 3), ((128, 8, 64), 3), ((64, 16, 4), 3)])      # z columns on 16, 8, 4 lanes (ZXInv)
def test_narrow_meshes_with_their_own_launch_geometry(shape, path):
    """2-D: rows per block of the x kernels and columns per YFused tile follow the block count (make_launch_cfg);
    slabs: extra ky residues while the blocks still fit the SMs at once (plane_geom).  Same parity bar."""
    nz, ny, nx = shape
    h, Ms = (3e-9, 2e-9, 1e-9), 8e5
    M_host = W.make_texture("random", shape, Ms, seed=151)
    plan = binding.DemagPlan(nx, ny, nz, *h)
    assert plan.layout()["path"] == path
    H, E = gpu_apply(plan, M_host, want_energy=True)
    H_ref = demag_fft(M_host, h)
    assert_parity(H, H_ref, Ms)
    assert abs(E - demag_energy(M_host, H_ref, h)) <= TOL_E * abs(E)
    M = torch.from_numpy(M_host).cuda()
    H2 = torch.full_like(M, float("nan"))
    E2 = plan.apply_energy(M, H2)
    torch.cuda.synchronize()
    assert np.array_equal(H2.cpu().numpy(), H)
    assert abs(E2.item() - E) <= 1e-12 * abs(E)
    plan.close()
