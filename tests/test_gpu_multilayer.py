"""GPU parity of the multi-layered convolution (include/boris_demag_ml.h; Eq. 4) with oracle/multilayer.py.

fp32 plans are held to the north_star gate (max|dH| <= 1e-5 Ms, relative L2 <= 2e-6), fp64 plans to the fp64 gate of
tests/test_gpu_f64.py (1e-10 sqrt(N) Ms, relative L2 1e-9).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import multilayer as ML
from oracle.demag_fft import demag_fft
from paper_2008_02478_b200 import binding, build, workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def cuda_library():
    build.build()
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(0)


def run(plan, M_host):
    M = torch.from_numpy(M_host).cuda()
    H = torch.full_like(M, float("nan"))
    plan.apply(M, H)
    E = plan.energy(M, H)
    torch.cuda.synchronize()
    return H.cpu().numpy().astype(np.float64), float(E.item())


def check(H, H_ref, Ms, fp64):
    assert np.isfinite(H).all()
    err = np.abs(H - H_ref)
    rel = np.sqrt((err ** 2).sum() / (H_ref ** 2).sum())
    if fp64:
        assert err.max() <= 1e-10 * np.sqrt(H.size / 3) * Ms and rel <= 1e-9, (err.max() / Ms, rel)
    else:
        assert err.max() <= 1e-5 * Ms and rel <= 2e-6, (err.max() / Ms, rel)


# the paper's kind of stack (L76): CoFe 4.9 nm / Ru 0.6 nm / CoFe 2.9 nm / Ru 0.6 nm, repeated
def cofe_ru_stack(repeats):
    t, z, z0 = [], [], 0.0
    for _ in range(repeats):
        for th in (4.9e-9, 2.9e-9):
            t.append(th)
            z.append(z0 + th / 2)
            z0 += th + 0.6e-9
    return t, z


@pytest.mark.parametrize("fp64", [False, True])
@pytest.mark.parametrize("ny,nx,stack", [(4, 8, ([3e-9, 1e-9], [1.5e-9, 5e-9])), (6, 5, ([2e-9, 2e-9, 1e-9], [1e-9, 3.5e-9, 7e-9])),
                                         (16, 32, cofe_ru_stack(2))])
def test_small_stacks_against_the_written_out_sum(ny, nx, stack, fp64):
    t, z = stack
    Ms = 1.4e6
    M_host = W.make_texture("random", (len(t), ny, nx), Ms, seed=111)
    M_host = M_host.astype(np.float64) if fp64 else M_host
    plan = binding.MultiLayerPlan(nx, ny, 5e-9, 4e-9, t, z, fp64=fp64)
    H, E = run(plan, M_host)
    H_ref = ML.multilayer_direct(M_host, 5e-9, 4e-9, t, z) if ny * nx <= 64 else ML.multilayer_fft(M_host, 5e-9, 4e-9, t, z)
    check(H, H_ref, Ms, fp64)
    E_ref = ML.multilayer_energy(M_host, H_ref, 5e-9, 4e-9, t)
    assert abs(E - E_ref) <= (1e-9 if fp64 else 1e-5) * abs(E_ref)
    plan.close()


@pytest.mark.parametrize("fp64", [False, True])
def test_the_papers_ten_repeat_stack_at_film_size(fp64):
    """[CoFe 4.9 / Ru 0.6 / CoFe 2.9 / Ru 0.6] x 10: 20 magnetic layers of 128 x 128 cells."""
    t, z = cofe_ru_stack(10)
    ny = nx = 128
    Ms = 1.4e6
    M_host = W.make_texture("vortex", (len(t), ny, nx), Ms, seed=112)
    # antiparallel alignment of neighbouring layers, as the RKKY-coupled stack of the paper prefers
    M_host[:, 1::2] *= -1
    M_host = M_host.astype(np.float64) if fp64 else M_host
    plan = binding.MultiLayerPlan(nx, ny, 4e-9, 4e-9, t, z, fp64=fp64)
    H, _ = run(plan, M_host)
    check(H, ML.multilayer_fft(M_host, 4e-9, 4e-9, t, z), Ms, fp64)
    plan.close()


def test_a_stack_on_a_common_grid_matches_the_single_mesh_engine_and_oracle():
    """Equal thickness, integer levels: Eq. 4 is the single 3-D mesh with empty layers — oracle.demag_fft and the fp32
    single-mesh engine (boris_demag_apply) must agree with the multi-layer engine."""
    levels, (ny, nx), h, Ms = (0, 1, 3), (32, 64), (3e-9, 3e-9, 2e-9), 8e5
    M_host = W.make_texture("random", (len(levels), ny, nx), Ms, seed=113)
    t = [h[2]] * len(levels)
    z = [(lv + 0.5) * h[2] for lv in levels]
    plan = binding.MultiLayerPlan(nx, ny, h[0], h[1], t, z)
    H, _ = run(plan, M_host)
    M3 = np.zeros((3, 4, ny, nx), np.float32)
    M3[:, list(levels)] = M_host
    want = demag_fft(M3, h)[:, list(levels)]
    check(H, want, Ms, False)
    p3 = binding.DemagPlan(nx, ny, 4, *h)
    H3 = torch.empty(3, 4, ny, nx, device="cuda")
    p3.apply(torch.from_numpy(M3).cuda(), H3)
    assert np.abs(H3.cpu().numpy()[:, list(levels)] - H).max() <= 2e-5 * Ms
    p3.close()
    plan.close()


def test_sizes_that_are_not_powers_of_two_and_invalid_arguments():
    t, z = [2e-9, 3e-9], [1e-9, 4e-9]
    M_host = W.make_texture("random", (2, 10, 21), 8e5, seed=114)
    plan = binding.MultiLayerPlan(21, 10, 3e-9, 2e-9, t, z)
    H, _ = run(plan, M_host)
    check(H, ML.multilayer_fft(M_host, 3e-9, 2e-9, t, z), 8e5, False)
    plan.close()
    with pytest.raises(binding.DemagError, match="overlap"):
        binding.MultiLayerPlan(8, 8, 3e-9, 2e-9, [2e-9, 2e-9], [1e-9, 2e-9])
    with pytest.raises(binding.DemagError, match="nlayers"):
        binding.MultiLayerPlan(8, 8, 3e-9, 2e-9, [1e-9] * 33, list(np.arange(33) * 2e-9))
    assert binding.lib().boris_demag_ml_apply(None, None, None, None) == -1
