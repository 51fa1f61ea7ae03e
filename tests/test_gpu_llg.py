"""GPU parity of the LLG evaluation around the demag path (include/boris_llg.h) with oracle/llg.py."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import llg as O
from paper_2008_02478_b200 import binding, build, workloads as W

pytestmark = pytest.mark.gpu

MU0 = 4e-7 * np.pi
MS, A_EX = 8e5, 1.3e-11


@pytest.fixture(scope="module", autouse=True)
def cuda_library():
    build.build()
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(0)


def unit_field(shape, seed):
    return W.make_texture("vortex" if shape[0] == 1 else "helix", shape, 1.0, seed=seed)     # |m| = 1, fp32


# the last two: more rows than the stage kernel has blocks to spare per row group, plane strides of 16 K and
# 64 K elements (the stencil's +-plane neighbours), and the 2-D row walk of a 256 x 256 film
@pytest.mark.parametrize("shape,h", [((1, 32, 64), (4e-9, 4e-9, 3e-9)), ((8, 16, 32), (3e-9, 3e-9, 2e-9)),
                                     ((3, 10, 6), (4e-9, 5e-9, 3e-9)), ((32, 128, 128), (3e-9, 3e-9, 2e-9)),
                                     ((1, 256, 256), (4e-9, 4e-9, 4e-9))])
def test_effective_field_matches_the_oracle(shape, h):
    nz, ny, nx = shape
    m_host = unit_field(shape, 61)
    Hext = (2e4, -1e4, 3e4)
    plan = binding.DemagPlan(nx, ny, nz, *h)
    solver = binding.LLG(plan, MS, A_EX, 0.02, Hext=Hext)
    m = torch.from_numpy(m_host).cuda()
    H = torch.full_like(m, float("nan"))
    solver.effective_field(m, H)
    torch.cuda.synchronize()
    H_ref = O.effective_field(m_host, h, MS, A_EX, Hext)
    # demag: north_star's 1e-5 Ms.  Exchange: the fp32 differences m[i+1] - m[i] of unit vectors carry an
    # absolute error of 2^-24 each, six of them scaled by 2A / (mu0 Ms h^2)
    tol = 1e-5 * MS + 6 * 2.0 ** -23 * 2 * A_EX / (MU0 * MS * min(h) ** 2)
    assert np.abs(H.cpu().numpy() - H_ref).max() <= tol
    solver.close()
    plan.close()


@pytest.mark.parametrize("shape,h,n", [((1, 16, 32), (4e-9, 4e-9, 3e-9), 10), ((4, 8, 16), (3e-9, 3e-9, 3e-9), 10),
                                       ((2, 5, 7), (4e-9, 4e-9, 4e-9), 10), ((32, 128, 128), (3e-9, 3e-9, 2e-9), 3),
                                       ((1, 256, 256), (4e-9, 4e-9, 4e-9), 5)])
def test_rk4_steps_match_the_oracle(shape, h, n):
    nz, ny, nx = shape
    m_host = unit_field(shape, 62)
    Hext, alpha, dt = (-2e4, 4e3, 0.0), 0.1, 1e-13
    plan = binding.DemagPlan(nx, ny, nz, *h)
    solver = binding.LLG(plan, MS, A_EX, alpha, Hext=Hext)
    m = torch.from_numpy(m_host).cuda()
    solver.rk4(m, dt, n)
    torch.cuda.synchronize()
    ref = m_host.astype(np.float64)
    Khat = O.precompute(shape, h)
    for _ in range(n):
        ref = O.rk4_step(ref, dt, h, MS, A_EX, Hext, O.GAMMA, alpha, Khat)
    got = m.cpu().numpy()
    assert np.abs((got.astype(np.float64) ** 2).sum(0) - 1).max() <= 1e-6
    assert np.abs(got - ref).max() <= 2e-5                      # 40 fp32 evaluations of fields of ~1e6 A/m
    assert np.abs(ref - m_host).max() >= 1e-4 * n               # the steps did move the magnetization
    solver.close()
    plan.close()


def test_single_cubic_cell_follows_the_closed_form_damped_precession():
    """Same closed form as tests/test_oracle_llg.py (N = 1/3 I: the demag field exerts no torque)."""
    h = (2e-9, 2e-9, 2e-9)
    alpha, Hz, th0, dt, n = 0.1, 2e5, 1.0, 5e-14, 400
    plan = binding.DemagPlan(1, 1, 1, *h)
    solver = binding.LLG(plan, MS, A_EX, alpha, Hext=(0.0, 0.0, Hz))
    m = torch.tensor([np.sin(th0), 0.0, np.cos(th0)], dtype=torch.float32).reshape(3, 1, 1, 1).cuda()
    solver.rk4(m, dt, n)
    torch.cuda.synchronize()
    t = n * dt
    mz = np.tanh(alpha * O.GAMMA * Hz / (1 + alpha ** 2) * t + np.arctanh(np.cos(th0)))
    phi = O.GAMMA * Hz * t / (1 + alpha ** 2)
    ref = np.array([np.sqrt(1 - mz ** 2) * np.cos(phi), np.sqrt(1 - mz ** 2) * np.sin(phi), mz])
    assert np.abs(m.cpu().numpy().ravel() - ref).max() <= 2e-5
    solver.close()
    plan.close()


def test_solver_rejects_a_mesh_or_cell_that_differs_from_the_plan():
    plan = binding.DemagPlan(16, 8, 4, 3e-9, 3e-9, 2e-9)
    L = binding.lib()
    assert not L.boris_llg_create(plan._h, 16, 8, 8, 3e-9, 3e-9, 2e-9, MS, A_EX, 0.1, O.GAMMA)
    assert "differ from the mesh" in binding.last_error()
    assert not L.boris_llg_create(plan._h, 16, 8, 4, 3e-9, 4e-9, 2e-9, MS, A_EX, 0.1, O.GAMMA)
    assert "cell sides" in binding.last_error()
    assert not L.boris_llg_create(plan._h, 16, 8, 4, 3e-9, 3e-9, 2e-9, -1.0, A_EX, 0.1, O.GAMMA)
    assert "invalid argument" in binding.last_error()
    assert plan.mesh() == ((16, 8, 4), (3e-9, 3e-9, 2e-9))
    plan.close()
