"""boris_demag_energy_noalloc (include/boris_demag_noalloc.h): the energy entry point that allocates nothing — its
reduction scratch is a static device array of the library — against the existing path (boris_demag_energy, whose
scratch belongs to a plan) and the fp64 oracle.  Collected last on purpose (the suite runs with pytest -x).

Two calls in a row share the array: the second call runs on a SMALLER mesh than the first, so stale block sums of the
first call sit behind the ones it writes, and on different data.
"""
import numpy as np
import pytest
import torch

from oracle.energy import demag_energy
from paper_2008_02478_b200 import binding, build
from paper_2008_02478_b200 import workloads as W

TOL_E = 1e-5        # relative, energy against the oracle (tests/test_gpu_parity.py)
TOL_SAME = 1e-12    # against the existing GPU path: both are fp64 sums of the same products in a different order


@pytest.fixture(scope="module", autouse=True)
def cuda_library():
    build.build()
    binding.lib()


def fields(shape, h, seed):
    """M and the field the EXISTING path computes for it, on the device, plus that path's energy."""
    nz, ny, nx = shape
    M_host = W.make_texture("random", shape, 8e5, seed=seed)
    plan = binding.DemagPlan(nx, ny, nz, *h)
    M = torch.from_numpy(M_host).cuda()
    H = torch.empty_like(M)
    plan.apply(M, H)
    E_plan = plan.energy(M, H)
    torch.cuda.synchronize()
    E_plan = float(E_plan.item())
    plan.close()
    return M_host, M, H, E_plan


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path():
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(0)
    h1, h2 = (2e-9, 3e-9, 1e-9), (4e-9, 4e-9, 2e-9)
    # 24576 float4 items = 12 full blocks; then 20 x 12 x 7 x 3 = 5040 values: one partial block, stale sums behind it
    M1h, M1, H1, E1_plan = fields((8, 32, 128), h1, seed=41)
    M2h, M2, H2, E2_plan = fields((7, 12, 20), h2, seed=42)
    E = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    E3 = torch.zeros(1, dtype=torch.float64, device="cuda")
    binding.energy_noalloc(M1, H1, h1, E[0:1])
    binding.energy_noalloc(M2, H2, h2, E[1:2])
    torch.cuda.synchronize()
    E1, E2 = float(E[0].item()), float(E[1].item())
    assert abs(E1 - E1_plan) <= TOL_SAME * abs(E1_plan), (E1, E1_plan)
    assert abs(E2 - E2_plan) <= TOL_SAME * abs(E2_plan), (E2, E2_plan)
    # and against the oracle's energy of the same fields (fp64 on the host)
    for Ev, Mh, Hd, h in ((E1, M1h, H1, h1), (E2, M2h, H2, h2)):
        E_ref = demag_energy(Mh.astype(np.float64), Hd.cpu().numpy().astype(np.float64), h)
        assert abs(Ev - E_ref) <= TOL_E * abs(E_ref), (Ev, E_ref)
    # a repeated call gives the same bits (fixed summation order), whatever the array held before
    # (the module that holds the kernel and the array is loaded by now: free device memory must not move any more)
    free_before = torch.cuda.mem_get_info()[0]
    binding.energy_noalloc(M1, H1, h1, E3)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before            # the call took no device memory
    assert float(E3.item()) == E1


@pytest.mark.gpu
def test_values_that_are_not_a_multiple_of_four_and_rejected_sizes():
    torch.cuda.set_device(0)
    h = (1e-9, 2e-9, 3e-9)
    g = torch.Generator(device="cpu").manual_seed(7)
    n = 3 * 8192 + 8192 - 1                                        # three full blocks, one short of a fourth: 3 trailing values
    M = (torch.rand(n, generator=g) - 0.5).mul_(8e5)
    H = (-0.3 * M + (torch.rand(n, generator=g) - 0.5).mul_(1e5)).cuda()      # M.H mostly of one sign: no cancellation
    M = M.cuda()
    E = torch.zeros(1, dtype=torch.float64, device="cuda")
    binding.energy_noalloc(M, H, h, E)
    torch.cuda.synchronize()
    want = -0.5 * 4e-7 * np.pi * h[0] * h[1] * h[2] * float(np.dot(M.cpu().numpy().astype(np.float64), H.cpu().numpy().astype(np.float64)))
    assert abs(float(E.item()) - want) <= 1e-12 * abs(want)
    L = binding.lib()
    too_many = binding.NOALLOC_MAX_VALUES + 1
    assert L.boris_demag_energy_noalloc(M.data_ptr(), H.data_ptr(), too_many, *h, E.data_ptr(), None) == -1
    assert "BORIS_DEMAG_NOALLOC_MAX_VALUES" in binding.last_error()
    assert L.boris_demag_energy_noalloc(M.data_ptr() + 4, H.data_ptr(), 16, *h, E.data_ptr(), None) == -1
    assert "aligned" in binding.last_error()
    assert L.boris_demag_energy_noalloc(None, H.data_ptr(), 16, *h, E.data_ptr(), None) == -1
    assert L.boris_demag_energy_noalloc(M.data_ptr(), H.data_ptr(), 0, *h, E.data_ptr(), None) == -1
    assert L.boris_demag_energy_noalloc(M.data_ptr(), H.data_ptr(), 16, 0.0, 1e-9, 1e-9, E.data_ptr(), None) == -1
    # the error paths left the array usable
    binding.energy_noalloc(M, H, h, E)
    torch.cuda.synchronize()
    assert abs(float(E.item()) - want) <= 1e-12 * abs(want)


def test_entry_point_is_exported_and_documented():
    import ctypes
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    assert hasattr(ctypes.CDLL(binding.LIB_PATH), "boris_demag_energy_noalloc")
    src = open(os.path.join(root, "paper_2008_02478_b200", "csrc", "boris_demag_noalloc.cu")).read()
    code = "\n".join(line.split("//")[0] for line in src.splitlines())
    assert "cudaMalloc" not in code and "cudaFree" not in code        # the entry point allocates nothing
    assert "static __device__ __align__(256)" in code and "cudaGetSymbolAddress" in code
