"""The C-ABI library loads and exports every symbol include/boris_demag.h declares (no GPU needed)."""
import ctypes
import os
import re

import pytest

from paper_2008_02478_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "boris_demag.h")
HEADER_LLG = os.path.join(ROOT, "include", "boris_llg.h")
HEADER_MICRO = os.path.join(ROOT, "include", "boris_micro.h")
HEADER_F64 = os.path.join(ROOT, "include", "boris_demag_f64.h")
HEADER_ML = os.path.join(ROOT, "include", "boris_demag_ml.h")
HEADER_NOALLOC = os.path.join(ROOT, "include", "boris_demag_noalloc.h")


@pytest.fixture(scope="session", autouse=True)
def built_library():
    build.build()


def declared_symbols():
    text = open(HEADER).read() + open(HEADER_LLG).read() + open(HEADER_MICRO).read() + open(HEADER_F64).read() + open(HEADER_ML).read() + open(HEADER_NOALLOC).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(boris_(?:demag|llg|micro)_\w+)\s*\(", text)))


def test_header_declares_the_entry_points_the_north_star_names():
    syms = declared_symbols()
    for name in ("boris_demag_plan_create", "boris_demag_apply", "boris_demag_energy", "boris_demag_plan_destroy",
                 "boris_demag_last_error", "boris_demag_plan_info", "boris_demag_apply_host"):
        assert name in syms


def test_library_exports_every_declared_symbol():
    lib = ctypes.CDLL(binding.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_header_has_no_torch_or_cxx_types():
    text = open(HEADER).read()
    assert "torch" not in text and "at::" not in text and "std::" not in text
    assert 'extern "C"' in text


def test_version_and_invalid_arguments():
    assert "sm_100a" in binding.version()
    L = binding.lib()
    for bad in [(2048, 4, 1), (4, 1025, 1), (4, 4, 1024), (0, 4, 1), (4, -2, 1), (4, 4, 0)]:
        assert not L.boris_demag_plan_create(*bad, 1e-9, 1e-9, 1e-9)
        assert "must be in [1," in binding.last_error()
    assert not L.boris_demag_plan_create(4, 4, 1, 0.0, 1e-9, 1e-9)
    assert "positive" in binding.last_error()
    assert L.boris_demag_apply(None, None, None, None) == -1
    assert L.boris_demag_energy(None, None, None, None, None) == -1
    L.boris_demag_plan_destroy(None)


def test_no_cpu_fallback_plan_create_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(binding.DemagError, match="CUDA|cuda"):
        binding.DemagPlan(32, 32, 1, 5e-9, 5e-9, 3e-9)


def test_product_package_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2008_02478_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".h", ".cu", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2008_02478_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "``paper_2008_02478_b200/``", ""), f
