"""The C-ABI library loads without a GPU and exports every symbol include/gravidy_b200.h declares; calls that
need a device fail loudly (no CPU fallback).  No compute is run here."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = ROOT / "include" / "gravidy_b200.h"


@pytest.fixture(scope="module")
def binding():
    from paper_1702_00440_b200 import build, binding
    build.build_library()
    binding.load()
    return binding


def declared_symbols():
    text = HEADER.read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"GD_API[^;(]*?\b(gd_\w+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for must in ("gd_init", "gd_predict", "gd_force_jerk", "gd_correct_and_timestep", "gd_next_block", "gd_energy"):
        assert must in names


def test_library_exports_every_declared_symbol(binding):
    lib = C.CDLL(str(binding.LIB_PATH))
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in the header but not exported"


def test_binding_covers_every_declared_symbol(binding):
    assert sorted(binding.SYMBOLS) == declared_symbols()


def test_version_and_workspace_size(binding):
    assert "sm_100a" in binding.version()
    assert binding.workspace_bytes(0) == 0
    b1, b2 = binding.workspace_bytes(1024), binding.workspace_bytes(1025)
    assert b1 > 1024 * 184 and b2 > b1 and b1 % 256 == 0
    # C5 fits one GPU with a wide margin (180 GB HBM)
    assert binding.workspace_bytes(1048577) < 2 << 30


def test_bad_arguments_are_rejected_before_any_cuda_call(binding):
    lib = binding.load()
    h = C.c_void_p(None)
    assert lib.gd_init(C.byref(h), 0, 1, 1, 1, 1e-4, 0.01, 256, 1 << 20, None) == binding.GD_EINVAL
    assert lib.gd_init(C.byref(h), 16, None, 1, 1, 1e-4, 0.01, 256, 1 << 20, None) == binding.GD_EINVAL
    assert lib.gd_init(C.byref(h), 16, 1, 1, 1, 1e-4, -1.0, 256, 1 << 30, None) == binding.GD_EINVAL
    assert lib.gd_init(C.byref(h), 16, 1, 1, 1, 1e-4, 0.01, 256, 16, None) == binding.GD_EINVAL      # too small
    assert lib.gd_init(C.byref(h), 16, 1, 1, 1, 1e-4, 0.01, 264, 1 << 30, None) == binding.GD_EINVAL  # misaligned
    assert b"gd_init" in lib.gd_last_error(None)
    # ranges: n beyond the capacity of the active-set scan (2^25); a softening so small that eps^3 underflows the self pair
    assert lib.gd_init(C.byref(h), (1 << 25) + 1, 1, 1, 1, 1e-4, 0.01, 256, 1 << 40, None) == binding.GD_EINVAL
    assert lib.gd_init(C.byref(h), 16, 1, 1, 1, 1e-150, 0.01, 256, 1 << 30, None) == binding.GD_EINVAL
    assert b"eps" in lib.gd_last_error(None)
    assert lib.gd_predict(None, 0.0) == binding.GD_EINVAL
    lib.gd_destroy(None)


def test_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import numpy as np
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.Hermite(np.ones(4), np.zeros((4, 3)), np.zeros((4, 3)), 1e-4, 0.01)
    with pytest.raises(binding.GravidyError):
        binding.fp64_peak_probe(16)
