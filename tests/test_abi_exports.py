"""CPU-only: the C-ABI library builds, loads, and exports every symbol include/clover.h declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "clover.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(\w+)\s*\([^;{]*\)\s*;", src)))


def test_library_exports_every_declared_symbol():
    from paper_1405_4524_b200 import build
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert {"clover_create", "clover_destroy", "dslash_apply", "clover_solve", "clover_solve_host", "noise_fill",
            "clover_bench_kernel", "clover_get_stats", "clover_last_error", "stochastic_operators", "stochastic_correlator", "stochastic_fill", "timeslice_norm2"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_binding_lists_the_same_names():
    from paper_1405_4524_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()


def test_no_device_fails_loudly():
    """Without a GPU every entry point reports CLOVER_ECUDA / raises: there is no CPU fallback."""
    import pytest
    import torch
    from paper_1405_4524_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(binding.CloverError):
        binding.noise_fill((4, 4, 4, 8), 1, 1)
    out = ctypes.c_void_p()
    lib = ctypes.CDLL(binding.LIB_PATH)
    lib.clover_last_error.restype = ctypes.c_char_p
    dims = (ctypes.c_int * 4)(4, 4, 4, 8)
    rc = lib.noise_fill(ctypes.c_void_p(16), 64, dims, ctypes.c_uint64(1), 1, 0, 0, ctypes.c_double(1.0), None)
    assert rc == -2 and b"no CPU fallback" in lib.clover_last_error(None)
    bad = (ctypes.c_int * 4)(4, 3, 4, 8)
    assert lib.noise_fill(ctypes.c_void_p(16), 64, bad, ctypes.c_uint64(1), 1, 0, 0, ctypes.c_double(1.0), None) == -1
