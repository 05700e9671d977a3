"""CPU-side checks of the C-ABI boundary (no compute calls): libfizzy.so builds for sm_100a,
loads without a GPU, exports every symbol include/fizzy.h declares, sizes workspaces, rejects
bad arguments, and fails loudly (FIZZY_ECUDA) when no CUDA device is present."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2502_04189_b200 import build as fz_build
from paper_2502_04189_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    fz_build.build()
    from paper_2502_04189_b200 import binding as b
    return b


def declared_functions():
    text = open(os.path.join(ROOT, "include", "fizzy.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fizzy_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(binding):
    names = declared_functions()
    assert set(names) == set(binding.EXPORTS)
    lib = C.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n


def test_abi_version_matches_the_header(binding):
    text = open(os.path.join(ROOT, "include", "fizzy.h")).read()
    declared = int(re.search(r"#define\s+FIZZY_ABI_VERSION\s+(\d+)", text).group(1))
    assert binding._lib.fizzy_abi_version() == declared == binding.FIZZY_ABI_VERSION


def test_only_sm100a_code_in_the_library(binding):
    import subprocess
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_workspace_bytes_and_validation(binding):
    cfg, _, _, _ = W.make(0)
    n = cfg["nx"] * cfg["ny"] * cfg["nz"]
    b = binding.fizzy_workspace_bytes(cfg)
    assert 20 * 8 * n < b < 40 * 8 * n
    cfg5, _, _, _ = W.make(4, grid=(64, 32, 48), ndrops=1, radius=0.3)
    assert binding.fizzy_workspace_bytes(cfg5) > 0
    for key, val in [("nx", 24), ("ny", 4), ("nz", 3), ("rho1", -1.0), ("eps", 0.0), ("lx", 0.0)]:
        bad = dict(cfg)
        bad[key] = val
        assert binding.fizzy_workspace_bytes(bad) == 0, key
    bad = dict(cfg5)
    bad["zf"] = np.array(cfg5["zf"])[::-1].copy()
    assert binding.fizzy_workspace_bytes(bad) == 0
    bad = dict(cfg5)
    bad["z_wall"] = 0  # stretched grid needs walls
    assert binding.fizzy_workspace_bytes(bad) == 0


def test_null_context_calls_are_safe(binding):
    lib = binding._lib
    assert lib.fizzy_rk3_substep(None, 0, 1.0) == binding.FIZZY_EINVAL
    assert lib.fizzy_destroy(None) == binding.FIZZY_EINVAL
    assert lib.fizzy_launch_count(None) == 0
    assert lib.fizzy_last_error(None) == b"null context"
    assert np.isnan(lib.fizzy_gamma(None))


def test_no_cpu_fallback_without_a_device(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    cfg, _, _, _ = W.make(0)
    with pytest.raises(binding.FizzyError) as e:
        binding.Fizzy(cfg)
    assert e.value.status == binding.FIZZY_ECUDA
    # and straight through the C ABI with a fake (aligned) workspace address
    g, bc, pr, _keep = binding.structs_from_cfg(cfg)
    h = C.c_void_p()
    st = binding._lib.fizzy_create(C.byref(g), C.byref(bc), C.byref(pr), 4096, 1 << 40, None, C.byref(h))
    assert st == binding.FIZZY_ECUDA and not h.value


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2502_04189_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), fn
                assert "fizzy_oracle" not in text and "liborc" not in text, fn


def test_variable_coefficient_entry_points_reject_null_contexts(binding):
    """SURVEY.md 8(f)-4 calls: argument errors come back as status codes without a GPU."""
    lib = C.CDLL(binding.LIB_PATH)
    lib.fizzy_varcoef_workspace_bytes.restype = C.c_size_t
    lib.fizzy_varcoef_workspace_bytes.argtypes = [C.c_void_p]
    assert lib.fizzy_varcoef_workspace_bytes(None) == 0
    lib.fizzy_poisson_solve_varcoef.restype = C.c_int
    lib.fizzy_poisson_solve_varcoef.argtypes = [C.c_void_p] * 5 + [C.c_size_t, C.c_double, C.c_int, C.c_void_p, C.c_void_p]
    assert lib.fizzy_poisson_solve_varcoef(None, None, None, None, None, 0, 1e-10, 10, None, None) == binding.FIZZY_EINVAL
    lib.fizzy_set_pressure_solver.restype = C.c_int
    lib.fizzy_set_pressure_solver.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_size_t, C.c_double, C.c_int]
    assert lib.fizzy_set_pressure_solver(None, 1, None, 0, 1e-10, 10) == binding.FIZZY_EINVAL
