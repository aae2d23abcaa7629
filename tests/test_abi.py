"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/p3t.h declares.

No compute call is made here (there is no GPU in the CPU test run): only the build, the symbol
table, the host-only sizing function and the layering rules (product never touches oracle/).
"""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1506_04553_b200 import build

    return build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "p3t.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(p3t_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    names = _declared_symbols()
    for must in ("p3t_create", "p3t_destroy", "p3t_set_params", "p3t_load_particles", "p3t_build_tree",
                 "p3t_eval_soft", "p3t_get_acc_pot", "p3t_get_neighbours", "p3t_get_neighbour_counts",
                 "p3t_get_stats", "p3t_eval_direct", "p3t_workspace_bytes", "p3t_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/p3t.h but not exported"


def test_binding_lists_the_same_symbols(libpath):
    from paper_1506_04553_b200 import binding

    assert sorted(binding.SYMBOLS) == _declared_symbols()


def test_workspace_bytes_is_host_only_and_monotone(libpath):
    lib = ctypes.CDLL(libpath)
    f = lib.p3t_workspace_bytes
    f.restype = ctypes.c_size_t
    f.argtypes = [ctypes.c_size_t, ctypes.c_int, ctypes.c_size_t]
    assert f(0, 63, 0) == 0 and f(1024, 31, 0) == 0          # invalid arguments
    a, b, c = f(4096, 30, 0), f(1 << 20, 63, 0), f(1 << 20, 63, 1 << 20)
    assert 0 < a < b < c
    assert c - b >= 12 * (1 << 20) - 4096                            # pairs (8 B) + CSR entries (4 B)
    assert b < 1024 * (1 << 20)                             # < 1 KiB per particle at 1M


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1506_04553_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "p3t_oracle" not in text and "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1506_04553_b200 import" not in text and "libp3t.so" not in text, f


def test_binding_fails_loudly_without_a_gpu(libpath):
    import torch

    from paper_1506_04553_b200 import binding

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.P3T(1024)
