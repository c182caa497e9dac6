"""CPU-only checks of the C-ABI boundary: the library builds (nvcc cross-compiles sm_100a without a GPU),
loads, exports every symbol include/bie.h declares, and fails loudly -- never falls back -- without a device."""
import ctypes
import os
import re
import subprocess

import pytest

from paper_2108_01786_b200 import bie, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    return build.build_library()


def _declared():
    src = open(os.path.join(ROOT, "include", "bie.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bie_[a-z_0-9]+)\s*\(", src)))


def test_header_and_binding_agree():
    assert _declared() == sorted(bie.EXPORTS)


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for name in _declared():
        assert hasattr(L, name), name


def test_library_is_sm100a_only(libpath):
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_strerror_and_sizes(libpath):
    assert bie.strerror(0) == "ok"
    assert "aligned" in bie.strerror(-3)
    n, m = 1000, 50
    ws = bie.Context.bie_gmres_workspace_bytes(n, m)
    assert ws >= 8 * (m + 1) * n
    assert bie.Context.bie_solve_workspace_bytes(n, m, False) >= ws + 8 * n * n
    assert bie.Context.bie_solve_workspace_bytes(n, m, True) < 8 * n * n
    assert bie.Context.bie_gmres_workspace_bytes(0, m) == 0


def test_no_cpu_fallback_without_a_device(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(bie.BieError) as e:
        bie.Context(0)
    assert e.value.code == -5


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2108_01786_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "bie_oracle" not in txt, f
