"""CPU-side checks of the C-ABI boundary: the library builds, loads, and exports every symbol that
include/ca.h declares; struct layouts agree; argument validation that needs no GPU."""
import ctypes as C
import os
import re

import pytest

from paper_2303_08123_b200 import binding, build, workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def _declared():
    src = open(os.path.join(ROOT, "include", "ca.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ca_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(binding.EXPORTS)


def test_workspace_bytes_and_validation(lib):
    assert lib.ca_workspace_bytes(0, 32, 32, 32, 10) == 0
    assert lib.ca_workspace_bytes(1, 2, 32, 32, 10) == 0
    assert lib.ca_workspace_bytes(1, 32, 32, 32, 65) == 0
    n = 64 * 64 ** 3
    need = lib.ca_workspace_bytes(64, 64, 64, 64, 10)
    assert need >= 29 * n and need < 29 * n * 1.1 + (1 << 22)       # 29 B/site resident + small tables


def test_create_rejects_bad_arguments_without_a_gpu(lib):
    p = binding.make_params(workloads.default_params())
    ctx = C.c_void_p()
    assert lib.ca_create(C.byref(ctx), 1, 2, 8, 8, C.byref(p), 10, None, 0, None) == binding.CA_EINVAL
    bad = binding.make_params(workloads.default_params(**{"lambda": [0.2, 0.05, 0.1]}))
    assert lib.ca_create(C.byref(ctx), 1, 8, 8, 8, C.byref(bad), 10, None, 0, None) == binding.CA_EINVAL
    assert b"lambda" in lib.ca_last_error(None)
    assert lib.ca_create(C.byref(ctx), 1, 8, 8, 8, C.byref(p), 10, None, 0, None) == binding.CA_EINVAL   # no workspace
    assert ctx.value is None


def test_struct_layouts():
    assert C.sizeof(binding.CaParams) == 4 * (2 + 3 + 3 + 12 + 5 + 4 + 4 + 4 + 4 + 2 + 2 + 1 + 1 + 1)      # ... + well_mixed_medium
    assert C.sizeof(binding.CaInit) == 24


def test_product_never_imports_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2303_08123_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "ca_oracle" not in txt, f
