"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol that
include/flutas.h declares, and rejects bad arguments without touching a GPU."""
import os
import re

import pytest

import paper_2204_08834_b200 as fl
from paper_2204_08834_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "flutas.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(flutas_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = _declared()
    assert len(names) >= 14
    for n in names:
        assert hasattr(binding.lib, n), n          # ctypes resolves the symbol lazily -> AttributeError if absent
    assert sorted(binding.EXPORTS) == names


def test_oracle_library_exports_every_declared_symbol(oracle_mod):
    src = open(os.path.join(ROOT, "oracle", "oracle.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    from oracle import oracle as o
    for n in set(re.findall(r"\b(oracle_[a-z_]+)\s*\(", src)):
        assert hasattr(o._lib, n), n


@pytest.mark.parametrize("args,code", [
    ((33, 32, 32, 1.0, 1.0, 1.0, 0, 1.0, 1.0), 2),      # nx not a power of two
    ((4, 32, 32, 1.0, 1.0, 1.0, 0, 1.0, 1.0), 2),       # nx too small
    ((32, 32, 5000, 1.0, 1.0, 1.0, 1, 1.0, 1.0), 2),    # wall nz above the documented maximum
    ((32, 32, 32, 1.0, 1.0, 1.0, 0, 1e-200, 1.0), 1),   # density outside the documented range
    ((32, 32, 12, 1.0, 1.0, 1.0, 0, 1.0, 1.0), 2),      # periodic nz must be a power of two
    ((32, 32, 1, 1.0, 1.0, 1.0, 1, 1.0, 1.0), 2),       # wall nz >= 2
    ((4096, 32, 32, 1.0, 1.0, 1.0, 0, 1.0, 1.0), 2),    # too large
    ((32, 32, 32, 0.0, 1.0, 1.0, 0, 1.0, 1.0), 1),      # lx
    ((32, 32, 32, 1.0, 1.0, 1.0, 0, -1.0, 1.0), 1),     # rho1
    ((32, 32, 32, 1.0, 1.0, 1.0, 7, 1.0, 1.0), 1),      # bc_z
])
def test_plan_create_rejects_bad_arguments(args, code):
    for ws in ("torch", "library"):
        with pytest.raises(fl.FlutasError) as e:
            fl.Plan(*args, workspace=ws)
        assert e.value.code == code
    if code == 2:
        assert binding.workspace_bytes(args[0], args[1], args[2], args[6]) == 0


def test_workspace_size_query_needs_no_plan_and_no_device():
    """flutas_workspace_bytes: one padded half-spectrum + four fields (+ the wall table), every part 1 KiB aligned"""
    up = lambda b: (b + 1023) // 1024 * 1024
    for (nx, ny, nz) in ((32, 32, 32), (512, 512, 512), (8, 8, 8)):
        spec = 16 * (nx // 2 + 8) * (ny + 1) * nz
        assert binding.workspace_bytes(nx, ny, nz, 0) == up(spec) + 4 * up(8 * nx * ny * nz)
    per, wall = binding.workspace_bytes(256, 256, 128, 0), binding.workspace_bytes(256, 256, 128, 1)
    assert 0 < wall - per <= 0.30 * 8 * 256 * 256 * 128           # the elimination table: about a quarter of a field
    assert binding.workspace_bytes(1024, 1024, 512, 1) < 22 * 2**30
    assert binding.lib.flutas_plan_set_workspace(None, None, 0) == 1
    assert binding.lib.flutas_plan_kernel_symbol(None, 0) is None


def test_null_plan_is_rejected_and_destroy_null_is_noop():
    binding.lib.flutas_plan_destroy(None)
    assert binding.lib.flutas_projection_step(None, None, None, None, None, None, None, 1e-3, None) == 1
    assert binding.lib.flutas_plan_kernel_launches(None) == 0
    assert binding.lib.flutas_plan_workspace_bytes(None) == 0
    assert b"NULL plan" in binding.lib.flutas_last_error()


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    for ws in ("torch", "library"):
        with pytest.raises(fl.FlutasError) as e:
            fl.Plan(32, 32, 32, 1.0, 1.0, 1.0, 0, 1.0, 1.0, workspace=ws)
        assert e.value.code == 4 and "no CPU fallback" in str(e.value)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2204_08834_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inl")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), f
    text = open(os.path.join(ROOT, "workloads.py")).read()          # the shared input generators import neither side
    assert "import oracle" not in text and "from oracle" not in text and "paper_2204_08834_b200" not in text
