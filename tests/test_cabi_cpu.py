"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/dpi.h declares, validates
arguments before touching a device, and fails loudly (no CPU fallback) when there is no GPU."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

from paper_2606_21101_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "dpi.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dpi_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    declared = _declared_functions()
    assert len(declared) >= 15
    assert sorted(binding.EXPORTS) == declared
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.dpi_version() == 100
    assert lib.dpi_status_string(2) == b"DPI_ERR_UNSUPPORTED"


def test_no_torch_types_in_the_boundary():
    for header in ("dpi.h", "dpi_nongemm.h"):
        text = open(os.path.join(ROOT, "include", header)).read()
        assert "torch" not in re.sub(r"/\*.*?\*/", "", text, flags=re.S).lower()
        assert "cuda_runtime" not in text


def test_library_exports_every_symbol_of_the_nongemm_header(lib):
    from paper_2606_21101_b200 import nongemm
    text = open(os.path.join(ROOT, "include", "dpi_nongemm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = sorted(set(re.findall(r"\b(dpi_[a-z_0-9]+)\s*\(", text)))
    assert sorted(nongemm.EXPORTS) == declared
    for name in declared:
        assert hasattr(lib, name), name


def test_nongemm_argument_validation_and_host_schedule_need_no_device(lib):
    from paper_2606_21101_b200 import nongemm
    nongemm._lib()
    buf = np.zeros(64, dtype=np.float32)
    p = buf.ctypes.data - buf.ctypes.data % 16 + 16
    assert lib.dpi_fm_interaction(None, 0, 4, 2, 4, 0, p, None, None) == 1          # NULL x
    assert lib.dpi_fm_interaction(p, 0, 4, 2, 4, 0, None, None, None) == 1          # neither y nor v
    assert lib.dpi_fm_interaction(p, 0, 4, 2, 3, 0, p, None, None) == 2             # 12-byte field
    assert lib.dpi_fm_interaction(p, 0, 4, 2, 4, 6, p, None, None) == 1             # x_ld < T*D
    assert lib.dpi_fm_interaction(p, 9, 4, 2, 4, 0, p, None, None) == 1             # dtype
    assert lib.dpi_fm_interaction(p, 0, 0, 2, 4, 0, p, None, None) == 0             # B = 0: nothing to do, no launch
    assert lib.dpi_cross_combine(p, p, None, None, p, 0, 2, 4, None) == 1
    assert lib.dpi_cross_combine(p, p, p, None, p, 0, 2, 3, None) == 2
    assert lib.dpi_cross_combine(p + 4, p, p, None, p, 0, 2, 4, None) == 1          # misaligned
    assert lib.dpi_bias_act(p, None, p, 0, 2, 4, 5, None) == 1                      # unknown activation
    assert lib.dpi_bias_act(p, None, p, 1, 2, 4, 1, None) == 2                      # 8-byte fp16 row
    assert b"dpi_bias_act" in lib.dpi_last_error()
    assert nongemm.bfs_schedule(2, 4) == [(1, 0), (0, 0), (1, 1), (0, 1), (1, 2), (1, 3)]   # PAPER.md Alg. 2, by hand
    assert nongemm.bfs_schedule(0, 0) == []
    with pytest.raises(binding.DpiError):
        nongemm.bfs_schedule(-1, 2)
    assert lib.dpi_launcher_run(None, None, 0, None, 0, 2, None) == 1


def _create(lib, T, rows, dims, dtype, B, max_idx):
    rows = np.asarray(rows, dtype=np.int64)
    dims = np.asarray(dims, dtype=np.int32)
    h = ctypes.c_void_p()
    st = lib.dpi_plan_create(T, rows.ctypes.data, dims.ctypes.data, dtype, B, max_idx, ctypes.byref(h))
    return st, h, lib.dpi_last_error().decode()


def test_argument_validation_happens_before_any_device_work(lib):
    assert _create(lib, 0, [1], [16], 0, 4, 10)[0] == 1                      # T < 1
    assert _create(lib, 1, [1], [16], 0, 0, 10)[0] == 1                      # B < 1
    assert _create(lib, 1, [0], [16], 0, 4, 10)[0] == 1                      # empty table
    assert _create(lib, 1, [5], [16], 7, 4, 10)[0] == 1                      # unknown dtype
    assert _create(lib, 1, [5], [16], 0, 4, -1)[0] == 1                      # negative capacity
    assert _create(lib, 1, [5], [16], 0, 4, 2 ** 31)[0] == 1                 # N must stay below 2^31
    assert _create(lib, 2, [5, 5], [16, 30], 0, 4, 10)[0] == 2               # mixed dims are fine, a 120-byte row is not
    assert _create(lib, 1, [5], [3], 0, 4, 10)[0] == 2                       # 12-byte rows
    assert _create(lib, 1, [5], [4], 1, 4, 10)[0] == 2                       # 8-byte fp16 rows
    assert _create(lib, 1, [5], [256], 0, 4, 10)[0] == 2                     # 1 KiB rows
    st, _, msg = _create(lib, 2049, [5] * 2049, [16] * 2049, 0, 1, 10)
    assert st == 2 and "DPI_MAX_TABLES" in msg
    assert lib.dpi_plan_destroy(None) == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful on a box without a GPU")
def test_no_gpu_means_loud_failure_not_cpu_fallback(lib):
    st, h, msg = _create(lib, 1, [5], [16], 0, 4, 10)
    assert st == 4 and not h.value
    assert "no CPU fallback" in msg
    with pytest.raises(binding.DpiError):
        binding.Plan([5], 16, 0, 4, 10)


def test_missing_library_is_loud(tmp_path):
    with pytest.raises(binding.DpiLibraryMissing):
        binding.load_library(str(tmp_path / "libdpi.so"))


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_21101_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".inc", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert not re.search(r"#\s*include[^\n]*oracle", src), f
                assert "liboracle" not in src, f
    src = (open(os.path.join(ROOT, "oracle", "__init__.py")).read()
           + open(os.path.join(ROOT, "oracle", "dpi_oracle.c")).read())
    assert "paper_2606_21101_b200 import" not in src and "import paper_2606_21101_b200" not in src
    assert "dpi.h" not in src and "dpi_internal" not in src
