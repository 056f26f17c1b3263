"""CPU-only checks of the boundary: libtdx.so loads and exports every symbol include/tdx.h declares, the host-only
entry points work, and (without a device) the solve path fails loudly instead of falling back."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle as orc
from paper_1812_01178_b200 import binding as tdx

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "tdx.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tdx_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_all_exported_and_bound():
    names = declared_symbols()
    assert len(names) >= 14
    L = tdx.lib()
    for n in names:
        assert hasattr(L, n), "libtdx.so does not export %s" % n
    assert sorted(tdx.EXPORTS) == names


def test_version_and_status_strings():
    assert "tdx" in tdx.version()
    assert tdx.status_string(0) == "TDX_OK" and tdx.status_string(-2) == "TDX_ERR_BAD_PARTITION"


@pytest.mark.parametrize("n,P", [(12, 4), (32, 4), (288, 16), (288, 32), (100, 7), (4096, 128), (17, 8), (9, 4), (64, 1)])
def test_partition_bounds_bit_exact_vs_oracle(n, P):
    assert np.array_equal(tdx.partition_bounds(n, P), orc.partition_bounds(n, P))


def test_partition_bounds_errors():
    with pytest.raises(tdx.TdxError) as e:
        tdx.partition_bounds(7, 4)
    assert e.value.status == tdx.ERR_BAD_PARTITION
    with pytest.raises(tdx.TdxError):
        tdx.partition_bounds(64, 0)
    with pytest.raises(tdx.TdxError):
        tdx.partition_bounds(1, 1)


def test_grid_create_argument_errors_precede_device_use():
    f = np.linspace(0, 1, 9)
    bad = f.copy(); bad[3] = bad[2]
    with pytest.raises(tdx.TdxError) as e:
        tdx.Grid(8, 8, 8, bad, f, f)
    assert e.value.status == tdx.ERR_INVALID_ARG
    with pytest.raises(tdx.TdxError) as e:
        tdx.Grid(1, 8, 8, np.linspace(0, 1, 2), f, f)
    assert e.value.status == tdx.ERR_INVALID_ARG


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    f = np.linspace(0, 1, 9)
    with pytest.raises(tdx.TdxError) as e:
        tdx.Grid(8, 8, 8, f, f, f)
    assert e.value.status == tdx.ERR_CUDA and "no CPU fallback" in str(e.value)


def test_product_package_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1812_01178_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), fn
                assert "liboracle" not in src and "oracle.c" not in src, fn
