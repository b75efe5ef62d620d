"""The C-ABI libraries load without a GPU and export every symbol the headers declare (no compute calls)."""
import ctypes
import os
import re

import pytest

from paper_1211_3991_b200 import _build, binding, levy

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared(header):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(xy_[a-z0-9_]+)\s*\(", src)))


def test_xy_b200_exports_every_declared_symbol():
    names = declared("xy_b200.h")
    assert set(names) == set(binding.SYMBOLS), set(names) ^ set(binding.SYMBOLS)
    for n in ("xy_graph_load", "xy_pt_create", "xy_sweep", "xy_overrelax", "xy_pt_swap", "xy_measure"):
        assert n in names            # the six calls BASELINE.json north_star names
    L = ctypes.CDLL(_build.build_xy())
    for n in names:
        assert hasattr(L, n), n
    assert binding.xy_abi_version() == 1


def test_xy_levy_exports_every_declared_symbol():
    L = levy.lib()
    for n in declared("xy_levy.h"):
        assert hasattr(L, n), n


def test_no_cpu_fallback_without_device():
    """the product path must fail loudly, not fall back: without a CUDA device graph_load returns XY_ECUDA."""
    import numpy as np
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(binding.XYError) as e:
        binding.xy_graph_load(np.array([0, 1, 2], np.int32), np.array([1, 0], np.int32), np.array([0, 1], np.int32))
    assert e.value.code == binding.XY_ECUDA
    with pytest.raises(binding.XYError):
        binding.Ensemble(np.array([0, 1, 2], np.int32), np.array([1, 0], np.int32), np.array([0, 1], np.int32), [1.0], 1)


def test_product_does_not_import_oracle():
    """neither side imports the other: nothing under the package mentions oracle/, and oracle/ never
    mentions the package."""
    pkg = os.path.join(ROOT, "paper_1211_3991_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                txt = open(os.path.join(d, f)).read()
                assert "import oracle" not in txt and "xy_oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1211_3991_b200" not in txt and "xy_b200" not in txt and "xy_kernels" not in txt, f
