"""CPU-side checks of the boundary: libnb.so builds, loads and exports every symbol that
include/nb.h declares; without a GPU every entry point fails loudly (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1207_2367_b200 as nbmod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "nb.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nb_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported():
    names = _declared()
    assert len(names) >= 20 and "nb_force" in names and "nb_correct_and_step" in names
    L = ctypes.CDLL(nbmod.lib_path() if os.path.exists(nbmod.lib_path()) else nbmod.lib()._name)
    for n in names:
        assert hasattr(L, n), "libnb.so does not export %s" % n


def test_binding_mirrors_header():
    assert nbmod.exported_symbols() == _declared()
    for n in _declared():
        assert hasattr(nbmod, n), "binding lacks %s" % n


def test_north_star_calls_present():
    for n in ("nb_init", "nb_predict", "nb_force", "nb_correct_and_step", "nb_energy"):
        assert n in _declared()


def test_version_string():
    assert "sm_100a" in nbmod.nb_version()


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less box")
    z = np.zeros((4, 3)); m = np.ones(4)
    with pytest.raises(nbmod.NBError) as e:
        nbmod.nb_init(z, z, m, 1e-3, 0.45)
    assert e.value.code == nbmod.nb.NB_ECUDA
    with pytest.raises(RuntimeError):
        nbmod.NBody(z, z, m, 1e-3, 0.45)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1207_2367_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower(), (dirpath, f)


def test_paper_flop_convention_is_consistent():
    """tests/golden/paper_flop_convention.txt: the printed counts add up, Eq. 27 gives the
    printed mixed peak, and bench.py quotes Tflop/s in exactly that convention."""
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_flop_convention.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                vals[k] = float(v)
    assert vals["dp_ops_per_pair"] + vals["sp_ops_per_pair"] == vals["flops_per_pair"] == 97
    r_peak = (vals["sp_ops_per_pair"] * vals["S_peak_gflops"] + vals["dp_ops_per_pair"] * vals["D_peak_gflops"]) / vals["flops_per_pair"]
    assert abs(r_peak - vals["R_peak_gflops"]) < 1.0                       # Eq. 27: "~950 GFLOPS"
    assert abs(vals["reported_gflops_per_gpu"] / r_peak - 0.42) < 0.03      # "around 40% of the claimed peak"
    import bench
    assert bench.FLOPS_PER_PAIR_PAPER == vals["flops_per_pair"]
