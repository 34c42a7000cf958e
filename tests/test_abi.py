"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol that
include/flashvan.h declares; shape validation works without touching the device."""
import ctypes
import os
import re

import pytest

from paper_2606_22984_b200 import binding as fv
from paper_2606_22984_b200 import build as fvbuild
from paper_2606_22984_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def library():
    fvbuild.build()
    return fv.lib()


def test_header_symbols_are_exported(library):
    header = open(os.path.join(ROOT, "include", "flashvan.h")).read()
    declared = set(re.findall(r"\b(fv_[a-z_0-9]+)\s*\(", header))
    assert declared == set(fv.SYMBOLS), declared ^ set(fv.SYMBOLS)
    for name in declared:
        assert hasattr(library, name), name


def test_n_weights_matches_generators(library):
    for w in W.CONFIGS.values():
        cfg = fv.make_config(w, 8)
        assert library.fv_n_weights(ctypes.byref(cfg)) == W.n_weights(w)
    bad = fv.make_config(W.CONFIGS["cfg1"], 8)
    bad.d_model = 48
    assert library.fv_n_weights(ctypes.byref(bad)) < 0
    assert library.fv_launch_count() >= 0 and library.fv_kv_bytes(None) == 0


def test_no_cpu_fallback_in_product():
    """The product package never imports the oracle."""
    pkg = os.path.join(ROOT, "paper_2606_22984_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower() or f == "workloads.py", f
