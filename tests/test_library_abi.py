"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/pcmd.h declares; host-side argument checks that need no GPU; separation of the
oracle and the CUDA path."""
import ctypes as C
import os
import re

import numpy as np

import paper_1904_00011_b200.build as B
from paper_1904_00011_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_every_declared_symbol():
    path = B.build()
    L = C.CDLL(path)
    names = binding.exported_symbols()
    assert {"pcmd_create", "pcmd_destroy", "pcmd_simulate", "pcmd_hess", "pcmd_loglike",
            "pcmd_evaluate_host"} <= set(names)
    for n in names:
        assert hasattr(L, n), n


def test_struct_layouts_match_header():
    assert C.sizeof(binding.HessStats) == 32 and binding.STATS_DTYPE.itemsize == 32
    assert C.sizeof(binding.HessSpec) == 56
    assert C.sizeof(binding.Params) == 48


def test_strerror_and_null_arguments():
    L = binding.lib()
    assert L.pcmd_strerror(0) == b"ok"
    assert L.pcmd_strerror(-2).startswith(b"expected star count")
    ctx = C.c_void_p()
    assert L.pcmd_create(C.byref(ctx), None) == -1          # PCMD_EINVAL before any CUDA call
    assert L.pcmd_hess_bins_total(None) == 0
    assert L.pcmd_launch_count(None) == 0


def test_oracle_and_cuda_path_share_no_code():
    pk = os.path.join(ROOT, "paper_1904_00011_b200")
    for dirpath, _, files in os.walk(pk):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|#include\s+\"[^\"]*oracle", src, re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1904_00011_b200" not in src.replace("under paper_1904_00011_b200/", "") \
                .replace("from paper_1904_00011_b200 (the CUDA path)", "") or f.endswith((".h", ".py")), f
            assert not re.search(r"^\s*(from|import)\s+paper_1904_00011_b200", src, re.M), f
    for f in ("workloads/synthetic.py",):
        src = open(os.path.join(ROOT, f)).read()
        assert not re.search(r"^\s*(from|import)\s+(oracle|paper_1904_00011_b200)", src, re.M)
