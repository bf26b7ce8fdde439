"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/dp.h declares (no GPU needed)."""
import ctypes
import os
import re

from paper_2005_00223_b200 import binding, build


def test_library_builds_and_exports_header_symbols():
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    header = open(os.path.join(os.path.dirname(__file__), "..", "include", "dp.h")).read()
    declared = set(re.findall(r"\b(dp_[a-z_]+)\s*\(", header))
    declared -= {"dp_model"}
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_strerror_and_argument_validation_without_gpu():
    L = binding.lib()
    assert L.dp_strerror(0) == b"ok"
    assert b"box" in L.dp_strerror(-2)
    assert L.dp_workspace_bytes(None, 100, None) == 0
    assert L.dp_create(None, None, None, 0, 6.0, 0.5, None, 0) == -1     # DP_EINVAL before any CUDA call
