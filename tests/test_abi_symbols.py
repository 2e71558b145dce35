"""The C-ABI library loads and exports every symbol include/mpmi.h declares (no compute, no GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "mpmi.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mpmi_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_1906_02318_b200 import build
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert len(names) == 18, names
    for name in names:
        assert hasattr(lib, name), name


def test_binding_names_match_header():
    from paper_1906_02318_b200 import mpmi
    assert sorted(mpmi.EXPORTS) == _declared()
    assert ctypes.sizeof(mpmi.Result) == 56


def test_errors_without_gpu_are_statuses_not_crashes():
    """mpmi_create validates before touching CUDA; on a box without a GPU it returns a status."""
    from paper_1906_02318_b200 import mpmi
    lib = mpmi.load_library()
    assert lib.mpmi_create(None, None) == mpmi.ERR_INVALID
    assert lib.mpmi_strerror(mpmi.ERR_INVALID) == b"invalid argument"
    assert lib.mpmi_strerror(0) == b"ok"
    import numpy as np
    import workloads as W
    w = W.make("C1")
    bad = dict(vars(w)); bad["N"] = 0
    try:
        mpmi.Context(bad)
        assert False
    except mpmi.MpmiError as e:
        assert e.status == mpmi.ERR_INVALID
    bad = dict(vars(w)); bad["K"] = np.full((8, 8), np.nan, np.float32)
    try:
        mpmi.Context(bad)
        assert False
    except mpmi.MpmiError as e:
        assert e.status == mpmi.ERR_INVALID and "non-finite" in str(e)
    bad = dict(vars(W.make("C3"))); bad["grid_counts"] = np.array([10, 10], np.int32)
    try:
        mpmi.Context(bad)
        assert False
    except mpmi.MpmiError as e:
        assert e.status == mpmi.ERR_INVALID and "grid" in str(e)
