"""The C-ABI library builds here (nvcc cross-compiles sm_100a without a GPU), loads, and exports every
function include/ut_compass.h declares.  No compute call is made: there is no GPU on this box."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ut_compass.h")


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)          # comments
    text = re.sub(r"^\s*#.*$", " ", text, flags=re.M)           # preprocessor lines
    text = re.sub(r"typedef\s+struct\s*\{.*?\}\s*\w+\s*;", " ", text, flags=re.S)
    names = re.findall(r"\b(?:int32_t|uint32_t|size_t|void|const\s+char\s*\*)\s+(\w+)\s*\(", text)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    from paper_2002_11529_b200 import build
    path = build.build()
    assert os.path.exists(path)
    return path


def test_header_declares_the_hot_path_calls():
    names = declared_functions()
    assert "ut_decode" in names and "compass_track" in names
    assert len(names) >= 10


def test_library_exports_every_declared_symbol(lib):
    handle = ctypes.CDLL(lib)
    missing = [n for n in declared_functions() if not hasattr(handle, n)]
    assert not missing, f"declared in ut_compass.h but not exported: {missing}"


def test_exports_are_plain_c_symbols(lib):
    out = subprocess.run(["nm", "-D", "--defined-only", lib], capture_output=True, text=True, check=True).stdout
    syms = {line.split()[-1] for line in out.splitlines() if line.strip()}
    for n in declared_functions():
        assert n in syms                                          # unmangled: extern "C"


def test_binding_names_match_the_header(lib):
    from paper_2002_11529_b200 import binding as B
    assert sorted(B.EXPORTS) == declared_functions()
    assert B.ut_version().startswith("ut-compass-b200")
    for n in ("ut_decode", "compass_track", "ut_geometry_upload", "compass_config_default"):
        assert callable(getattr(B, n))


def test_built_for_sm_100a_only(lib):
    out = subprocess.run(["cuobjdump", "-lelf", lib], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_host_argument_checks_need_no_gpu(lib):
    """Host-detected errors are returned before any CUDA call."""
    from paper_2002_11529_b200 import binding as B
    L = ctypes.CDLL(lib)
    L.ut_decode.restype = ctypes.c_int32
    L.compass_track.restype = ctypes.c_int32
    assert L.ut_decode(None, None, 1, None, None, None, None) == -1            # UT_ERR_NULL
    assert L.compass_track(None, None, None, None, 1, None, None, None) == -1
    cfg = B.compass_config()
    g = B.ut_geometry()
    L.compass_config_default.restype = ctypes.c_int32
    L.compass_config_default.argtypes = [ctypes.c_float, ctypes.c_float, ctypes.c_int32, ctypes.c_int32,
                                         ctypes.c_void_p, ctypes.c_void_p]
    assert L.compass_config_default(-1.0, 1.0, 3, 16, ctypes.byref(g), ctypes.byref(cfg)) == -2   # UT_ERR_ARG
    g.layer_z[:] = [2327.5, 2372.5, 2597.5, 2642.5]
    assert L.compass_config_default(2000.0, 1.0, 3, 16, ctypes.byref(g), ctypes.byref(cfg)) == 0
    import synth
    p = synth.make_compass_params()
    assert [cfg.win_half[i] for i in range(4)] == list(p.win_half)
    assert cfg.max_slope == p.max_slope and cfg.kappa == p.kappa and cfg.z_mag == p.z_mag
