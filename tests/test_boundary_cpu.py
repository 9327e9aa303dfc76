"""Host-side checks that need no GPU: libcwo.so builds, loads, and exports every symbol include/cwo.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1107_5578_b200 import build
    return build.build()


def _declared(header="cwo.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cwo_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_calls_of_the_scope_table():
    names = _declared()
    for must in ("cwo_plan", "cwo_asm", "cwo_fresnel_conv", "cwo_propagate_stack", "cwo_gs",
                 "cwo_plan_workspace_bytes", "cwo_plan_set_workspace", "cwo_plan_set_stream", "cwo_strerror",
                 # SURVEY 8(f) rows f1-f4
                 "cwo_plan_set_offset", "cwo_fresnel_fourier", "cwo_fresnel_shifted", "cwo_plan_set_dst_pitch_xy",
                 "cwo_scale255", "cwo_pls_cgh"):
        assert must in names


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for name in _declared() + _declared("cwo_debug.h"):
        assert hasattr(L, name), name


def test_product_header_has_no_measurement_hooks():
    names = _declared()
    assert not [n for n in names if "debug" in n or "timing" in n or "launch_count" in n]
    src = open(os.path.join(ROOT, "include", "cwo.h")).read()
    assert "EXPERIMENT" not in src and "CWO_OPT_TIMING" not in src


def test_binding_lists_the_same_names(libpath):
    from paper_1107_5578_b200 import api
    assert sorted(api.EXPORTS) == _declared()
    assert sorted(api.DEBUG_EXPORTS) == _declared("cwo_debug.h")
    for name in ("cwo_plan", "cwo_asm", "cwo_fresnel_conv", "cwo_propagate_stack", "cwo_gs"):
        assert callable(getattr(api, name))


def test_no_torch_types_or_cpp_in_the_abi():
    src = open(os.path.join(ROOT, "include", "cwo.h")).read()
    assert "torch" not in src.replace("torch.complex64 element", "") and "std::" not in src and "at::" not in src


def test_strerror_and_argument_checks_without_a_device(libpath):
    L = ctypes.CDLL(libpath)
    L.cwo_strerror.restype = ctypes.c_char_p
    assert L.cwo_strerror(0) == b"ok" and b"workspace" in L.cwo_strerror(-2)
    h = ctypes.c_void_p()
    L.cwo_plan.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.POINTER(ctypes.c_void_p)]
    assert L.cwo_plan(100, 128, 1e-5, 633e-9, ctypes.byref(h)) == -1          # not a power of two
    assert L.cwo_plan(128, 128, -1.0, 633e-9, ctypes.byref(h)) == -1          # pitch <= 0
    assert L.cwo_plan(128, 128, 1e-5, 633e-9, None) == -1
    assert L.cwo_plan(32768, 128, 1e-5, 633e-9, ctypes.byref(h)) == -1        # too large
    L.cwo_plan_workspace_bytes.restype = ctypes.c_size_t
    L.cwo_plan_workspace_bytes.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int]
    assert L.cwo_plan_workspace_bytes(None, 1, 0) == 0


def test_product_path_does_not_reach_the_oracle():
    # the package must not import, call or link anything under oracle/ (and vice versa)
    pkg = os.path.join(ROOT, "paper_1107_5578_b200")
    for d, _, files in os.walk(pkg):
        if os.path.basename(d) == "_build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(d, f)).read()
                assert "import oracle" not in s and "from oracle" not in s and "cwo_oracle" not in s, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libcwo.so" not in s and "include/cwo.h\"" not in s and "import paper_1107_5578_b200" not in s
