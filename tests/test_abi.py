"""CPU-only checks of the boundary: libovl.so builds for sm_100a, loads, and exports every symbol include/ovl.h
declares; the Python binding declares exactly the same set; the product package does not touch oracle/."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ovl.h")
PKG = os.path.join(ROOT, "paper_1510_06897_b200")


def header_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ovl_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1510_06897_b200 import build
    return build.build_library()


def test_header_declares_the_boundary():
    fns = header_functions()
    for must in ["ovl_create", "ovl_destroy", "ovl_dw", "ovl_sign", "ovl_overlap", "ovl_cg", "ovl_set_chebyshev",
                 "ovl_set_deflation", "ovl_dw_native"]:
        assert must in fns


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for fn in header_functions():
        assert hasattr(lib, fn), fn
    lib.ovl_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.ovl_version()


def test_binding_signatures_match_header(lib_path):
    from paper_1510_06897_b200 import binding
    assert sorted(binding.SIGNATURES) == header_functions()
    lib = binding.load_library()
    for name in binding.SIGNATURES:
        assert callable(getattr(binding, name)), name
        assert getattr(lib, name).argtypes is not None


def test_library_is_sm100a_only(lib_path):
    out = subprocess.run(["cuobjdump", "-lelf", lib_path], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_host_side_argument_checks_without_gpu(lib_path):
    """Pure host logic reachable without a device: size arithmetic and EINVAL paths that return before any CUDA call."""
    from paper_1510_06897_b200 import binding as B
    lib = B.load_library()
    dims = (ctypes.c_int * 4)(20, 20, 20, 64)
    v = 20 * 20 * 20 * 64
    got = lib.ovl_device_bytes(dims, B.OVL_F64, B.OVL_RECON18, 50)
    assert got >= v * (4 * 9 * 16 + (50 + 10) * 12 * 16)
    assert lib.ovl_device_bytes(dims, 7, B.OVL_RECON18, 0) == 0
    bad = (ctypes.c_int * 4)(4, 4, 1, 4)
    assert lib.ovl_device_bytes(bad, B.OVL_F64, B.OVL_RECON18, 0) == 0
    # the workspace plan: monotone in every capacity, >= the sum of its big pieces, 0 for bad capacities
    w0 = lib.ovl_workspace_bytes(dims, B.OVL_F64, B.OVL_RECON18, 0, 1, 0)
    assert w0 == lib.ovl_device_bytes(dims, B.OVL_F64, B.OVL_RECON18, 0)
    assert w0 >= v * (4 * 9 * 16 + 10 * 12 * 16 + 2 * 12 * 16)
    w50 = lib.ovl_workspace_bytes(dims, B.OVL_F64, B.OVL_RECON18, 50, 1, 0)
    assert w50 - w0 >= 50 * v * 12 * 16 and w50 == got
    w12 = lib.ovl_workspace_bytes(dims, B.OVL_F64, B.OVL_RECON18, 50, 12, 0)
    assert w12 - w50 >= (8 * 11 + 2 * 12) * v * 12 * 16
    we = lib.ovl_workspace_bytes(dims, B.OVL_F64, B.OVL_RECON18, 50, 12, 104)
    assert we - w12 >= 5 * 104 * v * 12 * 16
    assert lib.ovl_workspace_bytes(dims, B.OVL_F32, B.OVL_RECON12, 0, 1, 0) < w0 // 2 + 2 * v * 12 * 16
    for bad_caps in [(-1, 1, 0), (0, 0, 0), (0, 13, 0), (0, 1, -1), (0, 1, 129)]:
        assert lib.ovl_workspace_bytes(dims, B.OVL_F64, B.OVL_RECON18, *bad_caps) == 0
    ctx = ctypes.c_void_p()
    assert lib.ovl_create_ws(ctypes.byref(ctx), dims, ctypes.c_void_p(16), B.OVL_F64, B.OVL_RECON18, 0, 1, 0, None, 0, None) == B.OVL_EINVAL
    assert lib.ovl_create(ctypes.byref(ctx), bad, ctypes.c_void_p(16), B.OVL_F64, B.OVL_RECON18, None) == B.OVL_EINVAL
    assert lib.ovl_create(ctypes.byref(ctx), dims, None, B.OVL_F64, B.OVL_RECON18, None) == B.OVL_EINVAL
    # the t-split group: slab arithmetic is refused before any CUDA call
    grp = ctypes.c_void_p()
    streams = (ctypes.c_void_p * 16)()
    for nslabs in (0, 17, 3, 64):  # out of range; Lt = 64 not divisible by 3; Lt / nslabs < 2
        assert lib.ovl_group_create(ctypes.byref(grp), dims, nslabs, ctypes.c_void_p(16), B.OVL_F64, B.OVL_RECON18, streams, None) == B.OVL_EINVAL
    assert lib.ovl_group_create(ctypes.byref(grp), dims, 2, None, B.OVL_F64, B.OVL_RECON18, streams, None) == B.OVL_EINVAL
    assert lib.ovl_group_destroy(None) == B.OVL_EINVAL and lib.ovl_group_slabs(None) == 0
    assert lib.ovl_group_last_error(None) == b"null group"
    assert lib.ovl_destroy(None) == B.OVL_EINVAL
    assert lib.ovl_last_error(None) == b"null context"


def test_product_never_references_the_oracle():
    """The CUDA path and its binding share no code with oracle/ and never import it (only tests/, smoke() and
    bench.py's cpu_baseline / --impl reference legs may)."""
    for dirpath, _, files in os.walk(PKG):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, flags=re.M), f
                assert "ovl_oracle" not in txt and "libovl_oracle" not in txt, f
    hdr = open(HEADER).read()
    assert "oracle" not in hdr.lower()
