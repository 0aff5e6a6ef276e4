"""CPU-side checks of the boundary: libmhd.so builds/loads, exports every symbol include/mhd.h declares, the Python
binding's struct matches the header, and argument checking that needs no device.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mhd.h")


@pytest.fixture(scope="module")
def libpath():
    from paper_1804_03479_b200 import build
    return build.build()


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mhd_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_contract_calls():
    fns = declared_functions()
    for must in ["mhd_create", "mhd_destroy", "mhd_sizes", "mhd_advance", "mhd_advance_host", "mhd_dt_reduce",
                 "mhd_get_stats", "mhd_strerror"]:
        assert must in fns


def test_library_exports_every_declared_symbol(libpath):
    L = C.CDLL(libpath)
    for fn in declared_functions():
        assert hasattr(L, fn), f"{fn} declared in include/mhd.h but not exported"


def test_binding_lists_the_same_names(libpath):
    from paper_1804_03479_b200 import mhd
    assert sorted(mhd.EXPORTS) == declared_functions()


def test_config_struct_matches_header_field_order():
    from paper_1804_03479_b200 import mhd
    src = open(HEADER).read()
    body = src[src.index("typedef struct {"):src.index("} mhd_config;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"\b(?:int|double)\s+([a-z_0-9]+)\s*;", body)
    assert fields == [f[0] for f in mhd.Config._fields_]
    ctype = {"int": C.c_int, "double": C.c_double}
    kinds = re.findall(r"\b(int|double)\s+[a-z_0-9]+\s*;", body)
    assert [ctype[k] for k in kinds] == [f[1] for f in mhd.Config._fields_]


def test_strerror_and_null_argument_checks_need_no_device(libpath):
    from paper_1804_03479_b200 import mhd
    L = mhd.lib()
    assert mhd.strerror(0) == "ok"
    assert "invalid" in mhd.strerror(mhd.EINVAL)
    assert L.mhd_create(None, None) == mhd.EINVAL
    h = C.c_void_p()
    bad = mhd.make_config(g=2)                       # ghost width below the minimum of DESIGN.md R8
    assert L.mhd_create(C.byref(bad), C.byref(h)) == mhd.EINVAL and not h
    bad = mhd.make_config(scheme=mhd.VL, recon=mhd.PPM, g=3)      # VL + PPM needs 4 ghost cells like CTU + PPM
    assert L.mhd_create(C.byref(bad), C.byref(h)) == mhd.EINVAL
    bad = mhd.make_config(limiter=3)
    assert L.mhd_create(C.byref(bad), C.byref(h)) == mhd.EINVAL
    bad = mhd.make_config(scheme=mhd.CTU, recon=mhd.PPM, g=3)
    assert L.mhd_create(C.byref(bad), C.byref(h)) == mhd.EINVAL
    assert L.mhd_destroy(None) == mhd.EINVAL
    assert L.mhd_advance(None, None, None, None, None, None, None, 1, 0.1, 0.1, None) == mhd.EINVAL
    assert L.mhd_launch_count(None) == 0
    # the no-allocation entry point checks its arguments and its size limit before it touches the device
    one = C.c_double()
    ptr = C.cast(C.pointer(one), C.c_void_p)
    assert L.mhd_dt_reduce_noalloc(0, None, ptr, 1, 16, 0, 5.0 / 3.0, 1e-10, 1e-10, 0.1, 0.3, ptr, None) == mhd.EINVAL
    assert L.mhd_dt_reduce_noalloc(0, ptr, ptr, 1, 15, 0, 5.0 / 3.0, 1e-10, 1e-10, 0.1, 0.3, ptr, None) == mhd.EINVAL
    assert L.mhd_dt_reduce_noalloc(0, ptr, ptr, mhd.NOALLOC_MAX_BLOCKS // 16 + 1, 16, 0, 5.0 / 3.0, 1e-10, 1e-10, 0.1, 0.3, ptr, None) == mhd.ELIMIT
    assert "MHD_NOALLOC_MAX_BLOCKS" in mhd.strerror(mhd.ELIMIT)


def test_no_cpu_fallback_create_fails_loudly_without_a_device(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("this box has a GPU")
    from paper_1804_03479_b200 import mhd
    with pytest.raises(mhd.MHDError) as ei:
        mhd.Solver(mhd.make_config())
    assert ei.value.code in (mhd.ECUDA, mhd.ENOMEM)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1804_03479_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".inl", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "mhdref" not in txt, f
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, flags=re.M), f
