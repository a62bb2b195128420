"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/dkd.h declares.
No compute calls (no GPU here); the product path must fail loudly, never fall back to a CPU path."""
import ctypes
import os
import re
import subprocess

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_01757_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "dkd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dkd_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    import paper_2607_01757_b200 as dkd
    syms = declared_symbols()
    assert "dkd_create" in syms and "dkd_extract" in syms and "dkd_destroy" in syms and "dkd_extract_host" in syms
    for s in syms:
        assert getattr(lib, s) is not None, s
    assert sorted(dkd.EXPORTED_SYMBOLS) == syms                  # the binding covers the whole header


def test_header_is_plain_c():
    out = os.path.join(ROOT, "tests", "_hdr_check.o")
    try:
        subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-x", "c", "-c",
                               os.path.join(ROOT, "include", "dkd.h"), "-o", out])
    finally:
        if os.path.exists(out):
            os.remove(out)


def test_library_is_sm100a_with_tma():
    from paper_2607_01757_b200 import build
    path = build.build()
    elf = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True).stdout
    assert "sm_100a" in elf
    full = subprocess.run(["cuobjdump", "-sass", path], capture_output=True, text=True).stdout
    funcs = [f for f in full.split("Function : ")[1:] if "k_nms_tma" in f.split("\n")[0]]
    assert len(funcs) == 16                                      # radius 1..4 x {thr_up > 0, thr_up <= 0} x {S, heat x reliability}
    sass = funcs[0]
    assert "UTMALDG" in sass                                     # TMA tile loads in the NMS kernel
    assert "FMNMX3" in sass                                      # 3-input max of the separable window maximum
    assert "SYNCS" in sass                                       # mbarrier pipeline


@pytest.mark.skipif(torch.cuda.is_available(), reason="CPU-only behaviour")
def test_fails_loudly_without_gpu(lib):
    import paper_2607_01757_b200 as dkd
    with pytest.raises(dkd.DKDError):
        dkd.DKD(1, 64, 64, 16)
    lib.dkd_last_error.restype = ctypes.c_char_p
    lib.dkd_last_error.argtypes = [ctypes.c_void_p]
    assert lib.dkd_destroy(None) == 0                            # NULL is a no-op


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_01757_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "oracle" not in txt.lower(), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2607_01757_b200" not in txt and "libdkd.so" not in txt


def test_static_matcher_limit_is_the_same_in_header_binding_and_readme():
    """DKD_MATCH_STATIC_MAX_RECS (the capacity of dkd_match_static's built-in scratch) is stated in three places."""
    import paper_2607_01757_b200 as dkd
    hdr = open(os.path.join(ROOT, "include", "dkd.h")).read()
    m = re.search(r"#define\s+DKD_MATCH_STATIC_MAX_RECS\s+(\d+)", hdr)
    assert m and int(m.group(1)) == dkd.MATCH_STATIC_MAX_RECS
    assert int(m.group(1)) * 16 == 1 << 20                       # "1 MiB" in the header and the README
    assert str(dkd.MATCH_STATIC_MAX_RECS) in open(os.path.join(ROOT, "README.md")).read()
