"""-m "not gpu": the C-ABI library builds for sm_100a, loads without a GPU and exports every symbol
that include/metad.h declares; host-side argument checks that need no device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2510_06873_b200 import build, metad
    build.build()
    return metad.load()


def test_library_exports_every_declared_symbol(lib):
    from paper_2510_06873_b200 import metad
    hdr = open(os.path.join(ROOT, "include", "metad.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(metad_[a-z0-9_]+)\s*\(", hdr))
    assert declared and declared == set(metad.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_layout_matches_header():
    """sizeof of the ctypes mirrors equals what a C compiler makes of include/metad.h."""
    import subprocess
    import tempfile
    from paper_2510_06873_b200 import metad
    src = '#include <stdio.h>\n#include "metad.h"\nint main(){printf("%zu %zu\\n", sizeof(metad_cv_desc), sizeof(metad_params));return 0;}\n'
    with tempfile.TemporaryDirectory() as td:
        c = os.path.join(td, "t.c")
        open(c, "w").write(src)
        exe = os.path.join(td, "t")
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        a, b = map(int, subprocess.check_output([exe]).split())
    assert a == ctypes.sizeof(metad.CvDesc) and b == ctypes.sizeof(metad.Params)


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2510_06873_b200 import metad
    p = metad.Params()
    p.natoms, p.precision, p.max_neigh, p.ncv, p.max_hills = 8, 64, 8, 1, 8
    p.sigma[0] = 1.0
    p.cv[0].kind = metad.CV_Q6_MEAN
    h = ctypes.c_void_p()
    code = lib.metad_create(ctypes.byref(h), ctypes.byref(p), None)
    assert code == metad.ERR_CUDA and b"no CPU fallback" in lib.metad_last_error()


def test_argument_checks_need_no_device(lib):
    from paper_2510_06873_b200 import metad
    p = metad.Params()
    h = ctypes.c_void_p()
    assert lib.metad_create(ctypes.byref(h), ctypes.byref(p), None) == metad.ERR_ARG   # natoms == 0
    p.natoms, p.precision = 8, 16
    assert lib.metad_create(ctypes.byref(h), ctypes.byref(p), None) == metad.ERR_ARG   # bad precision
    assert lib.metad_build_neighbors(None, None, None, 1.0) == metad.ERR_ARG
    assert lib.metad_version().startswith(b"metad-b200")


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2510_06873_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".c", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "metad_oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2510_06873_b200", txt, flags=re.M), f
            assert "libmetad_b200" not in txt and "metad.h" not in txt, f
