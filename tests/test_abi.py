"""No-GPU checks of the boundary: libmoto.so builds, loads and exports every symbol include/moto.h declares;
argument errors come back as status codes."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2509_26269_b200 import build, binding
    build.build()
    return binding.load_library()


def header_symbols():
    src = open(os.path.join(ROOT, "include", "moto.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(moto_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = header_symbols()
    assert len(names) >= 18
    for n in names:
        assert hasattr(lib, n), f"{n} declared in moto.h but not exported"


def test_binding_covers_header(lib):
    from paper_2509_26269_b200 import binding
    assert set(header_symbols()) == set(binding.EXPORTS)


def test_version_and_arg_errors_without_gpu(lib):
    from paper_2509_26269_b200 import binding as b
    assert b"sm_100a" in lib.moto_version()
    lat = b.Lattice(b.KIND_TRI2D, 8, 8, 1, 1, 0)
    assert lib.moto_workspace_bytes(C.byref(lat), 2) > 6 * 2 * 64 * 24
    assert lib.moto_workspace_bytes(C.byref(lat), 0) == 0
    assert lib.moto_workspace_bytes(C.byref(lat), b.KMAX + 1) == 0
    bad = b.Lattice(7, 8, 8, 1, 1, 0)
    assert lib.moto_workspace_bytes(C.byref(bad), 2) == 0
    h = C.c_void_p()
    p = b.SpinParams(1, 0.3, 0.05, (C.c_double * 3)(0, 0, 0.02), 1.0)
    assert lib.moto_create(C.byref(lat), C.addressof(p), None, 0, None, 2, C.byref(h)) == b.EINVAL
    assert lib.moto_hvp(None, None, None, 1, None) == b.EINVAL
    assert lib.moto_last_error(None) == b"null context"


def test_struct_sizes_match_header():
    from paper_2509_26269_b200 import binding as b
    assert C.sizeof(b.SpinParams) == 7 * 8
    assert C.sizeof(b.MorseParams) == 4 * 8
    assert C.sizeof(b.SolveInfo) == 8 + 8 * b.KMAX + 8
    assert C.sizeof(b.SolverOpts) == 16 + 16 + 8 + 8 + 8   # + method, ncv, cheb_mode, persistent
    assert C.sizeof(b.Lattice) == 24 + 32 + 8
    assert C.sizeof(b.RelaxInfo) == 16 + 24


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2509_26269_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2509_26269_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "arxiv", ""), f
