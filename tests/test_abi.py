"""-m "not gpu": the C-ABI library loads, exports every symbol include/homg.h declares, and its
host-only entry points (no device work) behave.  No compute calls are made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def H():
    from paper_1108_2045_b200 import build as B, homg
    B.build()
    homg.lib()
    return homg


def test_every_declared_symbol_is_exported(H):
    text = open(os.path.join(ROOT, "include", "homg.h")).read()
    declared = sorted(set(re.findall(r"HOMG_API[^;(]*?\b(homg_\w+)\s*\(", text)))
    assert declared == sorted(H.SYMBOLS), (declared, sorted(H.SYMBOLS))
    lib = C.CDLL(H.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name


def test_binding_struct_matches_header(H):
    text = open(os.path.join(ROOT, "include", "homg.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} homg_options;", text, re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = [re.search(r"(\w+)\s*$", d.strip()).group(1) for d in body.split(";") if d.strip()]
    assert names == [f[0] for f in H.HomgOptions._fields_]


def test_workspace_bytes_and_argument_checks(H):
    wb = H.workspace_bytes
    # cfg4: 513^3 fp32, 9 levels: level 0 has 6 arrays of 513*513*544*4 B; all levels < 8/7 * (8/6) of that + staging
    b = wb((513, 513, 513), 9, "poisson7", "f32")
    arr0 = 513 * 513 * 544 * 4
    assert 6 * arr0 + 513 ** 3 * 4 < b < 10 * arr0
    assert wb((129, 129), 7, "poisson5", "f64") > 6 * 129 * 144 * 8
    # bad arguments give 0 (no exception, no abort)
    assert wb((130, 129), 7, "poisson5", "f64") == 0          # not c*2^(L-1)+1
    assert wb((129, 129), 8, "poisson5", "f64") == 0          # coarsest level would have < 3 nodes
    assert wb((129, 129), 7, "poisson7", "f64") == 0          # stencil / ndim mismatch
    assert wb((129, 129, 129), 7, "poisson5", "f64") == 0
    assert wb((129, 129), 0, "poisson5", "f64") == 0
    # variable coefficient needs one more array per level
    assert wb((65, 65, 65), 6, "diffusion7", "f64") > wb((65, 65, 65), 6, "poisson7", "f64")


def test_missing_library_fails_loudly(H, monkeypatch):
    monkeypatch.setattr(H, "_lib", None)
    monkeypatch.setattr(H, "LIB_PATH", os.path.join(ROOT, "no_such_dir", "libhomg.so"))
    with pytest.raises(ImportError):
        H.lib()


def test_no_cpu_device(H):
    with pytest.raises(Exception):
        H.Solver((17, 17), 3, "poisson5", "f64", device="cpu")
