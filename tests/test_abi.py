"""The C-ABI library loads and exports every symbol include/clusco.h declares (no compute without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1302_4000_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def _declared():
    txt = open(os.path.join(ROOT, "include", "clusco.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(clusco_[a-z0-9_]+)\s*\(", txt)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert "clusco_crmsd_allpairs" in names and "clusco_center" in names and "clusco_crmsd_one_vs_all" in names
    for n in names:
        assert hasattr(lib, n), n
    import paper_1302_4000_b200 as pkg
    assert sorted(pkg.EXPORTS) == names


def test_status_strings_and_version(lib):
    lib.clusco_status_string.restype = ctypes.c_char_p
    lib.clusco_version.restype = ctypes.c_char_p
    assert lib.clusco_status_string(0) == b"ok"
    assert b"invalid" in lib.clusco_status_string(1)
    assert lib.clusco_version().decode().count(".") == 1


def test_workspace_query_is_host_only(lib):
    f = lib.clusco_crmsd_allpairs_workspace
    f.argtypes = [ctypes.c_int64, ctypes.c_int32]
    f.restype = ctypes.c_size_t
    assert f(-1, 10) == 0 and f(10, 0) == 0
    assert f(10000, 250) > 10000 * 250 * 3
    assert f(1, 10) > 0


def test_argument_validation_needs_no_gpu(lib):
    i64, i32, vp = ctypes.c_int64, ctypes.c_int32, ctypes.c_void_p
    lib.clusco_center.argtypes = [vp, i64, i32, vp, vp, vp]
    assert lib.clusco_center(None, -1, 10, None, None, None) == 1
    assert lib.clusco_center(None, 0, 10, None, None, None) == 0          # empty input: OK, no work
    assert lib.clusco_center(None, 5, 10, None, None, None) == 1          # NULL with non-empty extent
    lib.clusco_crmsd_allpairs.argtypes = [vp, i64, i32, vp, vp, ctypes.c_size_t, vp]
    assert lib.clusco_crmsd_allpairs(None, 1, 10, None, None, 0, None) == 0   # N < 2 writes nothing
    assert lib.clusco_crmsd_allpairs(None, 5, 0, None, None, 0, None) == 1
    assert lib.clusco_crmsd_allpairs(None, 5, 10, None, None, 0, None) == 1
    lib.clusco_crmsd_one_vs_all.argtypes = [vp, vp, i64, i32, vp, vp]
    assert lib.clusco_crmsd_one_vs_all(None, None, 0, 10, None, None) == 0
    assert lib.clusco_crmsd_one_vs_all(None, None, 3, 10, None, None) == 1


def test_partition_rows(lib):
    import paper_1302_4000_b200 as pkg
    for N, parts in ((10000, 2), (30000, 8), (200, 4), (1000, 1)):
        b = pkg.clusco_partition_rows(N, parts)
        assert b[0] == 0 and b[-1] == N and len(b) == parts + 1
        assert all(x <= y for x, y in zip(b, b[1:]))
        assert all(x % 128 == 0 for x in b[:-1])
        if N >= 10000:
            pairs = [hi * (2 * N - hi - 1) // 2 - lo * (2 * N - lo - 1) // 2 for lo, hi in zip(b, b[1:])]
            assert max(pairs) < 1.15 * (N * (N - 1) // 2) / parts
