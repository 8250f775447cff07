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


def test_host_consumer_calls_validate_without_a_gpu(lib):
    i64, i32, vp, f = ctypes.c_int64, ctypes.c_int32, ctypes.c_void_p, ctypes.c_float
    lib.clusco_crmsd_allpairs_below_host.argtypes = [vp, i64, i32, f, i64, vp, vp, vp, vp]
    lib.clusco_crmsd_rowstats_host.argtypes = [vp, i64, i32, f, vp, vp]
    count = ctypes.c_ulonglong(7)
    cp = ctypes.cast(ctypes.byref(count), vp)
    assert lib.clusco_crmsd_allpairs_below_host(None, 1, 10, 3.2, 0, None, None, None, cp) == 0 and count.value == 0
    assert lib.clusco_crmsd_allpairs_below_host(None, 5, 10, 3.2, 0, None, None, None, None) == 1     # no count
    assert lib.clusco_crmsd_allpairs_below_host(None, 5, 10, 3.2, 4, None, None, None, cp) == 1       # capacity, no arrays
    assert lib.clusco_crmsd_allpairs_below_host(None, 5, 0, 3.2, 0, None, None, None, cp) == 1
    assert lib.clusco_crmsd_rowstats_host(None, 0, 10, 3.2, None, None) == 0
    assert lib.clusco_crmsd_rowstats_host(None, 5, 10, 3.2, None, None) == 1
    assert lib.clusco_crmsd_rowstats_host(None, -1, 10, 3.2, None, None) == 1


def test_binding_rejects_bad_buffers_before_the_library_sees_them():
    """The binding passes raw pointers: a short, wrong-dtype, non-contiguous or host tensor must raise, not corrupt memory.
    (Checked on host tensors: the checks run before any device work.)"""
    import torch
    import paper_1302_4000_b200 as pkg
    x = torch.zeros((4, 5, 3), dtype=torch.float32)
    with pytest.raises(pkg.CluscoError):
        pkg.clusco_crmsd_allpairs(x)                                   # not a CUDA tensor
    with pytest.raises(pkg.CluscoError):
        pkg.clusco_crmsd_allpairs_host(x.double())
    with pytest.raises(pkg.CluscoError):
        pkg.clusco_crmsd_allpairs_host(x, torch.zeros(3))              # needs 6 results
    with pytest.raises(pkg.CluscoError):
        pkg.clusco_crmsd_allpairs_host(x[:, :, :2])
    with pytest.raises(pkg.CluscoError):
        pkg.clusco_crmsd_one_vs_all_host(torch.zeros((4, 3)), x)        # native of the wrong length
    with pytest.raises(pkg.CluscoError):
        pkg.clusco_crmsd_rowstats_host(x, 3.0, out=(torch.zeros(4), torch.zeros(4, dtype=torch.int32)))   # float32 sums
    with pytest.raises(pkg.CluscoError):
        pkg.clusco_crmsd_allpairs_below_host(x, 3.0, 8, out=(torch.zeros(8, dtype=torch.int32),) * 3)


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


def test_i8tc_geometry_counts_the_upper_triangle_tiles():
    """Row tile I (32 models) meets column tiles J >= 2 I (16 models each): the host-only geometry query must report exactly
    that many tiles, the k-step count ceil(L / 32), and refuse chains the tensor-core engine does not serve."""
    import paper_1302_4000_b200 as clusco
    for N, L in ((2, 1), (33, 5), (200, 76), (2000, 120), (10000, 250), (30000, 100), (4097, 256)):
        geo = clusco.i8tc_geometry(N, L)
        rows, cols = (N + 31) // 32, (N + 15) // 16
        assert geo["tiles"] == sum(max(0, cols - 2 * I) for I in range(rows))
        assert geo["ksteps"] == (L + 31) // 32
        assert geo["mma_columns_per_kstep"] == 144 + 96 + 48
    assert clusco.engine_supported(clusco.ENGINE_I8TC, 256) and not clusco.engine_supported(clusco.ENGINE_I8TC, 257)
    with pytest.raises(clusco.CluscoError):
        clusco.i8tc_geometry(100, 300)
