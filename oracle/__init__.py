"""FP64 CPU oracle for cRMSD -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this package.  It shares no code with `paper_1302_4000_b200/` (the CUDA path)
and imports nothing from it.

`oracle.crmsd_oracle.c` is the oracle proper (plain C, double precision, Jacobi SVD per pair; see
its header for the algorithm and the PAPER.md citations).  This file only builds it with gcc and
marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "crmsd_oracle.c")
_LIB = os.path.join(_HERE, "libcrmsd_oracle.so")
_lib = None

_f32p = ctypes.POINTER(ctypes.c_float)
_f64p = ctypes.POINTER(ctypes.c_double)
_i64p = ctypes.POINTER(ctypes.c_int64)


_SRC_D = os.path.join(_HERE, "drmsd_oracle.c")
_LIB_D = os.path.join(_HERE, "libdrmsd_oracle.so")
_lib_d = None


_SRC_C = os.path.join(_HERE, "cmo_oracle.c")
_LIB_C = os.path.join(_HERE, "libcmo_oracle.so")
_lib_c = None


_SRC_G = os.path.join(_HERE, "gdt_oracle.c")
_LIB_G = os.path.join(_HERE, "libgdt_oracle.so")
_lib_g = None


def _compile(src: str, lib: str, force: bool) -> str:
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src):
        tmp = lib + f".tmp{os.getpid()}"
        subprocess.run(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", tmp, src, "-lm"],
                       check=True)
        os.replace(tmp, lib)
    return lib


def build(force: bool = False) -> str:
    """Compile crmsd_oracle.c and drmsd_oracle.c (gcc -O2 -fopenmp, no fast-math); returns the cRMSD library."""
    _compile(_SRC_D, _LIB_D, force)
    _compile(_SRC_C, _LIB_C, force)
    _compile(_SRC_G, _LIB_G, force)
    return _compile(_SRC, _LIB, force)


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_center.argtypes = [_f32p, ctypes.c_int64, ctypes.c_int32, _f64p, _f64p]
        lib.oracle_center.restype = None
        for name in ("oracle_crmsd_pair",):
            f = getattr(lib, name)
            f.argtypes = [_f32p, _f32p, ctypes.c_int32, _f64p]
            f.restype = ctypes.c_double
        lib.oracle_crmsd_pair_eq2.argtypes = [_f32p, _f32p, ctypes.c_int32, _f64p, _f64p, _f64p]
        lib.oracle_crmsd_pair_eq2.restype = ctypes.c_double
        lib.oracle_crmsd_pair_eq1.argtypes = [_f32p, _f32p, ctypes.c_int32, _f64p, _f64p]
        lib.oracle_crmsd_pair_eq1.restype = ctypes.c_double
        lib.oracle_pair_spectrum.argtypes = [_f32p, _f32p, ctypes.c_int32, _f64p, _f64p, _f64p]
        lib.oracle_pair_spectrum.restype = None
        lib.oracle_crmsd_rows.argtypes = [_f32p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64,
                                          ctypes.c_int64, _f64p, _f64p]
        lib.oracle_crmsd_rows.restype = None
        lib.oracle_crmsd_pairs.argtypes = [_f32p, ctypes.c_int64, ctypes.c_int32, _i64p, _i64p,
                                           ctypes.c_int64, _f64p, _f64p]
        lib.oracle_crmsd_pairs.restype = None
        lib.oracle_crmsd_one_vs_all.argtypes = [_f32p, _f32p, ctypes.c_int64, ctypes.c_int32, _f64p, _f64p]
        lib.oracle_crmsd_one_vs_all.restype = None
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = lib
    return _lib


def _f32(x, shape_tail=None):
    x = np.ascontiguousarray(x, dtype=np.float32)
    return x


def _p(a, t):
    return a.ctypes.data_as(t)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def center(coords):
    """coords[N][L][3] fp32 -> (centred[N][L][3] fp64, r2[N] fp64).  Steps 1-2."""
    x = _f32(coords)
    N, L, _ = x.shape
    cen = np.empty((N, L, 3), np.float64)
    r2 = np.empty(N, np.float64)
    _load().oracle_center(_p(x, _f32p), N, L, _p(cen, _f64p), _p(r2, _f64p))
    return cen, r2


def crmsd_pair(xa, xb):
    """(c, c2) of one pair by the definition route (centre, covariance, Jacobi SVD, sign det)."""
    a, b = _f32(xa), _f32(xb)
    assert a.shape == b.shape and a.shape[1] == 3
    c2 = ctypes.c_double()
    c = _load().oracle_crmsd_pair(_p(a, _f32p), _p(b, _f32p), a.shape[0], ctypes.byref(c2))
    return float(c), float(c2.value)


def crmsd_pair_eq2(xa, xb):
    """eq. 2 literally: returns (c, c2, lambdas[3] of M^T M descending, S)."""
    a, b = _f32(xa), _f32(xb)
    c2 = ctypes.c_double()
    S = ctypes.c_double()
    lam = np.empty(3, np.float64)
    c = _load().oracle_crmsd_pair_eq2(_p(a, _f32p), _p(b, _f32p), a.shape[0], ctypes.byref(c2),
                                      _p(lam, _f64p), ctypes.byref(S))
    return float(c), float(c2.value), lam, float(S.value)


def crmsd_pair_eq1(xa, xb):
    """eq. 1 literally: explicit optimal rotation, residual summed per atom.  (c, c2, R[3][3])."""
    a, b = _f32(xa), _f32(xb)
    c2 = ctypes.c_double()
    R = np.empty((3, 3), np.float64)
    c = _load().oracle_crmsd_pair_eq1(_p(a, _f32p), _p(b, _f32p), a.shape[0], ctypes.byref(c2),
                                      _p(R, _f64p))
    return float(c), float(c2.value), R


def pair_spectrum(xa, xb):
    """(singular values of M descending, det M, M[3][3]) of one pair."""
    a, b = _f32(xa), _f32(xb)
    s = np.empty(3, np.float64)
    M = np.empty((3, 3), np.float64)
    d = ctypes.c_double()
    _load().oracle_pair_spectrum(_p(a, _f32p), _p(b, _f32p), a.shape[0], _p(s, _f64p), ctypes.byref(d),
                                 _p(M, _f64p))
    return s, float(d.value), M


def crmsd_rows(coords, row_begin, row_end):
    """Rows [row_begin,row_end) of the packed all-vs-all matrix: (c, c2) fp64, row-major, j>i."""
    x = _f32(coords)
    N, L, _ = x.shape
    n = (row_begin * (2 * N - row_begin - 1) // 2, row_end * (2 * N - row_end - 1) // 2)
    c = np.empty(n[1] - n[0], np.float64)
    c2 = np.empty(n[1] - n[0], np.float64)
    _load().oracle_crmsd_rows(_p(x, _f32p), N, L, int(row_begin), int(row_end), _p(c, _f64p), _p(c2, _f64p))
    return c, c2


def crmsd_allpairs(coords):
    """Whole packed upper triangle, N(N-1)/2 values: (c, c2) fp64."""
    x = _f32(coords)
    return crmsd_rows(x, 0, x.shape[0])


def crmsd_pairs(coords, pi, pj):
    """Listed pairs: (c, c2) with c[k] = cRMSD(model pi[k], model pj[k])."""
    x = _f32(coords)
    N, L, _ = x.shape
    pi = np.ascontiguousarray(pi, np.int64)
    pj = np.ascontiguousarray(pj, np.int64)
    c = np.empty(pi.size, np.float64)
    c2 = np.empty(pi.size, np.float64)
    _load().oracle_crmsd_pairs(_p(x, _f32p), N, L, _p(pi, _i64p), _p(pj, _i64p), pi.size,
                               _p(c, _f64p), _p(c2, _f64p))
    return c, c2


def crmsd_one_vs_all(native, coords):
    """One native[L][3] against coords[N][L][3]: (c, c2) fp64."""
    nat = _f32(native)
    x = _f32(coords)
    N, L, _ = x.shape
    assert nat.shape == (L, 3)
    c = np.empty(N, np.float64)
    c2 = np.empty(N, np.float64)
    _load().oracle_crmsd_one_vs_all(_p(nat, _f32p), _p(x, _f32p), N, L, _p(c, _f64p), _p(c2, _f64p))
    return c, c2


# ---- consumers of the matrix, written out from their definitions -------------------
def pairs_below(coords, cutoff):
    """The paper's first use case: all-versus-all cRMSD, keep the pairs below a cut-off.
    Returns (i, j, c) of every i < j with c(i,j) < cutoff, in row-major order, from the FP64 matrix."""
    x = _f32(coords)
    N = x.shape[0]
    c, _ = crmsd_allpairs(x)
    ii, jj, cc = [], [], []
    k = 0
    for i in range(N):                      # plain loops over the packed triangle, row by row
        row = c[k:k + N - 1 - i]
        hit = np.nonzero(row < cutoff)[0]
        ii.extend([i] * hit.size)
        jj.extend((hit + i + 1).tolist())
        cc.extend(row[hit].tolist())
        k += N - 1 - i
    return np.asarray(ii, np.int64), np.asarray(jj, np.int64), np.asarray(cc, np.float64)


def rowstats(coords, cutoff):
    """Per-model reductions used by representative selection: rowsum[i] = sum_{j != i} c(i,j) and
    below[i] = #{j != i : c(i,j) < cutoff}, both from the FP64 matrix (symmetric: c(i,j) = c(j,i))."""
    x = _f32(coords)
    N = x.shape[0]
    c, _ = crmsd_allpairs(x)
    rowsum = np.zeros(N, np.float64)
    below = np.zeros(N, np.int64)
    k = 0
    for i in range(N):
        for j in range(i + 1, N):
            v = c[k]
            rowsum[i] += v
            rowsum[j] += v
            if v < cutoff:
                below[i] += 1
                below[j] += 1
            k += 1
    return rowsum, below


# ---- dRMSD (oracle = eq. 5 literally, drmsd_oracle.c) ------------------------------
def _load_d():
    global _lib_d
    if _lib_d is None:
        lib = ctypes.CDLL(_compile(_SRC_D, _LIB_D, False))
        lib.oracle_drmsd_pair.argtypes = [_f32p, _f32p, ctypes.c_int32, _f64p]
        lib.oracle_drmsd_pair.restype = ctypes.c_double
        lib.oracle_drmsd_rows.argtypes = [_f32p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64,
                                          _f64p, _f64p]
        lib.oracle_drmsd_rows.restype = None
        lib.oracle_drmsd_pairs.argtypes = [_f32p, ctypes.c_int64, ctypes.c_int32, _i64p, _i64p, ctypes.c_int64,
                                           _f64p, _f64p]
        lib.oracle_drmsd_pairs.restype = None
        lib.oracle_drmsd_one_vs_all.argtypes = [_f32p, _f32p, ctypes.c_int64, ctypes.c_int32, _f64p, _f64p]
        lib.oracle_drmsd_one_vs_all.restype = None
        _lib_d = lib
    return _lib_d


def drmsd_pair(xa, xb):
    """eq. 5 for one pair: (d, d2)."""
    a, b = _f32(xa), _f32(xb)
    assert a.shape == b.shape
    d2 = ctypes.c_double()
    d = _load_d().oracle_drmsd_pair(_p(a, _f32p), _p(b, _f32p), a.shape[0], ctypes.byref(d2))
    return float(d), float(d2.value)


def drmsd_rows(coords, row_begin, row_end):
    """Rows [row_begin,row_end) of the packed all-vs-all dRMSD matrix: (d, d2) fp64, row-major, j>i."""
    x = _f32(coords)
    N, L, _ = x.shape
    n = (row_begin * (2 * N - row_begin - 1) // 2, row_end * (2 * N - row_end - 1) // 2)
    d = np.empty(n[1] - n[0], np.float64)
    d2 = np.empty(n[1] - n[0], np.float64)
    _load_d().oracle_drmsd_rows(_p(x, _f32p), N, L, int(row_begin), int(row_end), _p(d, _f64p), _p(d2, _f64p))
    return d, d2


def drmsd_allpairs(coords):
    x = _f32(coords)
    return drmsd_rows(x, 0, x.shape[0])


def drmsd_pairs(coords, pi, pj):
    """Listed pairs: (d, d2)."""
    x = _f32(coords)
    N, L, _ = x.shape
    pi = np.ascontiguousarray(pi, np.int64)
    pj = np.ascontiguousarray(pj, np.int64)
    d = np.empty(pi.size, np.float64)
    d2 = np.empty(pi.size, np.float64)
    _load_d().oracle_drmsd_pairs(_p(x, _f32p), N, L, _p(pi, _i64p), _p(pj, _i64p), pi.size, _p(d, _f64p), _p(d2, _f64p))
    return d, d2


# ---- CMO (oracle = eq. 6-7 literally, cmo_oracle.c) --------------------------------
def _load_c():
    global _lib_c
    if _lib_c is None:
        lib = ctypes.CDLL(_compile(_SRC_C, _LIB_C, False))
        lib.oracle_cmo_pair.argtypes = [_f32p, _f32p, ctypes.c_int32, ctypes.c_double, _i64p]
        lib.oracle_cmo_pair.restype = ctypes.c_double
        lib.oracle_cmo_rows.argtypes = [_f32p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double, ctypes.c_int64,
                                        ctypes.c_int64, _f64p]
        lib.oracle_cmo_rows.restype = None
        lib.oracle_cmo_pairs.argtypes = [_f32p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double, _i64p, _i64p,
                                         ctypes.c_int64, _f64p]
        lib.oracle_cmo_pairs.restype = None
        lib.oracle_cmo_one_vs_all.argtypes = [_f32p, _f32p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double, _f64p]
        lib.oracle_cmo_one_vs_all.restype = None
        _lib_c = lib
    return _lib_c


def _cut(cutoff):
    return float(np.float32(cutoff))          # the C ABI takes the cut-off as fp32; both sides widen that value


def cmo_pair(xa, xb, cutoff):
    """eq. 6-7 for one pair: (S, [n(A), n(B), n(A and B)])."""
    a, b = _f32(xa), _f32(xb)
    cnt = np.zeros(3, np.int64)
    s = _load_c().oracle_cmo_pair(_p(a, _f32p), _p(b, _f32p), a.shape[0], _cut(cutoff), _p(cnt, _i64p))
    return float(s), cnt


def cmo_rows(coords, cutoff, row_begin, row_end):
    x = _f32(coords)
    N, L, _ = x.shape
    n = (row_begin * (2 * N - row_begin - 1) // 2, row_end * (2 * N - row_end - 1) // 2)
    s = np.empty(n[1] - n[0], np.float64)
    _load_c().oracle_cmo_rows(_p(x, _f32p), N, L, _cut(cutoff), int(row_begin), int(row_end), _p(s, _f64p))
    return s


def cmo_allpairs(coords, cutoff):
    x = _f32(coords)
    return cmo_rows(x, cutoff, 0, x.shape[0])


def cmo_pairs(coords, cutoff, pi, pj):
    x = _f32(coords)
    N, L, _ = x.shape
    pi = np.ascontiguousarray(pi, np.int64)
    pj = np.ascontiguousarray(pj, np.int64)
    s = np.empty(pi.size, np.float64)
    _load_c().oracle_cmo_pairs(_p(x, _f32p), N, L, _cut(cutoff), _p(pi, _i64p), _p(pj, _i64p), pi.size, _p(s, _f64p))
    return s


# ---- GDT_TS / TM-score / MaxSub versus a reference (gdt_oracle.c) ------------------
def _load_g():
    global _lib_g
    if _lib_g is None:
        lib = ctypes.CDLL(_compile(_SRC_G, _LIB_G, False))
        lib.oracle_gdt_pair.argtypes = [_f32p, _f32p, ctypes.c_int32, _f64p, _f64p]
        lib.oracle_gdt_pair.restype = None
        lib.oracle_gdt_pair_trace.argtypes = [_f32p, _f32p, ctypes.c_int32, _f64p, _f64p, _i64p]
        lib.oracle_gdt_pair_trace.restype = None
        lib.oracle_gdt_one_vs_all.argtypes = [_f32p, _f32p, ctypes.c_int64, ctypes.c_int32, _f64p]
        lib.oracle_gdt_one_vs_all.restype = None
        _lib_g = lib
    return _lib_g


def gdt_pair(ref, model):
    """The paper's search for one model: ((GDT_TS %, TM-score, MaxSub), max counts C_1, C_2, C_4, C_8)."""
    a, b = _f32(ref), _f32(model)
    assert a.shape == b.shape
    out = np.empty(3, np.float64)
    cnt = np.empty(4, np.float64)
    _load_g().oracle_gdt_pair(_p(a, _f32p), _p(b, _f32p), a.shape[0], _p(out, _f64p), _p(cnt, _f64p))
    return out, cnt


def gdt_pair_trace(ref, model):
    """gdt_pair plus the search-control diagnostics: (scores, counts, (seed fragments, superpositions evaluated in total,
    most superpositions spent on one seed))."""
    a, b = _f32(ref), _f32(model)
    assert a.shape == b.shape
    out = np.empty(3, np.float64)
    cnt = np.empty(4, np.float64)
    tr = np.zeros(3, np.int64)
    _load_g().oracle_gdt_pair_trace(_p(a, _f32p), _p(b, _f32p), a.shape[0], _p(out, _f64p), _p(cnt, _f64p), _p(tr, _i64p))
    return out, cnt, tuple(int(v) for v in tr)


def gdt_one_vs_all(ref, coords):
    """Reference against coords[N][L][3]: float64 [N, 3] = (GDT_TS %, TM-score, MaxSub) per model."""
    a, x = _f32(ref), _f32(coords)
    N, L, _ = x.shape
    out = np.empty((N, 3), np.float64)
    _load_g().oracle_gdt_one_vs_all(_p(a, _f32p), _p(x, _f32p), N, L, _p(out, _f64p))
    return out


def drmsd_one_vs_all(ref, coords):
    """eq. 5 of one reference against coords[N][L][3]: (d, d2) fp64 [N]."""
    a, x = _f32(ref), _f32(coords)
    N, L, _ = x.shape
    d = np.empty(N, np.float64)
    d2 = np.empty(N, np.float64)
    _load_d().oracle_drmsd_one_vs_all(_p(a, _f32p), _p(x, _f32p), N, L, _p(d, _f64p), _p(d2, _f64p))
    return d, d2


def cmo_one_vs_all(ref, coords, cutoff):
    """eq. 6-7 of one reference against coords[N][L][3]: S fp64 [N]."""
    a, x = _f32(ref), _f32(coords)
    N, L, _ = x.shape
    s = np.empty(N, np.float64)
    _load_c().oracle_cmo_one_vs_all(_p(a, _f32p), _p(x, _f32p), N, L, _cut(cutoff), _p(s, _f64p))
    return s


def gdt_allpairs(coords):
    """All-versus-all form: for i < j model i is the reference; float64 [N(N-1)/2, 3], packed row-major."""
    x = _f32(coords)
    N = x.shape[0]
    rows = [gdt_one_vs_all(x[i], x[i + 1:]) for i in range(N - 1)]
    return np.concatenate(rows) if rows else np.zeros((0, 3))
