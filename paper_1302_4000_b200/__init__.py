"""paper_1302_4000_b200 -- B200-native (sm_100a) cRMSD: thin Python binding over the C ABI in include/clusco.h.

Argument marshalling only: every step of the path (centring, covariance/Gram, the eq. 2 closed form,
packed store, one-vs-all) runs in the CUDA kernels of `csrc/`, reached through `libclusco.so`.
PyTorch is used for device memory and streams, nothing else.  There is NO CPU fallback: if the library
is missing or the device is not a B200-class GPU the calls raise.

    import paper_1302_4000_b200 as clusco
    out = clusco.clusco_crmsd_allpairs(coords)            # coords: cuda float32 [N, L, 3] -> [N(N-1)/2]
    d   = clusco.clusco_crmsd_one_vs_all(native, coords)  # -> [N]
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libclusco.so")
_lib = None

ENGINE_AUTO, ENGINE_FFMA, ENGINE_I8TC = 0, 1, 2

EXPORTS = (
    "clusco_status_string", "clusco_last_cuda_error", "clusco_version", "clusco_center",
    "clusco_crmsd_allpairs_workspace", "clusco_crmsd_allpairs", "clusco_crmsd_allpairs_ex",
    "clusco_crmsd_one_vs_all", "clusco_crmsd_allpairs_host", "clusco_crmsd_one_vs_all_host",
    "clusco_partition_rows", "clusco_engine_supported", "clusco_allpairs_prepare", "clusco_allpairs_compute",
    "clusco_host_release", "clusco_crmsd_allpairs_below", "clusco_crmsd_rowstats",
    "clusco_drmsd_allpairs_workspace", "clusco_drmsd_allpairs", "clusco_cmo_allpairs_workspace", "clusco_cmo_allpairs",
    "clusco_gdt_one_vs_all", "clusco_drmsd_one_vs_all", "clusco_cmo_one_vs_all", "clusco_gdt_allpairs",
    "clusco_crmsd_allpairs_below_host", "clusco_crmsd_rowstats_host", "clusco_i8tc_geometry",
)


class CluscoError(RuntimeError):
    pass


def lib_path() -> str:
    return _LIB_PATH


def load(build_if_missing: bool = False):
    """dlopen libclusco.so (built in-tree by `python -m paper_1302_4000_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        if not build_if_missing:
            raise CluscoError(f"{_LIB_PATH} is missing: run `python -m paper_1302_4000_b200.build` "
                              "(there is no CPU fallback)")
        from . import build as _build
        _build.build()
    lib = ctypes.CDLL(_LIB_PATH)
    vp, i64, i32, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_size_t
    lib.clusco_status_string.argtypes = [ctypes.c_int]
    lib.clusco_status_string.restype = ctypes.c_char_p
    lib.clusco_last_cuda_error.restype = ctypes.c_int
    lib.clusco_version.restype = ctypes.c_char_p
    lib.clusco_center.argtypes = [vp, i64, i32, vp, vp, vp]
    lib.clusco_crmsd_allpairs_workspace.argtypes = [i64, i32]
    lib.clusco_crmsd_allpairs_workspace.restype = sz
    lib.clusco_crmsd_allpairs.argtypes = [vp, i64, i32, vp, vp, sz, vp]
    lib.clusco_crmsd_allpairs_ex.argtypes = [vp, i64, i32, i64, i64, vp, vp, sz, ctypes.c_int, vp]
    lib.clusco_crmsd_one_vs_all.argtypes = [vp, vp, i64, i32, vp, vp]
    lib.clusco_crmsd_allpairs_host.argtypes = [vp, i64, i32, vp]
    lib.clusco_crmsd_one_vs_all_host.argtypes = [vp, vp, i64, i32, vp]
    lib.clusco_partition_rows.argtypes = [i64, i32, ctypes.POINTER(ctypes.c_int64)]
    lib.clusco_engine_supported.argtypes = [ctypes.c_int, i32]
    lib.clusco_allpairs_prepare.argtypes = [vp, i64, i32, vp, sz, ctypes.c_int, vp]
    lib.clusco_allpairs_compute.argtypes = [i64, i32, i64, i64, vp, vp, sz, ctypes.c_int, vp]
    lib.clusco_crmsd_allpairs_below.argtypes = [vp, i64, i32, ctypes.c_float, i64, vp, vp, vp, vp, vp, sz, vp]
    lib.clusco_crmsd_rowstats.argtypes = [vp, i64, i32, ctypes.c_float, vp, vp, vp, sz, vp]
    lib.clusco_drmsd_allpairs_workspace.argtypes = [i64, i32]
    lib.clusco_drmsd_allpairs_workspace.restype = sz
    lib.clusco_drmsd_allpairs.argtypes = [vp, i64, i32, vp, vp, sz, vp]
    lib.clusco_cmo_allpairs_workspace.argtypes = [i64, i32]
    lib.clusco_cmo_allpairs_workspace.restype = sz
    lib.clusco_cmo_allpairs.argtypes = [vp, i64, i32, ctypes.c_float, vp, vp, sz, vp]
    lib.clusco_gdt_one_vs_all.argtypes = [vp, vp, i64, i32, vp, vp]
    lib.clusco_drmsd_one_vs_all.argtypes = [vp, vp, i64, i32, vp, vp]
    lib.clusco_cmo_one_vs_all.argtypes = [vp, vp, i64, i32, ctypes.c_float, vp, vp]
    lib.clusco_gdt_allpairs.argtypes = [vp, i64, i32, vp, vp]
    lib.clusco_crmsd_allpairs_below_host.argtypes = [vp, i64, i32, ctypes.c_float, i64, vp, vp, vp, vp]
    lib.clusco_crmsd_rowstats_host.argtypes = [vp, i64, i32, ctypes.c_float, vp, vp]
    lib.clusco_i8tc_geometry.argtypes = [i64, i32, ctypes.POINTER(ctypes.c_int64)]
    for name in EXPORTS:                       # every declared symbol must be exported
        getattr(lib, name)
    _lib = lib
    return lib


def _check(status: int, what: str):
    if status != 0:
        lib = load()
        msg = lib.clusco_status_string(status).decode()
        extra = f" (cudaError {lib.clusco_last_cuda_error()})" if status == 4 else ""
        raise CluscoError(f"{what}: {msg}{extra}")


def _torch():
    import torch
    return torch


def _stream_ptr(t):
    torch = _torch()
    return ctypes.c_void_p(torch.cuda.current_stream(t.device).cuda_stream)


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else ctypes.c_void_p(0)


def _check_coords(coords, name="coords"):
    torch = _torch()
    if not (isinstance(coords, torch.Tensor) and coords.is_cuda and coords.dtype == torch.float32
            and coords.dim() == 3 and coords.shape[2] == 3 and coords.is_contiguous()):
        raise CluscoError(f"{name} must be a contiguous CUDA float32 tensor of shape [N, L, 3]")
    return int(coords.shape[0]), int(coords.shape[1])


def _check_buf(t, name, numel, dtype, device=None, cuda=True):
    """A caller-supplied buffer goes to the library as a raw pointer: check everything the pointer cannot say."""
    torch = _torch()
    if not isinstance(t, torch.Tensor) or t.is_cuda != cuda or t.dtype != dtype or not t.is_contiguous() \
            or t.numel() < numel or (cuda and device is not None and t.device != device):
        where = f"CUDA (on {device})" if cuda else "host"
        raise CluscoError(f"{name} must be a contiguous {where} {dtype} tensor with at least {numel} elements")
    return t


def _check_workspace(ws, nbytes, device):
    torch = _torch()
    if not isinstance(ws, torch.Tensor) or not ws.is_cuda or ws.device != device or not ws.is_contiguous() \
            or ws.numel() * ws.element_size() < nbytes or ws.data_ptr() % 256:
        raise CluscoError(f"workspace must be a contiguous CUDA tensor on {device} of at least {nbytes} bytes, "
                          "256-byte aligned")
    return ws


def _check_host_coords(coords_host, name="coords_host"):
    torch = _torch()
    if not (isinstance(coords_host, torch.Tensor) and not coords_host.is_cuda and coords_host.dtype == torch.float32
            and coords_host.dim() == 3 and coords_host.shape[2] == 3 and coords_host.is_contiguous()):
        raise CluscoError(f"{name} must be a contiguous host float32 tensor of shape [N, L, 3]")
    return int(coords_host.shape[0]), int(coords_host.shape[1])


def version() -> str:
    return load().clusco_version().decode()


def engine_supported(engine: int, L: int) -> bool:
    return bool(load().clusco_engine_supported(engine, L))


def i8tc_geometry(N: int, L: int) -> dict:
    """The tensor-core engine's work decomposition for (N, L) (include/clusco.h: clusco_i8tc_geometry)."""
    o = (ctypes.c_int64 * 5)()
    _check(load().clusco_i8tc_geometry(N, L, o), "clusco_i8tc_geometry")
    return {"tiles": int(o[0]), "ksteps": int(o[1]), "mma_columns_per_kstep": int(o[2]), "row_models": int(o[3]),
            "col_models": int(o[4])}


def n_pairs(N: int) -> int:
    return N * (N - 1) // 2


def clusco_center(coords, centred=None, r2=None):
    """coords[N][L][3] -> (centred[N][L][3], r2[N]); see include/clusco.h."""
    torch = _torch()
    N, L = _check_coords(coords)
    if centred is None:
        centred = torch.empty_like(coords)
    if r2 is None:
        r2 = torch.empty(N, dtype=torch.float32, device=coords.device)
    _check_buf(centred, "centred", N * L * 3, torch.float32, coords.device)
    _check_buf(r2, "r2", N, torch.float32, coords.device)
    with torch.cuda.device(coords.device):
        _check(load().clusco_center(_ptr(coords), N, L, _ptr(centred), _ptr(r2), _stream_ptr(coords)),
               "clusco_center")
    return centred, r2


def clusco_crmsd_allpairs_workspace(N: int, L: int) -> int:
    return int(load().clusco_crmsd_allpairs_workspace(N, L))


def clusco_crmsd_allpairs(coords, out=None, workspace=None, engine: int = ENGINE_AUTO,
                          row_begin: int = 0, row_end: int | None = None):
    """All-versus-all cRMSD: packed upper triangle float32[N(N-1)/2] (rows [row_begin,row_end) if given)."""
    torch = _torch()
    N, L = _check_coords(coords)
    row_end = N if row_end is None else row_end
    lo = row_begin * (2 * N - row_begin - 1) // 2
    hi = row_end * (2 * N - row_end - 1) // 2
    if not (0 <= row_begin <= row_end <= N):
        raise CluscoError("need 0 <= row_begin <= row_end <= N")
    if out is None:
        out = torch.empty(max(hi - lo, 0), dtype=torch.float32, device=coords.device)
    nbytes = clusco_crmsd_allpairs_workspace(N, L)
    if workspace is None:
        workspace = torch.empty(nbytes, dtype=torch.uint8, device=coords.device)
    _check_buf(out, "out", max(hi - lo, 0), torch.float32, coords.device)
    _check_workspace(workspace, nbytes, coords.device)
    with torch.cuda.device(coords.device):
        st = load().clusco_crmsd_allpairs_ex(_ptr(coords), N, L, row_begin, row_end, _ptr(out), _ptr(workspace),
                                             workspace.numel() * workspace.element_size(), engine,
                                             _stream_ptr(coords))
    _check(st, "clusco_crmsd_allpairs")
    return out


def clusco_allpairs_prepare(coords, workspace, engine: int = ENGINE_AUTO):
    """Stage 1 of the all-pairs call (centring, R^2, operand planes) into `workspace`."""
    torch = _torch()
    N, L = _check_coords(coords)
    _check_workspace(workspace, clusco_crmsd_allpairs_workspace(N, L), coords.device)
    with torch.cuda.device(coords.device):
        st = load().clusco_allpairs_prepare(_ptr(coords), N, L, _ptr(workspace),
                                            workspace.numel() * workspace.element_size(), engine,
                                            _stream_ptr(coords))
    _check(st, "clusco_allpairs_prepare")


def clusco_allpairs_compute(N: int, L: int, out, workspace, engine: int = ENGINE_AUTO, row_begin: int = 0,
                            row_end: int | None = None):
    """Stage 2 of the all-pairs call (Gram + eq. 2 + packed store) from a prepared workspace."""
    torch = _torch()
    row_end = N if row_end is None else row_end
    if not (0 <= row_begin <= row_end <= N):
        raise CluscoError("need 0 <= row_begin <= row_end <= N")
    need = row_end * (2 * N - row_end - 1) // 2 - row_begin * (2 * N - row_begin - 1) // 2
    if not (isinstance(out, torch.Tensor) and out.is_cuda):
        raise CluscoError("out must be a CUDA tensor")
    _check_buf(out, "out", need, torch.float32, out.device)
    _check_workspace(workspace, clusco_crmsd_allpairs_workspace(N, L), out.device)
    with torch.cuda.device(out.device):
        st = load().clusco_allpairs_compute(N, L, row_begin, row_end, _ptr(out), _ptr(workspace),
                                            workspace.numel() * workspace.element_size(), engine,
                                            _stream_ptr(out))
    _check(st, "clusco_allpairs_compute")
    return out


def clusco_crmsd_allpairs_below(coords, cutoff: float, capacity: int, workspace=None):
    """Pairs with cRMSD < cutoff, compacted: returns (pair_i int32[capacity], pair_j, pair_c float32, count int64[1]);
    the first min(count, capacity) slots are valid, in unspecified order (include/clusco.h)."""
    torch = _torch()
    N, L = _check_coords(coords)
    dev = coords.device
    pi = torch.empty(capacity, dtype=torch.int32, device=dev)
    pj = torch.empty(capacity, dtype=torch.int32, device=dev)
    pc = torch.empty(capacity, dtype=torch.float32, device=dev)
    count = torch.empty(1, dtype=torch.int64, device=dev)
    if workspace is None:
        workspace = torch.empty(clusco_crmsd_allpairs_workspace(N, L), dtype=torch.uint8, device=dev)
    _check_workspace(workspace, clusco_crmsd_allpairs_workspace(N, L), dev)
    with torch.cuda.device(dev):
        st = load().clusco_crmsd_allpairs_below(_ptr(coords), N, L, float(cutoff), capacity, _ptr(pi), _ptr(pj), _ptr(pc),
                                                _ptr(count), _ptr(workspace),
                                                workspace.numel() * workspace.element_size(), _stream_ptr(coords))
    _check(st, "clusco_crmsd_allpairs_below")
    return pi, pj, pc, count


def clusco_crmsd_rowstats(coords, cutoff: float, workspace=None):
    """Per-model reductions of the all-vs-all matrix: (rowsum float64[N], below int32[N]) (include/clusco.h)."""
    torch = _torch()
    N, L = _check_coords(coords)
    dev = coords.device
    rowsum = torch.empty(N, dtype=torch.float64, device=dev)
    below = torch.empty(N, dtype=torch.int32, device=dev)
    if workspace is None:
        workspace = torch.empty(clusco_crmsd_allpairs_workspace(N, L), dtype=torch.uint8, device=dev)
    _check_workspace(workspace, clusco_crmsd_allpairs_workspace(N, L), dev)
    with torch.cuda.device(dev):
        st = load().clusco_crmsd_rowstats(_ptr(coords), N, L, float(cutoff), _ptr(rowsum), _ptr(below), _ptr(workspace),
                                          workspace.numel() * workspace.element_size(), _stream_ptr(coords))
    _check(st, "clusco_crmsd_rowstats")
    return rowsum, below


def clusco_drmsd_allpairs(coords, out=None, workspace=None):
    """All-versus-all dRMSD (eq. 5): packed upper triangle float32[N(N-1)/2] (include/clusco.h)."""
    torch = _torch()
    N, L = _check_coords(coords)
    if out is None:
        out = torch.empty(n_pairs(N), dtype=torch.float32, device=coords.device)
    nbytes = int(load().clusco_drmsd_allpairs_workspace(N, L))
    if workspace is None:
        workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=coords.device)
    _check_buf(out, "out", n_pairs(N), torch.float32, coords.device)
    _check_workspace(workspace, nbytes, coords.device)
    with torch.cuda.device(coords.device):
        st = load().clusco_drmsd_allpairs(_ptr(coords), N, L, _ptr(out), _ptr(workspace),
                                          workspace.numel() * workspace.element_size(), _stream_ptr(coords))
    _check(st, "clusco_drmsd_allpairs")
    return out


def clusco_cmo_allpairs(coords, cutoff: float, out=None, workspace=None):
    """All-versus-all contact map overlap (eq. 6-7): packed upper triangle float32[N(N-1)/2] (include/clusco.h)."""
    torch = _torch()
    N, L = _check_coords(coords)
    if out is None:
        out = torch.empty(n_pairs(N), dtype=torch.float32, device=coords.device)
    nbytes = int(load().clusco_cmo_allpairs_workspace(N, L))
    if workspace is None:
        workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=coords.device)
    _check_buf(out, "out", n_pairs(N), torch.float32, coords.device)
    _check_workspace(workspace, nbytes, coords.device)
    with torch.cuda.device(coords.device):
        st = load().clusco_cmo_allpairs(_ptr(coords), N, L, float(cutoff), _ptr(out), _ptr(workspace),
                                        workspace.numel() * workspace.element_size(), _stream_ptr(coords))
    _check(st, "clusco_cmo_allpairs")
    return out


def clusco_crmsd_one_vs_all(native, coords, out=None):
    """One native[L][3] against coords[N][L][3] -> float32[N]."""
    torch = _torch()
    N, L = _check_coords(coords)
    if not (native.is_cuda and native.dtype == torch.float32 and tuple(native.shape) == (L, 3)
            and native.is_contiguous()):
        raise CluscoError("native must be a contiguous CUDA float32 tensor of shape [L, 3]")
    if out is None:
        out = torch.empty(N, dtype=torch.float32, device=coords.device)
    _check_buf(out, "out", N, torch.float32, coords.device)
    with torch.cuda.device(coords.device):
        st = load().clusco_crmsd_one_vs_all(_ptr(native), _ptr(coords), N, L, _ptr(out), _stream_ptr(coords))
    _check(st, "clusco_crmsd_one_vs_all")
    return out


def _check_native(native, coords):
    torch = _torch()
    N, L = _check_coords(coords)
    if not (native.is_cuda and native.dtype == torch.float32 and tuple(native.shape) == (L, 3)
            and native.is_contiguous()):
        raise CluscoError("native must be a contiguous CUDA float32 tensor of shape [L, 3]")
    return N, L


def clusco_drmsd_one_vs_all(native, coords, out=None):
    """dRMSD (eq. 5) of coords[N][L][3] against native[L][3] -> float32[N]."""
    torch = _torch()
    N, L = _check_native(native, coords)
    if out is None:
        out = torch.empty(N, dtype=torch.float32, device=coords.device)
    _check_buf(out, "out", N, torch.float32, coords.device)
    with torch.cuda.device(coords.device):
        st = load().clusco_drmsd_one_vs_all(_ptr(native), _ptr(coords), N, L, _ptr(out), _stream_ptr(coords))
    _check(st, "clusco_drmsd_one_vs_all")
    return out


def clusco_cmo_one_vs_all(native, coords, cutoff: float, out=None):
    """Contact map overlap (eq. 6-7) of coords[N][L][3] against native[L][3] -> float32[N]."""
    torch = _torch()
    N, L = _check_native(native, coords)
    if out is None:
        out = torch.empty(N, dtype=torch.float32, device=coords.device)
    _check_buf(out, "out", N, torch.float32, coords.device)
    with torch.cuda.device(coords.device):
        st = load().clusco_cmo_one_vs_all(_ptr(native), _ptr(coords), N, L, float(cutoff), _ptr(out), _stream_ptr(coords))
    _check(st, "clusco_cmo_one_vs_all")
    return out


def clusco_gdt_one_vs_all(native, coords, out=None):
    """GDT_TS (percent), TM-score, MaxSub of coords[N][L][3] against native[L][3] -> float32 [N, 3] (include/clusco.h)."""
    torch = _torch()
    N, L = _check_coords(coords)
    if not (native.is_cuda and native.dtype == torch.float32 and tuple(native.shape) == (L, 3)
            and native.is_contiguous()):
        raise CluscoError("native must be a contiguous CUDA float32 tensor of shape [L, 3]")
    if out is None:
        out = torch.empty((N, 3), dtype=torch.float32, device=coords.device)
    _check_buf(out, "out", 3 * N, torch.float32, coords.device)
    with torch.cuda.device(coords.device):
        st = load().clusco_gdt_one_vs_all(_ptr(native), _ptr(coords), N, L, _ptr(out), _stream_ptr(coords))
    _check(st, "clusco_gdt_one_vs_all")
    return out


def clusco_gdt_allpairs(coords, out=None):
    """All-versus-all GDT_TS (percent), TM-score, MaxSub -> float32 [N(N-1)/2, 3], packed upper triangle."""
    torch = _torch()
    N, L = _check_coords(coords)
    if out is None:
        out = torch.empty((n_pairs(N), 3), dtype=torch.float32, device=coords.device)
    _check_buf(out, "out", 3 * n_pairs(N), torch.float32, coords.device)
    with torch.cuda.device(coords.device):
        st = load().clusco_gdt_allpairs(_ptr(coords), N, L, _ptr(out), _stream_ptr(coords))
    _check(st, "clusco_gdt_allpairs")
    return out


def clusco_crmsd_allpairs_host(coords_host, out_host=None):
    """Host-buffer call (blocking): CPU float32 tensors in and out; copies are inside the call."""
    torch = _torch()
    N, L = _check_host_coords(coords_host)
    if out_host is None:
        out_host = torch.empty(n_pairs(N), dtype=torch.float32, pin_memory=True)
    _check_buf(out_host, "out_host", n_pairs(N), torch.float32, cuda=False)
    _check(load().clusco_crmsd_allpairs_host(_ptr(coords_host), N, L, _ptr(out_host)),
           "clusco_crmsd_allpairs_host")
    return out_host


def clusco_crmsd_one_vs_all_host(native_host, coords_host, out_host=None):
    torch = _torch()
    N, L = _check_host_coords(coords_host)
    if not (isinstance(native_host, torch.Tensor) and not native_host.is_cuda and native_host.dtype == torch.float32
            and tuple(native_host.shape) == (L, 3) and native_host.is_contiguous()):
        raise CluscoError("native_host must be a contiguous host float32 tensor of shape [L, 3]")
    if out_host is None:
        out_host = torch.empty(N, dtype=torch.float32, pin_memory=True)
    _check_buf(out_host, "out_host", N, torch.float32, cuda=False)
    _check(load().clusco_crmsd_one_vs_all_host(_ptr(native_host), _ptr(coords_host), N, L, _ptr(out_host)),
           "clusco_crmsd_one_vs_all_host")
    return out_host


def clusco_crmsd_allpairs_below_host(coords_host, cutoff: float, capacity: int, out=None):
    """Host-buffer form of clusco_crmsd_allpairs_below (blocking): returns (pair_i int32[capacity], pair_j, pair_c
    float32 -- host tensors -- and the count as a Python int); the first min(count, capacity) slots are valid."""
    torch = _torch()
    N, L = _check_host_coords(coords_host)
    if capacity < 0:
        raise CluscoError("capacity must be >= 0")
    if out is None:
        out = (torch.empty(capacity, dtype=torch.int32, pin_memory=capacity > 0),
               torch.empty(capacity, dtype=torch.int32, pin_memory=capacity > 0),
               torch.empty(capacity, dtype=torch.float32, pin_memory=capacity > 0))
    pi, pj, pc = out
    _check_buf(pi, "pair_i", capacity, torch.int32, cuda=False)
    _check_buf(pj, "pair_j", capacity, torch.int32, cuda=False)
    _check_buf(pc, "pair_c", capacity, torch.float32, cuda=False)
    count = ctypes.c_ulonglong(0)
    _check(load().clusco_crmsd_allpairs_below_host(_ptr(coords_host), N, L, float(cutoff), capacity, _ptr(pi), _ptr(pj),
                                                   _ptr(pc), ctypes.cast(ctypes.byref(count), ctypes.c_void_p)),
           "clusco_crmsd_allpairs_below_host")
    return pi, pj, pc, int(count.value)


def clusco_crmsd_rowstats_host(coords_host, cutoff: float, out=None):
    """Host-buffer form of clusco_crmsd_rowstats (blocking): (rowsum float64[N], below int32[N]) host tensors."""
    torch = _torch()
    N, L = _check_host_coords(coords_host)
    if out is None:
        out = (torch.empty(N, dtype=torch.float64, pin_memory=N > 0), torch.empty(N, dtype=torch.int32, pin_memory=N > 0))
    rowsum, below = out
    _check_buf(rowsum, "rowsum", N, torch.float64, cuda=False)
    _check_buf(below, "below", N, torch.int32, cuda=False)
    _check(load().clusco_crmsd_rowstats_host(_ptr(coords_host), N, L, float(cutoff), _ptr(rowsum), _ptr(below)),
           "clusco_crmsd_rowstats_host")
    return rowsum, below


def clusco_host_release():
    """Return the device memory pool kept by the *_host calls to the driver."""
    _check(load().clusco_host_release(), "clusco_host_release")


def clusco_partition_rows(N: int, parts: int):
    """Row boundaries (multiples of 128) giving each of `parts` ranks about the same number of pairs."""
    b = (ctypes.c_int64 * (parts + 1))()
    _check(load().clusco_partition_rows(N, parts, b), "clusco_partition_rows")
    return [int(v) for v in b]
