"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain CPU statement of LUMEN's KV checkpoint pack (section 4.2,
step 3 of the incremental checkpoint pipeline) and restore unpack
(section 4.3, KV-reuse recovery), in the buffer layout
[req][layer][K|V][token][head][dim] (BASELINE.json configs[0]; SURVEY.md
section 8(c) C1/C2).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It imports nothing from
paper_2606_17787_b200 and shares no source with it.

Two independent statements live here:
  * lumen_oracle.c  -- the five-loop definition in plain C (ctypes-loaded);
  * oracle_np.py    -- the same definition as a NumPy gather on slot ids.
They are cross-checked against each other and against pins P1-P10 in
tests/test_oracle_pins.py.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "lumen_oracle.c"
_SRCS = [_HERE / "lumen_oracle.c", _HERE / "tags_oracle.c"]
_SO = _HERE / "liblumen_oracle.so"

OK, EARG, EPAGE, ESIZE, EOVERLAP = 0, -1, -2, -3, -4


class OracleError(RuntimeError):
    def __init__(self, code: int):
        super().__init__(f"oracle error {code}")
        self.code = code


def build(force: bool = False) -> Path:
    """Compile lumen_oracle.c into oracle/liblumen_oracle.so with gcc."""
    if force or not _SO.exists() or any(_SO.stat().st_mtime < p.stat().st_mtime for p in _SRCS):
        tmp = _SO.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra",
             "-o", str(tmp), *map(str, _SRCS)])
        os.replace(tmp, _SO)
    return _SO


class _Geom(ctypes.Structure):
    _fields_ = [("L", ctypes.c_int32), ("H", ctypes.c_int32),
                ("D", ctypes.c_int32), ("S", ctypes.c_int32),
                ("N", ctypes.c_int64)]


class _Req(ctypes.Structure):
    _fields_ = [("PT", ctypes.POINTER(ctypes.c_int32)),
                ("PT_len", ctypes.c_int64),
                ("tb", ctypes.c_int64), ("te", ctypes.c_int64)]


class _Layout(ctypes.Structure):
    _fields_ = [("off_elems", ctypes.c_int64), ("stride_tokens", ctypes.c_int64)]


class _Tag(ctypes.Structure):
    _fields_ = [("hash", ctypes.c_uint64), ("end_pos", ctypes.c_int64)]


TAG_DTYPE = np.dtype([("hash", np.uint64), ("end_pos", np.int64)])

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(str(build()))
        PP = ctypes.POINTER(ctypes.c_void_p)
        G, Rq = ctypes.POINTER(_Geom), ctypes.POINTER(_Req)
        i32, i64, vp = ctypes.c_int32, ctypes.c_int64, ctypes.c_void_p
        _lib.lumen_oracle_total_elems.restype = i64
        _lib.lumen_oracle_total_elems.argtypes = [G, Rq, i32]
        _lib.lumen_oracle_req_offset_elems.restype = i64
        _lib.lumen_oracle_req_offset_elems.argtypes = [G, Rq, i32]
        for name in ("lumen_oracle_pack", "lumen_oracle_pack_omp",
                     "lumen_oracle_unpack_omp"):
            f = getattr(_lib, name)
            f.restype = ctypes.c_int
            f.argtypes = [G, PP, PP, Rq, i32, vp, i64]
        _lib.lumen_oracle_unpack.restype = ctypes.c_int
        _lib.lumen_oracle_unpack.argtypes = [G, PP, PP, Rq, i32, vp, i64,
                                             ctypes.c_int]
        _lib.lumen_oracle_buffer_index.restype = i64
        _lib.lumen_oracle_buffer_index.argtypes = [G, Rq, i32, i32, i32, i64, i64]
        _lib.lumen_oracle_pool_index.restype = i64
        _lib.lumen_oracle_pool_index.argtypes = [G, Rq, i32, i64, i64]
        _lib.lumen_oracle_omp_threads.restype = ctypes.c_int
        Ly = ctypes.POINTER(_Layout)
        for name in ("lumen_oracle_pack_layout", "lumen_oracle_unpack_layout"):
            f = getattr(_lib, name)
            f.restype = ctypes.c_int
            f.argtypes = [G, PP, PP, Rq, Ly, i32, vp, i64]
        T = ctypes.POINTER(_Tag)
        _lib.tags_oracle_fnv1a64.restype = ctypes.c_uint64
        _lib.tags_oracle_fnv1a64.argtypes = [ctypes.c_char_p, i64]
        _lib.tags_oracle_num_pages.restype = i64
        _lib.tags_oracle_num_pages.argtypes = [i64, i64]
        _lib.tags_oracle_page_tags.restype = ctypes.c_int
        _lib.tags_oracle_page_tags.argtypes = [ctypes.POINTER(ctypes.c_int32), i64, i64, T]
        _lib.tags_oracle_longest_prefix.restype = i64
        _lib.tags_oracle_longest_prefix.argtypes = [T, i64, T, i64]
    return _lib


# ---------------------------------------------------------------------------
# marshalling: geometry is (L, H, D, S, N); requests are (page_table, tb, te)
# with page_table a 1-D int32 array; planes are lists of L uint16 arrays of
# N*S*H*D words each (any shape, C-contiguous).
# ---------------------------------------------------------------------------

def _geom(geom) -> _Geom:
    L, H, D, S, N = (int(x) for x in geom)
    return _Geom(L, H, D, S, N)


def _reqs(reqs):
    keep = []
    arr = (_Req * max(len(reqs), 1))()
    for i, (pt, tb, te) in enumerate(reqs):
        pt = np.ascontiguousarray(pt, dtype=np.int32)
        keep.append(pt)
        arr[i].PT = pt.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
        arr[i].PT_len = pt.size
        arr[i].tb, arr[i].te = int(tb), int(te)
    return arr, keep


def _planes(planes, L, words, writable):
    if len(planes) != L:
        raise ValueError("need one plane per layer")
    out = (ctypes.c_void_p * L)()
    for i, p in enumerate(planes):
        if p.dtype != np.uint16 or not p.flags.c_contiguous:
            raise ValueError("planes must be C-contiguous uint16")
        if writable and not p.flags.writeable:
            raise ValueError("plane not writable")
        if p.size < words:
            raise ValueError("plane smaller than N*S*H*D")
        out[i] = p.ctypes.data
    return out


def total_elems(geom, reqs) -> int:
    g = _geom(geom)
    arr, _keep = _reqs(reqs)
    return int(lib().lumen_oracle_total_elems(ctypes.byref(g), arr, len(reqs)))


def req_offset_elems(geom, reqs, r: int) -> int:
    g = _geom(geom)
    arr, _keep = _reqs(reqs)
    return int(lib().lumen_oracle_req_offset_elems(ctypes.byref(g), arr, r))


def pack(geom, k_planes, v_planes, reqs, *, omp: bool = False) -> np.ndarray:
    """C1.  Returns the checkpoint buffer as a 1-D uint16 array."""
    g = _geom(geom)
    L, H, D, S, N = (int(x) for x in geom)
    arr, _keep = _reqs(reqs)
    words = N * S * H * D
    kp = _planes(k_planes, L, words, False)
    vp = _planes(v_planes, L, words, False)
    n = int(lib().lumen_oracle_total_elems(ctypes.byref(g), arr, len(reqs)))
    B = np.zeros(max(n, 0), dtype=np.uint16)
    fn = lib().lumen_oracle_pack_omp if omp else lib().lumen_oracle_pack
    rc = fn(ctypes.byref(g), kp, vp, arr, len(reqs), B.ctypes.data, B.size)
    if rc:
        raise OracleError(rc)
    return B


def unpack(geom, k_planes, v_planes, reqs, B, *, omp: bool = False,
           check_overlap: bool = False) -> None:
    """C2.  Scatters buffer B into the planes in place."""
    g = _geom(geom)
    L, H, D, S, N = (int(x) for x in geom)
    arr, _keep = _reqs(reqs)
    words = N * S * H * D
    kp = _planes(k_planes, L, words, True)
    vp = _planes(v_planes, L, words, True)
    B = np.ascontiguousarray(B, dtype=np.uint16)
    if omp:
        rc = lib().lumen_oracle_unpack_omp(ctypes.byref(g), kp, vp, arr,
                                           len(reqs), B.ctypes.data, B.size)
    else:
        rc = lib().lumen_oracle_unpack(ctypes.byref(g), kp, vp, arr, len(reqs),
                                       B.ctypes.data, B.size,
                                       1 if check_overlap else 0)
    if rc:
        raise OracleError(rc)


def _layouts(layouts):
    arr = (_Layout * max(len(layouts), 1))()
    for i, (off, stride) in enumerate(layouts):
        arr[i].off_elems, arr[i].stride_tokens = int(off), int(stride)
    return arr


def pack_layout(geom, k_planes, v_planes, reqs, layouts, B: np.ndarray) -> None:
    """Pack into B (uint16, modified in place) with request r's block at element offset
    layouts[r][0] and plane stride layouts[r][1] tokens; other words of B are left alone."""
    g = _geom(geom)
    L, H, D, S, N = (int(x) for x in geom)
    arr, _keep = _reqs(reqs)
    words = N * S * H * D
    kp = _planes(k_planes, L, words, False)
    vp = _planes(v_planes, L, words, False)
    if B.dtype != np.uint16 or not B.flags.c_contiguous or not B.flags.writeable:
        raise ValueError("B must be a writable C-contiguous uint16 array")
    rc = lib().lumen_oracle_pack_layout(ctypes.byref(g), kp, vp, arr, _layouts(layouts), len(reqs),
                                        B.ctypes.data, B.size)
    if rc:
        raise OracleError(rc)


def unpack_layout(geom, k_planes, v_planes, reqs, layouts, B: np.ndarray) -> None:
    g = _geom(geom)
    L, H, D, S, N = (int(x) for x in geom)
    arr, _keep = _reqs(reqs)
    words = N * S * H * D
    kp = _planes(k_planes, L, words, True)
    vp = _planes(v_planes, L, words, True)
    B = np.ascontiguousarray(B, dtype=np.uint16)
    rc = lib().lumen_oracle_unpack_layout(ctypes.byref(g), kp, vp, arr, _layouts(layouts), len(reqs),
                                          B.ctypes.data, B.size)
    if rc:
        raise OracleError(rc)


def buffer_index(geom, reqs, r, l, c, j, e) -> int:
    g = _geom(geom)
    arr, _keep = _reqs(reqs)
    return int(lib().lumen_oracle_buffer_index(ctypes.byref(g), arr, r, l, c, j, e))


def pool_index(geom, reqs, r, j, e) -> int:
    g = _geom(geom)
    arr, _keep = _reqs(reqs)
    return int(lib().lumen_oracle_pool_index(ctypes.byref(g), arr, r, j, e))


def omp_threads() -> int:
    return int(lib().lumen_oracle_omp_threads())


# ---------------------------------------------------------------------------
# page tags (tags_oracle.c)
# ---------------------------------------------------------------------------

def fnv1a64(data: bytes) -> int:
    return int(lib().tags_oracle_fnv1a64(data, len(data)))


def page_tags(token_ids, S: int) -> np.ndarray:
    """Tags of every page of one request: structured array (hash u64, end_pos i64)."""
    tok = np.ascontiguousarray(token_ids, dtype=np.int32)
    n = int(lib().tags_oracle_num_pages(tok.size, int(S)))
    out = np.zeros(max(n, 0), dtype=TAG_DTYPE)
    rc = lib().tags_oracle_page_tags(tok.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), tok.size,
                                     int(S), out.ctypes.data_as(ctypes.POINTER(_Tag)))
    if rc:
        raise OracleError(rc)
    return out


def longest_prefix(regen: np.ndarray, stored: np.ndarray) -> int:
    """Tokens of the longest contiguous checkpointed prefix."""
    regen = np.ascontiguousarray(regen, dtype=TAG_DTYPE)
    stored = np.ascontiguousarray(stored, dtype=TAG_DTYPE)
    return int(lib().tags_oracle_longest_prefix(
        regen.ctypes.data_as(ctypes.POINTER(_Tag)), regen.size,
        stored.ctypes.data_as(ctypes.POINTER(_Tag)), stored.size))
