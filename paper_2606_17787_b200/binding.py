"""ctypes binding of include/lumen_kv.h -- argument marshalling only.

Every step of the path (plan flattening, pack, unpack) runs inside
liblumen_kv.so; this module converts Python objects to the C structs and raises
LumenKVError on a negative status.  There is no fallback of any kind: if the
shared library is missing the import fails.

torch is *not* imported here.  Callers pass raw integers: device pointers
(`tensor.data_ptr()`), host pointers of pinned memory, and the `cudaStream_t`
handle (`torch.cuda.Stream.cuda_stream`).  Page tables are numpy int32 arrays.
"""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Iterable, Sequence, Tuple

import numpy as np

_SO = Path(__file__).resolve().parent / "liblumen_kv.so"

# ---- constants mirrored from include/lumen_kv.h -----------------------------------
LUMEN_KV_OK, LUMEN_KV_EINVAL, LUMEN_KV_ERANGE = 0, -1, -2
LUMEN_KV_EOVERLAP, LUMEN_KV_ESIZE, LUMEN_KV_ENOMEM, LUMEN_KV_ECUDA, LUMEN_KV_ESINK = -3, -4, -5, -6, -7
LUMEN_KV_ECAPACITY = -8
LUMEN_KV_NOALLOC_MAX_RUNS, LUMEN_KV_NOALLOC_MAX_REQS = 65536, 4096
LUMEN_KV_DIR_PACK, LUMEN_KV_DIR_RESTORE = 0, 1
LUMEN_KV_VALIDATE_UNIQUE_DST = 0x1
LUMEN_KV_MERGE_ADJACENT = 0x2
LUMEN_KV_HOST_ONLY = 0x4
LUMEN_KV_NO_INLINE = 0x8
LUMEN_KV_KERNEL_AUTO, LUMEN_KV_KERNEL_WARP, LUMEN_KV_KERNEL_BULK = 0x000, 0x100, 0x200
LUMEN_KV_MEM_DEVICE, LUMEN_KV_MEM_HOST_MAPPED, LUMEN_KV_MEM_DEVICE_PEER = 0, 1, 2

EXPORTS = (
    "lumen_kv_plan_build", "lumen_kv_plan_build_layout", "lumen_kv_plan_bytes", "lumen_kv_plan_req_offset",
    "lumen_kv_plan_num_runs", "lumen_kv_plan_get_run", "lumen_kv_checkpoint_pack",
    "lumen_kv_restore_unpack", "lumen_kv_copy_noalloc", "lumen_kv_plan_free", "lumen_kv_trim", "lumen_kv_init", "lumen_kv_set_option",
    "lumen_kv_checkpoint_pack_staged_async", "lumen_kv_restore_unpack_staged_async",
    "lumen_kv_stager_query", "lumen_kv_stager_wait", "lumen_kv_stager_sync",
    "lumen_kv_strerror", "lumen_kv_last_cuda_error", "lumen_kv_version",
    "lumen_kv_stager_create", "lumen_kv_stager_destroy", "lumen_kv_checkpoint_pack_staged",
    "lumen_kv_restore_unpack_staged", "lumen_kv_plan_num_chunks", "lumen_kv_plan_get_chunks",
    "lumen_kv_checkpoint_pack_staged_commit", "lumen_kv_restore_unpack_staged_ready",
    "lumen_kv_tags_num_pages", "lumen_kv_page_tags", "lumen_kv_page_tags_host", "lumen_kv_longest_prefix",
    "lumen_kv_store_create", "lumen_kv_store_destroy", "lumen_kv_store_available",
    "lumen_kv_store_reserved", "lumen_kv_store_reserve", "lumen_kv_store_release",
    "lumen_kv_store_append", "lumen_kv_store_tokens", "lumen_kv_store_lookup",
    "lumen_kv_store_segments", "lumen_kv_store_sink", "lumen_kv_store_sink_errors",
    "lumen_kv_store_acquire", "lumen_kv_store_abort", "lumen_kv_store_arena", "lumen_kv_ckpt_set_direct",
    "lumen_kv_store_restore",
    "lumen_kv_choose_holder", "lumen_kv_recover",
    "lumen_kv_ckpt_create", "lumen_kv_ckpt_destroy", "lumen_kv_ckpt_track", "lumen_kv_ckpt_untrack",
    "lumen_kv_ckpt_notify", "lumen_kv_ckpt_flush", "lumen_kv_ckpt_progress",
)


class lumen_kv_geom(ctypes.Structure):
    _fields_ = [("num_layers", ctypes.c_int32), ("kv_heads", ctypes.c_int32),
                ("head_dim", ctypes.c_int32), ("page_size", ctypes.c_int32),
                ("elem_bytes", ctypes.c_int32), ("reserved", ctypes.c_int32),
                ("num_pages", ctypes.c_int64), ("page_stride_bytes", ctypes.c_int64)]


class lumen_kv_req(ctypes.Structure):
    _fields_ = [("page_table", ctypes.c_void_p), ("page_table_len", ctypes.c_int64),
                ("t_begin", ctypes.c_int64), ("t_end", ctypes.c_int64)]


class lumen_kv_req_layout(ctypes.Structure):
    _fields_ = [("buf_offset", ctypes.c_int64), ("plane_stride_tokens", ctypes.c_int64)]


class lumen_kv_run_info(ctypes.Structure):
    _fields_ = [("src_slot", ctypes.c_int64), ("dst_token", ctypes.c_int64),
                ("req", ctypes.c_int32), ("count", ctypes.c_int32)]


class lumen_kv_chunk_info(ctypes.Structure):
    _fields_ = [("run_begin", ctypes.c_int64), ("run_end", ctypes.c_int64),
                ("plane_begin", ctypes.c_int32), ("plane_end", ctypes.c_int32),
                ("byte_begin", ctypes.c_int64), ("byte_end", ctypes.c_int64)]


# lumen_kv_sink_fn: (user, request_id, t_begin, t_end, delta pointer, delta_bytes, tags, n_tags)
SINK_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int64, ctypes.c_int64,
                           ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int32)


class LumenKVError(RuntimeError):
    def __init__(self, status: int, where: str):
        msg = _lib().lumen_kv_strerror(status).decode()
        cuda = _lib().lumen_kv_last_cuda_error() if status == LUMEN_KV_ECUDA else 0
        super().__init__(f"{where}: {msg} (status {status}" +
                         (f", cudaError {cuda})" if cuda else ")"))
        self.status = status
        self.cuda_error = cuda


_handle = None


def _lib() -> ctypes.CDLL:
    global _handle
    if _handle is not None:
        return _handle
    if not _SO.exists():
        raise ImportError(
            f"{_SO} is missing: run `python -m paper_2606_17787_b200.build` "
            "(nvcc, sm_100a).  There is no fallback path.")
    L = ctypes.CDLL(str(_SO))
    vp, i32, i64, u32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_uint32
    L.lumen_kv_plan_build.restype = ctypes.c_int
    L.lumen_kv_plan_build.argtypes = [ctypes.POINTER(lumen_kv_geom), ctypes.POINTER(lumen_kv_req),
                                      i32, u32, vp, ctypes.POINTER(vp)]
    L.lumen_kv_plan_build_layout.restype = ctypes.c_int
    L.lumen_kv_plan_build_layout.argtypes = [ctypes.POINTER(lumen_kv_geom), ctypes.POINTER(lumen_kv_req),
                                             ctypes.POINTER(lumen_kv_req_layout), i32, u32, vp,
                                             ctypes.POINTER(vp)]
    L.lumen_kv_plan_bytes.restype = i64
    L.lumen_kv_plan_bytes.argtypes = [vp]
    L.lumen_kv_plan_req_offset.restype = i64
    L.lumen_kv_plan_req_offset.argtypes = [vp, i32]
    L.lumen_kv_plan_num_runs.restype = i64
    L.lumen_kv_plan_num_runs.argtypes = [vp]
    L.lumen_kv_plan_get_run.restype = ctypes.c_int
    L.lumen_kv_plan_get_run.argtypes = [vp, i64, ctypes.POINTER(lumen_kv_run_info)]
    for name in ("lumen_kv_checkpoint_pack", "lumen_kv_restore_unpack"):
        f = getattr(L, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), vp, i64, ctypes.c_int, vp]
    L.lumen_kv_copy_noalloc.restype = ctypes.c_int
    L.lumen_kv_copy_noalloc.argtypes = [vp, ctypes.c_int, ctypes.POINTER(vp), ctypes.POINTER(vp), vp, i64,
                                        ctypes.c_int, vp]
    L.lumen_kv_stager_create.restype = ctypes.c_int
    L.lumen_kv_stager_create.argtypes = [vp, i64, i32, ctypes.POINTER(vp)]
    L.lumen_kv_stager_destroy.restype = None
    L.lumen_kv_stager_destroy.argtypes = [vp]
    for name in ("lumen_kv_checkpoint_pack_staged", "lumen_kv_restore_unpack_staged"):
        f = getattr(L, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), vp, i64, vp, vp]
    for name in ("lumen_kv_checkpoint_pack_staged_commit", "lumen_kv_restore_unpack_staged_ready"):
        f = getattr(L, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), vp, i64, vp, vp, vp, ctypes.c_uint64]
    for name in ("lumen_kv_checkpoint_pack_staged_async", "lumen_kv_restore_unpack_staged_async"):
        f = getattr(L, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), vp, i64, vp, vp, vp, ctypes.c_uint64,
                      ctypes.POINTER(ctypes.c_uint64)]
    L.lumen_kv_stager_query.restype = ctypes.c_int
    L.lumen_kv_stager_query.argtypes = [vp, ctypes.c_uint64]
    L.lumen_kv_stager_wait.restype = ctypes.c_int
    L.lumen_kv_stager_wait.argtypes = [vp, ctypes.c_uint64, vp]
    L.lumen_kv_stager_sync.restype = ctypes.c_int
    L.lumen_kv_stager_sync.argtypes = [vp, ctypes.c_uint64]
    L.lumen_kv_init.restype = ctypes.c_int
    L.lumen_kv_init.argtypes = []
    L.lumen_kv_set_option.restype = ctypes.c_int
    L.lumen_kv_set_option.argtypes = [ctypes.c_char_p, ctypes.c_int]
    L.lumen_kv_tags_num_pages.restype = i64
    L.lumen_kv_tags_num_pages.argtypes = [vp, i32, i32]
    L.lumen_kv_page_tags.restype = ctypes.c_int
    L.lumen_kv_page_tags.argtypes = [vp, vp, i32, i32, vp, i64, vp]
    L.lumen_kv_longest_prefix.restype = i64
    L.lumen_kv_longest_prefix.argtypes = [vp, i64, vp, i64]
    u64 = ctypes.c_uint64
    L.lumen_kv_store_create.restype = ctypes.c_int
    L.lumen_kv_store_create.argtypes = [vp, i64, i64, i32, i32, ctypes.POINTER(vp)]
    L.lumen_kv_store_destroy.restype = None
    L.lumen_kv_store_destroy.argtypes = [vp]
    for name in ("lumen_kv_store_available", "lumen_kv_store_reserved"):
        getattr(L, name).restype = i64
        getattr(L, name).argtypes = [vp]
    L.lumen_kv_store_reserve.restype = ctypes.c_int
    L.lumen_kv_store_reserve.argtypes = [vp, u64, i64]
    L.lumen_kv_store_release.restype = ctypes.c_int
    L.lumen_kv_store_release.argtypes = [vp, u64]
    L.lumen_kv_store_append.restype = ctypes.c_int
    L.lumen_kv_store_append.argtypes = [vp, u64, i64, i64, vp, i64, vp, i32]
    L.lumen_kv_store_tokens.restype = i64
    L.lumen_kv_store_tokens.argtypes = [vp, u64]
    L.lumen_kv_store_lookup.restype = i64
    L.lumen_kv_store_lookup.argtypes = [vp, u64, vp, i64]
    L.lumen_kv_store_restore.restype = ctypes.c_int
    L.lumen_kv_store_restore.argtypes = [vp, u64, vp, i64, ctypes.POINTER(lumen_kv_geom), vp, i64,
                                         ctypes.POINTER(vp), ctypes.POINTER(vp), vp, vp,
                                         ctypes.POINTER(i64)]
    L.lumen_kv_store_sink_errors.restype = i64
    L.lumen_kv_store_sink_errors.argtypes = [vp]
    L.lumen_kv_store_segments.restype = i64
    L.lumen_kv_store_segments.argtypes = [vp, u64, i64, vp, i64]
    L.lumen_kv_choose_holder.restype = ctypes.c_int
    L.lumen_kv_choose_holder.argtypes = [vp, vp, vp, vp, i32, i32, i64, ctypes.c_double,
                                         ctypes.c_double, ctypes.POINTER(i32)]
    L.lumen_kv_recover.restype = ctypes.c_int
    L.lumen_kv_recover.argtypes = [vp, vp, i32, vp, vp, i32, vp, vp, vp]
    L.lumen_kv_ckpt_create.restype = ctypes.c_int
    L.lumen_kv_ckpt_create.argtypes = [ctypes.POINTER(lumen_kv_geom), ctypes.POINTER(vp),
                                       ctypes.POINTER(vp), vp, i64, i32, vp, i64, SINK_FN, vp,
                                       ctypes.POINTER(vp)]
    L.lumen_kv_store_acquire.restype = vp
    L.lumen_kv_store_acquire.argtypes = [vp, u64, i64, i64, i64]
    L.lumen_kv_store_abort.restype = None
    L.lumen_kv_store_abort.argtypes = [vp, u64]
    L.lumen_kv_store_arena.restype = vp
    L.lumen_kv_store_arena.argtypes = [vp, ctypes.POINTER(i64)]
    L.lumen_kv_ckpt_set_direct.restype = ctypes.c_int
    L.lumen_kv_ckpt_set_direct.argtypes = [vp, vp, i64, vp, vp, i64]
    L.lumen_kv_ckpt_destroy.restype = None
    L.lumen_kv_ckpt_destroy.argtypes = [vp]
    L.lumen_kv_ckpt_track.restype = ctypes.c_int
    L.lumen_kv_ckpt_track.argtypes = [vp, ctypes.c_uint64, i64]
    L.lumen_kv_ckpt_untrack.restype = ctypes.c_int
    L.lumen_kv_ckpt_untrack.argtypes = [vp, ctypes.c_uint64]
    L.lumen_kv_ckpt_notify.restype = ctypes.c_int
    L.lumen_kv_ckpt_notify.argtypes = [vp, vp, ctypes.POINTER(lumen_kv_req), ctypes.POINTER(vp), i32, vp]
    L.lumen_kv_page_tags_host.restype = i64
    L.lumen_kv_page_tags_host.argtypes = [vp, i64, i64, i64, i32, vp, i64]
    L.lumen_kv_ckpt_flush.restype = ctypes.c_int
    L.lumen_kv_ckpt_flush.argtypes = [vp]
    L.lumen_kv_ckpt_progress.restype = i64
    L.lumen_kv_ckpt_progress.argtypes = [vp, ctypes.c_uint64]
    L.lumen_kv_plan_num_chunks.restype = i64
    L.lumen_kv_plan_num_chunks.argtypes = [vp, i64]
    L.lumen_kv_plan_get_chunks.restype = i64
    L.lumen_kv_plan_get_chunks.argtypes = [vp, i64, ctypes.POINTER(lumen_kv_chunk_info), i64]
    L.lumen_kv_plan_free.restype = None
    L.lumen_kv_plan_free.argtypes = [vp]
    L.lumen_kv_trim.restype = None
    L.lumen_kv_trim.argtypes = []
    L.lumen_kv_strerror.restype = ctypes.c_char_p
    L.lumen_kv_strerror.argtypes = [ctypes.c_int]
    L.lumen_kv_last_cuda_error.restype = ctypes.c_int
    L.lumen_kv_version.restype = ctypes.c_int
    _handle = L
    return L


def library_path() -> Path:
    return _SO


def make_geom(num_layers, kv_heads, head_dim, page_size, num_pages, *, elem_bytes=2,
              page_stride_bytes=0) -> lumen_kv_geom:
    return lumen_kv_geom(int(num_layers), int(kv_heads), int(head_dim), int(page_size),
                         int(elem_bytes), 0, int(num_pages), int(page_stride_bytes))


Req = Tuple[np.ndarray, int, int]


class Plan:
    """Owner of a `lumen_kv_plan*`; freed on close() / garbage collection."""

    def __init__(self, handle: int, geom: lumen_kv_geom, num_reqs: int):
        self._h = ctypes.c_void_p(handle)
        self.geom = geom
        self.num_reqs = num_reqs

    @property
    def handle(self) -> ctypes.c_void_p:
        if not self._h:
            raise ValueError("plan already freed")
        return self._h

    @property
    def nbytes(self) -> int:
        return int(_lib().lumen_kv_plan_bytes(self.handle))

    @property
    def num_runs(self) -> int:
        return int(_lib().lumen_kv_plan_num_runs(self.handle))

    def req_offset(self, r: int) -> int:
        v = int(_lib().lumen_kv_plan_req_offset(self.handle, int(r)))
        if v < 0:
            raise LumenKVError(v, "lumen_kv_plan_req_offset")
        return v

    def run(self, i: int) -> lumen_kv_run_info:
        info = lumen_kv_run_info()
        rc = _lib().lumen_kv_plan_get_run(self.handle, int(i), ctypes.byref(info))
        if rc:
            raise LumenKVError(rc, "lumen_kv_plan_get_run")
        return info

    def chunks(self, slot_bytes: int):
        """The chunks a staged call with this slot size is cut into (list of lumen_kv_chunk_info)."""
        n = int(_lib().lumen_kv_plan_num_chunks(self.handle, int(slot_bytes)))
        if n < 0:
            raise LumenKVError(n, "lumen_kv_plan_num_chunks")
        arr = (lumen_kv_chunk_info * max(n, 1))()
        m = int(_lib().lumen_kv_plan_get_chunks(self.handle, int(slot_bytes), arr, n))
        if m != n:
            raise LumenKVError(min(m, -1), "lumen_kv_plan_get_chunks")
        return [arr[i] for i in range(n)]

    def close(self) -> None:
        if self._h:
            _lib().lumen_kv_plan_free(self._h)
            self._h = ctypes.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


REQ_DTYPE = np.dtype([("page_table", np.uint64), ("page_table_len", np.int64),
                      ("t_begin", np.int64), ("t_end", np.int64)])
assert REQ_DTYPE.itemsize == ctypes.sizeof(lumen_kv_req)


class ReqArray:
    """A C array of lumen_kv_req kept as a numpy structured array, so that a serving loop
    can advance every request's delta range with one vectorised op per iteration
    (step a1) instead of re-marshalling Python tuples.  Owns the page tables."""

    def __init__(self, reqs: Sequence[Req]):
        self._tables = [np.ascontiguousarray(pt, dtype=np.int32) for pt, _, _ in reqs]
        self.arr = np.zeros(len(reqs), dtype=REQ_DTYPE)
        for i, ((_, tb, te), pt) in enumerate(zip(reqs, self._tables)):
            self.arr[i] = (pt.ctypes.data if pt.size else 0, pt.size, int(tb), int(te))

    def __len__(self) -> int:
        return self.arr.size

    def set_ranges(self, t_begin, t_end) -> None:
        self.arr["t_begin"] = t_begin
        self.arr["t_end"] = t_end

    def advance(self, tokens: int) -> None:
        """[tb, te) <- [te, te + tokens): the next incremental delta."""
        self.arr["t_begin"] = self.arr["t_end"]
        self.arr["t_end"] += int(tokens)


def lumen_kv_plan_build(geom: lumen_kv_geom, reqs, flags: int = 0, stream: int = 0,
                        layouts=None) -> Plan:
    """reqs: a ReqArray, or a sequence of (page_table int32 ndarray, t_begin, t_end).
    layouts: None (dense buffer) or one (buf_offset bytes, plane_stride_tokens) per request
    (lumen_kv_plan_build_layout)."""
    lay = None
    if layouts is not None:
        if len(layouts) != len(reqs):
            raise ValueError("one layout per request")
        lay = (lumen_kv_req_layout * max(len(layouts), 1))()
        for i, (off, stride) in enumerate(layouts):
            lay[i].buf_offset, lay[i].plane_stride_tokens = int(off), int(stride)
    keep = []
    if isinstance(reqs, ReqArray):
        n = len(reqs)
        arr = ctypes.cast(reqs.arr.ctypes.data, ctypes.POINTER(lumen_kv_req))
    else:
        n = len(reqs)
        arr = (lumen_kv_req * max(n, 1))()
        for i, (pt, tb, te) in enumerate(reqs):
            pt = np.ascontiguousarray(pt, dtype=np.int32)
            keep.append(pt)
            arr[i].page_table = pt.ctypes.data if pt.size else None
            arr[i].page_table_len = pt.size
            arr[i].t_begin, arr[i].t_end = int(tb), int(te)
    out = ctypes.c_void_p()
    rc = _lib().lumen_kv_plan_build_layout(ctypes.byref(geom), arr, lay, n, int(flags),
                                           ctypes.c_void_p(int(stream)), ctypes.byref(out))
    del keep
    if rc:
        raise LumenKVError(rc, "lumen_kv_plan_build")
    return Plan(out.value, geom, n)


def _ptr_array(ptrs: Iterable[int], L: int):
    ptrs = list(ptrs)
    if len(ptrs) != L:
        raise ValueError(f"need {L} plane pointers, got {len(ptrs)}")
    return (ctypes.c_void_p * L)(*[int(p) for p in ptrs])


def plane_ptrs(ptrs: Iterable[int], L: int):
    """Pre-marshal a list of device pointers once (reuse it across calls)."""
    return _ptr_array(ptrs, L)


def _as_ptr_array(x, L):
    return x if isinstance(x, ctypes.Array) else _ptr_array(x, L)


def lumen_kv_checkpoint_pack(plan: Plan, k_planes, v_planes, dst: int, dst_bytes: int,
                             dst_kind: int = LUMEN_KV_MEM_DEVICE, stream: int = 0) -> None:
    L = plan.geom.num_layers
    rc = _lib().lumen_kv_checkpoint_pack(plan.handle, _as_ptr_array(k_planes, L),
                                         _as_ptr_array(v_planes, L), ctypes.c_void_p(int(dst)),
                                         int(dst_bytes), int(dst_kind),
                                         ctypes.c_void_p(int(stream)))
    if rc:
        raise LumenKVError(rc, "lumen_kv_checkpoint_pack")


def lumen_kv_restore_unpack(plan: Plan, k_planes, v_planes, src: int, src_bytes: int,
                            src_kind: int = LUMEN_KV_MEM_DEVICE, stream: int = 0) -> None:
    L = plan.geom.num_layers
    rc = _lib().lumen_kv_restore_unpack(plan.handle, _as_ptr_array(k_planes, L),
                                        _as_ptr_array(v_planes, L), ctypes.c_void_p(int(src)),
                                        int(src_bytes), int(src_kind),
                                        ctypes.c_void_p(int(stream)))
    if rc:
        raise LumenKVError(rc, "lumen_kv_restore_unpack")


def lumen_kv_copy_noalloc(plan: Plan, direction: int, k_planes, v_planes, buf: int, buf_bytes: int,
                          buf_kind: int = LUMEN_KV_MEM_DEVICE, stream: int = 0) -> None:
    """Pack (LUMEN_KV_DIR_PACK) or restore (LUMEN_KV_DIR_RESTORE) without any GPU allocation, for a
    worker whose HBM is all committed to its KV pool or whose decode loop cannot take the device-wide
    stall of a cudaMalloc: the descriptors go into an array built into the library (at most
    LUMEN_KV_NOALLOC_MAX_RUNS runs / LUMEN_KV_NOALLOC_MAX_REQS requests, else LUMEN_KV_ECAPACITY).
    Build the plan with LUMEN_KV_HOST_ONLY; keep all such calls of a device on one stream (they share
    the array).  Same bytes as lumen_kv_checkpoint_pack / lumen_kv_restore_unpack."""
    L = plan.geom.num_layers
    rc = _lib().lumen_kv_copy_noalloc(plan.handle, int(direction), _as_ptr_array(k_planes, L),
                                      _as_ptr_array(v_planes, L), ctypes.c_void_p(int(buf)),
                                      int(buf_bytes), int(buf_kind), ctypes.c_void_p(int(stream)))
    if rc:
        raise LumenKVError(rc, "lumen_kv_copy_noalloc")


class Stager:
    """Owner of a `lumen_kv_stager*` over caller-provided device staging memory."""

    def __init__(self, staging_ptr: int, slot_bytes: int, n_slots: int):
        out = ctypes.c_void_p()
        rc = _lib().lumen_kv_stager_create(ctypes.c_void_p(int(staging_ptr)), int(slot_bytes),
                                           int(n_slots), ctypes.byref(out))
        if rc:
            raise LumenKVError(rc, "lumen_kv_stager_create")
        self._h = out
        self.slot_bytes, self.n_slots = int(slot_bytes), int(n_slots)

    @property
    def handle(self) -> ctypes.c_void_p:
        if not self._h:
            raise ValueError("stager already destroyed")
        return self._h

    def query(self, ticket: int) -> bool:
        """True once the asynchronous call `ticket` is complete; raises if it failed."""
        rc = int(_lib().lumen_kv_stager_query(self.handle, int(ticket)))
        if rc < 0:
            raise LumenKVError(rc, "lumen_kv_stager_query")
        return rc == 1

    def wait(self, ticket: int, stream: int = 0) -> None:
        """Make `stream` wait for the ticket (blocks the host only until it has been issued)."""
        rc = int(_lib().lumen_kv_stager_wait(self.handle, int(ticket), ctypes.c_void_p(int(stream))))
        if rc:
            raise LumenKVError(rc, "lumen_kv_stager_wait")

    def sync(self, ticket: int) -> None:
        rc = int(_lib().lumen_kv_stager_sync(self.handle, int(ticket)))
        if rc:
            raise LumenKVError(rc, "lumen_kv_stager_sync")

    def close(self) -> None:
        if self._h:
            _lib().lumen_kv_stager_destroy(self._h)
            self._h = ctypes.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lumen_kv_checkpoint_pack_staged(plan: Plan, k_planes, v_planes, dst_host: int, dst_bytes: int,
                                    stager: Stager, stream: int = 0) -> None:
    L = plan.geom.num_layers
    rc = _lib().lumen_kv_checkpoint_pack_staged(
        plan.handle, _as_ptr_array(k_planes, L), _as_ptr_array(v_planes, L),
        ctypes.c_void_p(int(dst_host)), int(dst_bytes), stager.handle, ctypes.c_void_p(int(stream)))
    if rc:
        raise LumenKVError(rc, "lumen_kv_checkpoint_pack_staged")


def lumen_kv_restore_unpack_staged(plan: Plan, k_planes, v_planes, src_host: int, src_bytes: int,
                                   stager: Stager, stream: int = 0) -> None:
    L = plan.geom.num_layers
    rc = _lib().lumen_kv_restore_unpack_staged(
        plan.handle, _as_ptr_array(k_planes, L), _as_ptr_array(v_planes, L),
        ctypes.c_void_p(int(src_host)), int(src_bytes), stager.handle, ctypes.c_void_p(int(stream)))
    if rc:
        raise LumenKVError(rc, "lumen_kv_restore_unpack_staged")


def lumen_kv_checkpoint_pack_staged_commit(plan: Plan, k_planes, v_planes, dst_host: int,
                                           dst_bytes: int, stager: Stager, stream: int,
                                           flags_host: int, epoch: int) -> None:
    """flags_host: host pointer of a pinned uint64 array, one word per chunk."""
    L = plan.geom.num_layers
    rc = _lib().lumen_kv_checkpoint_pack_staged_commit(
        plan.handle, _as_ptr_array(k_planes, L), _as_ptr_array(v_planes, L),
        ctypes.c_void_p(int(dst_host)), int(dst_bytes), stager.handle, ctypes.c_void_p(int(stream)),
        ctypes.c_void_p(int(flags_host)), int(epoch))
    if rc:
        raise LumenKVError(rc, "lumen_kv_checkpoint_pack_staged_commit")


def lumen_kv_restore_unpack_staged_ready(plan: Plan, k_planes, v_planes, src_host: int,
                                         src_bytes: int, stager: Stager, stream: int,
                                         flags_host: int, epoch: int) -> None:
    L = plan.geom.num_layers
    rc = _lib().lumen_kv_restore_unpack_staged_ready(
        plan.handle, _as_ptr_array(k_planes, L), _as_ptr_array(v_planes, L),
        ctypes.c_void_p(int(src_host)), int(src_bytes), stager.handle, ctypes.c_void_p(int(stream)),
        ctypes.c_void_p(int(flags_host)), int(epoch))
    if rc:
        raise LumenKVError(rc, "lumen_kv_restore_unpack_staged_ready")


def _staged_async(name, plan, k_planes, v_planes, host, nbytes, stager, stream, flags_host, epoch) -> int:
    L = plan.geom.num_layers
    ticket = ctypes.c_uint64(0)
    rc = getattr(_lib(), name)(
        plan.handle, _as_ptr_array(k_planes, L), _as_ptr_array(v_planes, L), ctypes.c_void_p(int(host)),
        int(nbytes), stager.handle, ctypes.c_void_p(int(stream)),
        ctypes.c_void_p(int(flags_host)) if flags_host else None, int(epoch), ctypes.byref(ticket))
    if rc:
        raise LumenKVError(rc, name)
    return int(ticket.value)


def lumen_kv_checkpoint_pack_staged_async(plan: Plan, k_planes, v_planes, dst_host: int, dst_bytes: int,
                                          stager: Stager, stream: int = 0, flags_host: int = 0,
                                          epoch: int = 0) -> int:
    """Returns at once with a ticket; the stager's thread issues the chunk pipeline
    (Stager.query / wait / sync)."""
    return _staged_async("lumen_kv_checkpoint_pack_staged_async", plan, k_planes, v_planes, dst_host,
                         dst_bytes, stager, stream, flags_host, epoch)


def lumen_kv_restore_unpack_staged_async(plan: Plan, k_planes, v_planes, src_host: int, src_bytes: int,
                                         stager: Stager, stream: int = 0, flags_host: int = 0,
                                         epoch: int = 0) -> int:
    return _staged_async("lumen_kv_restore_unpack_staged_async", plan, k_planes, v_planes, src_host,
                         src_bytes, stager, stream, flags_host, epoch)


def lumen_kv_set_option(name: str, value: int) -> None:
    rc = _lib().lumen_kv_set_option(name.encode(), int(value))
    if rc:
        raise LumenKVError(rc, "lumen_kv_set_option")


def lumen_kv_init() -> None:
    rc = _lib().lumen_kv_init()
    if rc:
        raise LumenKVError(rc, "lumen_kv_init")


TAG_DTYPE = np.dtype([("hash", np.uint64), ("end_pos", np.int64)])   # lumen_kv_tag


def lumen_kv_tags_num_pages(tok_offset, page_size: int) -> int:
    off = np.ascontiguousarray(tok_offset, dtype=np.int64)
    n = int(_lib().lumen_kv_tags_num_pages(off.ctypes.data, off.size - 1, int(page_size)))
    if n < 0:
        raise LumenKVError(n, "lumen_kv_tags_num_pages")
    return n


def lumen_kv_page_tags(token_ids_dev: int, tok_offset, page_size: int, tags_out_dev: int,
                       tags_cap: int, stream: int = 0) -> None:
    """token_ids_dev / tags_out_dev: device pointers; tok_offset: host int64 array (R + 1)."""
    off = np.ascontiguousarray(tok_offset, dtype=np.int64)
    rc = _lib().lumen_kv_page_tags(ctypes.c_void_p(int(token_ids_dev)), off.ctypes.data, off.size - 1,
                                   int(page_size), ctypes.c_void_p(int(tags_out_dev)), int(tags_cap),
                                   ctypes.c_void_p(int(stream)))
    if rc:
        raise LumenKVError(rc, "lumen_kv_page_tags")


def lumen_kv_page_tags_host(token_ids, first_token: int, t_begin: int, t_end: int, page_size: int) -> np.ndarray:
    """Tags of the pages [t_begin, t_end) touches; token_ids[0] is token `first_token`."""
    tok = np.ascontiguousarray(token_ids, dtype=np.int32)
    cap = max(0, (int(t_end) - 1) // int(page_size) - int(t_begin) // int(page_size) + 1) if t_end > t_begin else 0
    out = np.zeros(cap, dtype=TAG_DTYPE)
    n = int(_lib().lumen_kv_page_tags_host(tok.ctypes.data, int(first_token), int(t_begin), int(t_end),
                                           int(page_size), out.ctypes.data, cap))
    if n < 0:
        raise LumenKVError(n, "lumen_kv_page_tags_host")
    return out[:n]


def lumen_kv_longest_prefix(regen: np.ndarray, stored: np.ndarray) -> int:
    """regen, stored: host arrays of TAG_DTYPE.  Returns tokens of the longest contiguous prefix."""
    a = np.ascontiguousarray(regen, dtype=TAG_DTYPE)
    b = np.ascontiguousarray(stored, dtype=TAG_DTYPE)
    n = int(_lib().lumen_kv_longest_prefix(a.ctypes.data, a.size, b.ctypes.data, b.size))
    if n < 0:
        raise LumenKVError(n, "lumen_kv_longest_prefix")
    return n


SEGMENT_DTYPE = np.dtype([("t_begin", np.int64), ("t_end", np.int64), ("buf_offset", np.int64),
                          ("plane_stride_tokens", np.int64)])          # lumen_kv_segment


class Store:
    """Owner of a `lumen_kv_store*` over a caller-provided host arena (pointer + size)."""

    def __init__(self, arena_ptr: int, arena_bytes: int, token_bytes: int, page_size: int,
                 copy_threads: int = 1):
        out = ctypes.c_void_p()
        rc = _lib().lumen_kv_store_create(ctypes.c_void_p(int(arena_ptr)), int(arena_bytes),
                                          int(token_bytes), int(page_size), int(copy_threads),
                                          ctypes.byref(out))
        if rc:
            raise LumenKVError(rc, "lumen_kv_store_create")
        self._h = out
        self.token_bytes = int(token_bytes)

    def _check(self, rc, where):
        if rc < 0:
            raise LumenKVError(int(rc), where)
        return int(rc)

    @property
    def available(self) -> int:
        return self._check(_lib().lumen_kv_store_available(self._h), "lumen_kv_store_available")

    @property
    def reserved(self) -> int:
        return self._check(_lib().lumen_kv_store_reserved(self._h), "lumen_kv_store_reserved")

    def reserve(self, request_id: int, max_tokens: int) -> None:
        self._check(_lib().lumen_kv_store_reserve(self._h, int(request_id), int(max_tokens)),
                    "lumen_kv_store_reserve")

    def release(self, request_id: int) -> None:
        self._check(_lib().lumen_kv_store_release(self._h, int(request_id)), "lumen_kv_store_release")

    def append(self, request_id: int, t_begin: int, t_end: int, delta_ptr: int, delta_bytes: int,
               tags: np.ndarray) -> None:
        t = np.ascontiguousarray(tags, dtype=TAG_DTYPE)
        self._check(_lib().lumen_kv_store_append(self._h, int(request_id), int(t_begin), int(t_end),
                                                 ctypes.c_void_p(int(delta_ptr)), int(delta_bytes),
                                                 t.ctypes.data, t.size), "lumen_kv_store_append")

    def tokens(self, request_id: int) -> int:
        return self._check(_lib().lumen_kv_store_tokens(self._h, int(request_id)), "lumen_kv_store_tokens")

    def lookup(self, request_id: int, regen: np.ndarray) -> int:
        t = np.ascontiguousarray(regen, dtype=TAG_DTYPE)
        return self._check(_lib().lumen_kv_store_lookup(self._h, int(request_id), t.ctypes.data, t.size),
                           "lumen_kv_store_lookup")

    def restore(self, request_id: int, token_ids, geom: lumen_kv_geom, page_table, k_planes, v_planes,
                stager: "Stager", stream: int = 0) -> int:
        """KV-reuse recovery of one request (lumen_kv_store_restore); returns the restored prefix."""
        tok = np.ascontiguousarray(token_ids, dtype=np.int32)
        pt = np.ascontiguousarray(page_table, dtype=np.int32)
        L = geom.num_layers
        out = ctypes.c_int64(0)
        rc = _lib().lumen_kv_store_restore(self._h, int(request_id), tok.ctypes.data, tok.size,
                                           ctypes.byref(geom), pt.ctypes.data, pt.size,
                                           _as_ptr_array(k_planes, L), _as_ptr_array(v_planes, L),
                                           stager.handle, ctypes.c_void_p(int(stream)), ctypes.byref(out))
        if rc:
            raise LumenKVError(rc, "lumen_kv_store_restore")
        return int(out.value)

    def acquire(self, request_id: int, t_begin: int, t_end: int) -> int:
        """Claim [t_begin, t_end) at the request's tail; returns the arena address (0: refused)."""
        p = _lib().lumen_kv_store_acquire(self._h, int(request_id), int(t_begin), int(t_end),
                                          (int(t_end) - int(t_begin)) * self.token_bytes)
        return int(p or 0)

    def abort(self, request_id: int) -> None:
        _lib().lumen_kv_store_abort(self._h, int(request_id))

    @property
    def sink_errors(self) -> int:
        return self._check(_lib().lumen_kv_store_sink_errors(self._h), "lumen_kv_store_sink_errors")

    def segments(self, request_id: int, prefix_tokens: int) -> np.ndarray:
        n = self._check(_lib().lumen_kv_store_segments(self._h, int(request_id), int(prefix_tokens),
                                                       None, 0), "lumen_kv_store_segments")
        out = np.zeros(n, dtype=SEGMENT_DTYPE)
        self._check(_lib().lumen_kv_store_segments(self._h, int(request_id), int(prefix_tokens),
                                                   out.ctypes.data, n), "lumen_kv_store_segments")
        return out

    def close(self) -> None:
        if self._h:
            _lib().lumen_kv_store_destroy(self._h)
            self._h = ctypes.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lumen_kv_choose_holder(q, held, available, serving: int, footprint: int, lam: float,
                           bandwidth: float) -> int:
    """Eq. (1).  held: per worker, the reserved footprints of the checkpoints it holds.
    Returns h(r), or -1 if no worker can hold the checkpoint."""
    qa = np.ascontiguousarray(q, dtype=np.float64)
    begin = np.zeros(len(held) + 1, dtype=np.int32)
    begin[1:] = np.cumsum([len(h) for h in held])
    flat = np.ascontiguousarray([x for h in held for x in h], dtype=np.int64)
    av = np.ascontiguousarray(available, dtype=np.int64)
    out = ctypes.c_int32(-1)
    rc = _lib().lumen_kv_choose_holder(qa.ctypes.data, flat.ctypes.data if flat.size else None,
                                       begin.ctypes.data, av.ctypes.data, qa.size, int(serving),
                                       int(footprint), float(lam), float(bandwidth), ctypes.byref(out))
    if rc:
        raise LumenKVError(rc, "lumen_kv_choose_holder")
    return int(out.value)


def lumen_kv_recover(load, alive, interrupted):
    """interrupted: (holder, checkpointed size) per request.  Returns (assign, reuse, final loads)."""
    la = np.ascontiguousarray(load, dtype=np.int64)
    al = np.ascontiguousarray(alive, dtype=np.uint8)
    n = len(interrupted)
    ho = np.ascontiguousarray([h for h, _ in interrupted], dtype=np.int32)
    sz = np.ascontiguousarray([s for _, s in interrupted], dtype=np.int64)
    assign, reuse = np.zeros(n, dtype=np.int32), np.zeros(n, dtype=np.uint8)
    final = np.zeros(la.size, dtype=np.int64)
    rc = _lib().lumen_kv_recover(la.ctypes.data, al.ctypes.data, la.size,
                                 ho.ctypes.data if n else None, sz.ctypes.data if n else None, n,
                                 assign.ctypes.data if n else None, reuse.ctypes.data if n else None,
                                 final.ctypes.data)
    if rc:
        raise LumenKVError(rc, "lumen_kv_recover")
    return assign.tolist(), [bool(x) for x in reuse], final.tolist()


class BackgroundCheckpointer:
    """Owner of a `lumen_kv_ckpt*` (the worker's background checkpointing thread).
    sink(request_id, t_begin, t_end, delta_ptr, delta_bytes, tags) is called on that thread
    (tags: a TAG_DTYPE array, empty unless notify() was given token IDs) and returns None / 0
    when it took the delta, another int to reject it (an exception rejects it too and is chained
    to the error flush() raises); or pass a Store."""

    def __init__(self, geom: lumen_kv_geom, k_planes, v_planes, staging_ptr: int, slot_bytes: int,
                 n_slots: int, pinned_ptr: int, pinned_bytes: int, sink, direct_min_bytes=1 << 20):
        """direct_min_bytes (Store sinks only): batches whose average delta is at least this large are
        copied straight into the store's arena (lumen_kv_ckpt_set_direct) when the arena is pinned;
        None switches that off.  `self.direct` tells whether it is on."""
        L = geom.num_layers
        self.direct = False
        self.sink_exception = None       # first exception a Python sink raised (re-raised by flush)
        if isinstance(sink, Store):      # native sink: deltas go straight into the store, no Python
            self._keep = sink
            self._cb = ctypes.cast(_lib().lumen_kv_store_sink, SINK_FN)
            user = sink._h
        else:
            def _call(_u, rid, tb, te, ptr, nb, tags, n_tags):
                t = (np.ctypeslib.as_array((ctypes.c_uint8 * (16 * n_tags)).from_address(tags)).view(TAG_DTYPE).copy()
                     if n_tags else np.zeros(0, dtype=TAG_DTYPE))
                # ctypes swallows an exception raised inside a callback and hands 0 to the C side,
                # which would read "taken" and drop the delta silently: reject it instead, and keep
                # the exception for flush()
                try:
                    rc = sink(int(rid), int(tb), int(te), int(ptr), int(nb), t)
                    return int(rc) if rc else 0      # None / 0: taken; anything else: rejected
                except BaseException as exc:         # noqa: BLE001
                    if self.sink_exception is None:
                        self.sink_exception = exc
                    return -1
            self._cb = SINK_FN(_call)
            user = None
        out = ctypes.c_void_p()
        rc = _lib().lumen_kv_ckpt_create(ctypes.byref(geom), _as_ptr_array(k_planes, L),
                                         _as_ptr_array(v_planes, L), ctypes.c_void_p(int(staging_ptr)),
                                         int(slot_bytes), int(n_slots), ctypes.c_void_p(int(pinned_ptr)),
                                         int(pinned_bytes), self._cb, user, ctypes.byref(out))
        if rc:
            raise LumenKVError(rc, "lumen_kv_ckpt_create")
        self._h = out
        if isinstance(sink, Store) and direct_min_bytes is not None:
            nb = ctypes.c_int64(0)
            arena = _lib().lumen_kv_store_arena(sink._h, ctypes.byref(nb))
            rc = _lib().lumen_kv_ckpt_set_direct(self._h, ctypes.c_void_p(arena), nb.value,
                                                 ctypes.cast(_lib().lumen_kv_store_acquire, ctypes.c_void_p),
                                                 ctypes.cast(_lib().lumen_kv_store_abort, ctypes.c_void_p),
                                                 int(direct_min_bytes))
            if rc not in (LUMEN_KV_OK, LUMEN_KV_EINVAL):     # EINVAL: the arena is not pinned memory
                raise LumenKVError(rc, "lumen_kv_ckpt_set_direct")
            self.direct = rc == LUMEN_KV_OK

    def _check(self, rc, where):
        if rc < 0:
            raise LumenKVError(int(rc), where)
        return int(rc)

    def track(self, request_id: int, t_prev: int = 0) -> None:
        self._check(_lib().lumen_kv_ckpt_track(self._h, int(request_id), int(t_prev)), "lumen_kv_ckpt_track")

    def untrack(self, request_id: int) -> None:
        self._check(_lib().lumen_kv_ckpt_untrack(self._h, int(request_id)), "lumen_kv_ckpt_untrack")

    def notify(self, ids, reqs, ready_event: int = 0, token_ids=None) -> None:
        """reqs: (page_table, _, t_cur) per id; ready_event: a cudaEvent_t handle or 0;
        token_ids: None or one int32 array (the request's token history [0, t_cur)) per id."""
        n = len(ids)
        toks = None
        if token_ids is not None:
            tk = [np.ascontiguousarray(t, dtype=np.int32) for t in token_ids]
            toks = (ctypes.c_void_p * max(n, 1))(*[t.ctypes.data for t in tk])
        ida = np.ascontiguousarray(ids, dtype=np.uint64)
        arr = (lumen_kv_req * max(n, 1))()
        keep = []
        for i, (pt, _tb, te) in enumerate(reqs):
            pt = np.ascontiguousarray(pt, dtype=np.int32)
            keep.append(pt)
            arr[i].page_table = pt.ctypes.data if pt.size else None
            arr[i].page_table_len = pt.size
            arr[i].t_begin, arr[i].t_end = 0, int(te)
        self._check(_lib().lumen_kv_ckpt_notify(self._h, ida.ctypes.data, arr, toks, n,
                                                ctypes.c_void_p(int(ready_event))), "lumen_kv_ckpt_notify")

    def flush(self) -> None:
        """Raises LumenKVError(LUMEN_KV_ESINK) if a delta was rejected; if the rejection was an
        exception raised by a Python sink, that exception is its __cause__ (once)."""
        try:
            self._check(_lib().lumen_kv_ckpt_flush(self._h), "lumen_kv_ckpt_flush")
        except LumenKVError as e:
            exc, self.sink_exception = self.sink_exception, None
            if exc is not None:
                raise e from exc
            raise

    def progress(self, request_id: int) -> int:
        return self._check(_lib().lumen_kv_ckpt_progress(self._h, int(request_id)), "lumen_kv_ckpt_progress")

    def close(self) -> None:
        if self._h:
            _lib().lumen_kv_ckpt_destroy(self._h)
            self._h = ctypes.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lumen_kv_plan_free(plan: Plan) -> None:
    plan.close()


def lumen_kv_trim() -> None:
    _lib().lumen_kv_trim()


def lumen_kv_strerror(status: int) -> str:
    return _lib().lumen_kv_strerror(int(status)).decode()


def lumen_kv_version() -> int:
    return int(_lib().lumen_kv_version())
