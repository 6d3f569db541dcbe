"""paper_2606_17787_b200 -- B200-native KV checkpoint pack / restore unpack.

The data-parallel hot path of LUMEN's load-aware KV checkpointing and recovery
(arxiv/paper_2606_17787; section 4.2 step 3, PAPER.md:157-163
section 4.3): hand-written sm_100a kernels behind the C ABI of
include/lumen_kv.h, plus this thin ctypes binding with the same names.
Build the library with `python -m paper_2606_17787_b200.build`.
"""
from .binding import (  # noqa: F401
    EXPORTS, LumenKVError, Plan, ReqArray, Stager, lumen_kv_chunk_info,
    lumen_kv_checkpoint_pack_staged, lumen_kv_restore_unpack_staged,
    lumen_kv_checkpoint_pack_staged_commit, lumen_kv_restore_unpack_staged_ready,
    lumen_kv_checkpoint_pack_staged_async, lumen_kv_restore_unpack_staged_async, lumen_kv_init, lumen_kv_set_option,
    TAG_DTYPE, SEGMENT_DTYPE, Store, BackgroundCheckpointer, lumen_kv_choose_holder, lumen_kv_recover, lumen_kv_tags_num_pages, lumen_kv_page_tags, lumen_kv_page_tags_host, lumen_kv_longest_prefix, library_path, lumen_kv_checkpoint_pack, lumen_kv_geom,
    lumen_kv_plan_build, lumen_kv_plan_free, lumen_kv_req, lumen_kv_restore_unpack, lumen_kv_copy_noalloc,
    lumen_kv_run_info, lumen_kv_req_layout, lumen_kv_strerror, lumen_kv_trim, lumen_kv_version, make_geom, plane_ptrs,
    LUMEN_KV_OK, LUMEN_KV_EINVAL, LUMEN_KV_ERANGE, LUMEN_KV_EOVERLAP, LUMEN_KV_ESIZE,
    LUMEN_KV_ENOMEM, LUMEN_KV_ECUDA, LUMEN_KV_ESINK, LUMEN_KV_ECAPACITY, LUMEN_KV_NOALLOC_MAX_RUNS,
    LUMEN_KV_NOALLOC_MAX_REQS, LUMEN_KV_DIR_PACK, LUMEN_KV_DIR_RESTORE, LUMEN_KV_VALIDATE_UNIQUE_DST, LUMEN_KV_MERGE_ADJACENT,
    LUMEN_KV_HOST_ONLY, LUMEN_KV_NO_INLINE, LUMEN_KV_KERNEL_AUTO, LUMEN_KV_KERNEL_WARP, LUMEN_KV_KERNEL_BULK,
    LUMEN_KV_MEM_DEVICE, LUMEN_KV_MEM_HOST_MAPPED, LUMEN_KV_MEM_DEVICE_PEER,
)
