"""Thin torch plumbing around the C ABI: device memory, pinned host memory, streams.

Nothing here moves KV bytes -- that is liblumen_kv.so's job.  KVPool allocates the
2L planes of a paged pool as separate torch CUDA tensors (one per (layer, K|V), as
vLLM/SGLang-style engines do; reading A9 of DESIGN.md) and keeps their device
pointers marshalled for the binding.  Checkpointer is the user-facing call: one
object per pool, pack()/unpack() taking request lists and a torch tensor buffer.
"""
from __future__ import annotations

from typing import List, Optional, Sequence

import torch

from . import binding as B


class KVPool:
    """2L planes [N, S, H, D] of 16-bit words on one CUDA device."""

    def __init__(self, num_layers: int, kv_heads: int, head_dim: int, page_size: int,
                 num_pages: int, device: Optional[torch.device] = None,
                 dtype: torch.dtype = torch.bfloat16):
        if not torch.cuda.is_available():
            raise RuntimeError("KVPool needs a CUDA device (there is no CPU path)")
        if torch.empty(0, dtype=dtype).element_size() != 2:
            raise ValueError("16-bit element types only")
        self.device = torch.device(device if device is not None else "cuda")
        self.geom = B.make_geom(num_layers, kv_heads, head_dim, page_size, num_pages)
        shape = (num_pages, page_size, kv_heads, head_dim)
        self.k: List[torch.Tensor] = [torch.empty(shape, dtype=dtype, device=self.device)
                                      for _ in range(num_layers)]
        self.v: List[torch.Tensor] = [torch.empty(shape, dtype=dtype, device=self.device)
                                      for _ in range(num_layers)]
        self.k_ptrs = B.plane_ptrs([t.data_ptr() for t in self.k], num_layers)
        self.v_ptrs = B.plane_ptrs([t.data_ptr() for t in self.v], num_layers)

    @property
    def num_layers(self) -> int:
        return self.geom.num_layers

    @property
    def row_bytes(self) -> int:
        return self.geom.kv_heads * self.geom.head_dim * self.geom.elem_bytes

    @property
    def token_bytes(self) -> int:
        return 2 * self.geom.num_layers * self.row_bytes

    def planes(self) -> List[torch.Tensor]:
        """K0, V0, K1, V1, ... (plane index = 2*layer + {0: K, 1: V})."""
        out = []
        for k, v in zip(self.k, self.v):
            out += [k, v]
        return out


def pinned_buffer(nbytes: int) -> torch.Tensor:
    """Page-locked, device-mapped host buffer (uint8) for LUMEN_KV_MEM_HOST_MAPPED."""
    return torch.empty(int(nbytes), dtype=torch.uint8, pin_memory=True)


def _kind_of(buf: torch.Tensor) -> int:
    if buf.is_cuda:
        return B.LUMEN_KV_MEM_DEVICE
    if buf.is_pinned():
        return B.LUMEN_KV_MEM_HOST_MAPPED
    raise ValueError("checkpoint buffer must be a CUDA tensor or a pinned host tensor")


class StagingRing:
    """Device staging memory + the library's stager for the two-stage host path
    (lumen_kv_checkpoint_pack_staged / lumen_kv_restore_unpack_staged)."""

    def __init__(self, slot_bytes: int = 32 << 20, n_slots: int = 3,
                 device: Optional[torch.device] = None):
        self.mem = torch.empty(int(slot_bytes) * int(n_slots), dtype=torch.uint8,
                               device=torch.device(device if device is not None else "cuda"))
        self.stager = B.Stager(self.mem.data_ptr(), slot_bytes, n_slots)

    def close(self) -> None:
        self.stager.close()


class Checkpointer:
    """pack()/unpack() on the current torch CUDA stream (or an explicit one)."""

    def __init__(self, pool: KVPool, flags: int = 0):
        self.pool = pool
        self.flags = int(flags)

    def plan(self, reqs: Sequence, *, unique_dst: bool = False, stream=None, layouts=None) -> B.Plan:
        s = stream if stream is not None else torch.cuda.current_stream(self.pool.device)
        f = self.flags | (B.LUMEN_KV_VALIDATE_UNIQUE_DST if unique_dst else 0)
        return B.lumen_kv_plan_build(self.pool.geom, reqs, f, s.cuda_stream, layouts)

    def pack(self, plan: B.Plan, buf: torch.Tensor, *, stream=None) -> None:
        s = stream if stream is not None else torch.cuda.current_stream(self.pool.device)
        B.lumen_kv_checkpoint_pack(plan, self.pool.k_ptrs, self.pool.v_ptrs, buf.data_ptr(),
                                   buf.numel() * buf.element_size(), _kind_of(buf), s.cuda_stream)

    def unpack(self, plan: B.Plan, buf: torch.Tensor, *, stream=None) -> None:
        s = stream if stream is not None else torch.cuda.current_stream(self.pool.device)
        B.lumen_kv_restore_unpack(plan, self.pool.k_ptrs, self.pool.v_ptrs, buf.data_ptr(),
                                  buf.numel() * buf.element_size(), _kind_of(buf), s.cuda_stream)

    def pack_staged(self, plan: B.Plan, host_buf: torch.Tensor, ring: StagingRing, *, stream=None) -> None:
        s = stream if stream is not None else torch.cuda.current_stream(self.pool.device)
        B.lumen_kv_checkpoint_pack_staged(plan, self.pool.k_ptrs, self.pool.v_ptrs,
                                          host_buf.data_ptr(), host_buf.numel() * host_buf.element_size(),
                                          ring.stager, s.cuda_stream)

    def unpack_staged(self, plan: B.Plan, host_buf: torch.Tensor, ring: StagingRing, *, stream=None) -> None:
        s = stream if stream is not None else torch.cuda.current_stream(self.pool.device)
        B.lumen_kv_restore_unpack_staged(plan, self.pool.k_ptrs, self.pool.v_ptrs,
                                         host_buf.data_ptr(), host_buf.numel() * host_buf.element_size(),
                                         ring.stager, s.cuda_stream)
