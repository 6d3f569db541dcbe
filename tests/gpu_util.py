"""Helpers shared by the -m gpu tests (imported lazily: needs torch + CUDA)."""
from __future__ import annotations

import numpy as np
import torch

import paper_2606_17787_b200 as lk
from paper_2606_17787_b200.pool import KVPool, Checkpointer, StagingRing, pinned_buffer
from workloads import device as wdev
from workloads import fill_plane_np

# "warp": plans of <= 1,024 runs / 512 requests travel in the kernel parameters; "warp_upload" forces the
# descriptor upload to device memory for those too, so both descriptor paths are compared
KERNELS = {"warp": lk.LUMEN_KV_KERNEL_WARP, "bulk": lk.LUMEN_KV_KERNEL_BULK,
           "auto": lk.LUMEN_KV_KERNEL_AUTO,
           "warp_upload": lk.LUMEN_KV_KERNEL_WARP | lk.LUMEN_KV_NO_INLINE}


def build_all():
    from paper_2606_17787_b200 import build
    build.build()
    wdev.build()


def make_pool(geom, seed) -> KVPool:
    L, H, D, S, N = geom
    pool = KVPool(L, H, D, S, N)
    for i, t in enumerate(pool.planes()):
        wdev.fill_plane(t, seed, i)
    torch.cuda.synchronize()
    return pool


def host_planes(geom, seed):
    """Same content as make_pool, on the host (for the oracle)."""
    L, H, D, S, N = geom
    words = N * S * H * D
    K = [fill_plane_np(seed, 2 * l, words) for l in range(L)]
    V = [fill_plane_np(seed, 2 * l + 1, words) for l in range(L)]
    return K, V


def plane_to_np(t: torch.Tensor) -> np.ndarray:
    return t.view(torch.int16).cpu().numpy().view(np.uint16).reshape(-1)


def buf_to_np(buf: torch.Tensor, nbytes: int) -> np.ndarray:
    if buf.is_cuda:
        buf = buf.cpu()
    return buf.numpy().view(np.uint8)[:nbytes].view(np.uint16).copy()


def alloc_buffer(nbytes: int, where: str, guard: int = 4096):
    """Buffer with canary guard bands before and after (C5).  Returns (whole, view).
    Host buffers of 1 GiB and more are registered at their exact size (see pinned_exact)."""
    total = nbytes + 2 * guard
    if where == "device":
        whole = torch.full((total,), 0xA5, dtype=torch.uint8, device="cuda")
    elif total >= (1 << 30):
        whole = wdev.pinned_exact(total)
        whole[:guard] = 0xA5
        whole[guard + nbytes:] = 0xA5
    else:
        whole = pinned_buffer(total)
        whole.fill_(0xA5)
    return whole, whole[guard: guard + nbytes]


def release(whole: torch.Tensor) -> None:
    if not whole.is_cuda:
        wdev.unpin(whole)


def guards_intact(whole: torch.Tensor, nbytes: int, guard: int = 4096) -> bool:
    lo, hi = whole[:guard], whole[guard + nbytes:]
    return bool((lo == 0xA5).all()) and bool((hi == 0xA5).all())
