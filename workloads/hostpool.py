"""Sparse host-side paged pool for running the CPU oracle at full BASELINE.json sizes.

A 146 GiB pool cannot be copied to the host, but the oracle only ever touches the
pages named by the page tables.  Each plane is an anonymous MAP_NORESERVE mapping of
the full [N, S, H, D] size (virtual address space only); the pages the given requests
touch are filled with the same pattern g the device pool holds, so the plain oracle
runs unmodified with the exact page tables.
Test / bench tooling only; no pack/unpack arithmetic.
"""
from __future__ import annotations

import mmap
from typing import List, Sequence, Tuple

import numpy as np

from .content import g_words


def touched_pages(S: int, reqs: Sequence) -> np.ndarray:
    pages = []
    for pt, tb, te in reqs:
        if te > tb:
            pages.append(np.asarray(pt[tb // S: (te - 1) // S + 1], dtype=np.int64))
    return np.unique(np.concatenate(pages)) if pages else np.zeros(0, dtype=np.int64)


def sparse_host_pool(geom, seed: int, fill_reqs: Sequence,
                     content: str = "g") -> Tuple[List[np.ndarray], List[np.ndarray], list]:
    """Returns (K planes, V planes, keepalive).  Pages touched by fill_reqs hold g.
    content="tiled": for timing-only samples of several GiB (bench.py's CPU baseline on the
    32 GiB configs) the touched pages get 64 seeded random page images per plane, tiled --
    numpy evaluates g at 0.2 GB/s, and what a timed gather reads does not change its speed."""
    L, H, D, S, N = (int(x) for x in geom)
    page_words = S * H * D
    plane_bytes = N * page_words * 2
    pages = touched_pages(S, fill_reqs)
    K, V, keep = [], [], []
    for plane in range(2 * L):
        mm = mmap.mmap(-1, plane_bytes, flags=mmap.MAP_PRIVATE | mmap.MAP_ANONYMOUS | getattr(mmap, "MAP_NORESERVE", 0))
        arr = np.frombuffer(mm, dtype=np.uint16)
        if content == "tiled":
            rng = np.random.Generator(np.random.PCG64([int(seed), plane]))
            block = rng.integers(0, 65536, size=64 * page_words, dtype=np.uint16)
            for i, p in enumerate(pages):
                arr[p * page_words:(p + 1) * page_words] = block[(i % 64) * page_words:(i % 64 + 1) * page_words]
        else:
            for p in pages:
                arr[p * page_words:(p + 1) * page_words] = g_words(seed, plane, int(p) * page_words, page_words)
        keep.append(mm)
        (K if plane % 2 == 0 else V).append(arr)
    return K, V, keep
