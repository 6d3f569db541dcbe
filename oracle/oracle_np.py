"""oracle_np -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Second, independently written statement of pack / unpack as a library gather
(pin P2): a plane viewed as [N*S, E] rows, indexed
by slot_ids = PT[t // S] * S + t % S for t in [tb, te), stacked into
[req][layer][K|V][token][head*dim] (PAPER.md:31 for "page", PAPER.md:145 for
the delta range, PAPER.md:157 for restore; layout BASELINE.json configs[0]).

It shares no code with lumen_oracle.c (different language, different loop
structure) and nothing with the CUDA path.  It also serves full-size parity
tests, where only the *index map* (slot_ids, request offsets) is needed.
"""
from __future__ import annotations

import numpy as np


def slot_ids(S: int, page_table, tb: int, te: int) -> np.ndarray:
    """Global slot index (page * S + slot) of every token t in [tb, te)."""
    t = np.arange(int(tb), int(te), dtype=np.int64)
    pt = np.asarray(page_table, dtype=np.int64)
    if t.size and (t[-1] // S) >= pt.size:
        raise IndexError("page table does not cover the token range")
    return pt[t // S] * S + t % S


def layout(geom, reqs):
    """Per request: (offset in elements, n tokens). off_{r+1} = off_r + n_r*2L*E."""
    L, H, D, S, N = (int(x) for x in geom)
    E = H * D
    out, off = [], 0
    for (_pt, tb, te) in reqs:
        n = int(te) - int(tb)
        out.append((off, n))
        off += n * 2 * L * E
    return out, off


def pack(geom, k_planes, v_planes, reqs) -> np.ndarray:
    L, H, D, S, N = (int(x) for x in geom)
    E = H * D
    parts = []
    for (pt, tb, te) in reqs:
        ids = slot_ids(S, pt, tb, te)
        if ids.size and (ids.min() < 0 or ids.max() >= N * S):
            raise IndexError("page index outside the pool")
        per_plane = []
        for l in range(L):
            per_plane.append(k_planes[l].reshape(N * S, E)[ids])
            per_plane.append(v_planes[l].reshape(N * S, E)[ids])
        # [2L, n, E] == [layer][K|V][token][head*dim]
        parts.append(np.stack(per_plane, axis=0).reshape(-1))
    if not parts:
        return np.zeros(0, dtype=np.uint16)
    return np.concatenate(parts).astype(np.uint16, copy=False)


def unpack(geom, k_planes, v_planes, reqs, B) -> None:
    L, H, D, S, N = (int(x) for x in geom)
    E = H * D
    B = np.asarray(B, dtype=np.uint16)
    lay, total = layout(geom, reqs)
    if B.size < total:
        raise ValueError("buffer too small")
    for (pt, tb, te), (off, n) in zip(reqs, lay):
        ids = slot_ids(S, pt, tb, te)
        blk = B[off: off + n * 2 * L * E].reshape(L, 2, n, E)
        for l in range(L):
            k_planes[l].reshape(N * S, E)[ids] = blk[l, 0]
            v_planes[l].reshape(N * S, E)[ids] = blk[l, 1]


def pack_layout(geom, k_planes, v_planes, reqs, layouts, B: np.ndarray) -> None:
    """Explicit buffer layout (checkpoint store), second restatement:
    request r's plane p occupies B[off_r + p*stride_r*E : ... + n_r*E] as a strided 3-D view."""
    L, H, D, S, N = (int(x) for x in geom)
    E = H * D
    for (pt, tb, te), (off, stride) in zip(reqs, layouts):
        n = int(te) - int(tb)
        if n == 0:
            continue
        ids = slot_ids(S, pt, tb, te)
        view = np.lib.stride_tricks.as_strided(B[off:], shape=(2 * L, n, E),
                                               strides=(stride * E * 2, E * 2, 2))
        for l in range(L):
            view[2 * l] = k_planes[l].reshape(N * S, E)[ids]
            view[2 * l + 1] = v_planes[l].reshape(N * S, E)[ids]


def unpack_layout(geom, k_planes, v_planes, reqs, layouts, B: np.ndarray) -> None:
    L, H, D, S, N = (int(x) for x in geom)
    E = H * D
    for (pt, tb, te), (off, stride) in zip(reqs, layouts):
        n = int(te) - int(tb)
        if n == 0:
            continue
        ids = slot_ids(S, pt, tb, te)
        view = np.lib.stride_tricks.as_strided(B[off:], shape=(2 * L, n, E),
                                               strides=(stride * E * 2, E * 2, 2))
        for l in range(L):
            k_planes[l].reshape(N * S, E)[ids] = view[2 * l]
            v_planes[l].reshape(N * S, E)[ids] = view[2 * l + 1]
