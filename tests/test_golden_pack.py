"""tests/golden/pack_tiny.txt is a pack + restore example worked out by hand from the definition
(every number in it can be read off its decimal digits).  Both oracles, the plan builder and --
on a GPU -- the CUDA kernels must reproduce it: the oracle is pinned to something that is not
code, and the CUDA path is compared with that same thing directly, without the oracle in between."""
from __future__ import annotations

from pathlib import Path

import numpy as np
import pytest

import oracle
from oracle import oracle_np

GOLDEN = Path(__file__).resolve().parent / "golden" / "pack_tiny.txt"


def load_golden():
    g = {"req": [], "run": [], "row": {}, "restore_req": [], "placed": [], "layout": [], "at": []}
    for line in GOLDEN.read_text().splitlines():
        line = line.split("#")[0].strip()
        if not line:
            continue
        key, val = (x.strip() for x in line.split("=", 1))
        parts = [[int(t) for t in p.split()] for p in val.split(":")]
        if key == "geom":
            g["geom"] = tuple(parts[0])
        elif key == "fill":
            g["fill"] = tuple(parts[0])
        elif key in ("restore_fill", "layout_fill", "layout_extent_bytes"):
            g[key] = parts[0][0]
        elif key == "layout":
            g["layout"].append((parts[1][0], parts[1][1]))          # (byte offset, plane stride tokens)
        elif key == "at":
            g["at"].append((parts[0][0], tuple(parts[1])))
        elif key in ("req", "restore_req"):
            g[key].append((np.asarray(parts[1], dtype=np.int32), parts[2][0], parts[2][1]))
        elif key == "run":
            g["run"].append(tuple(parts[0]))
        elif key == "row":
            g["row"][tuple(parts[0])] = parts[1]
        elif key == "placed":
            g["placed"].append((tuple(parts[0]), tuple(parts[1])))
        else:
            raise ValueError(key)
    return g


def source_planes(g):
    """word e of (plane p, page, slot) = fill[0]*p + fill[1]*page + fill[2]*slot + e"""
    L, H, D, S, N = g["geom"]
    a, b, c = g["fill"]
    E = H * D
    planes = []
    for p in range(2 * L):
        w = (a * p + b * np.arange(N)[:, None, None] + c * np.arange(S)[None, :, None]
             + np.arange(E)[None, None, :])
        assert w.max() < 65536
        planes.append(w.astype(np.uint16).reshape(-1).copy())
    return planes[0::2], planes[1::2]          # K planes, V planes


def golden_buffer(g):
    """The rows of the file in buffer order [req][plane][j]."""
    L = g["geom"][0]
    out = []
    for r, (_, tb, te) in enumerate(g["req"]):
        for p in range(2 * L):
            for j in range(te - tb):
                out.extend(g["row"][(r, p, j)])
    return np.asarray(out, dtype=np.uint16)


def golden_layout_buffer(g):
    """The 25-row buffer of the explicit-layout example: hand-placed rows, the fill elsewhere."""
    E = g["geom"][1] * g["geom"][2]
    B = np.full(g["layout_extent_bytes"] // 2, g["layout_fill"], dtype=np.uint16)
    for at, key in g["at"]:
        B[at * E:(at + 1) * E] = g["row"][key]
    return B


def golden_restored_planes(g):
    L, H, D, S, N = g["geom"]
    E = H * D
    planes = []
    for p in range(2 * L):
        w = np.full((N, S, E), g["restore_fill"], dtype=np.uint16)
        for (page, slot), (r, j) in g["placed"]:
            w[page, slot] = g["row"][(r, p, j)]
        planes.append(w.reshape(-1))
    return planes


def test_file_is_self_consistent():
    g = load_golden()
    L, H, D, S, N = g["geom"]
    assert len(g["row"]) == sum(te - tb for _, tb, te in g["req"]) * 2 * L
    assert all(len(v) == H * D for v in g["row"].values())
    assert len(g["placed"]) == sum(te - tb for _, tb, te in g["restore_req"])
    assert golden_buffer(g).size == 128


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_oracle_pack_and_unpack_equal_the_hand_worked_example(impl):
    g = load_golden()
    mod = oracle if impl == "c" else oracle_np
    K, V = source_planes(g)
    B = mod.pack(g["geom"], K, V, g["req"])
    assert np.array_equal(B, golden_buffer(g))
    L, H, D, S, N = g["geom"]
    K2 = [np.full(N * S * H * D, g["restore_fill"], dtype=np.uint16) for _ in range(L)]
    V2 = [np.full(N * S * H * D, g["restore_fill"], dtype=np.uint16) for _ in range(L)]
    mod.unpack(g["geom"], K2, V2, g["restore_req"], golden_buffer(g))
    want = golden_restored_planes(g)
    for l in range(L):
        assert np.array_equal(K2[l], want[2 * l])
        assert np.array_equal(V2[l], want[2 * l + 1])


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_oracle_layout_pack_and_unpack_equal_the_hand_worked_example(impl):
    g = load_golden()
    mod = oracle if impl == "c" else oracle_np
    L, H, D, S, N = g["geom"]
    K, V = source_planes(g)
    lay = [(off // 2, stride) for off, stride in g["layout"]]      # the oracles take element offsets
    B = np.full(g["layout_extent_bytes"] // 2, g["layout_fill"], dtype=np.uint16)
    mod.pack_layout(g["geom"], K, V, g["req"], lay, B)
    assert np.array_equal(B, golden_layout_buffer(g))
    K2 = [np.full(N * S * H * D, g["restore_fill"], dtype=np.uint16) for _ in range(L)]
    V2 = [np.full(N * S * H * D, g["restore_fill"], dtype=np.uint16) for _ in range(L)]
    mod.unpack_layout(g["geom"], K2, V2, g["restore_req"], lay, golden_layout_buffer(g))
    want = golden_restored_planes(g)
    for l in range(L):
        assert np.array_equal(K2[l], want[2 * l])
        assert np.array_equal(V2[l], want[2 * l + 1])


def test_plan_builder_produces_the_hand_worked_runs():
    from paper_2606_17787_b200 import build
    build.build()
    import paper_2606_17787_b200 as lk
    g = load_golden()
    L, H, D, S, N = g["geom"]
    plan = lk.lumen_kv_plan_build(lk.make_geom(L, H, D, S, N), g["req"], lk.LUMEN_KV_HOST_ONLY)
    assert plan.nbytes == golden_buffer(g).size * 2
    assert plan.req_offset(1) == 3 * 2 * L * H * D * 2
    got = []
    for i in range(plan.num_runs):
        r = plan.run(i)
        got.append((r.req, r.src_slot, r.dst_token, r.count))
    assert got == g["run"]
    plan.close()
    plan = lk.lumen_kv_plan_build(lk.make_geom(L, H, D, S, N), g["req"], lk.LUMEN_KV_HOST_ONLY,
                                  layouts=g["layout"])
    assert plan.nbytes == g["layout_extent_bytes"]
    assert [plan.req_offset(r) for r in range(3)] == [32, 288, 400]
    plan.close()


@pytest.mark.gpu
@pytest.mark.parametrize("where", ["device", "host", "staged"])
@pytest.mark.parametrize("kernel", ["warp", "warp_upload", "bulk"])
def test_cuda_path_equals_the_hand_worked_example(kernel, where):
    """No oracle between the CUDA result and the hand-written numbers."""
    import torch
    from tests import gpu_util as G
    G.build_all()
    g = load_golden()
    L, H, D, S, N = g["geom"]
    K, V = source_planes(g)
    pool_a, pool_b = G.KVPool(L, H, D, S, N), G.KVPool(L, H, D, S, N)
    src = [x for kv in zip(K, V) for x in kv]
    for t, a in zip(pool_a.planes(), src):
        t.view(torch.int16).reshape(-1).copy_(torch.from_numpy(a.view(np.int16)))
    for t in pool_b.planes():
        t.view(torch.int16).fill_(g["restore_fill"])
    flags = G.KERNELS[kernel]
    ck_a, ck_b = G.Checkpointer(pool_a, flags), G.Checkpointer(pool_b, flags)
    plan = ck_a.plan(g["req"])
    rplan = ck_b.plan(g["restore_req"], unique_dst=True)
    whole, buf = G.alloc_buffer(plan.nbytes, "device" if where == "device" else "host")
    ring = G.StagingRing(64, 2) if where == "staged" else None     # 64-byte slots: 4 rows per chunk
    if ring:
        ck_a.pack_staged(plan, buf, ring)
    else:
        ck_a.pack(plan, buf)
    torch.cuda.synchronize()
    assert np.array_equal(G.buf_to_np(buf, plan.nbytes), golden_buffer(g))
    assert G.guards_intact(whole, plan.nbytes)
    if ring:
        ck_b.unpack_staged(rplan, buf, ring)
    else:
        ck_b.unpack(rplan, buf)
    torch.cuda.synchronize()
    for t, want in zip(pool_b.planes(), golden_restored_planes(g)):
        assert np.array_equal(G.plane_to_np(t), want)
    plan.close(); rplan.close()
    if ring:
        ring.close()
    G.release(whole)


@pytest.mark.gpu
@pytest.mark.parametrize("kernel", ["warp", "warp_upload", "bulk"])
def test_cuda_layout_path_equals_the_hand_worked_example(kernel):
    import torch
    from tests import gpu_util as G
    G.build_all()
    g = load_golden()
    L, H, D, S, N = g["geom"]
    K, V = source_planes(g)
    pool_a, pool_b = G.KVPool(L, H, D, S, N), G.KVPool(L, H, D, S, N)
    for t, a in zip(pool_a.planes(), [x for kv in zip(K, V) for x in kv]):
        t.view(torch.int16).reshape(-1).copy_(torch.from_numpy(a.view(np.int16)))
    for t in pool_b.planes():
        t.view(torch.int16).fill_(g["restore_fill"])
    flags = G.KERNELS[kernel]
    ck_a, ck_b = G.Checkpointer(pool_a, flags), G.Checkpointer(pool_b, flags)
    plan = ck_a.plan(g["req"], layouts=g["layout"])
    rplan = ck_b.plan(g["restore_req"], unique_dst=True, layouts=g["layout"])
    assert plan.nbytes == g["layout_extent_bytes"]
    whole, buf = G.alloc_buffer(plan.nbytes, "device")
    buf.view(torch.int16).fill_(g["layout_fill"])
    ck_a.pack(plan, buf)
    torch.cuda.synchronize()
    assert np.array_equal(G.buf_to_np(buf, plan.nbytes), golden_layout_buffer(g))
    assert G.guards_intact(whole, plan.nbytes)
    ck_b.unpack(rplan, buf)
    torch.cuda.synchronize()
    for t, want in zip(pool_b.planes(), golden_restored_planes(g)):
        assert np.array_equal(G.plane_to_np(t), want)
    plan.close(); rplan.close()
