"""GPU parity, small and mid sizes: CUDA path through the C ABI vs the CPU oracle,
bit for bit, on the same seeded inputs (T2 of SURVEY.md section 4).

Every case runs both kernels (SIMT warp / TMA bulk), both buffer kinds (HBM, mapped
pinned host) and checks: the packed buffer equals oracle.pack element by element;
after unpack the WHOLE destination pool equals the oracle's pool (so every non-target
byte is untouched, including partial first/last pages); guard bands around the
buffer are intact.
"""
import numpy as np
import pytest

import oracle
from workloads import cfg0_tiny, cfg1_qwen14b, cfg2_qwen32b, cfg4_longctx, random_tiny, substream, MASTER_SEED

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    import torch
    assert torch.cuda.is_available()
    from tests import gpu_util
    gpu_util.build_all()
    return gpu_util


def run_case(G, w, kernel, where, *, merge=False, seed=MASTER_SEED):
    import torch
    lk = G.lk
    flags = G.KERNELS[kernel] | (lk.LUMEN_KV_MERGE_ADJACENT if merge else 0)
    # ---- oracle side -----------------------------------------------------------
    K, V = G.host_planes(w.geom, seed)
    B_ref = oracle.pack(w.geom, K, V, w.reqs)
    K2, V2 = G.host_planes(w.geom, seed + 1)
    oracle.unpack(w.geom, K2, V2, w.restore_reqs, B_ref, check_overlap=len(w.reqs) and w.tokens < 3000)
    # ---- CUDA side -------------------------------------------------------------
    pool_a = G.make_pool(w.geom, seed)
    pool_b = G.make_pool(w.geom, seed + 1)
    ck_a, ck_b = G.Checkpointer(pool_a, flags), G.Checkpointer(pool_b, flags)
    plan = ck_a.plan(w.reqs)
    assert plan.nbytes == B_ref.size * 2
    whole, buf = G.alloc_buffer(plan.nbytes, where)
    ck_a.pack(plan, buf)
    torch.cuda.synchronize()
    got = G.buf_to_np(buf, plan.nbytes)
    assert np.array_equal(got, B_ref), f"pack mismatch kernel={kernel} where={where}"
    assert G.guards_intact(whole, plan.nbytes)
    # source pool unchanged by pack
    for t, ref in zip(pool_a.planes(), [x for kv in zip(K, V) for x in kv]):
        assert np.array_equal(G.plane_to_np(t), ref)
    # ---- restore into pool B under the fresh page tables -----------------------
    rplan = ck_b.plan(w.restore_reqs, unique_dst=True)
    ck_b.unpack(rplan, buf)
    torch.cuda.synchronize()
    for t, ref in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
        assert np.array_equal(G.plane_to_np(t), ref), f"unpack mismatch kernel={kernel} where={where}"
    # P3 on the GPU: packing the restored pool returns the identical buffer
    whole2, buf2 = G.alloc_buffer(plan.nbytes, "device")
    ck_b.pack(rplan, buf2)
    torch.cuda.synchronize()
    assert np.array_equal(G.buf_to_np(buf2, plan.nbytes), B_ref)
    assert G.guards_intact(whole2, plan.nbytes)
    plan.close(); rplan.close()


@pytest.mark.parametrize("where", ["device", "host"])
@pytest.mark.parametrize("kernel", ["warp", "warp_upload", "bulk", "auto"])
def test_cfg0_tiny(G, kernel, where):
    run_case(G, cfg0_tiny(), kernel, where)
    run_case(G, cfg0_tiny(full_prefix=True), kernel, where)


@pytest.mark.parametrize("kernel", ["warp", "warp_upload", "bulk"])
def test_random_tiny_geometries(G, kernel):
    rng = substream(2024, "gpu_tiny")
    n = 0
    while n < 40:
        w = random_tiny(rng)
        if (w.geom[1] * w.geom[2] * 2) % 16:
            continue
        run_case(G, w, kernel, "device" if n % 3 else "host", merge=bool(n % 2), seed=n)
        n += 1


@pytest.mark.parametrize("kernel", ["warp", "warp_upload", "bulk"])
def test_mid_cfg1_shape(G, kernel):
    """Qwen3-14B row/page shape, fewer layers/pages: 32 KiB runs, ragged 16-token deltas."""
    w = cfg1_qwen14b(L=3, N=2048, n_reqs=24, grow_iters=2, median=200, hi=512, lo=20)
    run_case(G, w, kernel, "device")
    run_case(G, w.advanced(16), kernel, "host")
    run_case(G, cfg1_qwen14b(L=3, N=2048, n_reqs=24, grow_iters=2, median=200, hi=512, lo=20, aligned=True), kernel, "device")


@pytest.mark.parametrize("kernel", ["warp", "bulk"])
def test_mid_cfg2_shape_full_prefix(G, kernel):
    w = cfg2_qwen32b(L=2, N=1200, n_reqs=5, prompt=1000)      # 1000 tokens: ragged last page
    run_case(G, w, kernel, "device")


@pytest.mark.parametrize("kernel", ["warp", "bulk"])
def test_mid_cfg4_token_granular(G, kernel):
    w = cfg4_longctx(L=2, tokens=3001, wave_reqs=2)          # S = 1: 6002 runs of one 2 KiB row
    run_case(G, w, kernel, "device")
    run_case(G, w, kernel, "host", merge=True)


@pytest.mark.parametrize("kernel", ["warp", "bulk"])
def test_tp_rank_shape_and_odd_rows(G, kernel):
    # H = 4 (one TP2 rank of an 8-kv-head model); and a 48-byte row
    run_case(G, cfg1_qwen14b(L=2, H=4, N=512, n_reqs=8, grow_iters=2, median=100, hi=256, lo=20), kernel, "device")
    run_case(G, cfg1_qwen14b(L=2, H=1, D=24, N=512, n_reqs=8, grow_iters=2, median=100, hi=256, lo=20), kernel, "device")
    # page larger than the 32 KiB chunk: S = 64 tokens of 2 KiB
    run_case(G, cfg2_qwen32b(L=1, S=64, N=64, n_reqs=3, prompt=500), kernel, "device")


def test_pack_allows_shared_pages(G):
    import torch
    rng = substream(5, "shared")
    for i in range(10):
        w = random_tiny(rng, allow_shared=True)
        K, V = G.host_planes(w.geom, i)
        ref = oracle.pack(w.geom, K, V, w.reqs)
        pool = G.make_pool(w.geom, i)
        ck = G.Checkpointer(pool)
        plan = ck.plan(w.reqs)
        whole, buf = G.alloc_buffer(plan.nbytes, "device")
        ck.pack(plan, buf)
        torch.cuda.synchronize()
        assert np.array_equal(G.buf_to_np(buf, plan.nbytes), ref)


def test_empty_plan_and_errors(G):
    import torch
    lk = G.lk
    w = cfg0_tiny()
    pool = G.make_pool(w.geom, 1)
    ck = G.Checkpointer(pool)
    empty = ck.plan([])
    buf = torch.zeros(64, dtype=torch.uint8, device="cuda")
    ck.pack(empty, buf); ck.unpack(empty, buf)            # A4: launches nothing, returns OK
    zero = ck.plan([(w.reqs[0][0], 5, 5)])
    ck.pack(zero, buf)
    plan = ck.plan(w.reqs)
    small = torch.zeros(plan.nbytes - 16, dtype=torch.uint8, device="cuda")
    with pytest.raises(lk.LumenKVError) as e:
        ck.pack(plan, small)
    assert e.value.status == lk.LUMEN_KV_ESIZE
    big = torch.zeros(plan.nbytes + 16, dtype=torch.uint8, device="cuda")
    with pytest.raises(lk.LumenKVError) as e:
        ck.pack(plan, big[8:])                               # misaligned base
    assert e.value.status == lk.LUMEN_KV_EINVAL
    pageable = torch.zeros(plan.nbytes, dtype=torch.uint8)
    with pytest.raises(lk.LumenKVError) as e:                # pageable host memory is not mapped
        lk.lumen_kv_checkpoint_pack(plan, pool.k_ptrs, pool.v_ptrs, pageable.data_ptr(), plan.nbytes,
                                    lk.LUMEN_KV_MEM_HOST_MAPPED, 0)
    assert e.value.status == lk.LUMEN_KV_EINVAL
    torch.cuda.synchronize()


def test_delta_concat_on_gpu(G):
    """P4 form 2 on the CUDA path: unpack(delta_1); unpack(delta_2) == unpack(full)."""
    import torch
    w = cfg0_tiny(full_prefix=True)
    pool_src = G.make_pool(w.geom, 3)
    ck_src = G.Checkpointer(pool_src)
    pool_full, pool_inc = G.make_pool(w.geom, 4), G.make_pool(w.geom, 4)
    ck_full, ck_inc = G.Checkpointer(pool_full), G.Checkpointer(pool_inc)
    full = ck_src.plan(w.reqs)
    bfull = torch.empty(full.nbytes, dtype=torch.uint8, device="cuda")
    ck_src.pack(full, bfull)
    ck_full.unpack(ck_full.plan(w.restore_reqs), bfull)
    cuts = [0, 7, 16, 33, 10**9]
    for a, b in zip(cuts[:-1], cuts[1:]):
        d_src = [(pt, min(a, te), min(b, te)) for pt, tb, te in w.reqs]
        d_dst = [(pt, min(a, te), min(b, te)) for pt, tb, te in w.restore_reqs]
        p = ck_src.plan(d_src)
        bd = torch.empty(max(p.nbytes, 16), dtype=torch.uint8, device="cuda")
        ck_src.pack(p, bd)
        ck_inc.unpack(ck_inc.plan(d_dst), bd)
    torch.cuda.synchronize()
    for x, y in zip(pool_full.planes(), pool_inc.planes()):
        assert torch.equal(x.view(torch.int16), y.view(torch.int16))


def test_plan_reuse_and_free_while_in_flight(G):
    """build -> pack -> free in a loop with no host sync: the arena must keep descriptors
    alive until the enqueued work is done, and recycle them afterwards."""
    import torch
    w = cfg1_qwen14b(L=2, N=8192, n_reqs=32, grow_iters=40, median=200, hi=512, lo=20)
    K, V = G.host_planes(w.geom, 9)
    pool = G.make_pool(w.geom, 9)
    ck = G.Checkpointer(pool)
    bufs, refs, cur = [], [], w
    for it in range(32):
        plan = ck.plan(cur.reqs)
        buf = torch.empty(plan.nbytes, dtype=torch.uint8, device="cuda")
        ck.pack(plan, buf)
        plan.close()                                         # freed while possibly in flight
        bufs.append(buf); refs.append(oracle.pack(cur.geom, K, V, cur.reqs))
        cur = cur.advanced(16)
    torch.cuda.synchronize()
    for buf, ref in zip(bufs, refs):
        assert np.array_equal(G.buf_to_np(buf, buf.numel()), ref)
    G.lk.lumen_kv_trim()


def test_two_streams_concurrent(G):
    """a8 in miniature: unpack on stream 1 while packs of other requests run on stream 2."""
    import torch
    w = cfg2_qwen32b(L=2, N=1200, n_reqs=6, prompt=900)
    seed = 21
    K, V = G.host_planes(w.geom, seed)
    pool = G.make_pool(w.geom, seed)
    ck = G.Checkpointer(pool)
    # requests 0-2 are "running" (packed); requests 3-5's checkpoint is restored into fresh pages
    run_reqs, ckpt_reqs, fresh = w.reqs[:3], w.reqs[3:], w.restore_reqs[3:]
    B_ckpt = oracle.pack(w.geom, K, V, ckpt_reqs)
    B_run = oracle.pack(w.geom, K, V, run_reqs)
    oracle.unpack(w.geom, K, V, fresh, B_ckpt)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    src = torch.from_numpy(B_ckpt.view(np.uint8)).pin_memory()
    out = G.pinned_buffer(B_run.size * 2)
    torch.cuda.synchronize()
    p1 = ck.plan(fresh, unique_dst=True, stream=s1)
    p2 = ck.plan(run_reqs, stream=s2)
    ck.unpack(p1, src, stream=s1)
    ck.pack(p2, out, stream=s2)
    torch.cuda.synchronize()
    assert np.array_equal(G.buf_to_np(out, out.numel()), B_run)
    for t, ref in zip(pool.planes(), [x for kv in zip(K, V) for x in kv]):
        assert np.array_equal(G.plane_to_np(t), ref)


# ---- two-stage host path (device staging ring + copy engines) -----------------------------
def run_staged_case(G, w, slot_bytes, n_slots, *, seed=MASTER_SEED, kernel="auto"):
    """pack_staged -> pinned host buffer == oracle.pack; unpack_staged -> whole pool == oracle's;
    the one-shot mapped-host call reads back what the staged call wrote and vice versa."""
    import torch
    K, V = G.host_planes(w.geom, seed)
    B_ref = oracle.pack(w.geom, K, V, w.reqs)
    K2, V2 = G.host_planes(w.geom, seed + 1)
    oracle.unpack(w.geom, K2, V2, w.restore_reqs, B_ref)
    pool_a, pool_b = G.make_pool(w.geom, seed), G.make_pool(w.geom, seed + 1)
    ck_a, ck_b = G.Checkpointer(pool_a, G.KERNELS[kernel]), G.Checkpointer(pool_b, G.KERNELS[kernel])
    ring = G.StagingRing(slot_bytes, n_slots)
    ring.mem.fill_(0x5A)
    plan = ck_a.plan(w.reqs)
    n_chunks = len(plan.chunks(slot_bytes))
    whole, buf = G.alloc_buffer(plan.nbytes, "host")
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):                       # not the default stream
        ck_a.pack_staged(plan, buf, ring)
        done = torch.cuda.Event(); done.record(side)    # stream order alone must imply completion
    done.synchronize()
    assert np.array_equal(G.buf_to_np(buf, plan.nbytes), B_ref), "staged pack mismatch"
    assert G.guards_intact(whole, plan.nbytes)
    rplan = ck_b.plan(w.restore_reqs, unique_dst=True)
    with torch.cuda.stream(side):
        ck_b.unpack_staged(rplan, buf, ring)            # same ring, other direction
        done.record(side)
    done.synchronize()
    for t, ref in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
        assert np.array_equal(G.plane_to_np(t), ref), "staged unpack mismatch"
    # two staged calls back to back on one stream reuse the slots while copies are in flight
    whole2, buf2 = G.alloc_buffer(plan.nbytes, "host")
    with torch.cuda.stream(side):
        ck_b.pack_staged(rplan, buf2, ring)
        ck_b.pack_staged(rplan, buf, ring)
        done.record(side)
    done.synchronize()
    assert np.array_equal(G.buf_to_np(buf2, plan.nbytes), B_ref)
    assert np.array_equal(G.buf_to_np(buf, plan.nbytes), B_ref)
    assert G.guards_intact(whole2, plan.nbytes)
    plan.close(); rplan.close(); ring.close()
    return n_chunks


def test_staged_cfg0_and_tiny(G):
    assert run_staged_case(G, cfg0_tiny(), 4096, 2) > 8           # 256 B rows, 16-token pages
    assert run_staged_case(G, cfg0_tiny(full_prefix=True), 1 << 20, 3) == 1
    rng = substream(4242, "gpu_staged")
    n = 0
    while n < 25:
        w = random_tiny(rng)
        row = w.geom[1] * w.geom[2] * 2
        if row % 16 or not w.tokens:
            continue
        max_run = max(min(w.geom[3], te - tb) for _, tb, te in w.reqs if te > tb) * row
        slot = (max_run * int(rng.integers(1, 6)) + 15) // 16 * 16
        run_staged_case(G, w, slot, int(rng.integers(2, 5)), seed=n)
        n += 1


@pytest.mark.parametrize("kernel", ["auto", "warp_upload", "bulk"])
def test_staged_mid_shapes(G, kernel):
    """All three chunk kinds on the paper's shapes: groups of whole requests (cfg 1 deltas),
    plane ranges of one request (cfg 2 prefixes), token ranges of one plane (cfg 4, S = 1)."""
    w = cfg1_qwen14b(L=3, N=2048, n_reqs=24, grow_iters=2, median=200, hi=512, lo=20)
    assert run_staged_case(G, w, 1 << 20, 3, kernel=kernel) == 5        # 24 x 192 KiB requests, 5 per slot
    w = cfg2_qwen32b(L=2, N=1200, n_reqs=3, prompt=1000)                # 1000 x 2 KiB per plane
    assert run_staged_case(G, w, 5 << 20, 2, kernel=kernel) == 2 * 3    # 2 planes per chunk
    w = cfg4_longctx(L=2, tokens=3001, wave_reqs=2)
    assert run_staged_case(G, w, 1 << 20, 4, kernel=kernel) == 2 * 4 * 6  # 512 tokens per chunk


def test_staged_errors(G):
    import torch
    lk = G.lk
    w = cfg0_tiny()
    pool = G.make_pool(w.geom, 1)
    ck = G.Checkpointer(pool)
    plan = ck.plan(w.reqs)
    ring = G.StagingRing(1024, 2)                       # smaller than one 16-token run (4 KiB)
    whole, buf = G.alloc_buffer(plan.nbytes, "host")
    with pytest.raises(lk.LumenKVError) as e:
        ck.pack_staged(plan, buf, ring)
    assert e.value.status == lk.LUMEN_KV_ESIZE
    ring2 = G.StagingRing(8192, 2)
    with pytest.raises(lk.LumenKVError) as e:
        ck.pack_staged(plan, buf[: plan.nbytes - 16], ring2)
    assert e.value.status == lk.LUMEN_KV_ESIZE
    pageable = torch.empty(plan.nbytes, dtype=torch.uint8)
    with pytest.raises(lk.LumenKVError) as e:
        lk.lumen_kv_checkpoint_pack_staged(plan, pool.k_ptrs, pool.v_ptrs, pageable.data_ptr(),
                                           plan.nbytes, ring2.stager, 0)
    assert e.value.status == lk.LUMEN_KV_EINVAL
    empty = ck.plan([])
    ck.pack_staged(empty, buf, ring2)                   # A4: nothing to do, returns OK
    torch.cuda.synchronize()
    assert G.guards_intact(whole, plan.nbytes)


def test_staged_commit_and_ready_flags(G):
    """Per-chunk flags: a host consumer that sees flags[c] == epoch finds chunk c
    complete in the pinned buffer while later chunks are still in flight; a restore whose
    ready flags are raised chunk by chunk by a host producer never reads a chunk early."""
    import threading
    import time
    import torch
    lk = G.lk
    w = cfg2_qwen32b(L=3, N=1500, n_reqs=4, prompt=1200)               # 4 x 14 MiB
    slot = 1 << 20
    K, V = G.host_planes(w.geom, 11)
    B_ref = oracle.pack(w.geom, K, V, w.reqs)
    K2, V2 = G.host_planes(w.geom, 12)
    oracle.unpack(w.geom, K2, V2, w.restore_reqs, B_ref)
    ref_bytes = B_ref.view(np.uint8)
    pool_a, pool_b = G.make_pool(w.geom, 11), G.make_pool(w.geom, 12)
    ring = G.StagingRing(slot, 3)
    plan = lk.lumen_kv_plan_build(pool_a.geom, w.reqs, 0, 0)
    chunks = plan.chunks(slot)
    assert len(chunks) > 40
    whole, buf = G.alloc_buffer(plan.nbytes, "host")
    buf.fill_(0xEE)
    host = buf.numpy()
    flags_t = torch.zeros(len(chunks), dtype=torch.int64, pin_memory=True)
    flags = flags_t.numpy()
    EPOCH = 7
    seen, bad, stop = [], [], threading.Event()

    def consumer():                                     # stands in for the sender of step (4)
        nxt = 0
        while nxt < len(chunks) and not stop.is_set():
            if flags[nxt] == EPOCH:
                c = chunks[nxt]
                if not np.array_equal(host[c.byte_begin:c.byte_end], ref_bytes[c.byte_begin:c.byte_end]):
                    bad.append(nxt)
                seen.append((nxt, int((flags == EPOCH).sum())))
                nxt += 1

    th = threading.Thread(target=consumer)
    th.start()
    side = torch.cuda.Stream()
    try:
        lk.lumen_kv_checkpoint_pack_staged_commit(plan, pool_a.k_ptrs, pool_a.v_ptrs, buf.data_ptr(),
                                                  plan.nbytes, ring.stager, side.cuda_stream,
                                                  flags_t.data_ptr(), EPOCH)
        side.synchronize()
        th.join(timeout=60)
    finally:
        stop.set()
    assert not th.is_alive() and len(seen) == len(chunks) and not bad
    assert np.array_equal(G.buf_to_np(buf, plan.nbytes), B_ref) and G.guards_intact(whole, plan.nbytes)

    # ---- restore side: chunks become ready one by one, out of a buffer that starts as garbage ----
    rplan = lk.lumen_kv_plan_build(pool_b.geom, w.restore_reqs, lk.LUMEN_KV_VALIDATE_UNIQUE_DST, 0)
    rchunks = rplan.chunks(slot)
    buf.fill_(0xEE)
    flags[:] = 0
    READY = 9
    lk.lumen_kv_restore_unpack_staged_ready(rplan, pool_b.k_ptrs, pool_b.v_ptrs, buf.data_ptr(),
                                            rplan.nbytes, ring.stager, side.cuda_stream,
                                            flags_t.data_ptr(), READY)
    done = torch.cuda.Event(); done.record(side)
    try:
        for i, c in enumerate(rchunks):                 # "reception": fill the chunk, then raise its flag
            assert not done.query(), "restore finished before all chunks were ready"
            host[c.byte_begin:c.byte_end] = ref_bytes[c.byte_begin:c.byte_end]
            if i % 16 == 0:
                time.sleep(0.002)
            flags[i] = READY
    finally:
        flags[:] = READY                                # never leave the stream waiting
    side.synchronize()
    for t, ref in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
        assert np.array_equal(G.plane_to_np(t), ref), "restore read a chunk before it was ready"
    plan.close(); rplan.close(); ring.close()


# ---- asynchronous staged calls (a stager-owned thread issues the chunk pipeline) -------------
def test_staged_async_parity_and_ordering(G):
    """_async returns a ticket at once; the plan is freed immediately, the pool of the producing
    stream is filled by work enqueued BEFORE the call (begin ordering), stager_wait makes a
    consumer stream see the result, query flips to True, sync blocks; bytes equal the oracle's.
    All three chunk kinds, with slots reused many times per call."""
    import torch
    lk = G.lk
    cases = [(cfg1_qwen14b(L=3, N=2048, n_reqs=24, grow_iters=2, median=200, hi=512, lo=20), 1 << 20, 3),
             (cfg2_qwen32b(L=2, N=1200, n_reqs=3, prompt=1000), 5 << 20, 2),
             (cfg4_longctx(L=2, tokens=3001, wave_reqs=2), 1 << 20, 4),
             (cfg0_tiny(), 4096, 2)]
    for n, (w, slot, nslots) in enumerate(cases):
        seed = 300 + 2 * n
        K, V = G.host_planes(w.geom, seed)
        B_ref = oracle.pack(w.geom, K, V, w.reqs)
        K2, V2 = G.host_planes(w.geom, seed + 1)
        oracle.unpack(w.geom, K2, V2, w.restore_reqs, B_ref)
        L, H, D, S, N = w.geom
        pool_a = G.KVPool(L, H, D, S, N)
        pool_b = G.make_pool(w.geom, seed + 1)
        ring = G.StagingRing(slot, nslots)
        whole, buf = G.alloc_buffer(w.payload_bytes, "host")
        prod, cons = torch.cuda.Stream(), torch.cuda.Stream()
        with torch.cuda.stream(prod):                       # the pool is produced on `prod` ...
            for i, t in enumerate(pool_a.planes()):
                G.wdev.fill_plane(t, seed, i, prod.cuda_stream)
        plan = lk.lumen_kv_plan_build(pool_a.geom, w.reqs, 0, prod.cuda_stream)
        n_chunks = len(plan.chunks(slot))
        t1 = lk.lumen_kv_checkpoint_pack_staged_async(plan, pool_a.k_ptrs, pool_a.v_ptrs, buf.data_ptr(),
                                                      plan.nbytes, ring.stager, prod.cuda_stream)
        plan.close()                                        # ... and the plan is gone before it is issued
        rplan = lk.lumen_kv_plan_build(pool_b.geom, w.restore_reqs, lk.LUMEN_KV_VALIDATE_UNIQUE_DST,
                                       cons.cuda_stream)
        # the restore reads what ticket t1 writes: same stager, so it is ordered behind it
        t2 = lk.lumen_kv_restore_unpack_staged_async(rplan, pool_b.k_ptrs, pool_b.v_ptrs, buf.data_ptr(),
                                                     rplan.nbytes, ring.stager, cons.cuda_stream)
        rplan.close()
        assert t2 == t1 + 1
        ring.stager.wait(t2, cons.cuda_stream)              # consumer stream sees the restored pool
        with torch.cuda.stream(cons):
            snap = [t.clone() for t in pool_b.planes()]
        cons.synchronize()
        assert ring.stager.query(t1) and ring.stager.query(t2)
        ring.stager.sync(t2)
        assert np.array_equal(G.buf_to_np(buf, w.payload_bytes), B_ref), f"async pack mismatch, case {n}"
        assert G.guards_intact(whole, w.payload_bytes)
        for t, ref in zip(snap, [x for kv in zip(K2, V2) for x in kv]):
            assert np.array_equal(G.plane_to_np(t), ref), f"async unpack mismatch, case {n}"
        assert n_chunks >= 1
        ring.close()
        G.release(whole)


def test_uploaded_plan_used_from_several_threads_and_a_stager_at_once(G):
    """One plan whose descriptors were uploaded (NO_INLINE) is used by four host threads, each
    packing on a stream of its own, while a stager's thread issues an _async staged pack of the
    same plan: the plan's bookkeeping (upload seen, last use per stream) is shared by all of
    them.  Every buffer must equal the oracle's, round after round."""
    import threading
    import torch
    lk = G.lk
    w = cfg2_qwen32b(L=2, N=1200, n_reqs=5, prompt=1000)
    seed = 77
    K, V = G.host_planes(w.geom, seed)
    B_ref = oracle.pack(w.geom, K, V, w.reqs)
    pool = G.make_pool(w.geom, seed)
    ring = G.StagingRing(1 << 20, 3)
    host_whole, host_buf = G.alloc_buffer(w.payload_bytes, "host")
    n_threads, rounds = 4, 6
    bufs = [torch.zeros(w.payload_bytes, dtype=torch.uint8, device="cuda") for _ in range(n_threads)]
    streams = [torch.cuda.Stream() for _ in range(n_threads)]
    torch.cuda.synchronize()
    for rnd in range(rounds):
        plan = lk.lumen_kv_plan_build(pool.geom, w.reqs, lk.LUMEN_KV_KERNEL_WARP | lk.LUMEN_KV_NO_INLINE)
        errors = []
        start = threading.Barrier(n_threads + 1)

        def worker(i):
            try:
                start.wait()
                for _ in range(8):        # each call records a use of the plan on this thread's stream
                    lk.lumen_kv_checkpoint_pack(plan, pool.k_ptrs, pool.v_ptrs, bufs[i].data_ptr(),
                                                plan.nbytes, lk.LUMEN_KV_MEM_DEVICE, streams[i].cuda_stream)
            except Exception as e:        # noqa: BLE001
                errors.append(e)

        threads = [threading.Thread(target=worker, args=(i,)) for i in range(n_threads)]
        for t in threads:
            t.start()
        start.wait()
        ticket = lk.lumen_kv_checkpoint_pack_staged_async(plan, pool.k_ptrs, pool.v_ptrs, host_buf.data_ptr(),
                                                          plan.nbytes, ring.stager, 0)
        for t in threads:
            t.join()
        plan.close()                      # freed while the stager may still be issuing from it
        ring.stager.sync(ticket)
        torch.cuda.synchronize()
        assert not errors, errors
        for i in range(n_threads):
            assert np.array_equal(G.buf_to_np(bufs[i], w.payload_bytes), B_ref), f"round {rnd}, thread {i}"
            bufs[i].zero_()
        assert np.array_equal(G.buf_to_np(host_buf, w.payload_bytes), B_ref), f"round {rnd}, staged"
        assert G.guards_intact(host_whole, w.payload_bytes)
        host_buf.zero_()
    ring.close()
    G.release(host_whole)


def test_stager_wait_and_sync_race_ticket_pruning(G):
    """a stager keeps 64 tickets and prunes completed ones when a new call is
    submitted.  Threads that wait on / synchronise with old tickets while another thread keeps
    submitting must never be handed a destroyed event: every wait and sync returns OK and the
    last buffer equals the oracle's."""
    import threading
    import torch
    lk = G.lk
    w = cfg0_tiny()
    K, V = G.host_planes(w.geom, 9)
    B_ref = oracle.pack(w.geom, K, V, w.reqs)
    pool = G.make_pool(w.geom, 9)
    ring = G.StagingRing(4096, 2)
    whole, buf = G.alloc_buffer(w.payload_bytes, "host")
    plan = lk.lumen_kv_plan_build(pool.geom, w.reqs)
    n_calls = 600
    tickets, errors = [], []
    done = threading.Event()

    def waiter(k):
        side = torch.cuda.Stream()
        rng = np.random.default_rng(k)
        try:
            while True:
                if not tickets:
                    continue
                t = tickets[int(rng.integers(max(0, len(tickets) - 80), len(tickets)))]
                if rng.integers(2):
                    ring.stager.wait(t, side.cuda_stream)
                else:
                    ring.stager.sync(t)
                assert ring.stager.query(t) in (True, False)
                if done.is_set():
                    break
            side.synchronize()
        except Exception as e:            # noqa: BLE001
            errors.append(e)

    threads = [threading.Thread(target=waiter, args=(k,)) for k in range(3)]
    for t in threads:
        t.start()
    for _ in range(n_calls):
        tickets.append(lk.lumen_kv_checkpoint_pack_staged_async(plan, pool.k_ptrs, pool.v_ptrs, buf.data_ptr(),
                                                                plan.nbytes, ring.stager, 0))
    done.set()
    for t in threads:
        t.join()
    ring.stager.sync(tickets[-1])
    assert not errors, errors
    assert tickets == list(range(tickets[0], tickets[0] + n_calls))
    assert np.array_equal(G.buf_to_np(buf, w.payload_bytes), B_ref)
    assert G.guards_intact(whole, w.payload_bytes)
    plan.close(); ring.close()
    G.release(whole)


def test_staged_calls_fail_cleanly_and_the_stager_stays_usable(G):
    """Failure injection (lumen_kv_set_option("fail_after_chunks", n)): a staged call that fails
    after n chunks reports ECUDA -- synchronously, or through query / wait / sync of its ticket,
    with the cudaError_t on the asking thread -- and leaves its stager usable: the next calls on
    the SAME stager, synchronous and asynchronous, on other streams, are bit-exact; so is a new
    stager on the same ring memory."""
    import torch
    lk = G.lk
    w = cfg2_qwen32b(L=2, N=1200, n_reqs=3, prompt=1000)      # 12 chunks of <= 1 MiB
    seed = 41
    K, V = G.host_planes(w.geom, seed)
    B_ref = oracle.pack(w.geom, K, V, w.reqs)
    K2, V2 = G.host_planes(w.geom, seed + 1)
    oracle.unpack(w.geom, K2, V2, w.restore_reqs, B_ref)
    pool_a = G.make_pool(w.geom, seed)
    ring = G.StagingRing(1 << 20, 3)
    whole, buf = G.alloc_buffer(w.payload_bytes, "host")
    plan = lk.lumen_kv_plan_build(pool_a.geom, w.reqs)
    rplan = lk.lumen_kv_plan_build(pool_a.geom, w.restore_reqs, lk.LUMEN_KV_VALIDATE_UNIQUE_DST)
    assert len(plan.chunks(1 << 20)) > 5
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    try:
        for n in (0, 1, 4):
            buf.zero_()
            lk.lumen_kv_set_option("fail_after_chunks", n)
            with pytest.raises(lk.LumenKVError) as e:
                lk.lumen_kv_checkpoint_pack_staged(plan, pool_a.k_ptrs, pool_a.v_ptrs, buf.data_ptr(), plan.nbytes,
                                                   ring.stager, s1.cuda_stream)
            assert e.value.status == lk.LUMEN_KV_ECUDA and e.value.cuda_error != 0
            t_bad = lk.lumen_kv_checkpoint_pack_staged_async(plan, pool_a.k_ptrs, pool_a.v_ptrs, buf.data_ptr(),
                                                             plan.nbytes, ring.stager, s2.cuda_stream)
            for ask in (ring.stager.sync, lambda t: ring.stager.wait(t, s1.cuda_stream), ring.stager.query):
                with pytest.raises(lk.LumenKVError) as e:
                    ask(t_bad)
                assert e.value.status == lk.LUMEN_KV_ECUDA and e.value.cuda_error != 0
            lk.lumen_kv_set_option("fail_after_chunks", -1)
            # the same stager, another stream: synchronous pack, then an asynchronous restore
            lk.lumen_kv_checkpoint_pack_staged(plan, pool_a.k_ptrs, pool_a.v_ptrs, buf.data_ptr(), plan.nbytes,
                                               ring.stager, s2.cuda_stream)
            s2.synchronize()
            assert np.array_equal(G.buf_to_np(buf, w.payload_bytes), B_ref), f"pack after failure at chunk {n}"
            pool_b = G.make_pool(w.geom, seed + 1)
            t_ok = lk.lumen_kv_restore_unpack_staged_async(rplan, pool_b.k_ptrs, pool_b.v_ptrs, buf.data_ptr(),
                                                           rplan.nbytes, ring.stager, s1.cuda_stream)
            assert t_ok == t_bad + 1
            ring.stager.sync(t_ok)
            assert ring.stager.query(t_ok)
            for t, ref in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
                assert np.array_equal(G.plane_to_np(t), ref), f"restore after failure at chunk {n}"
            with pytest.raises(lk.LumenKVError):                  # the failed ticket stays failed
                ring.stager.query(t_bad)
        # a failing restore, then a second stager on the same ring memory
        lk.lumen_kv_set_option("fail_after_chunks", 2)
        pool_c = G.make_pool(w.geom, seed + 1)
        with pytest.raises(lk.LumenKVError):
            lk.lumen_kv_restore_unpack_staged(rplan, pool_c.k_ptrs, pool_c.v_ptrs, buf.data_ptr(), rplan.nbytes,
                                              ring.stager, s1.cuda_stream)
        lk.lumen_kv_set_option("fail_after_chunks", -1)
        second = lk.Stager(ring.mem.data_ptr(), 1 << 20, 3)
        lk.lumen_kv_restore_unpack_staged(rplan, pool_c.k_ptrs, pool_c.v_ptrs, buf.data_ptr(), rplan.nbytes,
                                          second, s2.cuda_stream)
        s2.synchronize()
        for t, ref in zip(pool_c.planes(), [x for kv in zip(K2, V2) for x in kv]):
            assert np.array_equal(G.plane_to_np(t), ref)
        second.close()
    finally:
        lk.lumen_kv_set_option("fail_after_chunks", -1)
    assert G.guards_intact(whole, w.payload_bytes)
    plan.close(); rplan.close(); ring.close()
    G.release(whole)


def test_staged_async_mixed_with_sync_errors_and_flags(G):
    import threading
    import torch
    lk = G.lk
    w = cfg2_qwen32b(L=3, N=1500, n_reqs=4, prompt=1200)               # 4 x 14 MiB
    slot = 1 << 20
    K, V = G.host_planes(w.geom, 21)
    B_ref = oracle.pack(w.geom, K, V, w.reqs)
    ref_bytes = B_ref.view(np.uint8)
    pool = G.make_pool(w.geom, 21)
    ring = G.StagingRing(slot, 3)
    plan = lk.lumen_kv_plan_build(pool.geom, w.reqs, 0, 0)
    chunks = plan.chunks(slot)
    whole, buf = G.alloc_buffer(plan.nbytes, "host")
    whole2, buf2 = G.alloc_buffer(plan.nbytes, "host")
    s = torch.cuda.Stream()
    # validation errors come back from the call itself, and hand out no ticket
    with pytest.raises(lk.LumenKVError) as e:
        lk.lumen_kv_checkpoint_pack_staged_async(plan, pool.k_ptrs, pool.v_ptrs, buf.data_ptr(),
                                                 plan.nbytes - 16, ring.stager, s.cuda_stream)
    assert e.value.status == lk.LUMEN_KV_ESIZE
    small = G.StagingRing(1024, 2)
    with pytest.raises(lk.LumenKVError) as e:
        lk.lumen_kv_checkpoint_pack_staged_async(plan, pool.k_ptrs, pool.v_ptrs, buf.data_ptr(),
                                                 plan.nbytes, small.stager, s.cuda_stream)
    assert e.value.status == lk.LUMEN_KV_ESIZE
    with pytest.raises(lk.LumenKVError):
        ring.stager.query(1)                               # no such ticket yet
    empty = lk.lumen_kv_plan_build(pool.geom, [], 0, 0)
    t0 = lk.lumen_kv_checkpoint_pack_staged_async(empty, pool.k_ptrs, pool.v_ptrs, buf.data_ptr(),
                                                  plan.nbytes, ring.stager, s.cuda_stream)
    assert ring.stager.query(t0)                           # A4: nothing to do, complete at once
    ring.stager.wait(t0, s.cuda_stream); ring.stager.sync(t0)
    # async with commit flags + a host consumer, then a synchronous call on the same stager
    flags_t = torch.zeros(len(chunks), dtype=torch.int64, pin_memory=True)
    flags, host = flags_t.numpy(), buf.numpy()
    bad, seen = [], []

    def consumer():
        for i, c in enumerate(chunks):
            while flags[i] != 5:
                pass
            if not np.array_equal(host[c.byte_begin:c.byte_end], ref_bytes[c.byte_begin:c.byte_end]):
                bad.append(i)
            seen.append(i)

    th = threading.Thread(target=consumer)
    th.start()
    t1 = lk.lumen_kv_checkpoint_pack_staged_async(plan, pool.k_ptrs, pool.v_ptrs, buf.data_ptr(),
                                                  plan.nbytes, ring.stager, s.cuda_stream,
                                                  flags_t.data_ptr(), 5)
    lk.lumen_kv_checkpoint_pack_staged(plan, pool.k_ptrs, pool.v_ptrs, buf2.data_ptr(), plan.nbytes,
                                       ring.stager, s.cuda_stream)        # issued after t1, same slots
    s.synchronize()
    ring.stager.sync(t1)
    th.join(timeout=60)
    assert not th.is_alive() and len(seen) == len(chunks) and not bad
    assert np.array_equal(G.buf_to_np(buf, plan.nbytes), B_ref)
    assert np.array_equal(G.buf_to_np(buf2, plan.nbytes), B_ref)
    assert G.guards_intact(whole, plan.nbytes) and G.guards_intact(whole2, plan.nbytes)
    # a stager destroyed with calls still queued issues them first
    ring3 = G.StagingRing(slot, 2)
    buf.fill_(0)
    for _ in range(3):
        lk.lumen_kv_checkpoint_pack_staged_async(plan, pool.k_ptrs, pool.v_ptrs, buf.data_ptr(),
                                                 plan.nbytes, ring3.stager, s.cuda_stream)
    ring3.close()
    torch.cuda.synchronize()
    assert np.array_equal(G.buf_to_np(buf, plan.nbytes), B_ref)
    plan.close(); empty.close(); ring.close(); small.close()


# ---- explicit buffer layout (checkpoint store, f3) ------------------------------------------
@pytest.mark.parametrize("kernel", ["warp", "warp_upload", "bulk"])
def test_layout_parity(G, kernel):
    """pack / unpack with per-request (offset, plane stride), one-shot (HBM, mapped host) and
    staged: the whole buffer (gaps included) and the whole restored pool equal the oracle's."""
    import torch
    rng = substream(99, "gpu_layout")
    done = 0
    while done < 18:
        w = random_tiny(rng) if done % 3 else cfg1_qwen14b(L=2, N=1024, n_reqs=12, grow_iters=8,
                                                           median=150, hi=400, lo=20).advanced(16 * (done // 3 + 1))
        L, H, D, S, N = w.geom
        row = H * D * 2
        if row % 16 or not w.tokens:
            continue
        lays, at = [], int(rng.integers(0, 4)) * row
        for _, tb, te in w.reqs:
            stride = (te - tb) + int(rng.integers(0, 4))
            lays.append((at, stride))
            at += 2 * L * stride * row + int(rng.integers(0, 3)) * row
        size = at + row
        seed = 200 + done
        K, V = G.host_planes(w.geom, seed)
        B_ref = np.full(size // 2, 0xA5A5, dtype=np.uint16)
        oracle.pack_layout(w.geom, K, V, w.reqs, [(o // 2, s) for o, s in lays], B_ref)
        K2, V2 = G.host_planes(w.geom, seed + 1)
        oracle.unpack_layout(w.geom, K2, V2, w.restore_reqs, [(o // 2, s) for o, s in lays], B_ref)
        pool_a, pool_b = G.make_pool(w.geom, seed), G.make_pool(w.geom, seed + 1)
        ck_a, ck_b = G.Checkpointer(pool_a, G.KERNELS[kernel]), G.Checkpointer(pool_b, G.KERNELS[kernel])
        plan = ck_a.plan(w.reqs, layouts=lays)
        rplan = ck_b.plan(w.restore_reqs, unique_dst=True, layouts=lays)
        assert plan.nbytes <= size
        mode = ("device", "host", "staged")[done % 3 if done >= 3 else done]
        whole, buf = G.alloc_buffer(size, "device" if mode == "device" else "host")
        if mode == "staged":
            max_run = max(plan.run(i).count for i in range(plan.num_runs)) * row
            ring = G.StagingRing((max_run * int(rng.integers(1, 5)) + 15) // 16 * 16, 3)
            ck_a.pack_staged(plan, buf, ring)
            ck_b.unpack_staged(rplan, buf, ring)
        else:
            ck_a.pack(plan, buf)
            ck_b.unpack(rplan, buf)
        torch.cuda.synchronize()
        assert np.array_equal(G.buf_to_np(buf, size), B_ref), f"layout pack mismatch ({mode})"
        assert G.guards_intact(whole, size)
        for t, ref in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
            assert np.array_equal(G.plane_to_np(t), ref), f"layout unpack mismatch ({mode})"
        plan.close(); rplan.close()
        done += 1


def test_host_threads_share_the_library(G):
    """The library holds no per-call global state: four host threads build, pack, restore and
    free their own plans on their own streams at once (uploaded descriptors, so the arena's
    cache is shared); every thread's bytes equal the oracle's."""
    import threading
    import torch
    lk = G.lk
    w = cfg1_qwen14b(L=2, N=2048, n_reqs=16, grow_iters=8, median=150, hi=400, lo=20)
    K, V = G.host_planes(w.geom, 77)
    pool = G.make_pool(w.geom, 77)
    errors = []

    def worker(tid):
        try:
            torch.cuda.set_device(0)
            stream = torch.cuda.Stream()
            flags = lk.LUMEN_KV_NO_INLINE if tid % 2 else 0
            for it in range(12):
                ww = w.advanced(16 * (1 + (tid + it) % 6))
                ref = oracle.pack(ww.geom, K, V, ww.reqs)
                plan = lk.lumen_kv_plan_build(pool.geom, ww.reqs, flags, stream.cuda_stream)
                buf = torch.empty(plan.nbytes, dtype=torch.uint8, device="cuda")
                lk.lumen_kv_checkpoint_pack(plan, pool.k_ptrs, pool.v_ptrs, buf.data_ptr(), plan.nbytes,
                                            lk.LUMEN_KV_MEM_DEVICE, stream.cuda_stream)
                plan.close()                                # freed while the kernel may still run
                stream.synchronize()
                if not np.array_equal(G.buf_to_np(buf, ref.size * 2), ref):
                    errors.append((tid, it))
        except Exception as e:                              # noqa: BLE001
            errors.append((tid, repr(e)))

    threads = [threading.Thread(target=worker, args=(t,)) for t in range(4)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=120)
    assert not errors and not any(t.is_alive() for t in threads)


@pytest.mark.parametrize("kernel", ["warp", "warp_upload", "bulk"])
def test_many_planes_and_huge_rows(G, kernel):
    """Edge geometries: 2L = 260 planes (more than the 256 plane pointers one launch carries, so
    the plane base of the second launch matters) and a 64 KiB row (one row is larger than the
    32 KiB run limit and than the TMA ring slot: the bulk kernel hands over to the SIMT one)."""
    import workloads.gen as gen
    rng = substream(7, "edge")
    perm = rng.permutation(64)
    reqs = [(perm[0:5].astype(np.int32), 3, 18), (perm[5:8].astype(np.int32), 0, 9)]
    rreqs = [(perm[8:13].astype(np.int32), 3, 18), (perm[13:16].astype(np.int32), 0, 9)]
    w = gen.Workload("many_planes", (130, 1, 8, 4, 64), reqs, rreqs)
    run_case(G, w, kernel, "device")
    run_case(G, w, kernel, "host")
    assert run_staged_case(G, w, 4096, 3, kernel=kernel) >= 2
    perm = rng.permutation(8)
    reqs = [(perm[0:3].astype(np.int32), 1, 5)]
    rreqs = [(perm[3:6].astype(np.int32), 1, 5)]
    w = gen.Workload("huge_rows", (1, 64, 512, 2, 8), reqs, rreqs)      # row = 64 KiB
    run_case(G, w, kernel, "device")
    run_staged_case(G, w, 1 << 16, 2, kernel=kernel)


def test_alignment_falls_back_to_16_byte_accesses(G):
    """The default SIMT kernel moves 32 bytes per access; a buffer, plane or page stride that is
    only 16-byte aligned must take the 16-byte kernel and still be bit-exact."""
    import torch
    lk = G.lk
    w = cfg1_qwen14b(L=2, N=512, n_reqs=8, grow_iters=2, median=100, hi=256, lo=20)
    L, H, D, S, N = w.geom
    K, V = G.host_planes(w.geom, 5)
    ref = oracle.pack(w.geom, K, V, w.reqs)
    pool = G.make_pool(w.geom, 5)
    ck = G.Checkpointer(pool)
    plan = ck.plan(w.reqs)
    for shift in (16, 32, 48):                                # buffer base = 256-aligned + shift
        raw = torch.full((plan.nbytes + 4096,), 0xA5, dtype=torch.uint8, device="cuda")
        view = raw[shift: shift + plan.nbytes]
        ck.pack(plan, view)
        torch.cuda.synchronize()
        assert np.array_equal(G.buf_to_np(view, plan.nbytes), ref)
        assert bool((raw[:shift] == 0xA5).all()) and bool((raw[shift + plan.nbytes:] == 0xA5).all())
    # page stride that is a multiple of 16 but not of 32: planes with 16 bytes of padding per page
    row = H * D * 2
    stride = S * row + 16
    geom = lk.make_geom(L, H, D, S, N, page_stride_bytes=stride)
    planes = [torch.zeros(N * stride, dtype=torch.uint8, device="cuda") for _ in range(2 * L)]
    for p, src in zip(planes, pool.planes()):
        p.view(N, stride)[:, : S * row] = src.view(torch.uint8).view(N, S * row)
    kp = lk.plane_ptrs([planes[2 * l].data_ptr() for l in range(L)], L)
    vp = lk.plane_ptrs([planes[2 * l + 1].data_ptr() for l in range(L)], L)
    splan = lk.lumen_kv_plan_build(geom, w.reqs, 0, 0)
    out = torch.empty(splan.nbytes, dtype=torch.uint8, device="cuda")
    lk.lumen_kv_checkpoint_pack(splan, kp, vp, out.data_ptr(), splan.nbytes, lk.LUMEN_KV_MEM_DEVICE, 0)
    torch.cuda.synchronize()
    assert np.array_equal(G.buf_to_np(out, splan.nbytes), ref)


@pytest.mark.parametrize("elem_bytes", [1, 4])
def test_other_element_widths(G, elem_bytes):
    """The payload is opaque: an fp8 KV cache (1-byte elements) or a 4-byte one is the same byte
    permutation.  The library gets (H, D, elem_bytes); the oracle sees the same rows as 16-bit
    words (E = H*D*elem_bytes/2) -- results must be identical bytes."""
    import torch
    lk = G.lk
    L, H, D, S, N = 3, 4, 32, 16, 256
    E16 = H * D * elem_bytes // 2
    geom16 = (L, 1, E16, S, N)                                  # what the oracle is told
    w = cfg1_qwen14b(L=L, H=1, D=E16, S=S, N=N, n_reqs=6, grow_iters=2, median=100, hi=200, lo=20)
    K, V = G.host_planes(geom16, 31)
    ref = oracle.pack(geom16, K, V, w.reqs)
    K2, V2 = G.host_planes(geom16, 32)
    oracle.unpack(geom16, K2, V2, w.restore_reqs, ref)
    pool_a, pool_b = G.make_pool(geom16, 31), G.make_pool(geom16, 32)
    g = lk.make_geom(L, H, D, S, N, elem_bytes=elem_bytes)      # what the library is told
    plan = lk.lumen_kv_plan_build(g, w.reqs, 0, 0)
    rplan = lk.lumen_kv_plan_build(g, w.restore_reqs, lk.LUMEN_KV_VALIDATE_UNIQUE_DST, 0)
    assert plan.nbytes == ref.size * 2
    buf = torch.empty(plan.nbytes, dtype=torch.uint8, device="cuda")
    lk.lumen_kv_checkpoint_pack(plan, pool_a.k_ptrs, pool_a.v_ptrs, buf.data_ptr(), plan.nbytes, 0, 0)
    lk.lumen_kv_restore_unpack(rplan, pool_b.k_ptrs, pool_b.v_ptrs, buf.data_ptr(), plan.nbytes, 0, 0)
    torch.cuda.synchronize()
    assert np.array_equal(G.buf_to_np(buf, plan.nbytes), ref)
    for t, r in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
        assert np.array_equal(G.plane_to_np(t), r)


@pytest.mark.parametrize("kernel", ["warp", "warp_upload", "bulk"])
def test_cuda_graph_capture(G, kernel):
    """pack + restore captured into a CUDA graph (with the programmatic-launch attribute on the
    SIMT kernel) and replayed: same bytes as the oracle, every replay."""
    import torch
    lk = G.lk
    w = cfg1_qwen14b(L=2, N=1024, n_reqs=8, grow_iters=2, median=100, hi=256, lo=20)
    K, V = G.host_planes(w.geom, 3)
    ref = oracle.pack(w.geom, K, V, w.reqs)
    K2, V2 = G.host_planes(w.geom, 4)
    oracle.unpack(w.geom, K2, V2, w.restore_reqs, ref)
    pool, pool_b = G.make_pool(w.geom, 3), G.make_pool(w.geom, 4)
    s = torch.cuda.Stream()
    plan = lk.lumen_kv_plan_build(pool.geom, w.reqs, G.KERNELS[kernel], s.cuda_stream)
    rplan = lk.lumen_kv_plan_build(pool.geom, w.restore_reqs, G.KERNELS[kernel], s.cuda_stream)
    buf = torch.zeros(plan.nbytes, dtype=torch.uint8, device="cuda")
    s.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        lk.lumen_kv_checkpoint_pack(plan, pool.k_ptrs, pool.v_ptrs, buf.data_ptr(), plan.nbytes, 0, s.cuda_stream)
        lk.lumen_kv_restore_unpack(rplan, pool_b.k_ptrs, pool_b.v_ptrs, buf.data_ptr(), plan.nbytes, 0,
                                   s.cuda_stream)
    for _ in range(3):
        buf.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(G.buf_to_np(buf, plan.nbytes), ref)
    for t, r in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
        assert np.array_equal(G.plane_to_np(t), r)
    del g
    plan.close(); rplan.close()


@pytest.mark.gpu
@pytest.mark.parametrize("shape", ["one_wave", "many_waves"])
@pytest.mark.parametrize("kernel", ["warp", "warp_upload"])
def test_l2_prefetch_is_only_a_hint(G, kernel, shape):
    """The SIMT kernel asks L2 for source bytes ahead of the stream-order wait (option
    "prefetch": -1 off, 0 own task, d > 0 the task d CTAs further on).  Whatever the distance,
    the bytes are the oracle's -- also when fill -> pack -> restore -> pack run back to back on
    one stream with no host synchronisation in between, so that every kernel's early prefetch
    meets the previous kernel's stores (the buffers are reused with new content every round:
    a stale line would show)."""
    import torch
    lk = G.lk
    # one_wave: 288 CTAs, all of them resident (and prefetching) while the previous kernel still
    # runs; many_waves: 3,700 CTAs = 5 waves, the steady state behind the first wave as well
    w = (cfg1_qwen14b(L=3, N=2048, n_reqs=24, grow_iters=2, median=200, hi=512, lo=20) if shape == "one_wave"
         else cfg1_qwen14b(L=8, N=3200, n_reqs=120, grow_iters=2, median=150, hi=400, lo=20))
    flags = G.KERNELS[kernel]
    pool_a, pool_b = G.make_pool(w.geom, 7), G.make_pool(w.geom, 8)
    ck_a, ck_b = G.Checkpointer(pool_a, flags), G.Checkpointer(pool_b, flags)
    plan, rplan = ck_a.plan(w.reqs), ck_b.plan(w.restore_reqs, unique_dst=True)
    whole, buf = G.alloc_buffer(plan.nbytes, "device")
    whole2, buf2 = G.alloc_buffer(plan.nbytes, "device")
    try:
        dists = [-1, 0, 1, 16, 37, 1000, 10 ** 6, 16, 16, 16] if shape == "one_wave" else [16, 0, 16]
        for rnd, dist in enumerate(dists):
            lk.lumen_kv_set_option("prefetch", dist)
            seed = 100 + rnd
            for i, t in enumerate(pool_a.planes()):
                G.wdev.fill_plane(t, seed, i, torch.cuda.current_stream().cuda_stream)
            ck_a.pack(plan, buf)
            ck_b.unpack(rplan, buf)
            ck_b.pack(rplan, buf2)
            torch.cuda.synchronize()
            K, V = G.host_planes(w.geom, seed)
            B_ref = oracle.pack(w.geom, K, V, w.reqs)
            assert np.array_equal(G.buf_to_np(buf, plan.nbytes), B_ref), dist
            assert np.array_equal(G.buf_to_np(buf2, plan.nbytes), B_ref), dist
            assert G.guards_intact(whole, plan.nbytes) and G.guards_intact(whole2, plan.nbytes)
    finally:
        lk.lumen_kv_set_option("prefetch", 16)
    # a buffer declared as peer memory takes the same kernels (no early prefetch of it)
    B = lk.binding
    s = torch.cuda.current_stream().cuda_stream
    buf.zero_()
    B.lumen_kv_checkpoint_pack(plan, pool_a.k_ptrs, pool_a.v_ptrs, buf.data_ptr(), plan.nbytes,
                               lk.LUMEN_KV_MEM_DEVICE_PEER, s)
    B.lumen_kv_restore_unpack(rplan, pool_b.k_ptrs, pool_b.v_ptrs, buf.data_ptr(), plan.nbytes,
                              lk.LUMEN_KV_MEM_DEVICE_PEER, s)
    ck_b.pack(rplan, buf2)
    torch.cuda.synchronize()
    assert np.array_equal(G.buf_to_np(buf, plan.nbytes), B_ref)
    assert np.array_equal(G.buf_to_np(buf2, plan.nbytes), B_ref)
    with pytest.raises(lk.LumenKVError):
        B.lumen_kv_checkpoint_pack(plan, pool_a.k_ptrs, pool_a.v_ptrs, buf.data_ptr(), plan.nbytes, 3, s)
    plan.close(); rplan.close()


@pytest.mark.parametrize("kernel", ["warp", "warp_upload", "bulk"])
def test_descriptor_size_classes(G, kernel):
    """Plans of 257 .. 1,024 runs / 129 .. 512 requests ride in the larger parameter block, plans
    beyond that (and NO_INLINE ones) upload their descriptors on the library's own stream: the three
    cases on the 32-byte kernel, the 16-byte kernel (48-byte rows) and the TMA kernel."""
    lk = G.lk
    shapes = [
        dict(L=2, N=4096, n_reqs=300, grow_iters=1, median=60, hi=200, lo=20),            # requests > 128
        dict(L=2, N=4096, n_reqs=100, grow_iters=1, median=120, hi=300, lo=40, delta=120),  # runs > 256
        dict(L=2, H=1, D=24, N=4096, n_reqs=300, grow_iters=1, median=60, hi=200, lo=20),  # 16-byte kernel
        dict(L=1, N=6000, n_reqs=600, grow_iters=1, median=40, hi=100, lo=20),            # > 512 requests: upload
    ]
    for i, kw in enumerate(shapes):
        w = cfg1_qwen14b(**kw)
        plan = lk.lumen_kv_plan_build(lk.make_geom(*w.geom), w.reqs, lk.LUMEN_KV_HOST_ONLY)
        runs, reqs = plan.num_runs, len(w.reqs)
        plan.close()
        if i < 3:
            assert 256 < runs <= 1024 or 128 < reqs <= 512, (runs, reqs)
        else:
            assert reqs > 512
        run_case(G, w, kernel, "device" if i % 2 == 0 else "host", seed=40 + i)


def test_upload_on_the_library_stream_orders_the_kernel(G):
    """A plan with uploaded descriptors is used at once, on a stream that has just been created,
    with no host synchronisation anywhere; descriptor blobs are recycled from plan to plan."""
    import torch
    lk = G.lk
    w = cfg1_qwen14b(L=2, N=8192, n_reqs=32, grow_iters=40, median=200, hi=512, lo=20)
    K, V = G.host_planes(w.geom, 11)
    pool = G.make_pool(w.geom, 11)
    ck = G.Checkpointer(pool, lk.LUMEN_KV_NO_INLINE)
    torch.cuda.synchronize()
    bufs, refs, cur, streams = [], [], w, []
    for it in range(24):
        s = torch.cuda.Stream()
        streams.append(s)
        plan = ck.plan(cur.reqs, stream=s)
        buf = torch.empty(plan.nbytes, dtype=torch.uint8, device="cuda")
        ck.pack(plan, buf, stream=s)
        plan.close()
        bufs.append(buf); refs.append(oracle.pack(cur.geom, K, V, cur.reqs))
        cur = cur.advanced(16)
    torch.cuda.synchronize()
    for buf, ref in zip(bufs, refs):
        assert np.array_equal(G.buf_to_np(buf, buf.numel()), ref)
    lk.lumen_kv_trim()
