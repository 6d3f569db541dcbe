"""The worker's background checkpointer (include/lumen_kv.h lumen_kv_ckpt_*):
host-side argument checks on the CPU; on the GPU a decode loop notifies it after every batch
without ever waiting, the sink (standing in for the network send) appends to a checkpoint
store, and what arrives equals the oracle's pack of exactly the ranges delivered; after a
"failure" the stored prefix is restored and equals the oracle's restore."""
import threading

import numpy as np
import pytest

import oracle
from workloads import cfg1_qwen14b, substream


@pytest.fixture(scope="module")
def lk():
    from paper_2606_17787_b200 import build
    build.build()
    import paper_2606_17787_b200 as lk
    return lk


def test_create_needs_a_device_and_valid_arguments(lk):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    g = lk.make_geom(2, 2, 64, 16, 64)
    host = np.zeros(1 << 16, dtype=np.uint8)
    with pytest.raises(lk.LumenKVError) as e:               # the stager's copy stream needs CUDA
        lk.BackgroundCheckpointer(g, [16, 16], [16, 16], 4096, 4096, 2, host.ctypes.data & ~15, 1 << 15,
                                  lambda *a: None)
    assert e.value.status == lk.LUMEN_KV_ECUDA
    bad = lk.make_geom(2, 2, 3, 16, 64)                      # 12-byte rows
    with pytest.raises(lk.LumenKVError) as e:
        lk.BackgroundCheckpointer(bad, [16, 16], [16, 16], 4096, 4096, 2, host.ctypes.data & ~15, 1 << 15,
                                  lambda *a: None)
    assert e.value.status == lk.LUMEN_KV_EINVAL


@pytest.mark.gpu
def test_background_checkpointing_decode_loop(lk):
    import torch
    from tests import gpu_util as G
    G.build_all()
    w = cfg1_qwen14b(L=3, N=1024, n_reqs=6, grow_iters=10, median=150, hi=300, lo=40)
    L, H, D, S, N = w.geom
    tokb = 2 * L * H * D * 2
    pool = G.make_pool(w.geom, 41)
    K, V = G.host_planes(w.geom, 41)
    lens = [te for _, _, te in w.reqs]
    steps, dtok = 8, 16
    ring_mem = torch.empty(3 << 20, dtype=torch.uint8, device="cuda")
    pinned = G.pinned_buffer(64 * tokb)                      # two halves of 32 tokens: every prefill delta splits
    arena = G.pinned_buffer(sum(n + steps * dtok for n in lens) * tokb)
    st = lk.Store(arena.data_ptr(), arena.numel(), tokb, S)
    for rid, n in enumerate(lens):
        st.reserve(rid, n + steps * dtok)
    delivered, errors = {rid: [] for rid in range(len(lens))}, []
    rng = substream(8, "ckpt_tokens")
    hist = [rng.integers(0, 151936, size=n + steps * dtok + 9).astype(np.int32) for n in lens]

    def sink(rid, tb, te, ptr, nbytes, tags):                # runs on the checkpointer's thread
        try:
            got = np.ctypeslib.as_array((np.ctypeslib.ctypes.c_uint16 * (nbytes // 2)).from_address(ptr))
            ref = oracle.pack(w.geom, K, V, [(w.reqs[rid][0], tb, te)])
            if nbytes != (te - tb) * tokb or not np.array_equal(got, ref):
                errors.append(("bytes", rid, tb, te))
            want = oracle.page_tags(hist[rid][:te], S)       # "each transferred page carries a page tag"
            if not np.array_equal(tags, want[want["end_pos"] > tb]):
                errors.append(("tags", rid, tb, te))
            st.append(rid, tb, te, ptr, nbytes, tags)        # step (4): into the holder's store
            delivered[rid].append((tb, te))
        except Exception as e:                               # noqa: BLE001
            errors.append((rid, repr(e)))

    bg = lk.BackgroundCheckpointer(pool.geom, pool.k_ptrs, pool.v_ptrs, ring_mem.data_ptr(), 1 << 20, 3,
                                   pinned.data_ptr(), pinned.numel(), sink)
    for rid in range(len(lens)):
        bg.track(rid, 0)
    compute = torch.cuda.Stream()
    scratch = torch.zeros(1 << 22, device="cuda")
    events = []
    ids = list(range(len(lens)))
    for step in range(steps + 1):                            # step 0: prefill completion
        with torch.cuda.stream(compute):
            scratch.add_(1.0)                                # "the batch that produced the tokens"
            ev = torch.cuda.Event()
            ev.record(compute)
        events.append(ev)
        cur = [(pt, 0, n + step * dtok) for (pt, _, n) in w.reqs]
        bg.notify(ids, cur, ev.cuda_event, token_ids=hist)   # never waits for the checkpointer
    with pytest.raises(lk.LumenKVError):                     # going backwards is refused
        bg.notify([0], [(w.reqs[0][0], 0, 5)])
    with pytest.raises(lk.LumenKVError):
        bg.notify([99], [(w.reqs[0][0], 0, 5)])
    bg.flush()
    assert not errors
    for rid, n in enumerate(lens):
        final = n + steps * dtok
        assert bg.progress(rid) == final and st.tokens(rid) == final
        spans = delivered[rid]
        assert spans[0][0] == 0 and spans[-1][1] == final
        assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))        # in order, no gap
        assert all(te - tb <= 32 for tb, te in spans)                      # never more than half the pinned buffer
    # ---- failure: KV-reuse recovery of every request on the holder, one call each ----
    pool_b = G.make_pool(w.geom, 42)
    K2, V2 = G.host_planes(w.geom, 42)
    ring = G.StagingRing(1 << 20, 3)
    side = torch.cuda.Stream()
    for rid, (pt_new, _, n) in enumerate(w.restore_reqs):
        final = n + steps * dtok
        # cross-check the host-regenerated tags the call uses with the CUDA kernel's
        d_tok = torch.from_numpy(hist[rid]).cuda()
        n_pg = lk.lumen_kv_tags_num_pages([0, hist[rid].size], S)
        d_tags = torch.empty((n_pg, 2), dtype=torch.int64, device="cuda")
        lk.lumen_kv_page_tags(d_tok.data_ptr(), [0, hist[rid].size], S, d_tags.data_ptr(), n_pg, 0)
        torch.cuda.synchronize()
        regen = d_tags.cpu().numpy().copy().view(lk.TAG_DTYPE).reshape(-1)
        assert np.array_equal(regen, lk.lumen_kv_page_tags_host(hist[rid], 0, 0, hist[rid].size, S))
        prefix = st.restore(rid, hist[rid], pool_b.geom, pt_new, pool_b.k_ptrs, pool_b.v_ptrs,
                            ring.stager, side.cuda_stream)
        assert prefix == st.lookup(rid, regen) == (final // S) * S   # the history is 9 tokens longer
        oracle.unpack(w.geom, K2, V2, [(pt_new, 0, prefix)],
                      oracle.pack(w.geom, K, V, [(w.reqs[rid][0], 0, prefix)]))
    side.synchronize()
    for t, ref in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
        assert np.array_equal(G.plane_to_np(t), ref)
    assert st.restore(0, hist[0][::-1].copy(), pool_b.geom, w.restore_reqs[0][0], pool_b.k_ptrs,
                      pool_b.v_ptrs, ring.stager, 0) == 0               # another history: nothing to reuse
    with pytest.raises(lk.LumenKVError):
        st.restore(77, hist[0], pool_b.geom, w.restore_reqs[0][0], pool_b.k_ptrs, pool_b.v_ptrs, ring.stager, 0)
    bg.untrack(0)
    with pytest.raises(lk.LumenKVError):
        bg.progress(0)
    bg.close()


@pytest.mark.gpu
def test_background_checkpointer_stress(lk):
    """Three producer threads notify their requests at random paces (tiny pinned buffer, so deltas
    are batched, split and superseded in every combination), some requests are untracked in
    mid-flight: every delivered delta is the oracle's, each request's deltas tile a prefix of its
    tokens in order, and what was not untracked is delivered completely."""
    import random
    import time
    import torch
    from tests import gpu_util as G
    G.build_all()
    w = cfg1_qwen14b(L=2, N=2048, n_reqs=12, grow_iters=20, median=120, hi=260, lo=30)
    L, H, D, S, N = w.geom
    tokb = 2 * L * H * D * 2
    pool = G.make_pool(w.geom, 51)
    K, V = G.host_planes(w.geom, 51)
    lens = [te for _, _, te in w.reqs]
    final = [n + 20 * 16 for n in lens]
    ring_mem = torch.empty(2 * (256 << 10), dtype=torch.uint8, device="cuda")
    pinned = G.pinned_buffer(48 * tokb)
    spans, errors, lock = {r: [] for r in range(len(lens))}, [], threading.Lock()

    def sink(rid, tb, te, ptr, nbytes, tags):
        got = np.ctypeslib.as_array((np.ctypeslib.ctypes.c_uint16 * (nbytes // 2)).from_address(ptr))
        if not np.array_equal(got, oracle.pack(w.geom, K, V, [(w.reqs[rid][0], tb, te)])):
            errors.append(("bytes", rid, tb, te))
        with lock:
            spans[rid].append((tb, te))

    bg = lk.BackgroundCheckpointer(pool.geom, pool.k_ptrs, pool.v_ptrs, ring_mem.data_ptr(), 256 << 10, 2,
                                   pinned.data_ptr(), pinned.numel(), sink)
    for rid in range(len(lens)):
        bg.track(rid, 0)
    dropped = {}

    def producer(tid):
        rnd = random.Random(tid)
        mine = [r for r in range(len(lens)) if r % 3 == tid]
        cur = {r: 0 for r in mine}
        try:
            while mine:
                batch = rnd.sample(mine, rnd.randint(1, len(mine)))
                for r in batch:
                    cur[r] = min(final[r], cur[r] + rnd.choice([1, 1, 16, 40, lens[r]]))
                bg.notify(batch, [(w.reqs[r][0], 0, cur[r]) for r in batch])
                if rnd.random() < 0.3:
                    time.sleep(rnd.random() * 0.002)
                if rnd.random() < 0.04 and len(mine) > 1:       # a request completes / is cancelled
                    r = mine.pop(rnd.randrange(len(mine)))
                    bg.untrack(r)
                    dropped[r] = cur[r]
                mine = [r for r in mine if cur[r] < final[r]]
        except Exception as e:                                   # noqa: BLE001
            errors.append((tid, repr(e)))

    threads = [threading.Thread(target=producer, args=(t,)) for t in range(3)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=120)
    bg.flush()
    assert not errors and not any(t.is_alive() for t in threads)
    for rid in range(len(lens)):
        sp = spans[rid]
        assert all(a[1] == b[0] for a, b in zip(sp, sp[1:])) and (not sp or sp[0][0] == 0)
        assert all(te - tb <= 24 for tb, te in sp)               # half of the 48-token pinned buffer
        end = sp[-1][1] if sp else 0
        if rid in dropped:
            assert end <= dropped[rid]                           # a prefix of what had been notified
        else:
            assert end == final[rid] and bg.progress(rid) == final[rid]
    bg.close()


@pytest.mark.gpu
def test_sink_rejection_keeps_progress_and_surfaces(lk):
    """a sink that rejects a delta must not advance the request's progress; the
    rest of that request (pending, and already in the next batch) is dropped, flush() reports
    LUMEN_KV_ESINK, other requests are unaffected, and the next notification packs again from
    the last delivered token so that the sink never sees a gap."""
    import ctypes
    import torch
    from tests import gpu_util as G
    G.build_all()
    w = cfg1_qwen14b(L=2, N=512, n_reqs=3, grow_iters=6, median=100, hi=120, lo=90)
    L, H, D, S, N = w.geom
    tokb = 2 * L * H * D * 2
    pool = G.make_pool(w.geom, 77)
    K, V = G.host_planes(w.geom, 77)
    lens = [te for _, _, te in w.reqs]
    ring_mem = torch.empty(3 << 20, dtype=torch.uint8, device="cuda")
    pinned = G.pinned_buffer(64 * tokb)                      # halves of 32 tokens: prefill deltas come in pieces
    got = {r: [] for r in range(3)}
    reject = {"on": True}

    def sink(rid, tb, te, ptr, nb, tags):
        if rid == 1 and reject["on"] and tb >= 32:           # request 1: second piece onwards
            return -1
        data = np.ctypeslib.as_array((ctypes.c_uint16 * (nb // 2)).from_address(ptr)).copy()
        got[rid].append((tb, te, data))
        return 0

    bg = lk.BackgroundCheckpointer(pool.geom, pool.k_ptrs, pool.v_ptrs, ring_mem.data_ptr(), 1 << 20, 3,
                                   pinned.data_ptr(), pinned.numel(), sink)
    for rid in range(3):
        bg.track(rid, 0)
    bg.notify([0, 1, 2], [(pt, 0, n) for (pt, _, n) in w.reqs])
    with pytest.raises(lk.LumenKVError) as e:
        bg.flush()
    assert e.value.status == lk.LUMEN_KV_ESINK
    assert bg.progress(0) == lens[0] and bg.progress(2) == lens[2]
    assert bg.progress(1) == 32                               # only the first piece was taken
    assert [(tb, te) for tb, te, _ in got[1]] == [(0, 32)]
    reject["on"] = False
    bg.notify([1], [(w.reqs[1][0], 0, lens[1] + 5)])          # the retry starts at token 32
    try:
        bg.flush()
    except lk.LumenKVError as e2:                             # first_error is sticky by design
        assert e2.status == lk.LUMEN_KV_ESINK
    assert bg.progress(1) == lens[1] + 5
    for rid in range(3):
        at = 0
        for tb, te, data in got[rid]:
            assert tb == at                                   # deltas tile [0, t) in order: no gap, no repeat
            at = te
            ref = oracle.pack(w.geom, K, V, [(w.reqs[rid][0], tb, te)])
            assert np.array_equal(data, ref)
        assert at == bg.progress(rid)
    bg.close()


@pytest.mark.gpu
def test_raising_sink_rejects_the_delta(lk):
    """ctypes turns an exception inside the sink callback into a return value of 0,
    which the checkpointer would read as "taken".  The binding must hand back a rejection instead:
    progress stays where it was, flush() raises ESINK with the sink's exception as its cause, and a
    later notification delivers the same tokens again."""
    import ctypes
    import torch
    from tests import gpu_util as G
    G.build_all()
    w = cfg1_qwen14b(L=2, N=512, n_reqs=2, grow_iters=4, median=60, hi=64, lo=50)
    L, H, D, S, N = w.geom
    tokb = 2 * L * H * D * 2
    pool = G.make_pool(w.geom, 5)
    K, V = G.host_planes(w.geom, 5)
    ring_mem = torch.empty(3 << 20, dtype=torch.uint8, device="cuda")
    pinned = G.pinned_buffer(256 * tokb)
    got = {0: [], 1: []}
    state = {"raise": True}

    def sink(rid, tb, te, ptr, nb, tags):
        if rid == 1 and state["raise"]:
            raise RuntimeError("sink broke")
        got[rid].append((tb, te, np.ctypeslib.as_array((ctypes.c_uint16 * (nb // 2)).from_address(ptr)).copy()))

    bg = lk.BackgroundCheckpointer(pool.geom, pool.k_ptrs, pool.v_ptrs, ring_mem.data_ptr(), 1 << 20, 3,
                                   pinned.data_ptr(), pinned.numel(), sink)
    lens = [te for _, _, te in w.reqs]
    bg.track(0, 0); bg.track(1, 0)
    bg.notify([0, 1], [(pt, 0, n) for (pt, _, n) in w.reqs])
    with pytest.raises(lk.LumenKVError) as e:
        bg.flush()
    assert e.value.status == lk.LUMEN_KV_ESINK
    assert isinstance(e.value.__cause__, RuntimeError) and "sink broke" in str(e.value.__cause__)
    assert bg.progress(0) == lens[0] and bg.progress(1) == 0 and got[1] == []
    state["raise"] = False
    bg.notify([1], [(w.reqs[1][0], 0, lens[1])])
    try:
        bg.flush()
    except lk.LumenKVError as e2:                             # first_error is sticky by design
        assert e2.status == lk.LUMEN_KV_ESINK and e2.__cause__ is None
    assert bg.progress(1) == lens[1]
    for rid in (0, 1):
        at = 0
        for tb, te, data in got[rid]:
            assert tb == at
            at = te
            assert np.array_equal(data, oracle.pack(w.geom, K, V, [(w.reqs[rid][0], tb, te)]))
        assert at == lens[rid]
    bg.close()


@pytest.mark.gpu
def test_blocking_sink_and_failing_pack_do_not_hang_the_checkpointer(lk):
    """(a) destroying a checkpointer whose sink is blocked for two
    seconds waits for the sink and returns -- no deadlock; (b) a staged pack that fails inside the
    background thread (failure injection) is reported by flush() as ECUDA, progress does not move,
    and after the fault is gone a new notification delivers the tokens."""
    import ctypes
    import threading
    import time
    import torch
    from tests import gpu_util as G
    G.build_all()
    w = cfg1_qwen14b(L=2, N=512, n_reqs=2, grow_iters=4, median=60, hi=64, lo=50)
    L, H, D, S, N = w.geom
    tokb = 2 * L * H * D * 2
    pool = G.make_pool(w.geom, 5)
    K, V = G.host_planes(w.geom, 5)
    lens = [te for _, _, te in w.reqs]
    ring_mem = torch.empty(3 << 20, dtype=torch.uint8, device="cuda")
    pinned = G.pinned_buffer(256 * tokb)
    entered = threading.Event()
    got = []

    def slow_sink(rid, tb, te, ptr, nb, tags):
        entered.set()
        time.sleep(2.0)
        got.append((rid, tb, te))

    bg = lk.BackgroundCheckpointer(pool.geom, pool.k_ptrs, pool.v_ptrs, ring_mem.data_ptr(), 1 << 20, 3,
                                   pinned.data_ptr(), pinned.numel(), slow_sink)
    bg.track(0, 0)
    bg.notify([0], [(w.reqs[0][0], 0, lens[0])])
    assert entered.wait(20.0)
    t0 = time.perf_counter()
    closer = threading.Thread(target=bg.close)
    closer.start()
    closer.join(30.0)
    assert not closer.is_alive(), "lumen_kv_ckpt_destroy hangs behind a blocked sink"
    assert time.perf_counter() - t0 < 25.0 and got and got[0][0] == 0

    data = {0: [], 1: []}

    def sink(rid, tb, te, ptr, nb, tags):
        data[rid].append((tb, te, np.ctypeslib.as_array((ctypes.c_uint16 * (nb // 2)).from_address(ptr)).copy()))

    bg = lk.BackgroundCheckpointer(pool.geom, pool.k_ptrs, pool.v_ptrs, ring_mem.data_ptr(), 1 << 20, 3,
                                   pinned.data_ptr(), pinned.numel(), sink)
    try:
        bg.track(0, 0); bg.track(1, 0)
        lk.lumen_kv_set_option("fail_after_chunks", 0)
        bg.notify([0, 1], [(pt, 0, n) for (pt, _, n) in w.reqs])
        with pytest.raises(lk.LumenKVError) as e:
            bg.flush()
        assert e.value.status == lk.LUMEN_KV_ECUDA
        assert bg.progress(0) == 0 and bg.progress(1) == 0 and not data[0] and not data[1]
    finally:
        lk.lumen_kv_set_option("fail_after_chunks", -1)
    bg.notify([0, 1], [(pt, 0, n) for (pt, _, n) in w.reqs])
    try:
        bg.flush()
    except lk.LumenKVError as e2:                             # first_error is sticky by design
        assert e2.status == lk.LUMEN_KV_ECUDA
    for rid in (0, 1):
        assert bg.progress(rid) == lens[rid]
        at = 0
        for tb, te, d in data[rid]:
            assert tb == at
            at = te
            assert np.array_equal(d, oracle.pack(w.geom, K, V, [(w.reqs[rid][0], tb, te)]))
        assert at == lens[rid]
    bg.close()
