"""Checkpoint store: reservation
arithmetic, append-only deltas, visibility, tags and segments -- on the CPU against a plain
Python model and the oracle; then the whole chain on the GPU: incremental packs -> store ->
failure -> tag lookup -> restore of the longest checkpointed prefix straight out of the arena,
equal to the oracle's restore of that prefix."""
import ctypes
import threading

import numpy as np
import pytest

import oracle
from workloads import MASTER_SEED, cfg0_tiny, cfg1_qwen14b, substream


@pytest.fixture(scope="module")
def lk():
    from paper_2606_17787_b200 import build
    build.build()
    import paper_2606_17787_b200 as lk
    return lk


def _arena(nbytes):
    a = np.zeros(nbytes + 16, dtype=np.uint8)
    off = (-a.ctypes.data) % 16
    return a, a[off:off + nbytes]


def test_reservation_arithmetic(lk):
    """Footprint = max context length x bytes per token, reserved at assignment, released at
    completion: closed forms, first fit, coalescing."""
    tokb = 1024                                              # cfg 0: 2 layers x 2 x 256 B rows
    keep, arena = _arena(100 * tokb)
    st = lk.Store(arena.ctypes.data, arena.size, tokb, 16)
    assert st.available == 100 * tokb and st.reserved == 0
    st.reserve(1, 40); st.reserve(2, 30); st.reserve(3, 30)
    assert st.available == 0 and st.reserved == 100 * tokb
    with pytest.raises(lk.LumenKVError) as e:
        st.reserve(4, 1)
    assert e.value.status == lk.LUMEN_KV_ENOMEM               # a holder never over-commits
    with pytest.raises(lk.LumenKVError) as e:
        st.reserve(1, 1)                                      # exactly one checkpoint per request
    assert e.value.status == lk.LUMEN_KV_EINVAL
    st.release(2)
    assert st.available == 30 * tokb
    with pytest.raises(lk.LumenKVError):
        st.reserve(5, 31)                                     # 30 free, contiguous
    st.release(1)
    st.reserve(6, 70)                                         # the two holes coalesced: 40 + 30
    assert st.available == 0
    st.release(3); st.release(6)
    assert st.available == 100 * tokb
    st.reserve(7, 100)
    with pytest.raises(lk.LumenKVError):
        st.release(99)


def test_append_segments_and_lookup_against_model(lk):
    rng = substream(5, "store")
    w = cfg0_tiny(full_prefix=True)
    L, H, D, S, N = w.geom
    E, tokb = H * D, 2 * L * H * D * 2
    from workloads import fill_plane_np
    K = [fill_plane_np(3, 2 * l, N * S * E) for l in range(L)]
    V = [fill_plane_np(3, 2 * l + 1, N * S * E) for l in range(L)]
    keep, arena = _arena(400 * tokb)
    st = lk.Store(arena.ctypes.data, arena.size, tokb, S, copy_threads=3)
    model = {}
    for rid, (pt, _, n) in enumerate(w.reqs):
        st.reserve(rid, n + 20)
        toks = rng.integers(0, 1000, size=n).astype(np.int32)
        cuts = sorted(set(rng.integers(1, n, size=3).tolist())) if n > 2 else []
        at, segs = 0, []
        for te in cuts + [n]:
            delta = oracle.pack(w.geom, K, V, [(pt, at, te)])
            tags = oracle.page_tags(toks[:te], S)              # tags as of this delta
            tags = tags[(tags["end_pos"] > at) & (tags["end_pos"] <= te)]
            st.append(rid, at, te, delta.ctypes.data, delta.nbytes, tags)
            segs.append((at, te, delta))
            at = te
        model[rid] = (toks, segs)
        assert st.tokens(rid) == n
    for rid, (toks, segs) in model.items():
        n = toks.size
        # history = exactly what was checkpointed: everything is reusable
        assert st.lookup(rid, oracle.page_tags(toks, S)) == n
        # history has grown: a partly filled last page no longer matches, the prefix is page aligned
        longer = np.concatenate([toks, rng.integers(0, 1000, size=S).astype(np.int32)])
        prefix = st.lookup(rid, oracle.page_tags(longer, S))
        assert prefix == (n // S) * S
        # a different token history shares no prefix beyond the common pages
        other = toks.copy()
        if n > S:
            other[S] += 1
            assert st.lookup(rid, oracle.page_tags(other, S)) == S
        segs_got = st.segments(rid, prefix)
        want = [(a, min(b, prefix), b - a) for a, b, _ in segs if a < prefix]
        assert [(int(s["t_begin"]), int(s["t_end"]), int(s["plane_stride_tokens"])) for s in segs_got] == want
        for s, (a, b, delta) in zip(segs_got, segs):           # bytes in the arena == the delta received
            off = int(s["buf_offset"])
            assert np.array_equal(arena[off:off + delta.nbytes].view(np.uint16), delta)
    # out-of-order / oversized / wrong-size deltas and bad tags are refused
    st.reserve(50, 10)
    d = np.zeros(4 * tokb // 2, dtype=np.uint16)
    none = np.zeros(0, dtype=lk.TAG_DTYPE)
    for args, code in (((50, 1, 5, d.ctypes.data, d.nbytes, none), lk.LUMEN_KV_EINVAL),
                       ((50, 0, 4, d.ctypes.data, d.nbytes - 2, none), lk.LUMEN_KV_ESIZE),
                       ((51, 0, 4, d.ctypes.data, d.nbytes, none), lk.LUMEN_KV_EINVAL)):
        with pytest.raises(lk.LumenKVError) as e:
            st.append(*args)
        assert e.value.status == code
    bad = np.array([(1, 9)], dtype=lk.TAG_DTYPE)               # end position outside (0, 4]
    with pytest.raises(lk.LumenKVError):
        st.append(50, 0, 4, d.ctypes.data, d.nbytes, bad)
    st.append(50, 0, 4, d.ctypes.data, d.nbytes, none)
    big = np.zeros(7 * tokb // 2, dtype=np.uint16)
    with pytest.raises(lk.LumenKVError):
        st.append(50, 4, 11, big.ctypes.data, big.nbytes, none)   # beyond the reserved footprint


def test_visibility_only_after_complete_reception(lk):
    """A lookup running while a large delta is being copied in sees either nothing of it or
    all of it."""
    tokb, S, n = 1 << 20, 16, 64                               # 64 MiB delta, copied by 4 threads
    keep, arena = _arena(n * tokb)
    st = lk.Store(arena.ctypes.data, arena.size, tokb, S, copy_threads=4)
    st.reserve(7, n)
    toks = np.arange(n, dtype=np.int32)
    tags = oracle.page_tags(toks, S)
    delta = np.full(n * tokb, 0x5C, dtype=np.uint8)
    seen, stop = set(), threading.Event()

    def poll():
        while not stop.is_set():
            seen.add((st.tokens(7), st.lookup(7, tags)))

    th = threading.Thread(target=poll)
    th.start()
    st.append(7, 0, n, delta.ctypes.data, delta.nbytes, tags)
    seen.add((st.tokens(7), st.lookup(7, tags)))
    stop.set(); th.join()
    # the two reads of a sample are separate calls, so (0, n) can straddle the publication;
    # a partial count or tags without their tokens ((n, 0), (k, .) with 0 < k < n) never appear
    assert seen <= {(0, 0), (0, n), (n, n)} and (n, n) in seen
    assert (arena[:n * tokb] == 0x5C).all()


@pytest.mark.gpu
def test_gpu_checkpoint_chain_end_to_end(lk):
    """Worker A packs a delta per step into a pinned buffer (3), the bytes reach the holder's
    store (4); A fails; the holder regenerates the tags from the token history, finds the
    longest checkpointed prefix and restores it into fresh pages straight out of the pinned
    arena (staged, explicit layout).  The restored pool equals the oracle's restore of that
    prefix; tags come from the CUDA kernel."""
    import torch
    from tests import gpu_util as G
    G.build_all()
    w = cfg1_qwen14b(L=3, N=1024, n_reqs=6, grow_iters=8, median=150, hi=300, lo=40)
    L, H, D, S, N = w.geom
    E, tokb = H * D, 2 * L * H * D * 2
    rng = substream(6, "chain")
    lens = [te for _, _, te in w.reqs]
    steps, delta_tok = 5, 16
    hist = [rng.integers(0, 32000, size=n + steps * delta_tok).astype(np.int32) for n in lens]
    pool_a = G.make_pool(w.geom, 21)
    ck_a = G.Checkpointer(pool_a)
    arena_t = G.pinned_buffer(sum(n + 8 * delta_tok for n in lens) * tokb)
    st = lk.Store(arena_t.data_ptr(), arena_t.numel(), tokb, S, copy_threads=2)
    for rid, n in enumerate(lens):
        st.reserve(rid, n + 8 * delta_tok)
    stage = G.pinned_buffer(max(lens) * tokb)                  # worker A's pinned staging buffer
    ring = G.StagingRing(1 << 20, 3)
    d_tags = torch.empty((4096, 2), dtype=torch.int64, device="cuda")

    def tags_of(tokens):                                       # CUDA tag kernel
        d_tok = torch.from_numpy(np.ascontiguousarray(tokens)).cuda()
        n = lk.lumen_kv_tags_num_pages([0, tokens.size], S)
        lk.lumen_kv_page_tags(d_tok.data_ptr(), [0, tokens.size], S, d_tags.data_ptr(), n, 0)
        torch.cuda.synchronize()
        return d_tags[:n].cpu().numpy().copy().view(lk.TAG_DTYPE).reshape(-1)

    sent = [0] * len(lens)
    for step in range(steps + 1):                              # step 0 = prefill-completion checkpoint
        for rid, (pt, _, n) in enumerate(w.reqs):
            te = n + step * delta_tok if step < steps else n + (steps - 1) * delta_tok + 5
            if te <= sent[rid]:
                continue
            plan = ck_a.plan([(pt, sent[rid], te)])
            ck_a.pack_staged(plan, stage, ring)
            torch.cuda.synchronize()
            tags = tags_of(hist[rid][:te])
            tags = tags[(tags["end_pos"] > sent[rid]) & (tags["end_pos"] <= te)]
            st.append(rid, sent[rid], te, stage.data_ptr(), plan.nbytes, tags)   # "network"
            plan.close()
            sent[rid] = te
    # ---- failure of worker A; the holder restores into its own pool under fresh page tables ----
    pool_b = G.make_pool(w.geom, 22)
    ck_b = G.Checkpointer(pool_b)
    K, V = G.host_planes(w.geom, 21)
    K2, V2 = G.host_planes(w.geom, 22)
    reqs, lays, total_prefix = [], [], 0
    for rid, (pt_new, _, _) in enumerate(w.restore_reqs):
        regen = tags_of(hist[rid])                             # full token history kept by the gateway
        assert np.array_equal(regen, oracle.page_tags(hist[rid], S))
        prefix = st.lookup(rid, regen)
        assert prefix == (sent[rid] // S) * S                  # the 5-token tail page does not match
        total_prefix += prefix
        for s in st.segments(rid, prefix):
            reqs.append((pt_new, int(s["t_begin"]), int(s["t_end"])))
            lays.append((int(s["buf_offset"]), int(s["plane_stride_tokens"])))
        # oracle: restore of exactly that prefix
        oracle.unpack(w.geom, K2, V2, [(pt_new, 0, prefix)], oracle.pack(w.geom, K, V, [(w.reqs[rid][0], 0, prefix)]))
    rplan = ck_b.plan(reqs, unique_dst=True, layouts=lays)
    assert rplan.nbytes <= arena_t.numel()
    ck_b.unpack_staged(rplan, arena_t, ring)
    torch.cuda.synchronize()
    for t, ref in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
        assert np.array_equal(G.plane_to_np(t), ref)
    assert total_prefix > 0
    for rid in range(len(lens)):                               # completion releases the footprint
        st.release(rid)
    assert st.reserved == 0


def test_concurrent_appends_and_churn(lk):
    """Eight host threads (receivers of different workers' streams) append deltas to their own
    requests while requests are reserved and released around them; every stored byte and every
    count matches, and the arena is whole again at the end."""
    tokb, S = 4096, 16
    n_req, per_req = 8, 200
    keep, arena = _arena((n_req * per_req + 300) * tokb)
    st = lk.Store(arena.ctypes.data, arena.size, tokb, S, copy_threads=2)
    for rid in range(n_req):
        st.reserve(rid, per_req)
    errors = []
    none = np.zeros(0, dtype=lk.TAG_DTYPE)

    def receiver(rid):
        try:
            rng = np.random.default_rng(rid)
            at = 0
            while at < per_req:
                n = int(min(per_req - at, rng.integers(1, 40)))
                delta = np.full(n * tokb, (rid * 37 + at) % 251, dtype=np.uint8)
                st.append(rid, at, at + n, delta.ctypes.data, delta.nbytes, none)
                at += n
            segs = st.segments(rid, per_req)
            for s in segs:
                blk = arena[int(s["buf_offset"]): int(s["buf_offset"]) + int(s["t_end"] - s["t_begin"]) * tokb]
                if not (blk == (rid * 37 + int(s["t_begin"])) % 251).all():
                    errors.append(("bytes", rid, int(s["t_begin"])))
        except Exception as e:                                   # noqa: BLE001
            errors.append((rid, repr(e)))

    def churn():
        try:
            for i in range(300):
                st.reserve(1000 + i, 1 + i % 90)
                st.release(1000 + i)
        except Exception as e:                                   # noqa: BLE001
            errors.append(("churn", repr(e)))

    threads = [threading.Thread(target=receiver, args=(r,)) for r in range(n_req)] + [threading.Thread(target=churn)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=120)
    assert not errors and not any(t.is_alive() for t in threads)
    assert all(st.tokens(r) == per_req for r in range(n_req))
    assert st.reserved == n_req * per_req * tokb
    for r in range(n_req):
        st.release(r)
    assert st.available == arena.size
    st.reserve(9999, arena.size // tokb)                          # coalesced back into one hole


def test_acquire_commit_abort_and_racing_lookup(lk):
    """Reserve-then-commit (lumen_kv_store_acquire): a writer gets the final position of a delta,
    fills it in place and commits with an append whose source IS that position.  Until the commit
    neither tokens(), lookup() nor segments() show the claim -- also while another thread keeps
    looking (visible only upon complete reception); claims stack in order; abort
    voids them; the stored bytes equal oracle.pack of each delta."""
    w = cfg0_tiny(full_prefix=True)
    L, H, D, S, N = w.geom
    tokb = 2 * L * H * D * 2
    from workloads import fill_plane_np
    E = H * D
    K = [fill_plane_np(3, 2 * l, N * S * E) for l in range(L)]
    V = [fill_plane_np(3, 2 * l + 1, N * S * E) for l in range(L)]
    pt, _, n_tok = w.reqs[1]                                     # 100 tokens
    toks = substream(7, "acq").integers(0, 5000, size=n_tok).astype(np.int32)
    keep, arena = _arena(2 * n_tok * tokb)
    st = lk.Store(arena.ctypes.data, arena.size, tokb, S)
    st.reserve(5, n_tok); st.reserve(6, n_tok)
    regen = lk.lumen_kv_page_tags_host(toks, 0, 0, n_tok, S)
    stop = threading.Event()
    seen, bad = [], []

    def looker():
        last = 0
        while not stop.is_set():
            t, p = st.tokens(5), st.lookup(5, regen)
            if t < last or p > t or p % S not in (0, t % S) and p != t:
                bad.append((t, p))
            last = t
            seen.append(t)

    th = threading.Thread(target=looker, daemon=True)
    th.start()
    try:
        _acquire_commit_abort_body(lk, st, w, K, V, pt, tokb, S, regen, arena, stop, th, seen, bad)
    finally:
        stop.set()
        th.join(10)


def _acquire_commit_abort_body(lk, st, w, K, V, pt, tokb, S, regen, arena, stop, th, seen, bad):
    cuts = [0, 37, 64, 100]
    # two stacked claims, filled and committed in order
    p0 = st.acquire(5, 0, 37)
    p1 = st.acquire(5, 37, 64)
    assert p0 and p1 == p0 + 37 * tokb
    assert st.acquire(5, 37, 64) == 0 and st.acquire(5, 70, 80) == 0     # must continue the claims
    assert st.acquire(5, 64, 101) == 0                                    # beyond the reservation
    assert st.tokens(5) == 0 and st.lookup(5, regen) == 0
    with pytest.raises(lk.LumenKVError):                                  # a copying append cannot jump the claims
        st.append(5, 0, 37, np.zeros(37 * tokb, dtype=np.uint8).ctypes.data, 37 * tokb, regen[:0])
    for (a, b), dst in (((0, 37), p0), ((37, 64), p1)):
        delta = oracle.pack(w.geom, K, V, [(pt, a, b)])
        view = np.ctypeslib.as_array((ctypes.c_uint16 * delta.size).from_address(dst))
        view[:] = delta                                                   # "the copy engine"
        assert st.tokens(5) == a                                          # filled, not committed
        tags = regen[(regen["end_pos"] > a) & (regen["end_pos"] <= b)]
        st.append(5, a, b, dst, delta.size * 2, tags)                     # the commit: no copy
        assert st.tokens(5) == b
    assert st.lookup(5, regen) == 64
    # a claim that is aborted leaves no trace; the next claim takes the same place
    p2 = st.acquire(5, 64, 100)
    assert p2 == p0 + 64 * tokb
    st.abort(5)
    assert st.tokens(5) == 64 and st.acquire(5, 64, 100) == p2
    with pytest.raises(lk.LumenKVError):                                  # commit with a foreign pointer
        st.append(5, 64, 100, p2 + 2, 36 * tokb, regen[:0])
    delta = oracle.pack(w.geom, K, V, [(pt, 64, 100)])
    np.ctypeslib.as_array((ctypes.c_uint16 * delta.size).from_address(p2))[:] = delta
    st.append(5, 64, 100, p2, delta.size * 2, regen[(regen["end_pos"] > 64)])
    stop.set(); th.join()
    assert not bad and st.tokens(5) == 100 and st.lookup(5, regen) == 100
    assert set(seen) <= set(cuts)                                         # only committed states were ever seen
    segs = st.segments(5, 100)
    assert [(int(s["t_begin"]), int(s["t_end"])) for s in segs] == [(0, 37), (37, 64), (64, 100)]
    base = arena.ctypes.data
    for s in segs:
        a, b = int(s["t_begin"]), int(s["t_end"])
        off = int(s["buf_offset"])
        got = arena[off: off + (b - a) * tokb].view(np.uint16)
        assert np.array_equal(got, oracle.pack(w.geom, K, V, [(pt, a, b)]))
    # the classic copying append still works on another request, and refuses to run under a claim
    assert st.acquire(6, 0, 10)
    with pytest.raises(lk.LumenKVError):
        st.release(6)                                                     # claimed: not releasable
    st.abort(6)
    d = oracle.pack(w.geom, K, V, [(pt, 0, 10)])
    st.append(6, 0, 10, d.ctypes.data, d.size * 2, regen[:0])
    assert st.tokens(6) == 10
    st.release(6); st.release(5)
    assert st.reserved == 0 and base == arena.ctypes.data


@pytest.mark.gpu
def test_gpu_background_checkpointer_writes_straight_into_the_store(lk):
    """lumen_kv_ckpt_set_direct: with a pinned arena the background checkpointer packs every
    delta to the position the store hands out (no second host copy) and commits it with the sink
    call.  Prefill in several pieces (stacked claims), decode deltas, a request whose reservation
    runs out (acquire refuses -> that batch goes the copying way and the store rejects it): the
    store's content equals oracle.pack of every delta, tags and progress are those of the copying
    path, and restore out of the store reproduces the oracle's pool."""
    import torch
    from tests import gpu_util as G
    G.build_all()
    w = cfg1_qwen14b(L=2, N=1024, n_reqs=5, grow_iters=8, median=150, hi=300, lo=60)
    L, H, D, S, N = w.geom
    tokb = 2 * L * H * D * 2
    lens = [te for _, _, te in w.reqs]
    steps, delta_tok = 6, 3
    rng = substream(8, "direct")
    hist = [rng.integers(0, 32000, size=n + steps * delta_tok).astype(np.int32) for n in lens]
    K, V = G.host_planes(w.geom, 31)
    results = {}
    for mode in ("direct", "copy"):
        pool = G.make_pool(w.geom, 31)
        arena_t = G.pinned_buffer(sum(n + steps * delta_tok for n in lens) * tokb)
        arena_t.zero_()
        st = lk.Store(arena_t.data_ptr(), arena_t.numel(), tokb, S, copy_threads=2)
        for rid, n in enumerate(lens):
            st.reserve(rid, n + steps * delta_tok - (4 if rid == 4 else 0))     # request 4 runs out of room
        ring_mem = torch.empty(3 << 20, dtype=torch.uint8, device="cuda")
        pinned = G.pinned_buffer(2 * 100 * tokb)                 # halves of 100 tokens: prefill comes in pieces
        bg = lk.BackgroundCheckpointer(pool.geom, pool.k_ptrs, pool.v_ptrs, ring_mem.data_ptr(), 1 << 20, 3,
                                       pinned.data_ptr(), pinned.numel(), st,
                                       direct_min_bytes=0 if mode == "direct" else None)
        assert bg.direct == (mode == "direct")
        for rid in range(len(lens)):
            bg.track(rid, 0)
        bg.notify(list(range(len(lens))), [(pt, 0, n) for (pt, _, n) in w.reqs], token_ids=hist)
        for step in range(1, steps + 1):
            bg.notify(list(range(len(lens))), [(pt, 0, n + step * delta_tok) for (pt, _, n) in w.reqs],
                      token_ids=hist)
            if step == 3:
                bg.flush()
        try:
            bg.flush()
            raised = None
        except lk.LumenKVError as e:
            raised = e.status
        assert raised == lk.LUMEN_KV_ESINK                       # request 4's last delta did not fit
        final = [n + steps * delta_tok for n in lens]
        for rid in range(4):
            assert bg.progress(rid) == final[rid] == st.tokens(rid)
        assert st.tokens(4) == bg.progress(4) < final[4]
        state = []
        for rid in range(len(lens)):
            segs = st.segments(rid, st.tokens(rid))
            at = 0
            for s in segs:
                a, b, off = int(s["t_begin"]), int(s["t_end"]), int(s["buf_offset"])
                assert a == at
                at = b
                got = arena_t[off: off + (b - a) * tokb].numpy().view(np.uint16)
                assert np.array_equal(got, oracle.pack(w.geom, K, V, [(w.reqs[rid][0], a, b)])), (mode, rid, a, b)
            assert at == st.tokens(rid)
            regen = lk.lumen_kv_page_tags_host(hist[rid], 0, 0, st.tokens(rid), S)
            state.append((st.tokens(rid), st.lookup(rid, regen)))
        results[mode] = state
        # recovery out of the store into fresh pages == the oracle's restore of the same prefix
        pool_b = G.make_pool(w.geom, 32)
        K2, V2 = G.host_planes(w.geom, 32)
        ringr = G.StagingRing(1 << 20, 3)
        for rid, (pt_new, _, _) in enumerate(w.restore_reqs):
            n = st.tokens(rid)
            got = st.restore(rid, hist[rid][:n], pool_b.geom, pt_new, pool_b.k_ptrs, pool_b.v_ptrs, ringr.stager)
            assert got == state[rid][1]
            if got:
                oracle.unpack(w.geom, K2, V2, [(pt_new, 0, got)],
                              oracle.pack(w.geom, K, V, [(w.reqs[rid][0], 0, got)]))
        torch.cuda.synchronize()
        for t, ref in zip(pool_b.planes(), [x for kv in zip(K2, V2) for x in kv]):
            assert np.array_equal(G.plane_to_np(t), ref), mode
        ringr.close(); bg.close(); st.close()
    assert results["direct"] == results["copy"]
