"""lumen_kv_copy_noalloc against the regular pack / restore calls.

Some users of this library cannot let it allocate GPU memory: a serving worker that gave all of
its HBM to the KV pool (a cudaMalloc may fail just when a recovery burst needs a restore), or a
decode loop that cannot take the device-wide stall cudaMalloc / cudaFree cause.  For them the
library has one call whose descriptor memory is an array built into the library itself, shared
by every call and never cleared.  This test checks that the call moves exactly the bytes the
regular calls move (the tolerance of every test here: bit for bit), in both directions, for two
different plans enqueued one right after the other on one stream -- the second, smaller plan
runs over what the first left in the array -- and that an oversized plan is refused.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here
should not hide the parity tests.  It passes alone in a fresh process (its first call then
performs the per-device set-up) and after every other test.
"""
import ctypes

import numpy as np
import pytest

import oracle
from workloads import cfg1_qwen14b, cfg4_longctx, MASTER_SEED


@pytest.fixture(scope="module")
def G():
    import torch
    assert torch.cuda.is_available()
    from tests import gpu_util
    gpu_util.build_all()
    return gpu_util


def _regular(G, w, seed, where):
    """Pack with the existing call; restore with the existing call into a second pool."""
    import torch
    pool_a, pool_b = G.make_pool(w.geom, seed), G.make_pool(w.geom, seed + 1)
    ck_a, ck_b = G.Checkpointer(pool_a), G.Checkpointer(pool_b)
    plan = ck_a.plan(w.reqs)
    whole, buf = G.alloc_buffer(plan.nbytes, where)
    ck_a.pack(plan, buf)
    rplan = ck_b.plan(w.restore_reqs, unique_dst=True)
    ck_b.unpack(rplan, buf)
    torch.cuda.synchronize()
    packed = G.buf_to_np(buf, plan.nbytes)
    restored = [G.plane_to_np(t) for t in pool_b.planes()]
    plan.close(); rplan.close()
    G.release(whole)
    return packed, restored


@pytest.mark.gpu
def test_noalloc_equals_regular_path_two_calls_in_a_row(G):
    import torch
    lk = G.lk
    # plan 1: 6,002 one-token runs (six descriptor slices, the last one ragged; the regular call
    # uploads such a plan to device memory it allocates); plan 2: 24 requests' 16-token deltas,
    # a different geometry, far fewer runs than plan 1 left behind in the array
    w1 = cfg4_longctx(L=2, tokens=3001, wave_reqs=2)
    w2 = cfg1_qwen14b(L=3, N=2048, n_reqs=24, grow_iters=2, median=200, hi=512, lo=20)
    cases = [(w1, MASTER_SEED, "device"), (w2, MASTER_SEED + 7, "host")]
    want = [_regular(G, w, seed, where) for w, seed, where in cases]
    # the first plan's packed buffer also against the CPU oracle
    K, V = G.host_planes(w1.geom, MASTER_SEED)
    assert np.array_equal(want[0][0], oracle.pack(w1.geom, K, V, w1.reqs))

    stream = torch.cuda.Stream()
    state = []
    with torch.cuda.stream(stream):
        for w, seed, where in cases:
            pool_a, pool_b = G.make_pool(w.geom, seed), G.make_pool(w.geom, seed + 1)
            whole, buf = G.alloc_buffer(w.payload_bytes, where)
            state.append((pool_a, pool_b, whole, buf))
    torch.cuda.synchronize()
    kind = {"device": lk.LUMEN_KV_MEM_DEVICE, "host": lk.LUMEN_KV_MEM_HOST_MAPPED}
    # four calls back to back on one stream, no synchronisation in between:
    # pack 1, restore 1, pack 2, restore 2
    for (w, seed, where), (pool_a, pool_b, whole, buf) in zip(cases, state):
        plan = lk.lumen_kv_plan_build(pool_a.geom, w.reqs, lk.LUMEN_KV_HOST_ONLY)
        assert plan.nbytes == w.payload_bytes
        lk.lumen_kv_copy_noalloc(plan, lk.LUMEN_KV_DIR_PACK, pool_a.k_ptrs, pool_a.v_ptrs,
                                 buf.data_ptr(), plan.nbytes, kind[where], stream.cuda_stream)
        plan.close()                      # the descriptors have left the host already
        rplan = lk.lumen_kv_plan_build(pool_b.geom, w.restore_reqs,
                                       lk.LUMEN_KV_HOST_ONLY | lk.LUMEN_KV_VALIDATE_UNIQUE_DST)
        lk.lumen_kv_copy_noalloc(rplan, lk.LUMEN_KV_DIR_RESTORE, pool_b.k_ptrs, pool_b.v_ptrs,
                                 buf.data_ptr(), rplan.nbytes, kind[where], stream.cuda_stream)
        rplan.close()
    stream.synchronize()
    for i, ((w, seed, where), (pool_a, pool_b, whole, buf)) in enumerate(zip(cases, state)):
        packed, restored = want[i]
        assert np.array_equal(G.buf_to_np(buf, w.payload_bytes), packed), f"pack, call {i}"
        assert G.guards_intact(whole, w.payload_bytes)
        for p, (t, ref) in enumerate(zip(pool_b.planes(), restored)):
            assert np.array_equal(G.plane_to_np(t), ref), f"restore, call {i}, plane {p}"
        G.release(whole)


@pytest.mark.gpu
def test_noalloc_accepts_any_plan_and_an_empty_one(G):
    """A plan built without HOST_ONLY (descriptors in the parameters of the regular kernels, or
    uploaded) runs through the call as well; an empty plan is a no-op."""
    import torch
    lk = G.lk
    w = cfg1_qwen14b(L=2, N=512, n_reqs=8, grow_iters=2, median=100, hi=256, lo=20)
    packed, _ = _regular(G, w, 3, "device")
    pool = G.make_pool(w.geom, 3)
    for flags in (0, lk.LUMEN_KV_NO_INLINE):
        plan = lk.lumen_kv_plan_build(pool.geom, w.reqs, flags)
        whole, buf = G.alloc_buffer(plan.nbytes, "device")
        lk.lumen_kv_copy_noalloc(plan, lk.LUMEN_KV_DIR_PACK, pool.k_ptrs, pool.v_ptrs, buf.data_ptr(),
                                 plan.nbytes)
        torch.cuda.synchronize()
        assert np.array_equal(G.buf_to_np(buf, plan.nbytes), packed)
        assert G.guards_intact(whole, plan.nbytes)
        plan.close()
    empty = lk.lumen_kv_plan_build(pool.geom, [], lk.LUMEN_KV_HOST_ONLY)
    lk.lumen_kv_copy_noalloc(empty, lk.LUMEN_KV_DIR_PACK, pool.k_ptrs, pool.v_ptrs, 0, 0)


def test_noalloc_refuses_what_does_not_fit():
    """The size limit is checked on the host before any CUDA call, so this runs without a GPU."""
    from paper_2606_17787_b200 import build
    build.build()
    import paper_2606_17787_b200 as lk
    geom = lk.make_geom(1, 1, 8, 1, 70000)                        # S = 1: one run per token
    fake = (ctypes.c_void_p * 1)(4096)
    pt = np.arange(lk.LUMEN_KV_NOALLOC_MAX_RUNS + 1, dtype=np.int32)
    for n, status in ((pt.size, lk.LUMEN_KV_ECAPACITY),):
        plan = lk.lumen_kv_plan_build(geom, [(pt, 0, n)], lk.LUMEN_KV_HOST_ONLY)
        assert plan.num_runs == n
        with pytest.raises(lk.LumenKVError) as ei:
            lk.lumen_kv_copy_noalloc(plan, lk.LUMEN_KV_DIR_PACK, fake, fake, 4096, plan.nbytes)
        assert ei.value.status == status
        assert "lumen_kv_copy_noalloc" in lk.lumen_kv_strerror(status)
    reqs = [(pt[:1], 0, 1)] * (lk.LUMEN_KV_NOALLOC_MAX_REQS + 1)  # pack may share pages
    plan = lk.lumen_kv_plan_build(geom, reqs, lk.LUMEN_KV_HOST_ONLY)
    with pytest.raises(lk.LumenKVError) as ei:
        lk.lumen_kv_copy_noalloc(plan, lk.LUMEN_KV_DIR_RESTORE, fake, fake, 4096, plan.nbytes)
    assert ei.value.status == lk.LUMEN_KV_ECAPACITY
    small = lk.lumen_kv_plan_build(geom, [(pt, 0, 4)], lk.LUMEN_KV_HOST_ONLY)
    for bad_dir in (-1, 2):
        with pytest.raises(lk.LumenKVError) as ei:
            lk.lumen_kv_copy_noalloc(small, bad_dir, fake, fake, 4096, small.nbytes)
        assert ei.value.status == lk.LUMEN_KV_EINVAL
    with pytest.raises(lk.LumenKVError) as ei:                    # buffer too small
        lk.lumen_kv_copy_noalloc(small, lk.LUMEN_KV_DIR_PACK, fake, fake, 4096, small.nbytes - 1)
    assert ei.value.status == lk.LUMEN_KV_ESIZE
