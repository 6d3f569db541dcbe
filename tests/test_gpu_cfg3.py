"""configs[3], the recovery burst (SURVEY.md section 8(a) a6-a8, 8(d) cfg 3): checkpointed
prefixes are restored from pinned host memory into pages popped from a seeded shuffled
free list of a 40 %-occupied pool, while a second stream keeps packing 1-token deltas of
the running requests to pinned host memory.  As written the burst needs 198 GiB of
restored KV, so it runs in waves: a wave admits interrupted
requests while the free list can hold the next one.

Checked against the oracle: (mid size) the whole pool after all restores and every
concurrent pack buffer, element by element; (full size) sampled restored words through
the oracle's index accessors, every restored row through the NumPy oracle's slot map,
per-page checksums of every non-target page (the running requests' pages among them),
and every concurrent pack buffer against the full C oracle on a sparse host pool.
"""
import numpy as np
import pytest

import oracle
from oracle import oracle_np
from workloads import MASTER_SEED, cfg3_burst, g_words, substream

pytestmark = pytest.mark.gpu

CKPT_PLANE = 0xC3            # "plane" id of the host-resident checkpoint content g(seed, 0xC3, w)


@pytest.fixture(scope="module")
def G():
    import torch
    assert torch.cuda.is_available()
    from tests import gpu_util
    gpu_util.build_all()
    return gpu_util


def _free():
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()


def run_wave(G, pool, ck, geom, wave_reqs, running, hbuf, nbytes, n_pack_iters, pack_bufs,
             s_restore, s_pack, t0, rings=None):
    """Restore one wave on s_restore while s_pack packs `n_pack_iters` 1-token deltas.
    rings = (restore ring, pack ring): both directions go through the two-stage path, as in
    bench.py --workload cfg3.  Returns the per-iteration running-request lists that were packed."""
    import torch
    lk = G.lk
    rplan = lk.lumen_kv_plan_build(pool.geom, wave_reqs, lk.LUMEN_KV_VALIDATE_UNIQUE_DST,
                                   s_restore.cuda_stream)
    assert rplan.nbytes == nbytes
    packed = []
    if rings:
        lk.lumen_kv_restore_unpack_staged(rplan, pool.k_ptrs, pool.v_ptrs, hbuf.data_ptr(), nbytes,
                                          rings[0].stager, s_restore.cuda_stream)
    else:
        lk.lumen_kv_restore_unpack(rplan, pool.k_ptrs, pool.v_ptrs, hbuf.data_ptr(), nbytes,
                                   lk.LUMEN_KV_MEM_HOST_MAPPED, s_restore.cuda_stream)
    for it in range(n_pack_iters):                      # a2-a4 on the second stream, meanwhile
        reqs = [(pt, te + t0 + it - 1, te + t0 + it) for pt, _, te in running]
        p = lk.lumen_kv_plan_build(pool.geom, reqs, 0, s_pack.cuda_stream)
        if rings:
            lk.lumen_kv_checkpoint_pack_staged(p, pool.k_ptrs, pool.v_ptrs, pack_bufs[it].data_ptr(),
                                               p.nbytes, rings[1].stager, s_pack.cuda_stream)
        else:
            lk.lumen_kv_checkpoint_pack(p, pool.k_ptrs, pool.v_ptrs, pack_bufs[it].data_ptr(),
                                        p.nbytes, lk.LUMEN_KV_MEM_HOST_MAPPED, s_pack.cuda_stream)
        p.close()
        packed.append(reqs)
    s_restore.synchronize(); s_pack.synchronize()
    rplan.close()
    return packed


@pytest.mark.parametrize("staged", [False, True])
def test_cfg3_mid_size_whole_pool(G, staged):
    """Burst shape at a size the full oracle finishes in seconds: every byte of the pool after
    all waves, and every concurrent pack buffer, equal the oracle's."""
    import torch
    rings = (G.StagingRing(1 << 20, 3), G.StagingRing(1 << 20, 3)) if staged else None
    b = cfg3_burst(MASTER_SEED + 3, L=2, N=768, n_running=8, n_interrupted=7, p_lo=40, p_hi=2500,
                   grow_iters=16)
    assert b.meta["n_waves"] >= 2
    L, H, D, S, N = b.geom
    pool = G.make_pool(b.geom, MASTER_SEED + 3)
    K, V = G.host_planes(b.geom, MASTER_SEED + 3)
    ck = G.Checkpointer(pool)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    tok_bytes = 2 * L * H * D * 2
    iters = 4
    for wv, wave in enumerate(b.waves):
        nbytes = sum(te - tb for _, tb, te in wave) * tok_bytes
        hbuf = G.pinned_buffer(nbytes)
        ref_ck = g_words(MASTER_SEED + 30 + wv, CKPT_PLANE, 0, nbytes // 2)
        hbuf.numpy().view(np.uint16)[:] = ref_ck
        pbufs = [G.pinned_buffer(len(b.running) * tok_bytes) for _ in range(iters)]
        packed = run_wave(G, pool, ck, b.geom, wave, b.running, hbuf, nbytes, iters, pbufs, s1, s2,
                          t0=(wv * iters) % 12, rings=rings)
        for reqs, pb in zip(packed, pbufs):             # packs read only the running requests' pages
            assert np.array_equal(pb.numpy().view(np.uint16), oracle.pack(b.geom, K, V, reqs))
        oracle.unpack(b.geom, K, V, wave, ref_ck, check_overlap=True)
        for t, ref in zip(pool.planes(), [x for kv in zip(K, V) for x in kv]):
            assert np.array_equal(G.plane_to_np(t), ref), f"pool mismatch after wave {wv}"


@pytest.mark.parametrize("staged", [False, True])
def test_cfg3_full_size_waves(G, staged):
    """configs[3] at full size: Qwen3-32B shape, N = 30,720 pages (120 GiB), 40 % occupied by
    64 running requests, 48 interrupted prefixes U{1024..32768} restored in waves from
    pinned host into a seeded shuffled free list, 1-token delta packs on a second stream."""
    import torch
    _free()
    rings = (G.StagingRing(32 << 20, 3), G.StagingRing(32 << 20, 3)) if staged else None
    b = cfg3_burst()
    L, H, D, S, N = b.geom
    E = H * D
    tok_bytes = 2 * L * E * 2
    free_b, _ = torch.cuda.mem_get_info()
    if free_b < N * S * tok_bytes + (6 << 30):
        pytest.skip("not enough free HBM for the 120 GiB pool")
    wave_bytes = [sum(te - tb for _, tb, te in w) * tok_bytes for w in b.waves]
    assert sum(wave_bytes) == sum(b.prefix_tokens) * tok_bytes
    try:
        hwhole = G.wdev.pinned_exact(max(wave_bytes) + 8192)
    except RuntimeError as e:
        pytest.skip(f"cannot pin {max(wave_bytes) >> 30} GiB: {e}")
    pool = G.make_pool(b.geom, MASTER_SEED + 3)
    ck = G.Checkpointer(pool)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    iters = 16
    pbufs = [G.pinned_buffer(len(b.running) * tok_bytes) for _ in range(iters)]
    from workloads.hostpool import sparse_host_pool
    Kh, Vh, keep = sparse_host_pool(b.geom, MASTER_SEED + 3,               # running pages only
                                    [(pt, te - 1, te + 64) for pt, _, te in b.running])
    rng = substream(3, "cfg3_samples")
    planes = pool.planes()
    page_bytes = S * E * 2
    for wv, wave in enumerate(b.waves):
        nbytes = wave_bytes[wv]
        seed_ck = MASTER_SEED + 30 + wv
        hwhole[:4096] = 0xA5
        hwhole[4096 + nbytes: 8192 + nbytes] = 0xA5
        hbuf = hwhole[4096: 4096 + nbytes]
        G.wdev.fill_host_checkpoint(hbuf, nbytes, seed_ck, CKPT_PLANE)
        before = torch.stack([G.wdev.page_checksums(t, N, page_bytes) for t in planes])
        tails = [(int(pt[(te - 1) // S]), te % S) for pt, _, te in wave if te % S]
        snaps = [[t.view(torch.int16).view(N, S, E)[pg, a:].clone() for t in planes] for pg, a in tails]
        packed = run_wave(G, pool, ck, b.geom, wave, b.running, hbuf, nbytes, iters, pbufs, s1, s2,
                          t0=(wv * iters) % 48, rings=rings)
        # concurrent packs: whole buffers against the C oracle
        for reqs, pb in zip(packed, pbufs):
            assert np.array_equal(pb.numpy().view(np.uint16), oracle.pack(b.geom, Kh, Vh, reqs))
        # restore: non-target pages (running requests' among them) unchanged
        after = torch.stack([G.wdev.page_checksums(t, N, page_bytes) for t in planes])
        target = torch.zeros(N, dtype=torch.bool, device="cuda")
        for pt, tb, te in wave:
            target[torch.from_numpy(pt[: (te - 1) // S + 1].astype(np.int64)).cuda()] = True
        assert int(target.sum()) == sum((te + S - 1) // S for _, _, te in wave)   # disjoint pages
        assert not bool(((before != after).any(dim=0) & ~target).any()), "a non-target page changed"
        # (1) sampled restored words, one by one through the oracle's accessors
        pidx, plane_of, expect = [], [], []
        for _ in range(1200):
            r = int(rng.integers(0, len(wave)))
            n = wave[r][2]
            l, c = int(rng.integers(0, L)), int(rng.integers(0, 2))
            j, e = int(rng.integers(0, n)), int(rng.integers(0, E))
            bi = oracle.buffer_index(b.geom, wave, r, l, c, j, e)
            expect.append(int(g_words(seed_ck, CKPT_PLANE, bi, 1)[0]))
            pidx.append(oracle.pool_index(b.geom, wave, r, j, e))
            plane_of.append(2 * l + c)
        got = [int(planes[p].view(torch.int16).view(-1)[i].item()) & 0xFFFF
               for p, i in zip(plane_of, pidx)]
        assert got == expect
        # (2) every restored row == its buffer row (NumPy oracle's slot map, torch as plumbing)
        lay, total = oracle_np.layout(b.geom, wave)
        assert total * 2 == nbytes
        words = hbuf.view(torch.int16)
        for (pt, tb, te), (off, n) in zip(wave, lay):
            ids = torch.from_numpy(oracle_np.slot_ids(S, pt, tb, te)).cuda()
            blk = words[off: off + n * 2 * L * E].cuda(non_blocking=True).view(2 * L, n, E)
            for p in range(2 * L):
                got_rows = planes[p].view(torch.int16).view(N * S, E).index_select(0, ids)
                assert torch.equal(got_rows, blk[p]), f"wave {wv}: restored rows differ, plane {p}"
            del blk
        # untouched tail slots of every request's last, partly filled page (a target page, so the
        # checksums above do not cover it): equal to the snapshot taken before the restore
        for (pg, a), old_rows in zip(tails, snaps):
            for p, old in zip(range(2 * L), old_rows):
                assert torch.equal(planes[p].view(torch.int16).view(N, S, E)[pg, a:], old)
        assert bool((hwhole[:4096] == 0xA5).all()) and bool((hwhole[4096 + nbytes: 8192 + nbytes] == 0xA5).all())
    G.release(hwhole)
    del pool, planes
    _free()
