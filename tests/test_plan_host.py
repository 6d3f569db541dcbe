"""CPU tests of the C-ABI library's host logic (no GPU, no compute calls).

T1 of SURVEY.md section 4: the plan builder's runs, expanded back to per-token
(request, token) -> (pool slot, buffer row), must equal the oracle's index map
(oracle.pool_index / oracle.buffer_index, i.e. definition C1).  Also: the library
loads and exports every symbol include/lumen_kv.h declares, sizes and offsets
match the closed forms, validation rules of section 8(b)/C6 return the documented
status codes, and compute entry points fail loudly without a CUDA device.
"""
import re
from pathlib import Path

import numpy as np
import pytest

import oracle
from oracle import oracle_np
from workloads import cfg0_tiny, cfg1_qwen14b, cfg2_qwen32b, cfg4_longctx, random_tiny, substream

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lk():
    from paper_2606_17787_b200 import build
    build.build()
    import paper_2606_17787_b200 as lk
    return lk


def geom_of(lk, w, **kw):
    L, H, D, S, N = w.geom
    return lk.make_geom(L, H, D, S, N, **kw)


def expand(plan, geom, reqs):
    """runs -> dict (req, j) -> (global pool slot, count bookkeeping)."""
    L, H, D, S, N = geom
    out = {}
    for i in range(plan.num_runs):
        r = plan.run(i)
        assert r.count >= 1
        for k in range(r.count):
            key = (r.req, r.dst_token + k)
            assert key not in out, "token covered twice"
            out[key] = r.src_slot + k
    return out


def test_exports_match_header(lk):
    import ctypes
    text = (ROOT / "include" / "lumen_kv.h").read_text()
    declared = set(re.findall(r"LUMEN_KV_API[^;(]*?\b(lumen_kv_\w+)\s*\(", text))
    assert declared == set(lk.EXPORTS)
    lib = ctypes.CDLL(str(lk.library_path()))
    for name in declared:
        assert hasattr(lib, name), name
    assert lk.lumen_kv_version() == int(re.search(r"#define LUMEN_KV_VERSION (\d+)", text).group(1))


def test_struct_layouts_match_header(lk):
    import ctypes
    assert ctypes.sizeof(lk.lumen_kv_geom) == 40
    assert ctypes.sizeof(lk.lumen_kv_req) == 32
    assert ctypes.sizeof(lk.lumen_kv_run_info) == 24


@pytest.mark.parametrize("merge", [False, True])
def test_t1_runs_equal_oracle_index_map(lk, merge):
    rng = substream(77, "t1")
    flags = lk.LUMEN_KV_HOST_ONLY | (lk.LUMEN_KV_MERGE_ADJACENT if merge else 0)
    cases = [cfg0_tiny(), cfg0_tiny(full_prefix=True)] + [random_tiny(rng, allow_shared=True) for _ in range(150)]
    for w in cases:
        L, H, D, S, N = w.geom
        E = H * D
        plan = lk.lumen_kv_plan_build(geom_of(lk, w), w.reqs, flags)
        assert plan.nbytes == 2 * oracle.total_elems(w.geom, w.reqs)
        m = expand(plan, w.geom, w.reqs)
        assert len(m) == w.tokens
        for r, (pt, tb, te) in enumerate(w.reqs):
            assert plan.req_offset(r) == 2 * oracle.req_offset_elems(w.geom, w.reqs, r)
            for j in range(te - tb):
                # oracle: word e=0 of token j lives at pool word slot*E
                assert m[(r, j)] * E == oracle.pool_index(w.geom, w.reqs, r, j, 0)
        assert plan.req_offset(len(w.reqs)) == plan.nbytes
        plan.close()


def test_runs_never_cross_pages_unless_merged_and_respect_chunk(lk):
    w = cfg2_qwen32b(N=2048, n_reqs=4, prompt=1000)
    L, H, D, S, N = w.geom
    row = H * D * 2
    plan = lk.lumen_kv_plan_build(geom_of(lk, w), w.reqs, lk.LUMEN_KV_HOST_ONLY)
    assert plan.num_runs == sum((te - 1) // S - tb // S + 1 for _, tb, te in w.reqs)
    for i in range(plan.num_runs):
        r = plan.run(i)
        assert r.src_slot // S == (r.src_slot + r.count - 1) // S
        assert r.count * row <= 32768


def test_p9_merge_adjacent_identity_table(lk):
    # identity page table: every page adjacent -> merged runs are chunk-sized (32 KiB)
    L, H, D, S, N = 1, 2, 8, 4, 4096          # row = 32 B, page = 128 B
    g = lk.make_geom(L, H, D, S, N)
    pt = np.arange(N, dtype=np.int32)
    a = lk.lumen_kv_plan_build(g, [(pt, 3, 4 * N - 5)], lk.LUMEN_KV_HOST_ONLY)
    b = lk.lumen_kv_plan_build(g, [(pt, 3, 4 * N - 5)], lk.LUMEN_KV_HOST_ONLY | lk.LUMEN_KV_MERGE_ADJACENT)
    assert a.num_runs == N - 1                            # last token 4N-6 lies in page N-2
    assert b.num_runs == -(-(4 * N - 8) // 1024)          # ceil(tokens / (32 KiB / 32 B))
    assert expand(a, (L, H, D, S, N), None) == expand(b, (L, H, D, S, N), None)


def test_page_stride(lk):
    L, H, D, S, N = 1, 2, 8, 4, 16
    row = H * D * 2
    g = lk.make_geom(L, H, D, S, N, page_stride_bytes=S * row + 64)
    pt = np.array([3, 4, 9], dtype=np.int32)
    p = lk.lumen_kv_plan_build(g, [(pt, 1, 11)], lk.LUMEN_KV_HOST_ONLY | lk.LUMEN_KV_MERGE_ADJACENT)
    # padded stride: adjacent pages are not byte-contiguous, so no merging
    assert [(p.run(i).src_slot, p.run(i).count) for i in range(p.num_runs)] == [(13, 3), (16, 4), (36, 3)]


def test_closed_form_sizes_big_configs(lk):
    w1 = cfg1_qwen14b()
    p1 = lk.lumen_kv_plan_build(geom_of(lk, w1), w1.reqs, lk.LUMEN_KV_HOST_ONLY)
    assert p1.nbytes == 167_772_160
    assert 64 <= p1.num_runs <= 128
    w2 = cfg2_qwen32b()
    p2 = lk.lumen_kv_plan_build(geom_of(lk, w2), w2.reqs,
                                lk.LUMEN_KV_HOST_ONLY | lk.LUMEN_KV_VALIDATE_UNIQUE_DST)
    assert p2.nbytes == 32 * 2**30 and p2.num_runs == 8192
    w4 = cfg4_longctx(tokens=4096, wave_reqs=2)
    p4 = lk.lumen_kv_plan_build(geom_of(lk, w4), w4.reqs,
                                lk.LUMEN_KV_HOST_ONLY | lk.LUMEN_KV_VALIDATE_UNIQUE_DST)
    assert p4.num_runs == 8192 and p4.nbytes == 8192 * 256 * 1024


def test_oracle_np_layout_equals_plan_offsets(lk):
    w = cfg1_qwen14b(N=4096, n_reqs=8, grow_iters=2, hi=2048)
    plan = lk.lumen_kv_plan_build(geom_of(lk, w), w.reqs, lk.LUMEN_KV_HOST_ONLY)
    lay, total = oracle_np.layout(w.geom, w.reqs)
    assert plan.nbytes == 2 * total
    assert [plan.req_offset(r) for r in range(len(w.reqs))] == [2 * o for o, _ in lay]


def test_validation_status_codes(lk):
    E = lk.LumenKVError
    H = lk.LUMEN_KV_HOST_ONLY
    g = lk.make_geom(2, 2, 8, 4, 16)
    pt = np.array([1, 2, 3], dtype=np.int32)

    def status(fn):
        with pytest.raises(E) as e:
            fn()
        return e.value.status

    # geometry
    assert status(lambda: lk.lumen_kv_plan_build(lk.make_geom(0, 2, 8, 4, 16), [], H)) == lk.LUMEN_KV_EINVAL
    assert status(lambda: lk.lumen_kv_plan_build(lk.make_geom(1, 1, 4, 4, 16), [], H)) == lk.LUMEN_KV_EINVAL  # row 8 B
    assert status(lambda: lk.lumen_kv_plan_build(lk.make_geom(1, 2, 8, 4, 0), [], H)) == lk.LUMEN_KV_EINVAL
    assert status(lambda: lk.lumen_kv_plan_build(lk.make_geom(1, 2, 8, 4, 2**31), [], H)) == lk.LUMEN_KV_EINVAL
    assert status(lambda: lk.lumen_kv_plan_build(lk.make_geom(1, 2, 8, 4, 16, page_stride_bytes=100), [], H)) == lk.LUMEN_KV_EINVAL
    # ranges
    assert status(lambda: lk.lumen_kv_plan_build(g, [(pt, 5, 4)], H)) == lk.LUMEN_KV_EINVAL
    assert status(lambda: lk.lumen_kv_plan_build(g, [(pt, -1, 4)], H)) == lk.LUMEN_KV_EINVAL
    assert status(lambda: lk.lumen_kv_plan_build(g, [(pt, 0, 13)], H)) == lk.LUMEN_KV_ERANGE
    assert status(lambda: lk.lumen_kv_plan_build(g, [(np.array([1, 16], np.int32), 0, 8)], H)) == lk.LUMEN_KV_ERANGE
    assert status(lambda: lk.lumen_kv_plan_build(g, [(np.array([1, -1], np.int32), 0, 8)], H)) == lk.LUMEN_KV_ERANGE
    # A6: entries outside the touched range are ignored
    lk.lumen_kv_plan_build(g, [(np.array([99, 2, 99], np.int32), 4, 8)], H).close()
    # unknown flag / kernel selector
    assert status(lambda: lk.lumen_kv_plan_build(g, [], H | 0x80)) == lk.LUMEN_KV_EINVAL
    assert status(lambda: lk.lumen_kv_plan_build(g, [], H | 0x300)) == lk.LUMEN_KV_EINVAL
    # A5: duplicate destination page, across and within requests
    U = H | lk.LUMEN_KV_VALIDATE_UNIQUE_DST
    assert status(lambda: lk.lumen_kv_plan_build(g, [(pt, 0, 4), (pt, 0, 4)], U)) == lk.LUMEN_KV_EOVERLAP
    assert status(lambda: lk.lumen_kv_plan_build(g, [(np.array([5, 5], np.int32), 0, 8)], U)) == lk.LUMEN_KV_EOVERLAP
    lk.lumen_kv_plan_build(g, [(pt, 0, 4), (pt, 0, 4)], H).close()        # pack may share pages
    lk.lumen_kv_plan_build(g, [(pt, 0, 4), (pt, 4, 12)], U).close()       # disjoint pages are fine
    # sparse path of the uniqueness check (huge N, few pages)
    big = lk.make_geom(1, 2, 8, 4, 2**31 - 1)
    far = np.array([2**31 - 2, 7], dtype=np.int32)
    assert status(lambda: lk.lumen_kv_plan_build(big, [(far, 0, 8), (far, 4, 8)], U)) == lk.LUMEN_KV_EOVERLAP
    lk.lumen_kv_plan_build(big, [(far, 0, 8)], U).close()


def test_empty_plans(lk):
    g = lk.make_geom(2, 2, 8, 4, 16)
    p = lk.lumen_kv_plan_build(g, [], lk.LUMEN_KV_HOST_ONLY)
    assert p.nbytes == 0 and p.num_runs == 0 and p.req_offset(0) == 0
    pt = np.array([1], dtype=np.int32)
    p = lk.lumen_kv_plan_build(g, [(pt, 2, 2), (np.zeros(0, np.int32), 0, 0)], lk.LUMEN_KV_HOST_ONLY)
    assert p.nbytes == 0 and p.num_runs == 0 and p.req_offset(2) == 0


def test_no_cpu_fallback(lk):
    """Without a CUDA device everything that would touch the device fails loudly (ECUDA):
    the descriptor upload of plan_build, and pack/unpack of a parameter-resident plan
    (whose build makes no CUDA call)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    g = lk.make_geom(2, 2, 8, 4, 16)
    pt = np.array([1], dtype=np.int32)
    with pytest.raises(lk.LumenKVError) as e:
        lk.lumen_kv_plan_build(g, [(pt, 0, 2)], lk.LUMEN_KV_NO_INLINE)
    assert e.value.status == lk.LUMEN_KV_ECUDA
    small = lk.lumen_kv_plan_build(g, [(pt, 0, 2)], 0)
    assert small.nbytes == 2 * 2 * 2 * 32 and small.num_runs == 1
    for call in (lk.lumen_kv_checkpoint_pack, lk.lumen_kv_restore_unpack):
        with pytest.raises(lk.LumenKVError) as e:
            call(small, [16, 16], [16, 16], 16, 1 << 20)
        assert e.value.status == lk.LUMEN_KV_ECUDA
    small.close()
    # the stager validates its arguments on the host, then needs a device for its copy stream
    for bad in ((0, 1024, 2), (16, 1000, 2), (16, 1024, 1), (16, 1024, 17), (24, 1024, 2)):
        with pytest.raises(lk.LumenKVError) as e:
            lk.Stager(*bad)
        assert e.value.status == lk.LUMEN_KV_EINVAL
    with pytest.raises(lk.LumenKVError) as e:
        lk.Stager(16, 1024, 2)
    assert e.value.status == lk.LUMEN_KV_ECUDA
    # a host-only plan cannot be executed
    p = lk.lumen_kv_plan_build(g, [(pt, 0, 2)], lk.LUMEN_KV_HOST_ONLY)
    with pytest.raises(lk.LumenKVError) as e:
        lk.lumen_kv_checkpoint_pack(p, [16, 16], [16, 16], 16, 1 << 20)
    assert e.value.status == lk.LUMEN_KV_EINVAL


def test_product_does_not_import_oracle():
    for p in (ROOT / "paper_2606_17787_b200").rglob("*"):
        if p.suffix in {".py", ".cu", ".cpp", ".hpp", ".h"}:
            s = p.read_text()
            assert "oracle" not in s.lower(), p
    for p in (ROOT / "oracle").rglob("*"):
        if p.suffix in {".py", ".c"}:
            s = p.read_text()
            assert "import paper_2606_17787_b200" not in s and "lumen_kv.h\"" not in s, p


def test_plan_build_speed_host(lk):
    """a2 must be microsecond-scale for per-decode-step deltas (SURVEY 7.3 hard part 2)."""
    import time
    w = cfg1_qwen14b()
    g = geom_of(lk, w)
    t0 = time.perf_counter()
    for _ in range(200):
        lk.lumen_kv_plan_build(g, w.reqs, lk.LUMEN_KV_HOST_ONLY).close()
    dt = (time.perf_counter() - t0) / 200
    assert dt < 2e-3, dt      # includes the ctypes marshalling of 64 requests


# ---- two-stage host path: the chunker (host arithmetic only) ---------------------------
def _check_chunks(plan, geom, reqs, slot):
    """Chunks tile the buffer in ascending order, fit the slot, and chunk (runs, planes) covers
    exactly its byte range according to the NumPy oracle's layout."""
    L, H, D, S, N = geom
    row = H * D * 2
    lay, total = oracle_np.layout(geom, reqs)             # (offset, n) per request, in words
    chunks = plan.chunks(slot)
    runs = [plan.run(i) for i in range(plan.num_runs)]
    at = 0
    for c in chunks:
        assert c.byte_begin == at and c.byte_end > c.byte_begin
        assert c.byte_end - c.byte_begin <= slot
        assert 0 <= c.plane_begin < c.plane_end <= 2 * L and c.run_begin < c.run_end
        covered = []
        for p in range(c.plane_begin, c.plane_end):
            for i in range(c.run_begin, c.run_end):
                r = runs[i]
                off_words, n = lay[r.req]
                b0 = off_words * 2 + (p * n + r.dst_token) * row
                covered.append((b0, b0 + r.count * row))
        covered.sort()
        assert covered[0][0] == c.byte_begin and covered[-1][1] == c.byte_end
        for (a0, a1), (b0, b1) in zip(covered, covered[1:]):
            assert a1 == b0, "chunk is not contiguous in the buffer"
        at = c.byte_end
    assert at == total * 2 == plan.nbytes
    return len(chunks)


def test_chunks_tile_the_buffer(lk):
    rng = substream(77, "chunks")
    seen = 0
    for _ in range(60):
        w = random_tiny(rng)
        row = w.geom[1] * w.geom[2] * 2
        if row % 16:
            continue
        plan = lk.lumen_kv_plan_build(geom_of(lk, w), w.reqs, lk.LUMEN_KV_HOST_ONLY)
        max_run = max([plan.run(i).count for i in range(plan.num_runs)] + [1]) * row
        for slot in (max_run, 2 * max_run + 16, 7 * row + max_run, 1 << 20):
            slot = (slot + 15) // 16 * 16
            seen += _check_chunks(plan, w.geom, w.reqs, slot)
        if plan.num_runs and max_run > 16:
            with pytest.raises(lk.LumenKVError) as e:       # a run must fit a slot
                plan.chunks(max_run - 16)
            assert e.value.status == lk.LUMEN_KV_ESIZE
    assert seen > 200


def test_chunks_of_the_big_configs(lk):
    """Closed forms: cfg1 step (64 x 2.5 MiB requests) in 32 MiB slots = whole-request groups of
    12; cfg2 request (2 GiB, 16 MiB per plane) = 2 planes per chunk; cfg4 (256 MiB per plane,
    one 2 KiB run per token) = 8 token ranges per plane."""
    slot = 32 << 20
    w = cfg1_qwen14b()
    p = lk.lumen_kv_plan_build(geom_of(lk, w), w.reqs, lk.LUMEN_KV_HOST_ONLY)
    ch = p.chunks(slot)
    assert len(ch) == 6 and all(c.plane_begin == 0 and c.plane_end == 80 for c in ch)
    assert [c.byte_end - c.byte_begin for c in ch] == [12 * 2621440] * 5 + [4 * 2621440]
    w = cfg2_qwen32b(n_reqs=2, N=4096)
    p = lk.lumen_kv_plan_build(geom_of(lk, w), w.reqs, lk.LUMEN_KV_HOST_ONLY)
    ch = p.chunks(slot)
    assert len(ch) == 2 * 64 and all(c.plane_end - c.plane_begin == 2 for c in ch)
    assert all(c.run_end - c.run_begin == 512 for c in ch)
    w = cfg4_longctx(wave_reqs=1)
    p = lk.lumen_kv_plan_build(geom_of(lk, w), w.reqs, lk.LUMEN_KV_HOST_ONLY)
    ch = p.chunks(slot)
    assert len(ch) == 128 * 8 and all(c.run_end - c.run_begin == 16384 for c in ch)
    assert p.chunks(1 << 40)[0].byte_end == 32 << 30 and len(p.chunks(1 << 40)) == 1


# ---- explicit buffer layout (checkpoint store, f3) ------------------------------------------
def _random_layouts(rng, w):
    """Non-overlapping blocks with random gaps and plane strides >= n (bytes, tokens)."""
    L, H, D, S, N = w.geom
    row = H * D * 2
    lays, at = [], int(rng.integers(0, 4)) * row
    for _, tb, te in w.reqs:
        stride = (te - tb) + int(rng.integers(0, 4))
        lays.append((at, stride))
        at += 2 * L * stride * row + int(rng.integers(0, 3)) * row
    return lays, at + row


def test_layout_plan_addresses_equal_oracle(lk):
    """Bytes addressed by (runs x planes) under a layout, and by the chunks of the staged path,
    are exactly the words the layout oracle writes into a sentinel buffer."""
    rng = substream(88, "layout_plan")
    for _ in range(40):
        w = random_tiny(rng)
        L, H, D, S, N = w.geom
        row = H * D * 2
        if row % 16:
            continue
        lays, size = _random_layouts(rng, w)
        plan = lk.lumen_kv_plan_build(geom_of(lk, w), w.reqs, lk.LUMEN_KV_HOST_ONLY, layouts=lays)
        K = [np.ones(N * S * H * D, np.uint16) for _ in range(L)]
        B = np.zeros(size // 2, dtype=np.uint16)
        oracle.pack_layout(w.geom, K, K, w.reqs, [(o // 2, s) for o, s in lays], B)
        want = np.repeat(B.astype(bool), 2)                       # byte mask of addressed bytes
        got = np.zeros(size, dtype=bool)
        runs = [plan.run(i) for i in range(plan.num_runs)]
        for r in runs:
            off, stride = lays[r.req]
            for p in range(2 * L):
                b0 = off + (p * stride + r.dst_token) * row
                assert not got[b0:b0 + r.count * row].any()
                got[b0:b0 + r.count * row] = True
        assert np.array_equal(got, want)
        extent = int(np.flatnonzero(want)[-1]) + 1 if want.any() else 0
        assert plan.nbytes == extent
        for i, (off, _) in enumerate(lays):
            assert plan.req_offset(i) == off
        max_run = max([r.count for r in runs] + [1]) * row
        for slot in (max_run, 3 * max_run + 16, 1 << 20):
            slot = (slot + 15) // 16 * 16
            cov = np.zeros(size, dtype=bool)
            for c in plan.chunks(slot):
                assert 0 < c.byte_end - c.byte_begin <= slot
                seg = np.zeros(size, dtype=bool)
                for p in range(c.plane_begin, c.plane_end):
                    for r in runs[c.run_begin:c.run_end]:
                        off, stride = lays[r.req]
                        b0 = off + (p * stride + r.dst_token) * row
                        seg[b0:b0 + r.count * row] = True
                assert seg[c.byte_begin:c.byte_end].all() and seg.sum() == c.byte_end - c.byte_begin
                assert not (cov & seg).any()
                cov |= seg
            assert np.array_equal(cov, want)


def test_layout_validation(lk):
    g = lk.make_geom(2, 2, 8, 4, 16)                              # row = 32 B
    pt = np.arange(4, dtype=np.int32)
    ok = lk.lumen_kv_plan_build(g, [(pt, 2, 9)], lk.LUMEN_KV_HOST_ONLY, layouts=[(64, 7)])
    assert ok.nbytes == 64 + (3 * 7 + 7) * 32 and ok.req_offset(0) == 64
    for bad in ((48, 7), (-32, 7), (64, 6)):                      # not a row multiple / negative / stride < n
        with pytest.raises(lk.LumenKVError) as e:
            lk.lumen_kv_plan_build(g, [(pt, 2, 9)], lk.LUMEN_KV_HOST_ONLY, layouts=[bad])
        assert e.value.status == lk.LUMEN_KV_EINVAL
    # dense layout given explicitly == no layout
    a = lk.lumen_kv_plan_build(g, [(pt, 2, 9), (pt, 0, 3)], lk.LUMEN_KV_HOST_ONLY,
                               layouts=[(0, 7), (7 * 4 * 32, 3)])
    b = lk.lumen_kv_plan_build(g, [(pt, 2, 9), (pt, 0, 3)], lk.LUMEN_KV_HOST_ONLY)
    spans = lambda p: [(c.byte_begin, c.byte_end) for c in p.chunks(1 << 20)]
    assert a.nbytes == b.nbytes and spans(a) == spans(b)


def test_unique_dst_is_slot_granular(lk):
    """Consecutive deltas of one request meet inside a page: disjoint token slots are legal,
    one shared slot is EOVERLAP (both the bitmap and the sort path)."""
    U = lk.LUMEN_KV_VALIDATE_UNIQUE_DST | lk.LUMEN_KV_HOST_ONLY
    pt = np.array([7, 3, 9], dtype=np.int32)
    for N in (16, 1 << 24):                                   # small pool: bitmap; huge pool: sort
        g = lk.make_geom(1, 1, 8, 4, N)
        lk.lumen_kv_plan_build(g, [(pt, 0, 6), (pt, 6, 7), (pt, 7, 12)], U).close()
        for bad in ([(pt, 0, 6), (pt, 5, 9)], [(pt, 0, 12), (pt, 7, 8)],
                    [(pt, 2, 3), (np.array([7], np.int32), 2, 3)]):
            with pytest.raises(lk.LumenKVError) as e:
                lk.lumen_kv_plan_build(g, bad, U)
            assert e.value.status == lk.LUMEN_KV_EOVERLAP
        # another request using the other half of the same physical page
        lk.lumen_kv_plan_build(g, [(pt, 0, 2), (np.array([7], np.int32), 2, 4)], U).close()


def test_maximum_sizes_are_64_bit_clean(lk):
    """Largest legal geometry: N = 2^31 - 1 pages of 32 KiB (a 64 TiB plane), page indices and
    token positions near the top, 128k-token ranges: offsets never wrap (SURVEY 7.3 hard part 5)."""
    N = (1 << 31) - 1
    g = lk.make_geom(64, 8, 128, 16, N)
    top = np.array([N - 1, 0, N - 2, 12345], dtype=np.int32)
    p = lk.lumen_kv_plan_build(g, [(top, 5, 60)], lk.LUMEN_KV_HOST_ONLY | lk.LUMEN_KV_VALIDATE_UNIQUE_DST)
    runs = [p.run(i) for i in range(p.num_runs)]
    assert [(r.src_slot, r.dst_token, r.count) for r in runs] == [
        ((N - 1) * 16 + 5, 0, 11), (0, 11, 16), ((N - 2) * 16, 27, 16), (12345 * 16, 43, 12)]
    assert p.nbytes == 55 * 128 * 2048
    # a 128k-token request in a token-granular pool of 2^31 - 1 slots, buffer offsets beyond 2^40
    g1 = lk.make_geom(64, 8, 128, 1, N)
    rng = substream(9, "max")
    pt = rng.integers(0, N, size=131072, dtype=np.int64).astype(np.int32)
    pt = np.unique(pt)[:100000].astype(np.int32)
    big = lk.lumen_kv_plan_build(g1, [(pt, 0, pt.size)] * 1 + [(pt[::-1].copy(), 0, 7)],
                                 lk.LUMEN_KV_HOST_ONLY, layouts=[(1 << 41, pt.size), (0, 7)])
    assert big.req_offset(0) == 1 << 41 and big.nbytes == (1 << 41) + (127 * pt.size + pt.size) * 2048
    r = big.run(99999)
    assert r.src_slot == int(pt[99999]) and r.dst_token == 99999 and r.count == 1
    with pytest.raises(lk.LumenKVError):                     # N = 2^31 is one too many
        lk.lumen_kv_plan_build(lk.make_geom(1, 1, 8, 1, 1 << 31), [], lk.LUMEN_KV_HOST_ONLY)


def test_layout_extent_overflow_is_rejected(lk):
    """buf_offset + ((planes-1)*stride + n)*row was evaluated without overflow
    checks, so a layout whose true extent is about 2^70 built and reported 1 GiB.  Every step is
    checked now and such a layout is EINVAL (it can never fit a real buffer)."""
    H = lk.LUMEN_KV_HOST_ONLY
    pt = np.zeros(1, dtype=np.int32)
    # probe 1: L = 1, row = 2^30, stride = 2^40 - 1, n = 2
    g = lk.make_geom(1, 1 << 15, 1 << 14, 2, 4)                 # row = 2^15 * 2^14 * 2 = 2^30
    with pytest.raises(lk.LumenKVError) as e:
        lk.lumen_kv_plan_build(g, [(pt, 0, 2)], H, layouts=[(0, (1 << 40) - 1)])
    assert e.value.status == lk.LUMEN_KV_EINVAL
    # probe 2: row = 16, L = 32767 (65,534 planes), stride = 2^40 - 1: about 2^60 bytes, which
    # 64 bits hold -- it builds, and the extent it reports is the true one (so a real buffer is ESIZE)
    g2 = lk.make_geom(32767, 1, 8, 4, 4)                        # row = 16
    big = lk.lumen_kv_plan_build(g2, [(pt, 0, 2)], H, layouts=[(16, (1 << 40) - 1)])
    assert big.nbytes == 16 + ((2 * 32767 - 1) * ((1 << 40) - 1) + 2) * 16
    # row = 2^20 with the same stride and planes does wrap 63 bits: EINVAL
    g3 = lk.make_geom(32767, 1 << 10, 1 << 9, 2, 4)             # row = 2^20
    with pytest.raises(lk.LumenKVError) as e:
        lk.lumen_kv_plan_build(g3, [(pt, 0, 2)], H, layouts=[(0, (1 << 40) - 1)])
    assert e.value.status == lk.LUMEN_KV_EINVAL


def test_run_reserve_is_exact_for_large_pages(lk):
    """the run list was reserved as if every touched page were used in full:
    S = 2^20, row = 16 KiB, 1-token deltas asked for 8 MiB of descriptors per page (false ENOMEM
    for many requests, std::length_error across the C boundary for extreme ones)."""
    g = lk.make_geom(1, 64, 128, 1 << 20, 4096)                 # row = 16 KiB, page = 16 GiB
    reqs = [(np.array([i], dtype=np.int32), 5, 6) for i in range(4096)]
    p = lk.lumen_kv_plan_build(g, reqs, lk.LUMEN_KV_HOST_ONLY)
    assert p.num_runs == 4096 and p.nbytes == 4096 * 2 * 16384


def test_async_staged_calls_validate_before_queueing(lk):
    """The asynchronous staged entry points reject what can be checked on the host without ever
    touching a device or starting the stager's thread (no GPU here: no stager can exist, so the
    NULL-stager / NULL-ticket paths are what is reachable)."""
    import ctypes
    L = lk.binding._lib()
    g = lk.make_geom(2, 2, 64, 16, 64)
    p = lk.lumen_kv_plan_build(g, [(np.arange(4, dtype=np.int32), 0, 40)], lk.LUMEN_KV_HOST_ONLY)
    t = ctypes.c_uint64(7)
    kv = (ctypes.c_void_p * 2)(16, 16)
    buf = np.zeros(1 << 16, dtype=np.uint8)
    for fn in (L.lumen_kv_checkpoint_pack_staged_async, L.lumen_kv_restore_unpack_staged_async):
        assert fn(p.handle, kv, kv, buf.ctypes.data, buf.size, None, None, None, 0, ctypes.byref(t)) == lk.LUMEN_KV_EINVAL
        assert t.value == 0                                     # no ticket was handed out
        assert fn(p.handle, kv, kv, buf.ctypes.data, buf.size, None, None, None, 0, None) == lk.LUMEN_KV_EINVAL
    assert L.lumen_kv_stager_query(None, 1) == lk.LUMEN_KV_EINVAL
    assert L.lumen_kv_stager_wait(None, 1, None) == lk.LUMEN_KV_EINVAL
    assert L.lumen_kv_stager_sync(None, 1) == lk.LUMEN_KV_EINVAL
    assert lk.lumen_kv_strerror(lk.LUMEN_KV_ESINK).startswith("the checkpointer's sink")
