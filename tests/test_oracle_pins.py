"""Pins for the oracle (CPU only).  SURVEY.md section 8(c) C7, P1-P10.

The paper prints no worked example for the pack/unpack path (PAPER.md:145,
157-163 give only the definition), so the oracle is pinned to what the
definition and the mathematics fix: special cases that reduce to a library
slice, an independently structured brute force, an address-coded fill that is
decoded with no oracle at all, closed-form sizes, and invariants.  Each pin is
chosen so that a plausible slip (K/V swapped, layer/token order swapped, wrong
offset prefix sum, t div S vs t mod S, transposed layout) fails it.
"""
import numpy as np
import pytest

import oracle
from oracle import oracle_np
from workloads import cfg0_tiny, random_tiny, substream, fill_plane_np, MASTER_SEED


def make_pool(geom, seed, *, salt=0):
    L, H, D, S, N = geom
    words = N * S * H * D
    K = [fill_plane_np(seed + salt, 2 * l, words) for l in range(L)]
    V = [fill_plane_np(seed + salt, 2 * l + 1, words) for l in range(L)]
    return K, V


def clone(planes):
    return [p.copy() for p in planes]


# ---- P1: identity page table => contiguous slice --------------------------------
@pytest.mark.parametrize("tb,te", [(0, 64), (5, 37), (16, 48), (63, 64), (7, 7)])
def test_p1_identity_page_table_is_contiguous_slice(tb, te):
    geom = (3, 2, 8, 4, 16)
    L, H, D, S, N = geom
    E = H * D
    K, V = make_pool(geom, 11)
    pt = np.arange(N, dtype=np.int32)
    B = oracle.pack(geom, K, V, [(pt, tb, te)])
    n = te - tb
    assert B.size == n * 2 * L * E
    B = B.reshape(L, 2, n, E)
    for l in range(L):
        assert np.array_equal(B[l, 0], K[l].reshape(N * S, E)[tb:te])
        assert np.array_equal(B[l, 1], V[l].reshape(N * S, E)[tb:te])


# ---- P2: library-routine restatement == loop oracle -------------------------------
def test_p2_numpy_gather_equals_loop_oracle_cfg0():
    w = cfg0_tiny()
    K, V = make_pool(w.geom, MASTER_SEED)
    a = oracle.pack(w.geom, K, V, w.reqs)
    b = oracle_np.pack(w.geom, K, V, w.reqs)
    assert np.array_equal(a, b)
    K2, V2 = make_pool(w.geom, MASTER_SEED, salt=1)
    K3, V3 = clone(K2), clone(V2)
    oracle.unpack(w.geom, K2, V2, w.restore_reqs, a, check_overlap=True)
    oracle_np.unpack(w.geom, K3, V3, w.restore_reqs, a)
    for x, y in zip(K2 + V2, K3 + V3):
        assert np.array_equal(x, y)


def test_p2_random_tiny_geometries():
    rng = substream(123, "p2")
    for _ in range(120):
        w = random_tiny(rng, allow_shared=True)
        K, V = make_pool(w.geom, 5)
        a = oracle.pack(w.geom, K, V, w.reqs)
        b = oracle_np.pack(w.geom, K, V, w.reqs)
        assert np.array_equal(a, b)
        assert a.size == oracle.total_elems(w.geom, w.reqs)
        K2, V2 = make_pool(w.geom, 6)
        K3, V3 = clone(K2), clone(V2)
        oracle.unpack(w.geom, K2, V2, w.restore_reqs, a, check_overlap=True)
        oracle_np.unpack(w.geom, K3, V3, w.restore_reqs, a)
        for x, y in zip(K2 + V2, K3 + V3):
            assert np.array_equal(x, y)


# ---- P3: round trip under any permutation; everything else untouched ------------
def test_p3_round_trip_and_untouched():
    rng = substream(7, "p3")
    for i in range(40):
        w = cfg0_tiny(seed=100 + i) if i < 5 else random_tiny(rng)
        L, H, D, S, N = w.geom
        E = H * D
        K, V = make_pool(w.geom, 1)
        B = oracle.pack(w.geom, K, V, w.reqs)
        K2, V2 = make_pool(w.geom, 2)
        K2_before, V2_before = clone(K2), clone(V2)
        oracle.unpack(w.geom, K2, V2, w.restore_reqs, B, check_overlap=True)
        B2 = oracle.pack(w.geom, K2, V2, w.restore_reqs)
        assert np.array_equal(B, B2)
        # target slots, built here from the *restore* page tables by hand
        target = np.zeros(N * S, dtype=bool)
        for pt, tb, te in w.restore_reqs:
            for t in range(tb, te):
                target[int(pt[t // S]) * S + t % S] = True
        for before, after in zip(K2_before + V2_before, K2 + V2):
            b = before.reshape(N * S, E)
            a = after.reshape(N * S, E)
            assert np.array_equal(b[~target], a[~target])


# ---- P4: delta concatenation ------------------------------------------------------
def test_p4_delta_concatenation():
    rng = substream(9, "p4")
    for i in range(30):
        w = cfg0_tiny(seed=i, full_prefix=True)
        L, H, D, S, N = w.geom
        E = H * D
        K, V = make_pool(w.geom, 3)
        full = oracle.pack(w.geom, K, V, w.reqs)
        # split each request's [0, len) into 1..5 deltas at random cut points
        n_deltas = int(rng.integers(1, 6))
        cuts = []
        for _, tb, te in w.reqs:
            c = np.sort(rng.integers(tb, te + 1, size=n_deltas - 1)).tolist()
            cuts.append([tb] + c + [te])
        deltas = []
        for d in range(n_deltas):
            reqs_d = [(pt, cuts[r][d], cuts[r][d + 1]) for r, (pt, _, _) in enumerate(w.reqs)]
            deltas.append((reqs_d, oracle.pack(w.geom, K, V, reqs_d)))
        # form 1: concat along the token axis per (req, layer, K|V)
        lay_full, _ = oracle_np.layout(w.geom, w.reqs)
        for r, (off, n) in enumerate(lay_full):
            blk = full[off: off + n * 2 * L * E].reshape(2 * L, n, E)
            pieces = []
            for reqs_d, Bd in deltas:
                lay_d, _ = oracle_np.layout(w.geom, reqs_d)
                o, m = lay_d[r]
                pieces.append(Bd[o: o + m * 2 * L * E].reshape(2 * L, m, E))
            assert np.array_equal(blk, np.concatenate(pieces, axis=1))
        # form 2: unpack(delta_1); unpack(delta_2); ... == unpack(full)
        Ka, Va = make_pool(w.geom, 4)
        Kb, Vb = clone(Ka), clone(Va)
        oracle.unpack(w.geom, Ka, Va, w.restore_reqs, full)
        for reqs_d, Bd in deltas:
            rr = [(w.restore_reqs[r][0], tb, te) for r, (_, tb, te) in enumerate(reqs_d)]
            oracle.unpack(w.geom, Kb, Vb, rr, Bd)
        for x, y in zip(Ka + Va, Kb + Vb):
            assert np.array_equal(x, y)


# ---- P5: brute force, inverse direction (walk the pool, find the owner) -----------
def test_p5_brute_force_inverse_walk():
    rng = substream(21, "p5")
    for i in range(25):
        w = cfg0_tiny(seed=i) if i < 3 else random_tiny(rng)
        L, H, D, S, N = w.geom
        E = H * D
        K, V = make_pool(w.geom, 8)
        B = oracle.pack(w.geom, K, V, w.reqs)
        expect = {}
        n_of = [te - tb for _, tb, te in w.reqs]
        # for every pool slot, find which (request, token) own it
        for page in range(N):
            for slot in range(S):
                for r, (pt, tb, te) in enumerate(w.reqs):
                    for lp in range(pt.size):
                        if int(pt[lp]) != page:
                            continue
                        t = lp * S + slot
                        if not (tb <= t < te):
                            continue
                        for l in range(L):
                            for c, planes in ((0, K), (1, V)):
                                row = planes[l].reshape(N, S, E)[page, slot]
                                expect[(r, l, c, t - tb)] = row
        assert len(expect) == sum(n_of) * 2 * L
        # walk the buffer in its declared order [req][layer][K|V][token][E]
        at = 0
        for r in range(len(w.reqs)):
            for l in range(L):
                for c in range(2):
                    for j in range(n_of[r]):
                        assert np.array_equal(B[at: at + E], expect[(r, l, c, j)])
                        at += E
        assert at == B.size


# ---- P6: address-coded fill, decoded with no oracle ------------------------------
def test_p6_address_coded_fill():
    w = cfg0_tiny()
    L, H, D, S, N = w.geom
    E = H * D                                            # 128
    # word = (plane id 0..3) << 14 | (page*S + slot)(10 bits) << 4 | (e mod 16)
    def coded(plane):
        slot = np.arange(N * S, dtype=np.uint32)[:, None]
        e = np.arange(E, dtype=np.uint32)[None, :]
        return ((plane << 14) | (slot << 4) | (e % 16)).astype(np.uint16).reshape(-1)
    K = [coded(2 * l) for l in range(L)]
    V = [coded(2 * l + 1) for l in range(L)]
    B = oracle.pack(w.geom, K, V, w.reqs)
    at = 0
    for pt, tb, te in w.reqs:
        n = te - tb
        for l in range(L):
            for c in range(2):
                for j in range(n):
                    t = tb + j
                    row = B[at: at + E].astype(np.uint32)
                    assert np.all(row >> 14 == 2 * l + c)
                    assert np.all((row >> 4) & 1023 == int(pt[t // S]) * S + t % S)
                    assert np.array_equal(row & 15, np.arange(E) % 16)
                    at += E
    assert at == B.size


# ---- P7: closed-form sizes ---------------------------------------------------------
def test_p7_closed_form_sizes():
    golden = {}
    for line in open(__file__.replace("test_oracle_pins.py", "golden/sizes.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            golden[k.strip()] = int(v)
    w = cfg0_tiny(full_prefix=True)
    assert 2 * oracle.total_elems(w.geom, w.reqs) == golden["cfg0_full_prefix_bytes"]
    assert sum(pt.size for pt, _, _ in w.reqs) == golden["cfg0_pages_used"]
    # sizes of the big configs from geometry only (no page table needed: PT unused by sizes)
    dummy = np.zeros(1, dtype=np.int32)
    g1 = (40, 8, 128, 16, 60000)
    assert 2 * oracle.total_elems(g1, [(dummy, 100, 116)] * 64) == golden["cfg1_iter_bytes"]
    g2 = (64, 8, 128, 16, 20000)
    assert 2 * oracle.total_elems(g2, [(dummy, 0, 8192)] * 16) == golden["cfg2_bytes"]
    assert 2 * oracle.total_elems((64, 8, 128, 1, 1 << 20), [(dummy, 0, 131072)] * 8) == golden["cfg4_bytes"]
    # per-request offsets are the exclusive prefix sum
    reqs = [(dummy, 3, 10), (dummy, 0, 0), (dummy, 5, 6)]
    g = (2, 2, 8, 16, 4)
    assert [oracle.req_offset_elems(g, reqs, r) for r in range(3)] == [0, 7 * 4 * 16, 7 * 4 * 16]


# ---- P8: conservation --------------------------------------------------------------
def test_p8_conservation_each_source_row_once():
    rng = substream(33, "p8")
    for _ in range(30):
        w = random_tiny(rng)
        L, H, D, S, N = w.geom
        E = H * D
        # every (plane,row) distinct in its first two words
        K, V = [], []
        for l in range(L):
            for c, dst in ((0, K), (1, V)):
                a = np.zeros((N * S, E), dtype=np.uint16)
                a[:, 0] = np.arange(N * S) & 0xFFFF
                a[:, 1] = ((np.arange(N * S) >> 16) << 8) | (2 * l + c)
                dst.append(a.reshape(-1))
        B = oracle.pack(w.geom, K, V, w.reqs).reshape(-1, E)
        keys = (B[:, 1].astype(np.int64) << 16) | B[:, 0]
        assert np.unique(keys).size == keys.size == w.tokens * 2 * L


# ---- P10: plan direction symmetry --------------------------------------------------
def test_p10_unpack_of_pack_into_same_pool_is_noop():
    rng = substream(44, "p10")
    for _ in range(30):
        w = random_tiny(rng)
        K, V = make_pool(w.geom, 9)
        K0, V0 = clone(K), clone(V)
        B = oracle.pack(w.geom, K, V, w.reqs)
        oracle.unpack(w.geom, K, V, w.reqs, B)
        for x, y in zip(K + V, K0 + V0):
            assert np.array_equal(x, y)


# ---- edge cases & errors -----------------------------------------------------------
def test_empty_and_zero_length():
    geom = (2, 2, 8, 4, 8)
    K, V = make_pool(geom, 1)
    assert oracle.pack(geom, K, V, []).size == 0
    pt = np.array([3, 1], dtype=np.int32)
    assert oracle.pack(geom, K, V, [(pt, 5, 5)]).size == 0
    B = oracle.pack(geom, K, V, [(pt, 5, 5), (pt, 0, 8)])
    assert np.array_equal(B, oracle.pack(geom, K, V, [(pt, 0, 8)]))


def test_errors():
    geom = (1, 1, 8, 4, 4)
    K, V = make_pool(geom, 1)
    with pytest.raises(oracle.OracleError) as e:
        oracle.pack(geom, K, V, [(np.array([4], dtype=np.int32), 0, 1)])
    assert e.value.code == oracle.EPAGE
    with pytest.raises(oracle.OracleError) as e:
        oracle.pack(geom, K, V, [(np.array([0], dtype=np.int32), 0, 5)])
    assert e.value.code == oracle.EPAGE
    with pytest.raises(oracle.OracleError) as e:
        oracle.pack(geom, K, V, [(np.array([0], dtype=np.int32), 3, 2)])
    assert e.value.code == oracle.EARG
    B = np.zeros(2 * 8 * 2, dtype=np.uint16)
    with pytest.raises(oracle.OracleError) as e:
        oracle.unpack(geom, K, V, [(np.array([1], dtype=np.int32), 0, 2),
                                   (np.array([1], dtype=np.int32), 1, 2)], np.zeros(3 * 16, np.uint16),
                      check_overlap=True)
    assert e.value.code == oracle.EOVERLAP
    # entries beyond ceil(te/S) are ignored (A6)
    ok = oracle.pack(geom, K, V, [(np.array([2, 99], dtype=np.int32), 0, 4)])
    assert ok.size == 4 * 2 * 8


# ---- one-by-one accessors agree with the dense definition --------------------------
def test_indexed_accessors_match_dense():
    rng = substream(55, "acc")
    for _ in range(20):
        w = random_tiny(rng)
        L, H, D, S, N = w.geom
        E = H * D
        if w.tokens == 0:
            continue
        K, V = make_pool(w.geom, 10)
        B = oracle.pack(w.geom, K, V, w.reqs)
        for _ in range(50):
            r = int(rng.integers(0, len(w.reqs)))
            n = w.reqs[r][2] - w.reqs[r][1]
            if n == 0:
                continue
            l, c = int(rng.integers(0, L)), int(rng.integers(0, 2))
            j, e = int(rng.integers(0, n)), int(rng.integers(0, E))
            bi = oracle.buffer_index(w.geom, w.reqs, r, l, c, j, e)
            pi = oracle.pool_index(w.geom, w.reqs, r, j, e)
            assert B[bi] == (K if c == 0 else V)[l][pi]


# ---- the OpenMP timing variants equal the plain oracle ------------------------------
def test_omp_variants_equal_plain():
    rng = substream(66, "omp")
    for i in range(10):
        w = cfg0_tiny(seed=i) if i < 2 else random_tiny(rng)
        K, V = make_pool(w.geom, 12)
        a = oracle.pack(w.geom, K, V, w.reqs)
        b = oracle.pack(w.geom, K, V, w.reqs, omp=True)
        assert np.array_equal(a, b)
        K2, V2 = make_pool(w.geom, 13)
        K3, V3 = clone(K2), clone(V2)
        oracle.unpack(w.geom, K2, V2, w.restore_reqs, a)
        oracle.unpack(w.geom, K3, V3, w.restore_reqs, a, omp=True)
        for x, y in zip(K2 + V2, K3 + V3):
            assert np.array_equal(x, y)


# ---- explicit buffer layout (checkpoint store, f3) ------------------------------------------
def _dense_layouts(geom, reqs):
    L, H, D, S, N = geom
    E, off, out = H * D, 0, []
    for _, tb, te in reqs:
        out.append((off, te - tb))
        off += (te - tb) * 2 * L * E
    return out, off


def test_layout_dense_special_case_equals_c1():
    rng = substream(31, "layout")
    for _ in range(40):
        w = random_tiny(rng)
        K, V = make_pool(w.geom, 5)
        lays, total = _dense_layouts(w.geom, w.reqs)
        B = np.full(total, 0xDEAD, dtype=np.uint16)
        oracle.pack_layout(w.geom, K, V, w.reqs, lays, B)
        assert np.array_equal(B, oracle.pack(w.geom, K, V, w.reqs))
        K2, V2 = make_pool(w.geom, 6)
        K3, V3 = [k.copy() for k in K2], [v.copy() for v in V2]
        oracle.unpack_layout(w.geom, K2, V2, w.restore_reqs, lays, B)
        oracle.unpack(w.geom, K3, V3, w.restore_reqs, B)
        assert all(np.array_equal(a, b) for a, b in zip(K2 + V2, K3 + V3))


def test_layout_strided_blocks_and_untouched_gaps():
    rng = substream(32, "layout2")
    for _ in range(40):
        w = random_tiny(rng)
        L, H, D, S, N = w.geom
        E = H * D
        K, V = make_pool(w.geom, 7)
        dense = oracle.pack(w.geom, K, V, w.reqs)
        lays, at, written = [], int(rng.integers(0, 9)), 0
        for _, tb, te in w.reqs:
            stride = (te - tb) + int(rng.integers(0, 5))
            lays.append((at, stride))
            at += 2 * L * stride * E + int(rng.integers(0, 7))
            written += (te - tb) * 2 * L * E
        B = np.full(at + 3, 0xDEAD, dtype=np.uint16)
        oracle.pack_layout(w.geom, K, V, w.reqs, lays, B)
        mask = np.zeros(B.size, dtype=bool)
        d_off = 0
        for (off, stride), (_, tb, te) in zip(lays, w.reqs):
            n = te - tb
            for p in range(2 * L):
                blk = slice(off + p * stride * E, off + p * stride * E + n * E)
                assert np.array_equal(B[blk], dense[d_off + p * n * E: d_off + (p + 1) * n * E])
                mask[blk] = True
            d_off += n * 2 * L * E
        assert mask.sum() == written and (B[~mask] == 0xDEAD).all()
        # round trip through the strided buffer == round trip through the dense one
        K2, V2 = make_pool(w.geom, 8)
        K3, V3 = [k.copy() for k in K2], [v.copy() for v in V2]
        oracle.unpack_layout(w.geom, K2, V2, w.restore_reqs, lays, B)
        oracle.unpack(w.geom, K3, V3, w.restore_reqs, dense)
        assert all(np.array_equal(a, b) for a, b in zip(K2 + V2, K3 + V3))


def test_layout_delta_append_in_place_and_prefix_cut():
    """P4 end to end: deltas packed one after another into ONE region (stride = final length)
    give the dense pack of the whole prefix; and a prefix that ends inside a stored delta is
    restored from that delta's own buffer through its plane stride."""
    w = cfg0_tiny(full_prefix=True)
    L, H, D, S, N = w.geom
    E = H * D
    K, V = make_pool(w.geom, 9)
    pt, _, n = w.reqs[1]                                     # 100 tokens
    full = oracle.pack(w.geom, K, V, [(pt, 0, n)])
    region = np.full(full.size, 0xDEAD, dtype=np.uint16)
    for tb, te in ((0, 37), (37, 53), (53, 100)):
        oracle.pack_layout(w.geom, K, V, [(pt, tb, te)], [(tb * E, n)], region)
    assert np.array_equal(region, full)
    # store keeps the delta [37, 53) as it arrived (dense, stride 16); recovery wants [37, 48)
    seg = oracle.pack(w.geom, K, V, [(pt, 37, 53)])
    pt2 = w.restore_reqs[1][0]
    K2, V2 = make_pool(w.geom, 10)
    K3, V3 = [k.copy() for k in K2], [v.copy() for v in V2]
    oracle.unpack_layout(w.geom, K2, V2, [(pt2, 37, 48)], [(0, 16)], seg)
    oracle.unpack(w.geom, K3, V3, [(pt2, 37, 48)], oracle.pack(w.geom, K, V, [(pt, 37, 48)]))
    assert all(np.array_equal(a, b) for a, b in zip(K2 + V2, K3 + V3))
    with pytest.raises(oracle.OracleError):                  # stride shorter than the range
        oracle.unpack_layout(w.geom, K2, V2, [(pt2, 37, 53)], [(0, 15)], seg)


def test_layout_numpy_restatement_equals_c_loops():
    """P2 for the explicit layout: strided-view NumPy restatement == the C loop nest."""
    rng = substream(33, "layout3")
    n = 0
    while n < 60:
        w = random_tiny(rng)
        if not w.tokens:
            continue
        L, H, D, S, N = w.geom
        E = H * D
        K, V = make_pool(w.geom, 11)
        lays, at = [], int(rng.integers(0, 9))
        for _, tb, te in w.reqs:
            stride = (te - tb) + int(rng.integers(0, 5))
            lays.append((at, stride))
            at += 2 * L * stride * E + int(rng.integers(0, 7))
        B1 = np.full(at + 3, 0xDEAD, dtype=np.uint16)
        B2 = B1.copy()
        oracle.pack_layout(w.geom, K, V, w.reqs, lays, B1)
        oracle_np.pack_layout(w.geom, K, V, w.reqs, lays, B2)
        assert np.array_equal(B1, B2)
        Ka, Va = make_pool(w.geom, 12)
        Kb, Vb = clone(Ka), clone(Va)
        oracle.unpack_layout(w.geom, Ka, Va, w.restore_reqs, lays, B1)
        oracle_np.unpack_layout(w.geom, Kb, Vb, w.restore_reqs, lays, B1)
        assert all(np.array_equal(a, b) for a, b in zip(Ka + Va, Kb + Vb))
        n += 1
