"""Page tags and the longest-contiguous-prefix lookup (
PAPER.md:147, 157).  Oracle pins first (published FNV-1a vectors, closed forms, brute force),
then the library's host lookup against the oracle on CPU, then the CUDA kernel against the
oracle on the GPU, bit for bit."""
import struct
from pathlib import Path

import numpy as np
import pytest

import oracle
from workloads import substream

ROOT = Path(__file__).resolve().parent.parent


# ---- oracle pins ------------------------------------------------------------------------
def test_fnv1a64_published_vectors():
    n = 0
    for line in (ROOT / "tests" / "golden" / "fnv1a64.txt").read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        text, hexval = line.rsplit(None, 1)
        assert oracle.fnv1a64(text.strip().strip('"').encode()) == int(hexval, 16), line
        n += 1
    assert n == 3


def test_page_hash_is_fnv_of_little_endian_token_bytes():
    rng = substream(1, "tags")
    for S in (1, 3, 16, 64):
        tok = rng.integers(-2**31, 2**31, size=5 * S + S // 2, dtype=np.int64).astype(np.int32)
        tags = oracle.page_tags(tok, S)
        for i, t in enumerate(tags):
            page = tok[i * S:(i + 1) * S]
            assert int(t["hash"]) == oracle.fnv1a64(struct.pack(f"<{page.size}i", *page.tolist()))
    # a byte-order or token-order slip changes the value: "foob" as one little-endian token
    assert int(oracle.page_tags([0x626F6F66], 1)[0]["hash"]) == oracle.fnv1a64(b"foob")
    assert int(oracle.page_tags([0x666F6F62], 1)[0]["hash"]) != oracle.fnv1a64(b"foob")


def test_end_positions_closed_form():
    for length, S in ((0, 16), (1, 16), (16, 16), (17, 16), (100, 16), (5, 1), (8192, 16), (37, 16)):
        tags = oracle.page_tags(np.zeros(length, np.int32), S)
        assert tags.size == -(-length // S)
        assert tags["end_pos"].tolist() == [min((i + 1) * S, length) for i in range(tags.size)]
    # equal content at different positions: equal hash, different tag (the end position differs)
    t = oracle.page_tags(np.zeros(48, np.int32), 16)
    assert len(set(t["hash"].tolist())) == 1 and len(set(t["end_pos"].tolist())) == 3
    # a partly filled last page hashes only the tokens it holds
    tok = np.arange(20, dtype=np.int32)
    assert oracle.page_tags(tok, 16)[1]["hash"] == oracle.page_tags(tok[16:], 16)[0]["hash"]
    # "derives purely from the request's token sequence": a longer history keeps earlier tags
    assert np.array_equal(oracle.page_tags(tok, 16)[:1], oracle.page_tags(np.arange(64, dtype=np.int32), 16)[:1])


def brute_prefix(regen, stored):
    have = {(int(h), int(e)) for h, e in zip(stored["hash"], stored["end_pos"])}
    out = 0
    for h, e in zip(regen["hash"], regen["end_pos"]):
        if (int(h), int(e)) not in have:
            break
        out = int(e)
    return out


def lookup_cases():
    rng = substream(2, "tags_lookup")
    for _ in range(200):
        S = int(rng.choice([1, 4, 16]))
        length = int(rng.integers(0, 12 * S))
        tok = rng.integers(0, 50, size=length).astype(np.int32)      # small vocabulary: repeated pages
        regen = oracle.page_tags(tok, S)
        keep = rng.random(regen.size) < rng.choice([0.3, 0.8, 1.0])
        stored = regen[keep]
        other = oracle.page_tags(rng.integers(0, 50, size=int(rng.integers(0, 5 * S))).astype(np.int32), S)
        stored = np.concatenate([stored, other, stored[:2]])          # foreign tags and duplicates
        rng.shuffle(stored)
        yield regen, stored


def test_longest_prefix_brute_force():
    for regen, stored in lookup_cases():
        assert oracle.longest_prefix(regen, stored) == brute_prefix(regen, stored)
    tok = np.arange(64, dtype=np.int32)
    t = oracle.page_tags(tok, 16)
    assert oracle.longest_prefix(t, t) == 64
    assert oracle.longest_prefix(t, t[[0, 1, 3]]) == 32        # halts at the first missing page
    assert oracle.longest_prefix(t, t[1:]) == 0
    assert oracle.longest_prefix(t, t[:0]) == 0 and oracle.longest_prefix(t[:0], t) == 0
    # an interrupted transfer: the store holds the tag of a SHORTER last page (end 40), the
    # history says the page is full (end 48): not the same tag, the lookup halts before it
    short = oracle.page_tags(tok[:40], 16)
    assert oracle.longest_prefix(t, short) == 32


# ---- library, host side ------------------------------------------------------------------
@pytest.fixture(scope="module")
def lk():
    from paper_2606_17787_b200 import build
    build.build()
    import paper_2606_17787_b200 as lk
    return lk


def test_library_lookup_equals_oracle(lk):
    assert lk.TAG_DTYPE == oracle.TAG_DTYPE
    for regen, stored in lookup_cases():
        assert lk.lumen_kv_longest_prefix(regen, stored) == oracle.longest_prefix(regen, stored)
    assert lk.lumen_kv_tags_num_pages([0, 37, 37, 137, 142], 16) == 3 + 0 + 7 + 1
    with pytest.raises(lk.LumenKVError):
        lk.lumen_kv_tags_num_pages([0, 5, 3], 16)


def test_host_tags_equal_oracle(lk):
    """lumen_kv_page_tags_host: the tags a sender attaches to a delta [tb, te) == the oracle's tags
    of a history of te tokens, restricted to the pages the delta touches."""
    rng = substream(4, "tags_host")
    for _ in range(200):
        S = int(rng.choice([1, 3, 16, 32]))
        te = int(rng.integers(1, 20 * S))
        tb = int(rng.integers(0, te))
        tok = rng.integers(-2**31, 2**31, size=te + 5, dtype=np.int64).astype(np.int32)
        ref = oracle.page_tags(tok[:te], S)
        ref = ref[ref["end_pos"] > tb]
        first = (tb // S) * S - S * int(rng.integers(0, 2)) * (tb // S > 0)      # any earlier page start
        got = lk.lumen_kv_page_tags_host(tok[first:], first, tb, te, S)
        assert np.array_equal(got, ref)
    assert lk.lumen_kv_page_tags_host(np.zeros(4, np.int32), 0, 3, 3, 16).size == 0
    with pytest.raises(lk.LumenKVError):                              # first_token not a page start
        lk.lumen_kv_page_tags_host(np.zeros(40, np.int32), 5, 6, 20, 16)
    with pytest.raises(lk.LumenKVError):                              # tokens start after the delta's page
        lk.lumen_kv_page_tags_host(np.zeros(40, np.int32), 16, 6, 20, 16)


# ---- CUDA kernel vs oracle -------------------------------------------------------------------
@pytest.mark.gpu
def test_gpu_page_tags_equal_oracle(lk):
    import torch
    rng = substream(3, "tags_gpu")
    for case in range(12):
        S = int(rng.choice([1, 3, 16, 16, 32]))
        R = int(rng.choice([0, 1, 7, 64, 600]))                        # 600 > one launch's 480 requests
        lens = rng.integers(0, 40 * S, size=R)
        if R and case % 3 == 0:
            lens[int(rng.integers(0, R))] = 131072 if S >= 16 else 5000  # one long request
        off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        tok = rng.integers(-2**31, 2**31, size=int(off[-1]) + 1, dtype=np.int64).astype(np.int32)
        n = lk.lumen_kv_tags_num_pages(off, S)
        d_tok = torch.from_numpy(tok).cuda()
        d_out = torch.full((n + 2, 2), -1, dtype=torch.int64, device="cuda")     # guard rows
        side = torch.cuda.Stream()
        lk.lumen_kv_page_tags(d_tok.data_ptr(), off, S, d_out[1:].data_ptr(), n, side.cuda_stream)
        side.synchronize()
        got = d_out.cpu().numpy()
        assert (got[0] == -1).all() and (got[-1] == -1).all()
        got = got[1:-1].copy().view(lk.TAG_DTYPE).reshape(-1)
        ref = np.concatenate([oracle.page_tags(tok[off[r]:off[r + 1]], S) for r in range(R)]
                             + [np.zeros(0, oracle.TAG_DTYPE)])
        assert np.array_equal(got, ref), f"case {case}"
    d_tok = torch.zeros(100, dtype=torch.int32, device="cuda")
    d_out = torch.zeros((8, 2), dtype=torch.int64, device="cuda")
    with pytest.raises(lk.LumenKVError) as e:                         # 7 pages, room for 6
        lk.lumen_kv_page_tags(d_tok.data_ptr(), [0, 100], 16, d_out.data_ptr(), 6, 0)
    assert e.value.status == lk.LUMEN_KV_ESIZE
    lk.lumen_kv_page_tags(d_tok.data_ptr(), [0, 0, 0], 16, 0, 0, 0)   # no pages: nothing to do
