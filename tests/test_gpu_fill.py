"""The pool content generator g has two implementations (numpy in workloads/content.py,
CUDA in workloads/csrc/kvfill.cu).  They must agree before any parity test relies on
them.  Also checks the checksum kernel detects any change."""
import numpy as np
import pytest

from workloads import g_words, substream

pytestmark = pytest.mark.gpu


def test_fill_kernel_matches_numpy_on_sampled_pages():
    import torch
    from workloads import device as wdev
    wdev.build()
    page_words = 16 * 8 * 128
    n_pages = 3000
    t = torch.empty(n_pages * page_words, dtype=torch.int16, device="cuda")
    for plane in (0, 7, 127):
        wdev.fill_plane(t, 0x4C554D454E, plane)
        torch.cuda.synchronize()
        rng = substream(plane, "fillchk")
        pages = rng.choice(n_pages, size=1000, replace=False)
        host = t.cpu().numpy().view(np.uint16)
        for p in pages:
            ref = g_words(0x4C554D454E, plane, int(p) * page_words, page_words)
            assert np.array_equal(host[p * page_words:(p + 1) * page_words], ref)
    # distribution sanity: bf16 NaN encodings are present on purpose
    h = t.cpu().numpy().view(np.uint16)
    assert ((h & 0x7F80) == 0x7F80).any()


def test_page_checksum_detects_single_word_change_and_swap():
    import torch
    from workloads import device as wdev
    wdev.build()
    page_bytes, n_pages = 4096, 64
    t = torch.empty(n_pages * page_bytes // 2, dtype=torch.int16, device="cuda")
    wdev.fill_plane(t, 1, 2)
    a = wdev.page_checksums(t, n_pages, page_bytes).clone()
    t[5 * 2048 + 17] += 1
    b = wdev.page_checksums(t, n_pages, page_bytes).clone()
    diff = (a != b).nonzero().flatten().tolist()
    assert diff == [5]
    t[5 * 2048 + 17] -= 1
    x, y = t[9 * 2048 + 3].clone(), t[9 * 2048 + 900].clone()
    t[9 * 2048 + 3], t[9 * 2048 + 900] = y, x
    c = wdev.page_checksums(t, n_pages, page_bytes)
    assert (a != c).nonzero().flatten().tolist() == ([9] if x != y else [])
