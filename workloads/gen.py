"""Seeded structure generators for the five BASELINE.json configs.

Everything here is plain index bookkeeping drawn from numpy PCG64 streams:
request lengths, page tables (chunks of a seeded permutation of the pool's
pages), delta ranges [t_prev, t_cur), fresh page tables for restore, free
lists.  No pack/unpack arithmetic.  Each generator accepts overrides so the
CPU test-suite can run the same recipe at a size the oracle finishes in
seconds; defaults are the BASELINE.json sizes (readings A14-A16 of SURVEY.md
section 8(c) C6: k = 1024, "60k pages" = 60,000, lognormal sigma = 1.0,
te = len, tb = len - 16).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

MASTER_SEED = 0x4C554D454E  # "LUMEN"

Req = Tuple[np.ndarray, int, int]  # (page table int32, t_begin, t_end)


def substream(seed: int, purpose: str) -> np.random.Generator:
    """Independent PCG64 stream per purpose (pool fill, lengths, perms, ...)."""
    tag = int.from_bytes(purpose.encode()[:8].ljust(8, b"\0"), "little")
    return np.random.Generator(np.random.PCG64([int(seed), tag]))


@dataclass
class Workload:
    name: str
    geom: Tuple[int, int, int, int, int]          # (L, H, D, S, N)
    reqs: List[Req]                               # pack side
    restore_reqs: List[Req]                       # same ranges, fresh pages
    meta: dict = field(default_factory=dict)

    @property
    def row_bytes(self) -> int:
        return self.geom[1] * self.geom[2] * 2

    @property
    def tokens(self) -> int:
        return sum(te - tb for _, tb, te in self.reqs)

    @property
    def payload_bytes(self) -> int:
        return self.tokens * 2 * self.geom[0] * self.row_bytes

    def advanced(self, tokens: int) -> "Workload":
        """Next iteration: every request grew by `tokens`; delta = the new tail."""
        def adv(rs):
            out = []
            for pt, tb, te in rs:
                S = self.geom[3]
                if (te + tokens + S - 1) // S > pt.size:
                    raise ValueError("page table too short to advance")
                out.append((pt, te, te + tokens))
            return out
        return Workload(self.name, self.geom, adv(self.reqs),
                        adv(self.restore_reqs), dict(self.meta))


def _pages(n_tokens: int, S: int) -> int:
    return (n_tokens + S - 1) // S


def _chunks(perm: np.ndarray, counts) -> List[np.ndarray]:
    out, at = [], 0
    for c in counts:
        out.append(np.ascontiguousarray(perm[at: at + c], dtype=np.int32))
        at += c
    if at > perm.size:
        raise ValueError("pool too small for the requested page tables")
    return out


# --------------------------------------------------------------------------
# cfg 0 -- tiny pool (BASELINE.json configs[0])
# --------------------------------------------------------------------------
def cfg0_tiny(seed: int = MASTER_SEED, *, full_prefix: bool = False) -> Workload:
    L, H, D, S, N = 2, 2, 64, 16, 64
    lens = [37, 100, 5, 64]
    counts = [_pages(n, S) for n in lens]             # 3 + 7 + 1 + 4 = 15
    perm_a = substream(seed, "perm_a").permutation(N)
    perm_b = substream(seed, "perm_b").permutation(N)
    rng = substream(seed, "t_prev")
    tprev = [0 if full_prefix else int(rng.integers(0, n)) for n in lens]
    pts_a, pts_b = _chunks(perm_a, counts), _chunks(perm_b, counts)
    reqs = [(pt, tp, n) for pt, tp, n in zip(pts_a, tprev, lens)]
    rreqs = [(pt, tp, n) for pt, tp, n in zip(pts_b, tprev, lens)]
    return Workload("cfg0_tiny", (L, H, D, S, N), reqs, rreqs,
                    {"lens": lens, "t_prev": tprev})


# --------------------------------------------------------------------------
# cfg 1 -- Qwen3-14B-shaped, 64 running requests, 16-token deltas
# --------------------------------------------------------------------------
def cfg1_qwen14b(seed: int = MASTER_SEED, *, L=40, H=8, D=128, S=16, N=60000,
                 n_reqs=64, delta=16, grow_iters=64, median=2048, sigma=1.0,
                 lo=128, hi=16384, aligned=False) -> Workload:
    rng = substream(seed, "lens")
    z = rng.standard_normal(n_reqs)
    lens = np.clip(np.rint(np.exp(np.log(median) + sigma * z)), lo, hi).astype(np.int64)
    if aligned:
        lens = np.maximum((lens // S) * S, max(S, delta))
    lens = np.maximum(lens, delta)
    counts = [_pages(int(n) + delta * grow_iters, S) for n in lens]
    perm = substream(seed, "perm_a").permutation(N)
    need = sum(counts)
    if 2 * need > N:
        raise ValueError(f"pool of {N} pages too small: need {2 * need}")
    pts_a = _chunks(perm[:need], counts)
    pts_b = _chunks(perm[need:], counts)              # fresh pages for restore
    reqs = [(pt, int(n) - delta, int(n)) for pt, n in zip(pts_a, lens)]
    rreqs = [(pt, int(n) - delta, int(n)) for pt, n in zip(pts_b, lens)]
    return Workload("cfg1_qwen3_14b", (L, H, D, S, N), reqs, rreqs,
                    {"lens": lens.tolist(), "delta": delta, "aligned": aligned,
                     "grow_iters": grow_iters, "sigma": sigma})


# --------------------------------------------------------------------------
# cfg 2 -- Qwen3-32B-shaped prefill-completion checkpoint + reverse restore
# --------------------------------------------------------------------------
def cfg2_qwen32b(seed: int = MASTER_SEED, *, L=64, H=8, D=128, S=16, N=20000,
                 n_reqs=16, prompt=8192) -> Workload:
    counts = [_pages(prompt, S)] * n_reqs
    perm = substream(seed, "perm_a").permutation(N)
    need = sum(counts)
    if 2 * need > N:
        raise ValueError(f"pool of {N} pages too small: need {2 * need}")
    pts_a = _chunks(perm[:need], counts)
    free = perm[need:].copy()
    substream(seed, "free").shuffle(free)             # seeded shuffled free list
    pts_b = _chunks(free, counts)
    reqs = [(pt, 0, prompt) for pt in pts_a]
    rreqs = [(pt, 0, prompt) for pt in pts_b]
    return Workload("cfg2_qwen3_32b", (L, H, D, S, N), reqs, rreqs,
                    {"prompt": prompt})


# --------------------------------------------------------------------------
# cfg 3 -- recovery burst: restore waves from host + concurrent 1-token packs
# --------------------------------------------------------------------------
@dataclass
class Burst:
    geom: Tuple[int, int, int, int, int]
    running: List[Req]                 # 1-token delta packs (stream 2)
    waves: List[List[Req]]             # restore requests per wave (stream 1)
    prefix_tokens: List[int]
    meta: dict


def cfg3_burst(seed: int = MASTER_SEED, *, L=64, H=8, D=128, S=16, N=30720,
               occupied_frac=0.4, n_running=64, n_interrupted=48,
               p_lo=1024, p_hi=32768, grow_iters=64) -> Burst:
    perm = substream(seed, "perm_a").permutation(N)
    n_occ = int(N * occupied_frac)
    per = n_occ // n_running                          # pages per running request
    pts_run = _chunks(perm[: per * n_running], [per] * n_running)
    # running request length: leaves `grow_iters` tokens of head-room in its pages
    run_len = per * S - grow_iters
    if run_len < 1:
        raise ValueError("pool too small for the running requests")
    running = [(pt, run_len - 1, run_len) for pt in pts_run]
    free0 = perm[n_occ:].copy()
    P = substream(seed, "prefix").integers(p_lo, p_hi + 1, size=n_interrupted)
    waves, cur, wave_no = [], [], 0
    free = free0.copy()
    substream(seed + wave_no, "free").shuffle(free)
    at = 0
    for p in P.tolist():
        need = _pages(p, S)
        if need > free0.size:
            raise ValueError("one restore does not fit the free list")
        if at + need > free.size:                     # wave full: release + reshuffle
            waves.append(cur)
            cur, wave_no, at = [], wave_no + 1, 0
            free = free0.copy()
            substream(seed + wave_no, "free").shuffle(free)
        cur.append((np.ascontiguousarray(free[at: at + need], dtype=np.int32), 0, int(p)))
        at += need
    if cur:
        waves.append(cur)
    return Burst((L, H, D, S, N), running, waves, P.tolist(),
                 {"occupied_pages": n_occ, "free_pages": int(free0.size),
                  "n_waves": len(waves)})


# --------------------------------------------------------------------------
# cfg 4 -- long context, token-granular pool (S = 1), fully shuffled slots
# --------------------------------------------------------------------------
def cfg4_longctx(seed: int = MASTER_SEED, *, L=64, H=8, D=128, tokens=131072,
                 wave_reqs=2, wave=0) -> Workload:
    S, N = 1, wave_reqs * tokens
    perm_a = substream(seed + wave, "perm_a").permutation(N)
    perm_b = substream(seed + wave, "perm_b").permutation(N)
    counts = [tokens] * wave_reqs
    reqs = [(pt, 0, tokens) for pt in _chunks(perm_a, counts)]
    rreqs = [(pt, 0, tokens) for pt in _chunks(perm_b, counts)]
    return Workload("cfg4_longctx_s1", (L, H, D, S, N), reqs, rreqs,
                    {"tokens": tokens, "wave_reqs": wave_reqs, "wave": wave})


# --------------------------------------------------------------------------
# random tiny geometries for property tests
# --------------------------------------------------------------------------
def random_tiny(rng: np.random.Generator, *, allow_shared=False) -> Workload:
    L = int(rng.integers(1, 4))
    H = int(rng.integers(1, 4))
    D = int(rng.choice([8, 16, 24, 64]))
    S = int(rng.choice([1, 2, 3, 16, 32]))
    R = int(rng.integers(0, 5))
    lens = [int(rng.integers(0, 3 * S + 8)) for _ in range(R)]
    counts = [_pages(n, S) + int(rng.integers(0, 2)) for n in lens]
    N = 2 * sum(counts) + int(rng.integers(1, 6))
    perm_a, perm_b = rng.permutation(N), rng.permutation(N)
    pts_a, pts_b = _chunks(perm_a, counts), _chunks(perm_b, counts)
    if allow_shared and R >= 2 and counts[0] and counts[1]:
        pts_a[1][0] = pts_a[0][0]                     # prefix sharing (pack only)
    reqs, rreqs = [], []
    for pa, pb, n in zip(pts_a, pts_b, lens):
        tb = int(rng.integers(0, n + 1))
        te = int(rng.integers(tb, n + 1))
        reqs.append((pa, tb, te))
        rreqs.append((pb, tb, te))
    return Workload("random_tiny", (L, H, D, S, N), reqs, rreqs, {"lens": lens})


def random_mid(rng: np.random.Generator) -> Workload:
    """Random geometry for differential fuzzing: up to 4 layers, rows of 16 B .. 2 KiB, page sizes
    1 .. 64, up to 200 requests with ragged ranges (some empty), page tables scattered or -- in a
    third of the cases -- physically consecutive (what MERGE_ADJACENT merges)."""
    L = int(rng.integers(1, 5))
    H = int(rng.integers(1, 9))
    D = int(rng.choice([8, 16, 24, 32, 64, 128]))
    while (H * D * 2) % 16:
        D = int(rng.choice([8, 16, 24, 32, 64, 128]))
    S = int(rng.choice([1, 2, 3, 7, 16, 32, 64]))
    R = int(rng.integers(1, 200))
    lens = [int(rng.integers(0, 6 * S + 40)) for _ in range(R)]
    counts = [_pages(n, S) + int(rng.integers(0, 2)) for n in lens]
    N = 2 * sum(counts) + int(rng.integers(1, 50))
    perm_a, perm_b = rng.permutation(N), rng.permutation(N)
    if rng.random() < 0.3:
        perm_a, perm_b = np.arange(N), np.arange(N)[::-1].copy()
    pts_a, pts_b = _chunks(perm_a, counts), _chunks(perm_b, counts)
    reqs, rreqs = [], []
    for pa, pb, n in zip(pts_a, pts_b, lens):
        tb = int(rng.integers(0, n + 1))
        te = int(rng.integers(tb, n + 1))
        reqs.append((pa, tb, te))
        rreqs.append((pb, tb, te))
    return Workload("random_mid", (L, H, D, S, N), reqs, rreqs, {"lens": lens})
