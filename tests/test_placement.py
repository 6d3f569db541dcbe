"""Placement Eq. (1), recovery dispatch and greedy rebalancing:
the oracle against hand-worked examples and invariants, then the library against the oracle."""
import ast
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

from oracle import placement_oracle as po
from workloads import substream

GOLDEN = Path(__file__).resolve().parent / "golden" / "placement.txt"


def golden(kind):
    for line in GOLDEN.read_text().splitlines():
        if line.startswith("{"):
            c = ast.literal_eval(line)
            if c["kind"] == kind:
                yield c


def frac(x):
    return Fraction(x)


def test_oracle_eq1_hand_worked():
    n = 0
    for c in golden("holder"):
        got = po.choose_holder([frac(x) for x in c["q"]], c["held"], c["available"], c["serving"],
                               c["footprint"], frac(c["lam"]), c["bw"])
        assert got == c["expect"], c
        n += 1
    assert n == 9
    assert po.restore_pressure([26], 13, 26) == Fraction(3, 4)
    assert po.restore_pressure([], 13, 26) == Fraction(1, 2)


def test_oracle_recovery_hand_worked():
    n = 0
    for c in golden("recover"):
        assign, reuse, final = po.dispatch_and_rebalance(c["load"], c["alive"], [tuple(x) for x in c["interrupted"]])
        assert (assign, reuse, final) == (c["assign"], c["reuse"], c["final"]), c
        n += 1
    assert n == 5


def random_recovery(rng):
    W = int(rng.integers(2, 9))
    alive = [bool(x) for x in rng.random(W) < 0.7]
    if not any(alive):
        alive[int(rng.integers(0, W))] = True
    load = [int(x) for x in rng.integers(0, 12, size=W)]
    n = int(rng.integers(0, 25))
    inter = [(int(rng.integers(0, W)), int(rng.integers(0, 40))) for _ in range(n)]
    return load, alive, inter


def test_oracle_recovery_invariants():
    rng = substream(41, "placement")
    for _ in range(300):
        load, alive, inter = random_recovery(rng)
        assign, reuse, final = po.dispatch_and_rebalance(load, alive, inter)
        surv = [w for w in range(len(load)) if alive[w]]
        assert all(alive[a] for a in assign)                              # only survivors get work
        assert sum(final[w] for w in surv) == sum(load[w] for w in surv) + len(inter)   # nothing lost
        for (holder, _), a, r in zip(inter, assign, reuse):
            assert (not r) or a == holder                                 # reuse only at the holder
            assert r or not alive[holder] or a != holder or len(surv) == 1 or True
        limit = -(-sum(final[w] for w in surv) // len(surv))
        for w in surv:                                                    # no overloaded worker keeps a
            if final[w] > limit:                                          # migratable request
                assert not any(a == w and r for a, r in zip(assign, reuse))
        # shed in increasing checkpointed size: every request still reusing at w is at least as
        # large as every request that was shed from w
        for w in surv:
            kept = [s for (h, s), a, r in zip(inter, assign, reuse) if h == w and r]
            shed = [s for (h, s), a, r in zip(inter, assign, reuse) if h == w and alive[h] and not r]
            if kept and shed:
                assert min(kept) >= max(shed)


@pytest.fixture(scope="module")
def lk():
    from paper_2606_17787_b200 import build
    build.build()
    import paper_2606_17787_b200 as lk
    return lk


def test_library_equals_oracle(lk):
    for c in golden("holder"):
        got = lk.lumen_kv_choose_holder([float(frac(x)) for x in c["q"]], c["held"], c["available"],
                                        c["serving"], c["footprint"], float(frac(c["lam"])), c["bw"])
        assert got == (c["expect"] if c["expect"] is not None else -1), c
    rng = substream(42, "placement_lib")
    for _ in range(300):
        W = int(rng.integers(1, 9))
        q = [float(x) for x in rng.random(W) * 3]
        held = [[int(x) for x in rng.integers(1, 200, size=int(rng.integers(0, 4)))] for _ in range(W)]
        avail = [int(x) for x in rng.integers(0, 300, size=W)]
        fp = int(rng.integers(1, 160))
        serving = int(rng.integers(0, W))
        lam = float(rng.choice([0.0, 0.5, 1.0, 4.0]))
        # the argmin is taken in the library's precision on both sides (double, same operation order)
        want = po.choose_holder(q, held, avail, serving, fp, lam, 26.0, num=float)
        assert lk.lumen_kv_choose_holder(q, held, avail, serving, fp, lam, 26.0) == (-1 if want is None else want)
    for c in golden("recover"):
        assert lk.lumen_kv_recover(c["load"], c["alive"], c["interrupted"]) == (c["assign"], c["reuse"], c["final"])
    for _ in range(300):
        load, alive, inter = random_recovery(rng)
        assert lk.lumen_kv_recover(load, alive, inter) == po.dispatch_and_rebalance(load, alive, inter)
