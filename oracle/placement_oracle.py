"""placement_oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain, step-by-step statement of LUMEN's checkpoint placement (Eq. (1)), recovery dispatch
and greedy load rebalancing, in the paper's order and
notation.  Pure Python with exact rational arithmetic (fractions.Fraction), no numpy.

What it follows (section 4.2):
  * "queueing delay q_w measures the average wait time on worker w"; "restore pressure
    p_w(r) ... the controller first averages the reserved KV footprints of the checkpoints
    that w would hold after assigning r, then divides this average by a fixed host-to-GPU
    bandwidth".
  * "The candidate set F(r) comprises all workers with sufficient storage to accommodate r's
    reserved KV footprint, excluding the worker currently serving r."
  * h(r) = argmin_{w in F(r)} (q_w + lambda * p_w(r))                                  (1)
and (section 4.3):
  * dispatch: "routes interrupted requests to their designated checkpoint holders. If a
    checkpoint holder has also failed, LUMEN marks the request for recomputation and assigns
    it to the least-loaded surviving worker."
  * rebalancing: "compares each surviving worker's total request load (i.e., queued, running,
    and newly assigned interrupted requests) against the cluster-wide average computed after
    the initial recovery dispatch. When a holder is overloaded, LUMEN migrates its assigned
    requests to the least-loaded worker, prioritizing requests in increasing order of their
    actual checkpointed size ... iteratively recomputes worker loads after each migration and
    always targets the most congested worker first, until no worker exceeds the cluster-wide
    average."

Readings where the paper is silent (F1-F4):
  F1  ties in argmin / "least-loaded" / "most congested": the lowest worker id wins.
  F2  loads are request counts (integers); with a fractional average "no worker exceeds the
      average" is unreachable, so a worker is overloaded iff load > ceil(average); for an
      integer average this is the paper's rule verbatim.
  F3  only interrupted requests dispatched to their checkpoint holder in the first step are
      migratable (they are what the holder was "assigned"); a migrated request has forfeited
      its checkpoint, becomes a recomputation at its new worker and is not moved again.  An
      overloaded worker with nothing migratable is skipped.
  F4  the migration target is the least-loaded surviving worker other than the source; a
      migration happens only while the source is overloaded, so it always ends.
"""
from __future__ import annotations

from fractions import Fraction
from math import ceil
from typing import Dict, List, Optional, Sequence, Tuple


def restore_pressure(held_footprints: Sequence[int], footprint_r: int, bandwidth, num=Fraction):
    """p_w(r): mean reserved footprint of the checkpoints w would hold after assigning r,
    divided by the fixed host-to-GPU bandwidth.  num = Fraction (exact) or float (the
    library's precision: IEEE double, operations in exactly this order)."""
    fps = list(held_footprints) + [footprint_r]
    return num(sum(fps)) / num(len(fps)) / num(bandwidth)


def choose_holder(q: Sequence, held: Sequence[Sequence[int]], available: Sequence[int],
                  serving: int, footprint_r: int, lam, bandwidth, num=Fraction) -> Optional[int]:
    """Eq. (1).  q[w]: queueing delay; held[w]: reserved footprints of the checkpoints w holds;
    available[w]: free checkpoint-store capacity; serving: the worker running r.
    Returns h(r), or None if F(r) is empty.  The argmin is an integer decided by real numbers:
    with num=float it is taken in the library's precision (double), as the parity rules ask."""
    best, best_score = None, None
    for w in range(len(q)):
        if w == serving or available[w] < footprint_r:      # F(r)
            continue
        score = num(q[w]) + num(lam) * restore_pressure(held[w], footprint_r, bandwidth, num)
        if best is None or score < best_score:              # F1: lowest id wins ties
            best, best_score = w, score
    return best


def dispatch_and_rebalance(load: Sequence[int], alive: Sequence[bool],
                           interrupted: Sequence[Tuple[int, int]]
                           ) -> Tuple[List[int], List[bool], List[int]]:
    """load[w]: queued + running requests of worker w before recovery (ignored for dead
    workers).  interrupted[i] = (holder, checkpointed_size).  Returns (worker assigned to each
    interrupted request, whether it still reuses its KV checkpoint, final loads)."""
    W = len(load)
    survivors = [w for w in range(W) if alive[w]]
    assert survivors
    cur = [load[w] if alive[w] else 0 for w in range(W)]
    assign: List[int] = [-1] * len(interrupted)
    reuse: List[bool] = [False] * len(interrupted)

    def least_loaded(exclude: int = -1) -> int:
        cands = [w for w in survivors if w != exclude]
        return min(cands, key=lambda w: (cur[w], w))        # F1

    # ---- recovery dispatch: locality first ---------------------------------------------
    for i, (holder, _size) in enumerate(interrupted):
        if 0 <= holder < W and alive[holder]:
            assign[i], reuse[i] = holder, True
        else:                                               # holder failed too: recompute
            assign[i], reuse[i] = least_loaded(), False
        cur[assign[i]] += 1
    # ---- load rebalancing ----------------------------------------------------------------
    average = Fraction(sum(cur[w] for w in survivors), len(survivors))   # after the dispatch
    limit = ceil(average)                                   # F2
    while True:
        over = [w for w in survivors if cur[w] > limit and
                any(assign[i] == w and reuse[i] for i in range(len(interrupted)))]   # F3
        if not over or len(survivors) < 2:
            break
        src = max(over, key=lambda w: (cur[w], -w))         # most congested first, F1
        movable = [i for i in range(len(interrupted)) if assign[i] == src and reuse[i]]
        i = min(movable, key=lambda k: (interrupted[k][1], k))   # smallest checkpointed size
        dst = least_loaded(exclude=src)                     # F4
        assign[i], reuse[i] = dst, False                    # forfeits its checkpoint
        cur[src] -= 1
        cur[dst] += 1
    return assign, reuse, cur
