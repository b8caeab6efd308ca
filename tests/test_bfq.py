"""Pins for oracle/bfq.py (§4.2, Eq. 1-3) and, when libfmx is built, exact agreement
of the C++ builder (fmx_bfq_*) with it on seeded traces."""
import math

import numpy as np
import pytest

from oracle.bfq import BFQ


def test_hand_computed_two_task_trace():
    """Weights w0 = 1, w1 = 2; B_max = 2; profile Lat(1) = 10 ms, Lat(2) = 12 ms; no SLO.
    Arithmetic written out (Eq. 1: S = max(F_prev, v); Eq. 2: F = S + l/w; Eq. 3 retag)."""
    q = BFQ(2, 2, [10.0, 12.0])
    q.set_task(0, 1.0); q.set_task(1, 2.0)
    q.enqueue(0, 100, 1, 0.0)      # v=0  S=max(0,0)=0    F=0+10/1=10
    q.enqueue(0, 101, 1, 0.0)      # v=0  S=max(10,0)=10  F=20
    q.enqueue(1, 102, 1, 0.0)      # v=0  S=0             F=0+10/2=5
    q.enqueue(1, 103, 1, 0.0)      #      S=5             F=10
    q.enqueue(1, 104, 1, 0.0)      #      S=10            F=15
    assert [(r["S"], r["F"]) for r in q.queue[0]] == [(0.0, 10.0), (10.0, 20.0)]
    assert [(r["S"], r["F"]) for r in q.queue[1]] == [(0.0, 5.0), (5.0, 10.0), (10.0, 15.0)]
    # order by (S, F, seq): 102 (0,5) < 100 (0,10) < 103 (5,10) < 104 (10,15) < 101 (10,20)
    assert q.next_batch(0.0, 8) == [(1, 1, 102), (0, 1, 100)]
    assert q.F_last == [10.0, 5.0]
    q.complete(12.0)               # l_i(b) = 12/2 = 6 per request
    # task 0: 100 -> S=max(0,0)=0, F=0+6/1=6 = F_last ; queued 101 -> S=max(6,0)=6, F=12
    # task 1: 102 -> S=0, F=0+6/2=3 = F_last ; queued 103 -> S=3, F=6 ; 104 -> S=6, F=9
    assert q.F_last == [6.0, 3.0]
    assert [(r["S"], r["F"]) for r in q.queue[0]] == [(6.0, 12.0)]
    assert [(r["S"], r["F"]) for r in q.queue[1]] == [(3.0, 6.0), (6.0, 9.0)]
    assert q.F_prev == [12.0, 9.0]
    q.enqueue(0, 105, 1, 1.0)      # v=max(6,3)=6  S=max(12,6)=12  F=12+10=22  (Eq. 2 uses l(1) again)
    assert (q.queue[0][-1]["S"], q.queue[0][-1]["F"], q.queue[0][-1]["v_arr"]) == (12.0, 22.0, 6.0)
    # 103 (3,6) < 104 (6,9) < 101 (6,12) < 105 (12,22)
    assert q.next_batch(1.0, 8) == [(1, 1, 103), (1, 1, 104)]
    q.complete(0.0)                # no measurement: profile Lat(2)/2 = 6 -> tags unchanged: 103 (3,6), 104 (6,9)
    assert q.F_last == [6.0, 9.0] and q.F_prev == [22.0, 9.0]
    assert q.next_batch(2.0, 8) == [(0, 1, 101), (0, 1, 105)]
    assert q.next_batch(3.0, 8) == []
    assert q.dispatched == [3, 3]


def test_slo_stops_extension_and_first_is_always_admitted():
    q = BFQ(1, 4, [10.0, 12.0, 14.0, 16.0])
    q.set_task(0, 1.0, slo_ms=13.0)
    for h in range(4):
        q.enqueue(0, h, 1, 0.0)
    # now=0: b=2 finishes at 12 <= 13 ok; b=3 finishes at 14 > 13 -> stop (Fig. 5 (a)/(b))
    assert [h for _, _, h in q.next_batch(0.0, 99)] == [0, 1]
    q.complete(0.0)
    # now=50: already late, the first is admitted anyway (work-conserving), nothing can join it
    assert [h for _, _, h in q.next_batch(50.0, 99)] == [2]


def test_cap_and_bmax_bound_the_batch():
    q = BFQ(2, 3, [1.0, 1.5, 2.0])
    for h in range(10):
        q.enqueue(h % 2, h, 1, 0.0)
    assert len(q.next_batch(0.0, 99)) == 3
    q.complete()
    assert len(q.next_batch(0.0, 2)) == 2
    q.complete()
    assert q.next_batch(0.0, 0) == []


def test_bmax_1_is_start_time_fair_queueing_order():
    rng = np.random.default_rng(11)
    q = BFQ(3, 1, [4.0])
    for i, w in enumerate((1.0, 2.0, 0.5)):
        q.set_task(i, w)
    h = 0
    for step in range(200):
        for _ in range(int(rng.integers(0, 3))):
            q.enqueue(int(rng.integers(0, 3)), h, 1, float(step)); h += 1
        queued = [r for qu in q.queue for r in qu]
        out = q.next_batch(float(step), 1)
        if queued:
            best = min(queued, key=lambda r: (r["S"], r["F"], r["seq"]))
            assert out == [(best["task"], 1, best["handle"])]      # min start tag first
        else:
            assert out == []                                       # work-conserving: idle only if empty
        q.complete(0.0)


@pytest.mark.parametrize("weights", [(1.0, 1.0), (2.0, 1.0), (3.0, 1.0)])
def test_weighted_share_under_backlog(weights):
    """PAPER.md Fig. 12 setting: all tasks backlogged; service follows the weights."""
    b_max = 4
    q = BFQ(2, b_max, [10.0, 11.0, 12.0, 13.0])
    for i, w in enumerate(weights):
        q.set_task(i, w)
    h = 0
    for i in range(2):
        for _ in range(400):
            q.enqueue(i, h, 1, 0.0); h += 1
    served = [0, 0]
    for step in range(60):
        batch = q.next_batch(float(step), 99)
        assert 1 <= len(batch) <= b_max
        for t, _, _ in batch:
            served[t] += 1
        q.complete(0.0)
        total = sum(served)
        for i in range(2):
            assert abs(served[i] - total * weights[i] / sum(weights)) <= b_max + 1
    for i in range(2):                                             # per-task FIFO and monotone tags
        S = [r["S"] for r in q.queue[i]]
        assert all(a <= b for a, b in zip(S, S[1:]))


def test_token_level_charging():
    q = BFQ(2, 8, [1.0] * 8, l_tok_ms=0.01)
    q.enqueue(0, 0, 1000, 0.0)     # l = 10  -> F = 10
    q.enqueue(1, 1, 100, 0.0)      # l = 1   -> F = 1
    q.enqueue(1, 2, 100, 0.0)      # S = 1, F = 2
    assert [(r["S"], r["F"]) for r in q.queue[1]] == [(0.0, 1.0), (1.0, 2.0)]
    assert [h for _, _, h in q.next_batch(0.0, 99)] == [1, 0, 2]
    q.complete(24.0)               # 1200 tokens -> 0.02 ms/token: 100-token requests cost 2, the 1000-token one 20
    assert q.F_last == [20.0, 4.0] and q.service_ms == [20.0, 4.0]


# ------------------------------------------------------------------------------------------------
# S0 parity of the PRODUCT code: the C++ builder (fmx_bfq_*, csrc/bfq.cpp) against oracle/bfq.py in
# lock-step on seeded traces (Eq. 1-3).  Tag arithmetic is IEEE
# double in the same order on both sides, so every comparison is `==`, not a tolerance.  Host only.
def _lockstep(seed, T, b_max, slo_choices, l_tok, steps=300):
    from paper_2606_09643_b200.binding import Bfq
    rng = np.random.default_rng(seed)
    lat = np.cumsum(rng.uniform(0.5, 3.0, b_max)).tolist()          # increasing latency profile Lat(1..b_max)
    o = BFQ(T, b_max, lat, l_tok_ms=l_tok)
    c = Bfq(T, b_max, lat, l_tok_ms=l_tok)
    for t in range(T):
        w = float(rng.choice([0.5, 1.0, 2.0, 3.0]))
        slo = float(rng.choice(slo_choices))
        o.set_task(t, w, slo); c.set_task(t, w, slo)
    h, now = 0, 0.0
    n_batches = n_nonempty = 0
    for step in range(steps):
        now += float(rng.uniform(0.0, 4.0))
        for _ in range(int(rng.integers(0, 2 * b_max + 1))):
            t = int(rng.integers(0, T))
            n = int(rng.integers(1, 1025)) if l_tok > 0 else int(rng.integers(1, 9))
            arr = now - float(rng.uniform(0.0, 2.0))
            o.enqueue(t, h, n, arr); c.enqueue(t, h, n, arr); h += 1
        # every queued request's (S, F, v_arr), every task
        for t in range(T):
            d, s_ms, queued = c.stats(t)
            assert queued == len(o.queue[t]) and d == o.dispatched[t] and s_ms == o.service_ms[t]
            for j, r in enumerate(o.queue[t]):
                assert c.peek(t, j) == (r["S"], r["F"], r["v_arr"]), (seed, step, t, j)
        cap = int(rng.choice([0, 1, b_max // 2 + 1, b_max, b_max + 3]))
        ref = o.next_batch(now, cap)
        ids, lens, handles = c.next_batch(now, cap)
        assert [(int(a), int(b), int(d)) for a, b, d in zip(ids, lens, handles)] == ref, (seed, step)
        n_batches += 1; n_nonempty += bool(ref)
        measured = 0.0 if rng.random() < 0.5 else float(rng.uniform(0.5, 40.0))
        o.complete(measured); c.complete(measured)
    for t in range(T):                                                # after the last retag
        for j, r in enumerate(o.queue[t]):
            assert c.peek(t, j) == (r["S"], r["F"], r["v_arr"])
        assert c.stats(t) == (o.dispatched[t], o.service_ms[t], len(o.queue[t]))
    assert n_nonempty > steps // 4                                    # the trace really exercised the builder
    return n_batches


@pytest.mark.parametrize("seed", range(12))
def test_cpp_builder_equals_oracle_in_lockstep(seed):
    rng = np.random.default_rng(1000 + seed)
    T = int(rng.integers(1, 9))
    b_max = int(rng.integers(1, 9))
    slo_choices = [[math.inf], [math.inf, 30.0, 12.0], [30.0, 12.0]][seed % 3]
    l_tok = 0.0 if seed % 2 == 0 else 0.01                            # both charging modes
    _lockstep(seed, T, b_max, slo_choices, l_tok)


def test_cpp_builder_equals_oracle_at_serving_scale():
    """92 tasks, B_max 512 (configs[4]'s batch), token charging: the shapes bench.py's `bfq` leg uses."""
    _lockstep(77, 92, 512, [math.inf, 500.0], 0.01, steps=12)
    _lockstep(78, 92, 512, [math.inf], 0.0, steps=12)
