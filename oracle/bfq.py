"""ORACLE (test infrastructure) — BFQ, the batch-aware fair-queue batch builder, step by step.

Follows PAPER.md §4.2 in the paper's order and notation:
  Eq. 1  S_i^j = max{F_i^{j-1}, v}                      (L156)
  Eq. 2  F_i^j = S_i^j + l / w_i                        (L158)
  v = max_i F_i^last over each task's most recently DISPATCHED request (L160)
  batch formation: order by start tag, extend until B_max or an SLO violation (L160)
  Eq. 3  F_i^j = S_i^j + l_i(b) / w_i  retag after a batch (L162-L166)
  token-based FMs: charge token-level work in service-time units (L168)
The readings of what the text leaves open (tie-break, stop-vs-skip, what b is, how the
retag chain restarts) are DESIGN.md §3 readings 24-29.  All tag arithmetic is IEEE double
in exactly the order written here; the C++ builder must agree bit for bit.

Pins (tests/test_bfq.py): a hand-computed two-task trace (arithmetic written out in the
test), B_max = 1 reduces to start-time fair queueing order, weighted share under backlog,
work conservation, per-task FIFO, batch <= B_max, SLO admission test.  The paper prints no
worked example; its fairness metric [16] has no formula in the text: unpinned.
"""
import math


class BFQ:
    def __init__(self, n_tasks, b_max, lat_ms, l_tok_ms=0.0):
        """lat_ms[b-1] = profiled latency (ms) of a batch of b requests, b = 1..b_max
        (the registration-time profile).  l_tok_ms > 0 selects token-level
        charging: a request of n tokens costs l_tok_ms * n (L168)."""
        assert len(lat_ms) == b_max and b_max >= 1
        self.n_tasks, self.b_max, self.lat_ms, self.l_tok = n_tasks, b_max, list(lat_ms), float(l_tok_ms)
        self.w = [1.0] * n_tasks
        self.slo = [math.inf] * n_tasks
        self.queue = [[] for _ in range(n_tasks)]     # FIFO of request dicts
        self.F_prev = [0.0] * n_tasks                 # F of most recently ENQUEUED request
        self.F_last = [0.0] * n_tasks                 # F of most recently DISPATCHED request
        self.seq = 0
        self.last_batch = []                          # admitted requests, admission order
        self.F_base = [0.0] * n_tasks                 # F_last before the last batch
        self.dispatched = [0] * n_tasks               # accounting (L121)
        self.service_ms = [0.0] * n_tasks

    def set_task(self, i, weight, slo_ms=math.inf):
        self.w[i], self.slo[i] = float(weight), float(slo_ms)

    # ---- service-time model ----------------------------------------------------
    def _l_single(self, n):
        return self.l_tok * n if self.l_tok > 0.0 else self.lat_ms[0]

    def _lat_batch(self, b, tokens):
        return self.l_tok * tokens if self.l_tok > 0.0 else self.lat_ms[b - 1]

    # ---- Eq. 1-2 -----------------------------------------------------------------
    def enqueue(self, i, handle, n, t_arr):
        v = max(self.F_last)
        S = max(self.F_prev[i], v)
        F = S + self._l_single(n) / self.w[i]
        self.queue[i].append(dict(task=i, handle=handle, n=n, arrival=t_arr, S=S, F=F, v_arr=v,
                                  seq=self.seq))
        self.seq += 1
        self.F_prev[i] = F

    # ---- batch formation -----------------------------------------------------------
    def next_batch(self, now, cap):
        heads = [0] * self.n_tasks
        selected = []
        tokens = 0
        limit = min(self.b_max, cap)
        while True:
            best = None
            for i in range(self.n_tasks):           # k-way merge of the queue heads
                if heads[i] < len(self.queue[i]):
                    r = self.queue[i][heads[i]]
                    key = (r["S"], r["F"], r["seq"])
                    if best is None or key < best[0]:
                        best = (key, r)
            if best is None:
                break
            c = best[1]
            b = len(selected)
            if b >= 1:
                if b + 1 > limit:
                    break
                done = now + self._lat_batch(b + 1, tokens + c["n"])
                if any(done > r["arrival"] + self.slo[r["task"]] for r in selected + [c]):
                    break
            elif limit < 1:
                break
            selected.append(c)
            tokens += c["n"]
            heads[c["task"]] += 1
        self.F_base = list(self.F_last)
        for r in selected:
            self.queue[r["task"]].pop(0)
            self.F_last[r["task"]] = r["F"]
            self.dispatched[r["task"]] += 1
        self.last_batch = selected
        return [(r["task"], r["n"], r["handle"]) for r in selected]

    # ---- Eq. 3 ---------------------------------------------------------------------
    def complete(self, measured_ms=0.0):
        batch = self.last_batch
        if not batch:
            return
        b_total = len(batch)
        tokens = sum(r["n"] for r in batch)
        total = measured_ms if measured_ms > 0.0 else self._lat_batch(b_total, tokens)
        unit = total / tokens if self.l_tok > 0.0 else total / b_total

        def l_b(r):
            return unit * r["n"] if self.l_tok > 0.0 else unit

        for i in sorted({r["task"] for r in batch}):
            F = self.F_base[i]
            for r in batch:
                if r["task"] != i:
                    continue
                r["S"] = max(F, r["v_arr"])
                r["F"] = r["S"] + l_b(r) / self.w[i]
                F = r["F"]
                self.service_ms[i] += l_b(r)
            self.F_last[i] = F
            for r in self.queue[i]:
                r["S"] = max(F, r["v_arr"])
                r["F"] = r["S"] + l_b(r) / self.w[i]
                F = r["F"]
            self.F_prev[i] = F
        self.last_batch = []
