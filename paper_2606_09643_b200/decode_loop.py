"""Host-side iteration scheduling for token decode: which sequences advance in the next decode
iteration, decided by the BFQ batch builder with token-level charging.

PAPER.md L168: "FMplex applies the same accounting principle to token-based FMs by charging token-level work in service-time
units", for runtimes with "continuous batching and long-lived decode iterations" (L127).  A live sequence is one request whose
service is consumed one token per iteration: before every iteration each live sequence holds exactly ONE queued BFQ item of
length 1 (cost l_tok_ms / weight), `next_iteration` lets BFQ pick up to `cap` of them by start tag, and `complete` retags with
the measured iteration time (Eq. 3).  Sequences that were not picked keep their tags and are served first later; a heavier task
decodes more tokens per unit time (the split is compressed relative to the weights because a queue that empties restarts at
v = max_i F_i^last, the paper's definition - tests/test_decode_loop.py).  Marshalling only: all arithmetic is in libfmx's `fmx_bfq_*`.
"""
from .binding import Bfq


class DecodeScheduler:
    def __init__(self, n_tasks, max_batch, l_tok_ms=1.0, weights=None, bfq_factory=None):
        lat = [l_tok_ms * (b + 1) for b in range(max_batch)]           # profiled latency of an iteration over b sequences
        make = bfq_factory or (lambda: Bfq(n_tasks, max_batch, lat, l_tok_ms))
        self.q = make()
        self.max_batch = max_batch
        for t in range(n_tasks):
            self.q.set_task(t, 1.0 if weights is None else float(weights[t]))
        self.task_of = {}            # live sequence handle -> task
        self.queued = set()          # handles that hold a queued item

    def add_sequence(self, handle, task):
        self.task_of[int(handle)] = int(task)

    def finish_sequence(self, handle):
        """The sequence produced its last token.  Its queued item (if any) stays in BFQ and is dropped when picked."""
        self.task_of.pop(int(handle), None)

    def next_iteration(self, now_ms, cap=None):
        """-> (handles, task ids) of the sequences that advance by one token in this iteration."""
        for h, t in self.task_of.items():
            if h not in self.queued:
                self.q.enqueue(t, h, 1, now_ms)
                self.queued.add(h)
        ids, _lens, handles = self.q.next_batch(now_ms, self.max_batch if cap is None else cap)
        picked, tasks = [], []
        for t, h in zip(ids.tolist(), handles.tolist()):
            self.queued.discard(h)
            if h in self.task_of:                                       # finished sequences' stale items are skipped
                picked.append(h)
                tasks.append(t)
        return picked, tasks

    def complete(self, measured_ms=0.0):
        self.q.complete(measured_ms)
