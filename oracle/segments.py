"""ORACLE (test infrastructure) — the task-sorted segment tables, written as their definition.

The paper has no such table; it is implied by executing adapter work "in compatible
sub-batches" (§6.2; L160 §4.2 "batches the requests across the common
backbone first then integrate adapter difference") and is required bit-exactly by
BASELINE.json north_star item (1).  Definition: a STABLE sort of request
indices by task id, then prefix sums.  All int32; comparisons are exact.

Pins (tests/test_oracle_pins.py): permutation/monotonicity/stability/prefix-sum properties,
exhaustive enumeration for B <= 6, T <= 3 against a brute-force insertion construction.
"""
import numpy as np


def segment_tables(task_ids, lengths, n_task_slots):
    """-> dict(perm, inv_perm, task_req_off, cu_tok, task_tok_off), all np.int32.

    perm[p]         original index of the request at sorted position p
    inv_perm[i]     sorted position of original request i
    task_req_off[t] #{i : task_ids[i] < t},  t = 0..T
    cu_tok[p]       sum of lengths of the requests at sorted positions < p,  p = 0..B
    task_tok_off[t] cu_tok[task_req_off[t]]
    """
    B = len(task_ids)
    perm = sorted(range(B), key=lambda i: (int(task_ids[i]), i))
    inv_perm = [0] * B
    for p, i in enumerate(perm):
        inv_perm[i] = p
    task_req_off = [sum(1 for i in range(B) if int(task_ids[i]) < t) for t in range(n_task_slots + 1)]
    cu_tok = [0] * (B + 1)
    for p in range(B):
        cu_tok[p + 1] = cu_tok[p] + int(lengths[perm[p]])
    task_tok_off = [cu_tok[task_req_off[t]] for t in range(n_task_slots + 1)]
    as32 = lambda v: np.array(v, dtype=np.int32)
    return dict(perm=as32(perm), inv_perm=as32(inv_perm), task_req_off=as32(task_req_off),
                cu_tok=as32(cu_tok), task_tok_off=as32(task_tok_off))
