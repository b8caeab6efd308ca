"""Pins for oracle/segments.py: properties + exhaustive brute force on tiny inputs."""
import itertools

import numpy as np

from oracle.segments import segment_tables


def _brute(task_ids, lengths, T):
    """Independent construction: repeated stable insertion, bucket by bucket."""
    perm = []
    for t in range(T):
        for i, tid in enumerate(task_ids):
            if tid == t:
                perm.append(i)
    return perm


def test_exhaustive_small():
    for B in range(0, 6):
        for T in (1, 2, 3):
            for ids in itertools.product(range(T), repeat=B):
                lengths = [(3 * i + 1) % 5 + 1 for i in range(B)]
                s = segment_tables(ids, lengths, T)
                perm = _brute(ids, lengths, T)
                assert s["perm"].tolist() == perm
                assert [s["inv_perm"][i] for i in perm] == list(range(B))
                assert s["task_req_off"].tolist() == [sum(1 for x in ids if x < t) for t in range(T + 1)]
                tok = np.concatenate([[0], np.cumsum([lengths[i] for i in perm])]).astype(np.int32)
                assert s["cu_tok"].tolist() == tok.tolist()
                assert s["task_tok_off"].tolist() == [int(tok[o]) for o in s["task_req_off"]]


def test_properties_random():
    rng = np.random.default_rng(7)
    for B, T in [(12, 3), (256, 10), (64, 92), (512, 92), (1, 5)]:
        ids = rng.integers(0, T, size=B)
        ids[ids == 2] = 3 if T > 3 else ids[ids == 2]          # leave a registered-but-absent task
        lengths = rng.integers(1, 1025, size=B)
        s = segment_tables(ids, lengths, T)
        perm = s["perm"]
        assert sorted(perm.tolist()) == list(range(B))
        sorted_ids = ids[perm]
        assert np.all(np.diff(sorted_ids) >= 0)
        same = np.diff(sorted_ids) == 0
        assert np.all(np.diff(perm)[same] > 0)                 # stable within equal ids
        assert s["task_req_off"][0] == 0 and s["task_req_off"][T] == B
        assert s["cu_tok"][B] == lengths.sum() and s["task_tok_off"][T] == lengths.sum()
        for t in range(T):
            lo, hi = s["task_req_off"][t], s["task_req_off"][t + 1]
            assert np.all(sorted_ids[lo:hi] == t)
        for v in s.values():
            assert v.dtype == np.int32
