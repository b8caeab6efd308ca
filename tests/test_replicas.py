"""Multi-GPU = replicas only: the only cross-rank logic is bench.py's barrier, the
max-over-ranks of the device time and the whole-job aggregation.  Covered here with world_size-2
gloo processes on CPU (no GPU needed)."""
import os
import socket
import subprocess
import sys
import textwrap

import pytest

from paper_2606_09643_b200 import replicas

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, {root!r})
    from paper_2606_09643_b200 import replicas
    rank, local_rank, world = replicas.init("gloo")
    assert world == 2 and rank == int(os.environ["RANK"])
    replicas.barrier()
    ms = [10.0, 12.5][rank]                       # rank 1 is the slow replica
    mx = replicas.max_over_ranks(ms)
    total = replicas.sum_over_ranks(256.0)
    lo, hi = replicas.shard_requests(7, rank, world)
    replicas.barrier()
    print(json.dumps(dict(rank=rank, mx=mx, total=total, lo=lo, hi=hi,
                          value=replicas.whole_job_throughput(256, 5, mx, world))))
    replicas.finalize()
""")


def test_two_replicas_gloo_max_and_aggregate(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0, err
        outs.append(__import__("json").loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["mx"] == 12.5 and o["total"] == 512.0           # MAX over ranks, SUM of units
        assert o["value"] == pytest.approx(2 * 256 * 5 / 12.5e-3)    # units of all ranks / max time
    assert [(o["lo"], o["hi"]) for o in sorted(outs, key=lambda o: o["rank"])] == [(0, 4), (4, 7)]


def test_single_process_identities():
    assert replicas.max_over_ranks(3.25) == 3.25 and replicas.sum_over_ranks(2.0) == 2.0
    assert replicas.whole_job_throughput(256, 10, 100.0, 1) == pytest.approx(25600.0)
    cover = []
    for r in range(3):
        lo, hi = replicas.shard_requests(10, r, 3)
        cover += list(range(lo, hi))
    assert cover == list(range(10))


def test_reference_arm_exits_quietly_on_nonzero_rank():
    """Under torchrun only rank 0 runs the oracle arm; other ranks exit 0 without work or output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"], env=env,
                       capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""
