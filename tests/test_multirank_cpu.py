"""N > 1 host logic of bench.py on CPU (gloo, world_size 2): the path shards by lines with no
data-path collective, so the only multi-rank logic is rendezvous, barrier, max-over-ranks of the
device time and the whole-job aggregate.  The reference arm must print on rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
sys.path.insert(0, %(root)r)
import bench
g = bench.RankGroup("gloo")
assert g.world == 2 and g.rank == int(os.environ["RANK"])
g.barrier()
sec = 0.010 if g.rank == 0 else 0.025          # rank 1 is the slow one
m = g.max(sec)
val = g.aggregate(1000, m)
g.barrier()
print(json.dumps({"rank": g.rank, "max": m, "value": val}))
g.close()
'''


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _spawn(code_or_args, world=2, is_code=True):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        cmd = [sys.executable, "-c", code_or_args] if is_code else [sys.executable] + code_or_args
        procs.append(subprocess.Popen(cmd, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = [p.communicate(timeout=300) for p in procs]
    return procs, outs


@pytest.mark.timeout(400)
def test_rank_group_max_and_aggregate_gloo_world2():
    procs, outs = _spawn(WORKER % {"root": ROOT})
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    recs = sorted((json.loads(o.strip().splitlines()[-1]) for o, _ in outs), key=lambda r: r["rank"])
    for r in recs:
        assert r["max"] == 0.025                       # max over ranks, seen by every rank
        assert r["value"] == pytest.approx(2 * 1000 / 0.025)   # all ranks' cells / slowest time


@pytest.mark.timeout(400)
def test_reference_arm_prints_on_rank0_only():
    args = [os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
            "--warmup", "1", "--ref-slices", "1", "--workload", "cfg1_tiny"]
    procs, outs = _spawn(args, is_code=False)
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    assert outs[1][0].strip() == ""
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
