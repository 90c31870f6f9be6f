"""Host logic of the N>1 path on CPU: two gloo ranks run bench.py's rendezvous / reduction helpers (the data path has
no collective: one prompt per rank, `value` = sum of per-rank work / max-over-ranks time) and the reference arm's
"rank 0 only" rule."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

RANK_SCRIPT = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import bench
from paper_2606_09441_b200 import workload as wl
rank, world, local = bench.dist_setup(2)
assert world == 2 and rank == int(os.environ["RANK"])
t = bench.max_over_ranks(1.0 + rank, world)          # slowest rank decides the step time
f = bench.sum_over_ranks(10.0 * (rank + 1), world)   # work of all ranks adds up
bench.barrier(world)
w = wl.custom("r", seed=wl.BASE_SEED + rank)         # one prompt per rank: seeds differ
print(json.dumps({{"rank": rank, "t": t, "f": f, "la0": int(w.la_blob[:8].sum())}}))
import torch.distributed as dist
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _env(rank, port):
    e = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
             MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
    return e


def test_two_rank_gloo_reductions():
    port = _free_port()
    procs = [subprocess.Popen([sys.executable, "-c", RANK_SCRIPT.format(root=ROOT)], env=_env(r, port),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    assert [d["t"] for d in outs] == [2.0, 2.0]
    assert [d["f"] for d in outs] == [30.0, 30.0]
    assert all("la0" in d for d in outs)


def test_reference_arm_runs_on_rank0_only():
    port = _free_port()
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--config", "tiny"]
    procs = [subprocess.Popen(cmd, env=_env(r, port), stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    res = [p.communicate(timeout=240) + (p.returncode,) for p in procs]
    assert all(rc == 0 for _, _, rc in res), res
    line = json.loads(res[0][0].strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0
    assert res[1][0].strip() == ""          # rank 1 exits 0 without work
