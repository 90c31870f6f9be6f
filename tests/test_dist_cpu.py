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


SHARD_SCRIPT = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch
import torch.distributed as dist
import bench
from oracle import sift_oracle as so
from paper_2606_09441_b200 import workload as wl, shard
rank, world, local = bench.dist_setup(2)
# ONE prompt, the same on every rank (same seed); 2 layers so that the layer part of the blob offsets is exercised
w = wl.custom("hs", n_layers=2, n_q_heads=4, n_kv_heads=2, head_dim=64, doc_lens=(150, 64, 200), query_len=33, tile=64,
              p_loc=0.5, p_cross=0.4, seed=77)
ps, layer = w.shape, 1
sh = shard.head_shard(ps.n_q_heads, ps.n_kv_heads, rank, world)
sub = shard.shard_prompt_shape(ps, sh)
la_off, ca_off = shard.shard_blob_offsets(w, sh, layer)
q, k, v = w.qkv(layer)
qs, ks, vs = shard.shard_views(q, k, v, sh)
rows = list(range(0, ps.n_tokens, 5)) + [ps.n_tokens - 1]
# the shard computes ITS heads from its own view of the inputs (sub-shape, shifted blob offsets, column views)
def vec(blob, off, nbytes, h, d):          # (layer 0, head h) of the sub-shape's blob of document d
    o = int(off[d]) + h * nbytes
    return blob[o:o + nbytes]
o_loc = torch.zeros((len(rows), sh.n_q, ps.head_dim), dtype=torch.float64)
for h in range(sh.n_q):
    la = [vec(w.la_blob, la_off, sub.la_bytes(d), h, d) for d in range(ps.n_docs)]
    ca = [vec(w.ca_blob, ca_off, sub.ca_bytes(d), h, d) for d in range(ps.n_docs)]
    o, _ = so.sift_attention_rows(qs, ks, vs, h, sub.doc_offsets, sub.query_len, sub.tile, sub.cross_gran, la, ca, rows, dtype=torch.float64)
    o_loc[:, h] = o
parts = [torch.zeros_like(o_loc) for _ in range(world)]
dist.all_gather(parts, o_loc)              # (test only: the path itself has no collective)
o_all = torch.cat(parts, dim=1)
# the unsharded prompt
ref = torch.zeros((len(rows), ps.n_q_heads, ps.head_dim), dtype=torch.float64)
for h in range(ps.n_q_heads):
    la, ca = so.head_vectors(w, layer, h)
    o, _ = so.sift_attention_rows(q, k, v, h, ps.doc_offsets, ps.query_len, ps.tile, ps.cross_gran, la, ca, rows, dtype=torch.float64)
    ref[:, h] = o
print(json.dumps({{"rank": rank, "heads": [sh.q0, sh.q1], "kv": [sh.kv0, sh.kv1], "err": float((o_all - ref).abs().max())}}))
dist.destroy_process_group()
"""


def test_head_sharded_prompt_two_ranks_concatenates_to_the_single_rank_result():
    """SURVEY 8(f)-4 / PAPER.md:L283: rank r owns a block of kv heads of ONE prompt; the shards' O columns, put side by
    side, are the unsharded O (computed here by the oracle on each shard's view of the inputs)."""
    port = _free_port()
    procs = [subprocess.Popen([sys.executable, "-c", SHARD_SCRIPT.format(root=ROOT)], env=_env(r, port),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    assert outs[0]["heads"] == [0, 2] and outs[1]["heads"] == [2, 4] and outs[0]["kv"] == [0, 1] and outs[1]["kv"] == [1, 2]
    assert outs[0]["err"] == 0.0 and outs[1]["err"] == 0.0


def test_head_shard_blocks_partition_the_heads():
    from paper_2606_09441_b200 import shard
    for hq, hkv, world in ((32, 8, 1), (32, 8, 2), (32, 8, 3), (32, 8, 8), (4, 4, 3)):
        blocks = [shard.head_shard(hq, hkv, r, world) for r in range(world)]
        assert blocks[0].kv0 == 0 and blocks[-1].kv1 == hkv
        for a, b in zip(blocks[:-1], blocks[1:]):
            assert a.kv1 == b.kv0 and a.q1 == b.q0
        assert all(b.q0 == b.kv0 * (hq // hkv) and b.q1 == b.kv1 * (hq // hkv) for b in blocks)
        assert max(b.n_kv for b in blocks) - min(b.n_kv for b in blocks) <= 1
