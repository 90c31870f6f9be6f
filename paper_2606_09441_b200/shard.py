"""Head-sharded run of ONE prompt over several GPUs (sec 7.1: TP = 1/4/8).

(layer, q-head) units are independent in decode and in attention, so the path shards by kv head with its q-heads and
needs NO collective: rank r of `world` takes a contiguous block of kv heads, decodes and attends on the sub-shape, and
writes its own columns of O (the tensor-parallel all-reduce of a model comes after o_proj, outside this path).
Host plumbing only (index arithmetic on shapes, byte offsets and tensor views); every step of the path runs in the
library through paper_2606_09441_b200.api."""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Tuple

import numpy as np


@dataclass(frozen=True)
class HeadShard:
    rank: int
    world: int
    kv0: int      # kv heads [kv0, kv1)
    kv1: int
    q0: int       # q heads [q0, q1) = the q-heads of those kv heads (GQA: q-head h uses kv head h // (Hq // Hkv))
    q1: int

    @property
    def n_kv(self) -> int:
        return self.kv1 - self.kv0

    @property
    def n_q(self) -> int:
        return self.q1 - self.q0


def head_shard(n_q_heads: int, n_kv_heads: int, rank: int, world: int) -> HeadShard:
    """Contiguous blocks of kv heads, sizes differing by at most one (ranks beyond n_kv_heads get an empty shard)."""
    assert n_q_heads % n_kv_heads == 0 and 0 <= rank < world
    hpg = n_q_heads // n_kv_heads
    base, rem = divmod(n_kv_heads, world)
    kv0 = rank * base + min(rank, rem)
    kv1 = kv0 + base + (1 if rank < rem else 0)
    return HeadShard(rank, world, kv0, kv1, kv0 * hpg, kv1 * hpg)


def shard_prompt_shape(ps, sh: HeadShard):
    """PromptShape of the shard: ONE layer (the blob offsets below select it), the shard's heads."""
    return replace(ps, n_layers=1, n_q_heads=sh.n_q, n_kv_heads=sh.n_kv)


def shard_blob_offsets(w, sh: HeadShard, layer: int) -> Tuple[np.ndarray, np.ndarray]:
    """Byte offsets of every document's blob as the sub-shape sees it: the blob of a document is laid out
    [layer][q_head][bytes], so the vectors of (layer, q0 + h) are those of (0, h) of a blob that starts
    (layer * Hq + q0) * bytes later (include/sift.h, "Bit vectors")."""
    ps = w.shape
    la = np.asarray([int(w.la_doc_off[d]) + (layer * ps.n_q_heads + sh.q0) * ps.la_bytes(d) for d in range(ps.n_docs)], np.int64)
    ca = np.asarray([int(w.ca_doc_off[d]) + (layer * ps.n_q_heads + sh.q0) * ps.ca_bytes(d) for d in range(ps.n_docs)], np.int64)
    return la, ca


def shard_views(q, k, v, sh: HeadShard):
    """Column views (no copies) of token-major Q [N, Hq, d], K, V [N, Hkv, d]: row stride stays the full row."""
    return q[:, sh.q0:sh.q1], k[:, sh.kv0:sh.kv1], v[:, sh.kv0:sh.kv1]
