"""Host-side accounting for bench.py: marked (query, key) pairs from decoded metadata, FLOP and byte models.
Pure integer arithmetic over the MD-v1 arrays the decode kernel wrote (no oracle code)."""
from __future__ import annotations

from typing import Dict

import numpy as np


def marked_pairs_per_head(md: Dict[str, np.ndarray], layer: int, n_docs: int, cross_gran: int = 1) -> np.ndarray:
    """True mask entries per q-head of one layer (reading A26: element level; the diagonal tile counts its causal
    half, ragged tiles their real rows).  md: numpy views of the MD-v1 arrays."""
    seg, row0, rows = md["tile_seg"], md["tile_row0"].astype(np.int64), md["tile_rows"].astype(np.int64)
    nt = len(seg)
    n_heads = md["cross_ptr"].shape[1]
    out = np.zeros(n_heads, dtype=np.int64)
    is_doc = seg < n_docs
    for h in range(n_heads):
        cp = md["cross_ptr"][layer, h].astype(np.int64)
        if cross_gran == 1:                          # entries are key rows
            keys_before = cp
        else:                                        # entries are pages: a page contributes its real rows
            ci = md["cross_idx"][layer, h][: cp[-1]].astype(np.int64)
            keys_before = np.concatenate([[0], np.cumsum(rows[ci])])[cp]
        tot = int((rows[is_doc] * keys_before[seg[is_doc]]).sum())
        lp = md["local_ptr"][layer, h].astype(np.int64)
        li = md["local_idx"][layer, h]
        owner = np.repeat(np.arange(nt), np.diff(lp))
        ent = li[: lp[-1]].astype(np.int64)
        doc_e = is_doc[owner]
        o, e = owner[doc_e], ent[doc_e]
        diag = o == e
        tot += int((rows[o[~diag]] * rows[e[~diag]]).sum())
        tot += int((rows[o[diag]] * (rows[o[diag]] + 1) // 2).sum())
        for t in np.nonzero(~is_doc)[0]:            # user-query rows: dense causal
            r0, r = int(row0[t]), int(rows[t])
            tot += r * r0 + r * (r + 1) // 2
        out[h] = tot
    return out


def dense_causal_pairs(n_tokens: int) -> int:
    return n_tokens * (n_tokens + 1) // 2


def attention_flops(pairs: int, head_dim: int) -> int:
    """4*d flop per marked pair: 2*d for q.k and 2*d for p*v."""
    return 4 * head_dim * int(pairs)


def decode_algorithmic_bytes(shape, lay, md: Dict[str, np.ndarray]) -> int:
    """Bit vectors read once + index lists / pointers written once (SURVEY.md 8(d) decode roofline)."""
    L, H = shape.n_layers, shape.n_q_heads
    off = shape.doc_offsets
    b = 0
    for d in range(len(off) - 1):
        ln = int(off[d + 1] - off[d])
        p = -(-ln // shape.tile)
        b += L * H * (-(-(p * (p + 1) // 2) // 8) + -(-(-(-ln // shape.cross_gran)) // 8))
    b += 4 * int(md["cross_ptr"][:, :, -1].astype(np.int64).sum())
    b += 4 * int(md["local_ptr"][:, :, -1].astype(np.int64).sum())
    b += 4 * L * H * (len(off) + 2 * lay.n_tiles + 1)
    return b
