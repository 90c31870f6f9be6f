"""CPU oracle for SIFT's decode + block-sparse prefill attention (arxiv/paper_2606_09441).

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this file.  It
shares no code with the CUDA path (``paper_2606_09441_b200/``) and does not import it;
the two only ever see the same seeded input arrays.

What it is: the plain definitions, written out.
  Part 1  ``expand_mask_rows``   -- the boolean mask the two bit vectors stand for
                                    (Fig 6; L201-203 sec 4.1; L209 sec 4.2).
  Part 2  ``attention_rows``     -- masked two-pass softmax attention, one row block at a time
                                    (north_star: "expands the bit vectors into an explicit boolean
                                    mask and runs fp32 masked softmax attention"; fp64 on request).
  Part 3  ``decode_metadata``    -- the decode kernel's output, pass 1 count -> offsets -> pass 2 fill,
                                    CA entries then LA entries, global coordinates
                                    (sec 5.1), in the container "MD-v1"
                                    (SURVEY.md 8(c) Part 3; the paper fixes no container).
  Sizes   ``la_vector_bytes`` .. -- PAPER.md:L213 sec 4.3 and Table 1 (L311-321).
  Part 4  ``encode_document``    -- offline metadata generation (L201, L209, L223).
  Part 5  ``*_batch``            -- several prompts in one call: a loop over prompts around Parts 1-3, shifted to
                                    batch coordinates (container "MD-v1b").
  Part 6  ``*_fp8``              -- e4m3 Q/K/V with per-head scales: decode the bytes by the format's definition, then
                                    Part 2 (reading R7).

Readings of the paper where it is silent or garbled are listed in DESIGN.md section 3
(A1..A26 of SURVEY.md 8(c)); the ones used here are cited inline.

Pins (tests/test_oracle_pins.py): byte patterns from the enumeration printed at L203, the
P=8 -> 36/8 bits example (L213), all of Table 1, all-ones == dense causal, CA cleared ==
block diagonal + dense query, brute-force fp64 softmax on tiny inputs, the torch SDPA
special case, metadata -> mask round trip, reorder invariance; batch: one prompt == MD-v1, block-diagonal mask,
MD-v1b -> mask round trip, brute force over the packed K/V.
Parity unpinned by the paper: the MD-v1 / MD-v1b *container layouts* (our definition; pinned only by
the round trips).
"""
from __future__ import annotations

import math
from typing import Callable, Dict, List, Optional, Sequence, Tuple

import numpy as np
import torch

VecFn = Callable[[int, int, int], np.ndarray]  # (layer, head, doc position) -> uint8 vector


# ------------------------------------------------------------------------------------------
# Sizes (Table 1)
# ------------------------------------------------------------------------------------------

def pages(doc_len: int, tile: int) -> int:
    """P = ceil(L / T)."""
    return -(-doc_len // tile)


def la_vector_bits(p: int) -> int:
    """Lower triangle of a PxP tile grid incl. the diagonal: P(P+1)/2 bits (L201-203, L213)."""
    return p * (p + 1) // 2


def la_vector_bytes(p: int) -> int:
    """ceil(P(P+1)/(2*8)) bytes (L213)."""
    return -(-la_vector_bits(p) // 8)


def ca_vector_bits(doc_len: int, tile: int, gran: int) -> int:
    """Paper (gran == tile): one bit per KV page -> P bits (L209, L213).
    BASELINE.json configs (gran == 1): one bit per key token -> L bits (reading A4)."""
    return -(-doc_len // gran)


def ca_vector_bytes(doc_len: int, tile: int, gran: int) -> int:
    return -(-ca_vector_bits(doc_len, tile, gran) // 8)


def sift_storage_bits(n_layers: int, n_heads: int, n_docs: int, p: int) -> int:
    """Unpadded bits for one prompt, page-granular CA (Table 1 reading: per q-head, A7)."""
    return n_layers * n_heads * n_docs * (la_vector_bits(p) + p)


# ------------------------------------------------------------------------------------------
# Bit access ("packed MSB-first, enumerated row-major in the lower triangle")
# ------------------------------------------------------------------------------------------

def get_bit(vec: np.ndarray, n: int) -> int:
    return (int(vec[n >> 3]) >> (7 - (n & 7))) & 1


def la_bit_index(i: int, j: int) -> int:
    """(0,0),(1,0),(1,1),(2,0)...: row i starts after 1+2+...+i = i(i+1)/2 bits."""
    assert 0 <= j <= i
    return i * (i + 1) // 2 + j


def la_tile_bit(vec: np.ndarray, i: int, j: int) -> int:
    return get_bit(vec, la_bit_index(i, j))


def read_bits(vec: np.ndarray, nbits: int) -> np.ndarray:
    """get_bit applied to n = 0..nbits-1 (same formula, element-wise). Padding bits beyond
    nbits are never looked at (reading A6)."""
    n = np.arange(nbits, dtype=np.int64)
    return ((vec[n >> 3].astype(np.int64) >> (7 - (n & 7))) & 1).astype(bool)


# ------------------------------------------------------------------------------------------
# Part 1: the mask
# ------------------------------------------------------------------------------------------

def segment_of(row: int, doc_offsets: Sequence[int]) -> int:
    """Index of the document holding global row `row`; len(doc_offsets)-1 (= D) for the user query."""
    d_total = len(doc_offsets) - 1
    for d in range(d_total):
        if doc_offsets[d] <= row < doc_offsets[d + 1]:
            return d
    return d_total


def expand_mask_rows(doc_offsets: Sequence[int], query_len: int, tile: int, gran: int,
                     la_vecs: Sequence[np.ndarray], ca_vecs: Sequence[np.ndarray],
                     rows: Sequence[int]) -> np.ndarray:
    """bool [len(rows), N] for one (layer, head). la_vecs[d] / ca_vecs[d] are that head's vectors.

    Rule (SURVEY.md 8(c) Part 1):
      1. k > q                     -> False   (causal; L201 "lower triangular ... due to causality")
      2. q in the user query       -> True    (L149 "query submatrix is always recomputed"; L243)
      3. q in doc d, k in doc d':
           d' == d -> LA_d bit of tile (floor(r/T), floor(c/T))          (L201-203)
           d' <  d -> CA_d' bit floor(c/G)                               (L177, L209; A16: every d'<d)
    """
    off = [int(x) for x in doc_offsets]
    n_docs = len(off) - 1
    n = off[-1] + query_len
    cross_allowed = [read_bits(ca_vecs[d], ca_vector_bits(off[d + 1] - off[d], tile, gran)) for d in range(n_docs)]
    out = np.zeros((len(rows), n), dtype=bool)
    for ri, q in enumerate(rows):
        q = int(q)
        d = segment_of(q, off)
        if d == n_docs:                      # user query row: dense causal
            out[ri, : q + 1] = True
            continue
        for dp in range(d):                  # earlier documents: per-key CA bit
            length = off[dp + 1] - off[dp]
            c = np.arange(length)
            out[ri, off[dp]: off[dp + 1]] = cross_allowed[dp][c // gran]
        r = q - off[d]
        i = r // tile
        for j in range(i + 1):               # own document: LA tile bit, then causality
            if la_tile_bit(la_vecs[d], i, j):
                c0 = off[d] + j * tile
                c1 = min(off[d] + (j + 1) * tile, off[d + 1])
                out[ri, c0: min(c1, q + 1)] = True
    return out


# ------------------------------------------------------------------------------------------
# Part 2: masked softmax attention (two-pass, no tiling, no online softmax)
# ------------------------------------------------------------------------------------------

def attention_rows(q_rows: torch.Tensor, k_all: torch.Tensor, v_all: torch.Tensor, mask: np.ndarray,
                   scale: float, dtype: torch.dtype = torch.float32) -> Tuple[torch.Tensor, torch.Tensor]:
    """q_rows [R,d], k_all/v_all [N,d] (any float dtype; widened exactly), mask bool [R,N].
    Returns O [R,d] and LSE [R] in `dtype`.
      s_k = scale * <q, k>;  m = max_k s_k;  l = sum_k exp(s_k - m);
      O = sum_k exp(s_k - m) v_k / l;  LSE = m + ln l   (natural log of scaled logits, A15).
    A row with no allowed key gives O = 0, LSE = -inf (A13)."""
    qf, kf, vf = q_rows.to(dtype), k_all.to(dtype), v_all.to(dtype)
    m_t = torch.from_numpy(np.ascontiguousarray(mask))
    s = (qf @ kf.T) * scale
    s = torch.where(m_t, s, torch.full_like(s, -math.inf))
    mx = s.max(dim=1).values
    empty = ~m_t.any(dim=1)
    mx_safe = torch.where(empty, torch.zeros_like(mx), mx)
    p = torch.exp(s - mx_safe[:, None])          # masked entries: exp(-inf) = 0
    l = p.sum(dim=1)
    o = (p @ vf) / torch.where(empty, torch.ones_like(l), l)[:, None]
    lse = torch.where(empty, torch.full_like(mx, -math.inf), mx_safe + torch.log(torch.where(empty, torch.ones_like(l), l)))
    return o, lse


def kv_head_of(h: int, n_q_heads: int, n_kv_heads: int) -> int:
    """Contiguous GQA groups: kv(h) = floor(h / (Hq/Hkv))  (A8)."""
    return h // (n_q_heads // n_kv_heads)


def sift_attention_rows(q: torch.Tensor, k: torch.Tensor, v: torch.Tensor, head: int,
                        doc_offsets: Sequence[int], query_len: int, tile: int, gran: int,
                        la_vecs: Sequence[np.ndarray], ca_vecs: Sequence[np.ndarray], rows: Sequence[int],
                        scale: Optional[float] = None, dtype: torch.dtype = torch.float32,
                        block: int = 64) -> Tuple[torch.Tensor, torch.Tensor]:
    """SIFT prefill attention for q-head `head` on the given global rows.
    q [N,Hq,d], k,v [N,Hkv,d].  The mask is materialised `block` rows at a time."""
    n, hq, d = q.shape
    hkv = k.shape[1]
    if scale is None:
        scale = 1.0 / math.sqrt(d)           # A14
    kvh = kv_head_of(head, hq, hkv)
    rows = [int(r) for r in rows]
    outs, lses = [], []
    for b0 in range(0, len(rows), block):
        rb = rows[b0: b0 + block]
        mask = expand_mask_rows(doc_offsets, query_len, tile, gran, la_vecs, ca_vecs, rb)
        kmax = max(rb) + 1                   # keys after the last row of the block are causally dead
        o, lse = attention_rows(q[rb, head, :], k[:kmax, kvh, :], v[:kmax, kvh, :], mask[:, :kmax], scale, dtype)
        outs.append(o)
        lses.append(lse)
    if not outs:
        return torch.zeros((0, d), dtype=dtype), torch.zeros((0,), dtype=dtype)
    return torch.cat(outs), torch.cat(lses)


def dense_causal_rows(q: torch.Tensor, k: torch.Tensor, v: torch.Tensor, head: int, rows: Sequence[int],
                      scale: Optional[float] = None, dtype: torch.dtype = torch.float32,
                      block: int = 64) -> Tuple[torch.Tensor, torch.Tensor]:
    """Plain dense causal attention (the "Full Recompute" comparator)."""
    n, hq, d = q.shape
    if scale is None:
        scale = 1.0 / math.sqrt(d)
    kvh = kv_head_of(head, hq, k.shape[1])
    rows = [int(r) for r in rows]
    outs, lses = [], []
    for b0 in range(0, len(rows), block):
        rb = rows[b0: b0 + block]
        kmax = max(rb) + 1
        mask = np.arange(kmax)[None, :] <= np.asarray(rb)[:, None]
        o, lse = attention_rows(q[rb, head, :], k[:kmax, kvh, :], v[:kmax, kvh, :], mask, scale, dtype)
        outs.append(o)
        lses.append(lse)
    return torch.cat(outs), torch.cat(lses)


def brute_force_row(q_row: np.ndarray, k_all: np.ndarray, v_all: np.ndarray, allowed: Sequence[int],
                    scale: float) -> Tuple[np.ndarray, float]:
    """Pure-Python fp64 loops, one row; for tiny pins only."""
    d = len(q_row)
    if len(allowed) == 0:
        return np.zeros(d), -math.inf
    s = []
    for kk in allowed:
        acc = 0.0
        for t in range(d):
            acc += float(q_row[t]) * float(k_all[kk][t])
        s.append(acc * scale)
    m = max(s)
    w = [math.exp(x - m) for x in s]
    l = sum(w)
    o = np.zeros(d)
    for wi, kk in zip(w, allowed):
        for t in range(d):
            o[t] += wi * float(v_all[kk][t])
    return o / l, m + math.log(l)


# ------------------------------------------------------------------------------------------
# Part 3: metadata decode (MD-v1)
# ------------------------------------------------------------------------------------------

def tile_tables(doc_offsets: Sequence[int], query_len: int, tile: int) -> Dict[str, np.ndarray]:
    """Doc-relative tiles (A2): tile (d,i) covers rows off[d]+iT .. ; the query is segment D.
    Returns P[D+1], tile_base[D+2], tile_seg[NT], tile_row0[NT], tile_rows[NT]."""
    off = [int(x) for x in doc_offsets]
    n_docs = len(off) - 1
    seg_len = [off[d + 1] - off[d] for d in range(n_docs)] + [query_len]
    seg_off = off[:-1] + [off[-1]]
    p = [pages(x, tile) for x in seg_len]
    base = [0]
    for x in p:
        base.append(base[-1] + x)
    seg, row0, nrows = [], [], []
    for d in range(n_docs + 1):
        for i in range(p[d]):
            seg.append(d)
            row0.append(seg_off[d] + i * tile)
            nrows.append(min(tile, seg_len[d] - i * tile))
    return {"P": np.asarray(p, np.int32), "tile_base": np.asarray(base, np.int32), "NT": base[-1],
            "tile_seg": np.asarray(seg, np.int32), "tile_row0": np.asarray(row0, np.int32),
            "tile_rows": np.asarray(nrows, np.int32)}


def cross_capacity(doc_offsets: Sequence[int], gran: int) -> int:
    """sum over documents of ceil(L_d / G), rounded up to a multiple of 128 (MD-v1, reading R5: SURVEY.md
    8(c) wrote ceil(off[D]/G), which is the same number for G = 1 but too small for G = tile with ragged documents,
    where every document contributes ceil(L_d / tile) pages)."""
    off = [int(x) for x in doc_offsets]
    n = sum(-(-(off[d + 1] - off[d]) // gran) for d in range(len(off) - 1))
    return -(-n // 128) * 128


def local_capacity(tt: Dict[str, np.ndarray]) -> int:
    """sum_d P_d(P_d+1)/2 over documents + sum over query tiles (global id t) of (t+1)."""
    p, base = tt["P"], tt["tile_base"]
    n_docs = len(p) - 1
    cap = sum(int(p[d]) * (int(p[d]) + 1) // 2 for d in range(n_docs))
    for t in range(int(base[n_docs]), int(base[n_docs + 1])):
        cap += t + 1
    return cap


def decode_metadata(doc_offsets: Sequence[int], query_len: int, tile: int, gran: int,
                    n_layers: int, n_heads: int, la_vec: VecFn, ca_vec: VecFn,
                    layers: Optional[Sequence[int]] = None) -> Dict[str, np.ndarray]:
    """Follows PAPER.md:L241-245: pass 1 counts marked CA and LA bits per (head, M-block)
    (query M-blocks: the number of causal N-blocks, L243); offsets = prefix sums of the counts;
    pass 2 scans CA then LA and writes the indices, offset to global coordinates, at their
    designated offset.  Container MD-v1: the CA entries of a document are a prefix of one
    per-head list (``cross_ptr``), instead of being replicated into every M-block's list;
    ``paper_view`` rebuilds the per-(head, M-block) list of L239.

    cross_idx: G == 1 -> global key row off[d']+c ; G == tile -> global tile id tile_base[d']+b.
    Entries of cross_idx at or beyond cross_ptr[..., D] and of local_idx beyond local_ptr[..., NT]
    are unspecified (-1 here; never compared)."""
    off = [int(x) for x in doc_offsets]
    n_docs = len(off) - 1
    tt = tile_tables(off, query_len, tile)
    nt, base, p = int(tt["NT"]), tt["tile_base"], tt["P"]
    ccap, lcap = cross_capacity(off, gran), local_capacity(tt)
    lay = list(range(n_layers)) if layers is None else list(layers)
    cross_ptr = np.zeros((n_layers, n_heads, n_docs + 1), np.int32)
    cross_idx = np.full((n_layers, n_heads, ccap), -1, np.int32)
    local_cnt = np.zeros((n_layers, n_heads, nt), np.int32)
    local_ptr = np.zeros((n_layers, n_heads, nt + 1), np.int32)
    local_idx = np.full((n_layers, n_heads, max(lcap, 1)), -1, np.int32)
    for l in lay:
        for h in range(n_heads):
            # ---- pass 1: count -------------------------------------------------------
            ca_bits = [read_bits(ca_vec(l, h, d), ca_vector_bits(off[d + 1] - off[d], tile, gran)) for d in range(n_docs)]
            ca_cnt = [int(b.sum()) for b in ca_bits]
            cnt = np.zeros(nt, np.int64)
            for d in range(n_docs):
                lv = la_vec(l, h, d)
                for i in range(int(p[d])):
                    c = 0
                    for j in range(i + 1):
                        c += la_tile_bit(lv, i, j)
                    cnt[int(base[d]) + i] = c
            for t in range(int(base[n_docs]), nt):      # query M-blocks: all causal N-blocks
                cnt[t] = t + 1
            # ---- offsets -------------------------------------------------------------
            cp = np.zeros(n_docs + 1, np.int64)
            for d in range(n_docs):
                cp[d + 1] = cp[d] + ca_cnt[d]
            lp = np.zeros(nt + 1, np.int64)
            for t in range(nt):
                lp[t + 1] = lp[t] + cnt[t]
            # ---- pass 2: fill (CA then LA, global coordinates) --------------------------
            for d in range(n_docs):
                w = int(cp[d])
                for b in np.nonzero(ca_bits[d])[0]:
                    cross_idx[l, h, w] = (off[d] + int(b)) if gran == 1 else (int(base[d]) + int(b))
                    w += 1
                assert w == cp[d + 1]
            for d in range(n_docs):
                lv = la_vec(l, h, d)
                for i in range(int(p[d])):
                    t = int(base[d]) + i
                    w = int(lp[t])
                    for j in range(i + 1):
                        if la_tile_bit(lv, i, j):
                            local_idx[l, h, w] = int(base[d]) + j
                            w += 1
            for t in range(int(base[n_docs]), nt):
                local_idx[l, h, int(lp[t]): int(lp[t + 1])] = np.arange(t + 1)
            cross_ptr[l, h], local_cnt[l, h], local_ptr[l, h] = cp, cnt, lp
    out = dict(tt)
    out.update(cross_ptr=cross_ptr, cross_idx=cross_idx, local_cnt=local_cnt, local_ptr=local_ptr,
               local_idx=local_idx, cross_cap=ccap, local_cap=lcap)
    return out


def paper_view(md: Dict[str, np.ndarray], layer: int, head: int, t: int) -> np.ndarray:
    """sparse_n_indices for (head, M-block t) as the paper lays it out (L239-245): the CA entries
    of all earlier documents, then the LA entries; a query M-block is all causal N-blocks."""
    n_docs = len(md["P"]) - 1
    d = int(md["tile_seg"][t])
    lo, hi = int(md["local_ptr"][layer, head, t]), int(md["local_ptr"][layer, head, t + 1])
    loc = md["local_idx"][layer, head, lo:hi]
    if d == n_docs:
        return loc.copy()
    return np.concatenate([md["cross_idx"][layer, head, : int(md["cross_ptr"][layer, head, d])], loc])


def metadata_to_mask_rows(md: Dict[str, np.ndarray], doc_offsets: Sequence[int], query_len: int, tile: int,
                          gran: int, layer: int, head: int, rows: Sequence[int]) -> np.ndarray:
    """Inverse of decode: rebuild the boolean mask rows from MD-v1 (round-trip pin)."""
    off = [int(x) for x in doc_offsets]
    n_docs = len(off) - 1
    n = off[-1] + query_len
    row0, nrows, seg, base = md["tile_row0"], md["tile_rows"], md["tile_seg"], md["tile_base"]
    out = np.zeros((len(rows), n), bool)
    for ri, q in enumerate(rows):
        q = int(q)
        d = segment_of(q, off)
        seg_start = off[d] if d < n_docs else off[-1]
        t = int(base[d]) + (q - seg_start) // tile
        if d < n_docs:
            for e in md["cross_idx"][layer, head, : int(md["cross_ptr"][layer, head, d])]:
                e = int(e)
                if gran == 1:
                    out[ri, e] = True
                else:
                    out[ri, int(row0[e]): int(row0[e]) + int(nrows[e])] = True
        lo, hi = int(md["local_ptr"][layer, head, t]), int(md["local_ptr"][layer, head, t + 1])
        for e in md["local_idx"][layer, head, lo:hi]:
            e = int(e)
            c0, c1 = int(row0[e]), int(row0[e]) + int(nrows[e])
            out[ri, c0: min(c1, q + 1)] = True
    return out


def marked_pairs(doc_offsets: Sequence[int], query_len: int, tile: int, gran: int,
                 la_vecs: Sequence[np.ndarray], ca_vecs: Sequence[np.ndarray], block: int = 256) -> int:
    """Number of True mask entries of one (layer, head) (A26: element level)."""
    n = int(doc_offsets[-1]) + query_len
    tot = 0
    for r0 in range(0, n, block):
        rows = list(range(r0, min(n, r0 + block)))
        tot += int(expand_mask_rows(doc_offsets, query_len, tile, gran, la_vecs, ca_vecs, rows).sum())
    return tot


# ------------------------------------------------------------------------------------------
# Part 5: several prompts in one call (sec 2 "TTFT gates decode batching", L267 sec 6)
# ------------------------------------------------------------------------------------------
# Plain definition: the prompts are packed back to back on the token axis (prompt p = its documents, then its query);
# a row of prompt p sees keys of prompt p only, by the single-prompt rule of Part 1.  Everything below is a loop over
# prompts around Parts 1-3 plus a shift to batch coordinates.  Container "MD-v1b" (ours, like MD-v1; for one prompt it
# IS MD-v1): segments are numbered in token order (documents and queries alike), documents are numbered in token order,
#   seg_doc[s]   document index of segment s, -1 for a query segment;  seg_first[s]  first segment of s's prompt
#   tile_base[S+1], tile_seg / tile_row0 / tile_rows [NT]               as in MD-v1, batch coordinates
#   cross_ptr[L][H][D+1]  running number of marked keys over the documents in token order, EXCEPT that the list of
#                         every prompt starts at a multiple of 128 (the attention kernel reads whole groups of 128
#                         entries): document d of a prompt whose first document is d0 attends entries
#                         [cross_ptr[d0], cross_ptr[d]); entries between a prompt's end and the next start: unspecified
#   local_*               per global tile; the list of query tile t of a prompt whose first tile is f is f .. t
# A prompt is given as (doc_offsets, query_len) with its own offsets starting at 0; vectors are addressed by the
# document's index in the batch.

Prompt = Tuple[Sequence[int], int]


def batch_layout(prompts: Sequence[Prompt], tile: int) -> Dict[str, list]:
    """row / document / segment / tile base of every prompt, and the segment tables of MD-v1b."""
    row_base, doc_base, seg_base, tile0 = [0], [0], [0], [0]
    seg_doc, seg_first, seg_off = [], [], [0]
    for off, qlen in prompts:
        off = [int(x) for x in off]
        n_docs = len(off) - 1
        tt = tile_tables(off, qlen, tile)
        for d in range(n_docs):
            seg_doc.append(doc_base[-1] + d)
            seg_first.append(seg_base[-1])
            seg_off.append(row_base[-1] + off[d + 1])
        seg_doc.append(-1)
        seg_first.append(seg_base[-1])
        seg_off.append(row_base[-1] + off[-1] + qlen)
        row_base.append(row_base[-1] + off[-1] + qlen)
        doc_base.append(doc_base[-1] + n_docs)
        seg_base.append(seg_base[-1] + n_docs + 1)
        tile0.append(tile0[-1] + int(tt["NT"]))
    return {"row_base": row_base, "doc_base": doc_base, "seg_base": seg_base, "tile0": tile0,
            "seg_doc": seg_doc, "seg_first": seg_first, "seg_off": seg_off}


def prompt_of_row(row: int, row_base: Sequence[int]) -> int:
    for p in range(len(row_base) - 1):
        if row_base[p] <= row < row_base[p + 1]:
            return p
    raise ValueError("row outside the batch")


def expand_mask_rows_batch(prompts: Sequence[Prompt], tile: int, gran: int, la_vecs: Sequence[np.ndarray],
                           ca_vecs: Sequence[np.ndarray], rows: Sequence[int]) -> np.ndarray:
    """bool [len(rows), N_total] for one (layer, head); la_vecs / ca_vecs are indexed by the document's batch index."""
    lay = batch_layout(prompts, tile)
    out = np.zeros((len(rows), lay["row_base"][-1]), dtype=bool)
    for ri, q in enumerate(rows):
        p = prompt_of_row(int(q), lay["row_base"])
        off, qlen = prompts[p]
        b, d0, d1 = lay["row_base"][p], lay["doc_base"][p], lay["doc_base"][p + 1]
        m = expand_mask_rows(off, qlen, tile, gran, la_vecs[d0:d1], ca_vecs[d0:d1], [int(q) - b])
        out[ri, b: b + m.shape[1]] = m[0]
    return out


def decode_metadata_batch(prompts: Sequence[Prompt], tile: int, gran: int, n_layers: int, n_heads: int,
                          la_vec: VecFn, ca_vec: VecFn) -> Dict[str, np.ndarray]:
    """MD-v1b: every prompt decoded on its own (Part 3), then shifted to batch coordinates."""
    lay = batch_layout(prompts, tile)
    n_docs, nt = lay["doc_base"][-1], lay["tile0"][-1]
    parts = []
    for p, (off, qlen) in enumerate(prompts):
        d0 = lay["doc_base"][p]
        parts.append(decode_metadata(off, qlen, tile, gran, n_layers, n_heads,
                                     lambda l, h, d, d0=d0: la_vec(l, h, d0 + d),
                                     lambda l, h, d, d0=d0: ca_vec(l, h, d0 + d)))
    ccap = sum(int(m["cross_cap"]) for m in parts)          # each prompt's list padded to whole groups of 128
    lcap = 0
    for p, m in enumerate(parts):                           # query tile t of a prompt lists its own tiles only
        npd = len(prompts[p][0]) - 1
        lcap += sum(int(x) * (int(x) + 1) // 2 for x in m["P"][:npd])
        lcap += sum(t + 1 for t in range(int(m["tile_base"][npd]), int(m["NT"])))
    cross_ptr = np.zeros((n_layers, n_heads, n_docs + 1), np.int32)
    cross_idx = np.full((n_layers, n_heads, max(ccap, 1)), -1, np.int32)
    local_cnt = np.zeros((n_layers, n_heads, nt), np.int32)
    local_ptr = np.zeros((n_layers, n_heads, nt + 1), np.int32)
    local_idx = np.full((n_layers, n_heads, max(lcap, 1)), -1, np.int32)
    tile_base, tile_seg, tile_row0, tile_rows = [0], [], [], []
    for p, m in enumerate(parts):
        npd = len(prompts[p][0]) - 1
        tile_base += [lay["tile0"][p] + int(x) for x in m["tile_base"][1:npd + 2]]
        tile_seg += [lay["seg_base"][p] + int(x) for x in m["tile_seg"]]
        tile_row0 += [lay["row_base"][p] + int(x) for x in m["tile_row0"]]
        tile_rows += [int(x) for x in m["tile_rows"]]
    for l in range(n_layers):
        for h in range(n_heads):
            cstart, lstart = 0, 0
            for p, m in enumerate(parts):
                npd = len(prompts[p][0]) - 1
                d0, t0, rb = lay["doc_base"][p], lay["tile0"][p], lay["row_base"][p]
                cstart = -(-cstart // 128) * 128                      # a prompt's list starts at a multiple of 128
                if npd > 0:
                    cross_ptr[l, h, d0: d0 + npd + 1] = cstart + m["cross_ptr"][l, h]
                tot = int(m["cross_ptr"][l, h, npd])
                cross_idx[l, h, cstart: cstart + tot] = m["cross_idx"][l, h, :tot] + (rb if gran == 1 else t0)
                cstart += tot
                ntp = int(m["NT"])
                local_cnt[l, h, t0: t0 + ntp] = m["local_cnt"][l, h]
                local_ptr[l, h, t0: t0 + ntp + 1] = lstart + m["local_ptr"][l, h]
                nl = int(m["local_ptr"][l, h, ntp])
                local_idx[l, h, lstart: lstart + nl] = m["local_idx"][l, h, :nl] + t0
                lstart += nl
            cross_ptr[l, h, n_docs] = cstart
    return {"seg_doc": np.asarray(lay["seg_doc"], np.int32), "seg_first": np.asarray(lay["seg_first"], np.int32),
            "tile_base": np.asarray(tile_base, np.int32), "NT": nt, "tile_seg": np.asarray(tile_seg, np.int32),
            "tile_row0": np.asarray(tile_row0, np.int32), "tile_rows": np.asarray(tile_rows, np.int32),
            "cross_ptr": cross_ptr, "cross_idx": cross_idx, "local_cnt": local_cnt, "local_ptr": local_ptr,
            "local_idx": local_idx, "cross_cap": ccap, "local_cap": max(lcap, 1)}


def metadata_batch_to_mask_rows(md: Dict[str, np.ndarray], prompts: Sequence[Prompt], tile: int, gran: int,
                                layer: int, head: int, rows: Sequence[int]) -> np.ndarray:
    """Inverse of MD-v1b, written against the container's own rules (not against Part 3): round-trip pin."""
    lay = batch_layout(prompts, tile)
    seg_off, seg_doc, seg_first = lay["seg_off"], md["seg_doc"], md["seg_first"]
    row0, nrows, base = md["tile_row0"], md["tile_rows"], md["tile_base"]
    out = np.zeros((len(rows), seg_off[-1]), bool)
    for ri, q in enumerate(rows):
        q = int(q)
        s = max(i for i in range(len(seg_off) - 1) if seg_off[i] <= q)
        while seg_off[s + 1] <= q:          # (zero-length segments share a start row)
            s += 1
        t = int(base[s]) + (q - seg_off[s]) // tile
        d = int(seg_doc[s])
        if d >= 0:
            d0 = int(seg_doc[int(seg_first[s])])
            lo, hi = int(md["cross_ptr"][layer, head, d0]), int(md["cross_ptr"][layer, head, d])
            assert lo % 128 == 0
            for e in md["cross_idx"][layer, head, lo:hi]:
                e = int(e)
                if gran == 1:
                    out[ri, e] = True
                else:
                    out[ri, int(row0[e]): int(row0[e]) + int(nrows[e])] = True
        lo, hi = int(md["local_ptr"][layer, head, t]), int(md["local_ptr"][layer, head, t + 1])
        for e in md["local_idx"][layer, head, lo:hi]:
            e = int(e)
            out[ri, int(row0[e]): min(int(row0[e]) + int(nrows[e]), q + 1)] = True
    return out


def sift_attention_rows_batch(q: torch.Tensor, k: torch.Tensor, v: torch.Tensor, head: int, prompts: Sequence[Prompt],
                              tile: int, gran: int, la_vecs: Sequence[np.ndarray], ca_vecs: Sequence[np.ndarray],
                              rows: Sequence[int], scale: Optional[float] = None,
                              dtype: torch.dtype = torch.float32) -> Tuple[torch.Tensor, torch.Tensor]:
    """(O [len(rows), d], LSE [len(rows)]) for rows of the packed batch: every row is computed inside its own prompt
    (slices of Q/K/V and of the vectors handed to Part 2's single-prompt routine)."""
    lay = batch_layout(prompts, tile)
    rows = [int(r) for r in rows]
    o_out = torch.zeros((len(rows), q.shape[2]), dtype=dtype)
    l_out = torch.zeros((len(rows),), dtype=dtype)
    for p, (off, qlen) in enumerate(prompts):
        b, e = lay["row_base"][p], lay["row_base"][p + 1]
        sel = [i for i, r in enumerate(rows) if b <= r < e]
        if not sel:
            continue
        d0, d1 = lay["doc_base"][p], lay["doc_base"][p + 1]
        o, lse = sift_attention_rows(q[b:e], k[b:e], v[b:e], head, off, qlen, tile, gran, la_vecs[d0:d1], ca_vecs[d0:d1],
                                     [rows[i] - b for i in sel], scale=scale, dtype=dtype)
        o_out[sel] = o
        l_out[sel] = lse
    return o_out, l_out


# ------------------------------------------------------------------------------------------
# Part 6: FP8 (e4m3) Q/K/V (sec 2.6 points at FP8/FP4 prefill)
# ------------------------------------------------------------------------------------------
# The paper fixes nothing here.  Definition (reading R7): Q, K, V arrive as OCP e4m3 bytes (1 sign, 4 exponent
# bits with bias 7, 3 mantissa bits; no infinities, S.1111.111 = NaN, largest finite 448) with one fp32 scale per q-head
# for Q and per kv-head for K and V.  The attention is Part 2's on the DEQUANTISED values q_scale[h] * Q8, k_scale[g] * K8,
# v_scale[g] * V8: the oracle decodes the bytes by the format's definition and calls Part 2 unchanged (fp64 on
# request).  What the GPU adds on top (P rounded to e4m3 before P*V) is an approximation the oracle does not imitate;
# its bound is derived in DESIGN.md and written into the parity test.

def e4m3_decode(b: np.ndarray) -> np.ndarray:
    """uint8 -> float64 by the OCP FP8 E4M3 definition: (-1)^s * 2^(e-7) * (1 + m/8) for e > 0, (-1)^s * 2^-6 * m/8
    for e = 0; e = 15, m = 7 is NaN."""
    b = np.asarray(b, np.uint8).astype(np.int64)
    sgn = np.where(b & 0x80, -1.0, 1.0)
    e, m = (b >> 3) & 0xF, b & 0x7
    val = np.where(e > 0, np.ldexp(1.0 + m / 8.0, e - 7), np.ldexp(m / 8.0, -6))
    val = np.where((e == 15) & (m == 7), np.nan, val)
    return sgn * val


def sift_attention_rows_fp8(q8: np.ndarray, k8: np.ndarray, v8: np.ndarray, q_scale: Sequence[float], k_scale: Sequence[float],
                            v_scale: Sequence[float], head: int, doc_offsets: Sequence[int], query_len: int, tile: int,
                            gran: int, la_vecs: Sequence[np.ndarray], ca_vecs: Sequence[np.ndarray], rows: Sequence[int],
                            scale: Optional[float] = None, dtype: torch.dtype = torch.float32) -> Tuple[torch.Tensor, torch.Tensor]:
    """q8 [N,Hq,d], k8, v8 [N,Hkv,d] uint8 (e4m3 bytes).  Dequantise, then Part 2 as it stands."""
    hq, hkv = q8.shape[1], k8.shape[1]
    q = torch.from_numpy(e4m3_decode(q8) * np.asarray(q_scale, np.float64)[None, :, None]).to(dtype)
    k = torch.from_numpy(e4m3_decode(k8) * np.asarray(k_scale, np.float64)[None, :, None]).to(dtype)
    v = torch.from_numpy(e4m3_decode(v8) * np.asarray(v_scale, np.float64)[None, :, None]).to(dtype)
    assert q.shape[1] == hq and k.shape[1] == hkv
    return sift_attention_rows(q, k, v, head, doc_offsets, query_len, tile, gran, la_vecs, ca_vecs, rows, scale=scale, dtype=dtype)


# ------------------------------------------------------------------------------------------
# Convenience for callers holding a workload-like object (duck-typed; no import of the package)
# ------------------------------------------------------------------------------------------

def head_vectors(w, layer: int, head: int) -> Tuple[List[np.ndarray], List[np.ndarray]]:
    n_docs = len(w.shape.doc_lens)
    return ([w.la_vec(layer, head, d) for d in range(n_docs)], [w.ca_vec(layer, head, d) for d in range(n_docs)])


# ------------------------------------------------------------------------------------------
# Part 4: offline metadata generation (sec 4.1, L209 sec 4.2, L223 sec 4.4)
# ------------------------------------------------------------------------------------------
# Plain definition, fp64: the standalone dense causal attention of ONE document gives a probability matrix p[q, k]
# (k <= q).  LA tile (i, j) is marked iff it holds at least one p >= alpha (L201).  CA (reading R6 of DESIGN.md; the
# paper words it per page at L209 and per key token at L185): a key group g (one key at G = 1, T keys at G = tile) is
# marked iff hits(g) > gamma * cells(g), hits = causal cells of its key columns with p >= beta, cells = all causal
# cells of those columns.  Pins (tests/test_oracle_pins.py): q = 0 gives p = 1/(q+1) in closed form; one-hot attention
# gives the diagonal-only LA vector 0xA4 of the paper's enumeration; alpha <= min p marks every tile.

def pack_bits_msb(bits: Sequence[int]) -> np.ndarray:
    """MSB-first packing, padded with zeros to the next byte boundary."""
    out = np.zeros((len(bits) + 7) // 8, dtype=np.uint8)
    for n, b in enumerate(bits):
        if b:
            out[n >> 3] |= 0x80 >> (n & 7)
    return out


def document_probabilities(q_doc: torch.Tensor, k_doc: torch.Tensor, scale: Optional[float] = None) -> np.ndarray:
    """p[q, k] of the dense causal attention of one document and head; q_doc, k_doc [L, d]; fp64; 0 above the diagonal."""
    n, d = q_doc.shape
    if scale is None:
        scale = 1.0 / math.sqrt(d)
    s = (q_doc.to(torch.float64) @ k_doc.to(torch.float64).T) * scale
    causal = torch.tril(torch.ones((n, n), dtype=torch.bool))
    s = torch.where(causal, s, torch.full_like(s, -math.inf))
    p = torch.softmax(s, dim=1)
    return p.numpy()


def encode_from_probabilities(p: np.ndarray, tile: int, gran: int, alpha: float, beta: float, gamma: float
                              ) -> Tuple[np.ndarray, np.ndarray, Dict[str, np.ndarray]]:
    """LA and CA vectors (packed) of one (document, head) from its probability matrix, plus the unpacked decisions
    and their margins (used by the GPU parity test to set aside cells that sit on a threshold)."""
    n = p.shape[0]
    pt = pages(n, tile)
    la_bits, la_max = [], []
    for i in range(pt):
        for j in range(i + 1):
            blk = p[i * tile: min(n, (i + 1) * tile), j * tile: min(n, (j + 1) * tile)]
            if i == j:
                blk = np.tril(blk)                       # cells above the diagonal are not part of the tile's triangle
            mx = float(blk.max())
            la_bits.append(1 if mx >= alpha else 0)
            la_max.append(mx)
    n_groups = -(-n // gran)
    hit = (p >= beta) & np.tril(np.ones((n, n), dtype=bool))
    col_hits = hit.sum(axis=0).astype(np.int64)          # per key column
    ca_bits, hits_g, cells_g = [], [], []
    for g in range(n_groups):
        ks = range(g * gran, min(n, (g + 1) * gran))
        hits = int(sum(int(col_hits[k]) for k in ks))
        cells = int(sum(n - k for k in ks))
        ca_bits.append(1 if hits > gamma * cells else 0)   # "exceeds gamma" (L209), gamma as given
        hits_g.append(hits)
        cells_g.append(cells)
    info = {"la_bits": np.array(la_bits), "la_max": np.array(la_max), "ca_bits": np.array(ca_bits),
            "hits": np.array(hits_g), "cells": np.array(cells_g), "col_hits": col_hits}
    return pack_bits_msb(la_bits), pack_bits_msb(ca_bits), info


def encode_document(q: torch.Tensor, k: torch.Tensor, head: int, tile: int, gran: int, alpha: float = 1e-3,
                    beta: float = 1e-2, gamma: float = 0.1, scale: Optional[float] = None):
    """q [L, Hq, d], k [L, Hkv, d] of one document; returns (la_vec, ca_vec, info) for q-head `head`."""
    kvh = kv_head_of(head, q.shape[1], k.shape[1])
    p = document_probabilities(q[:, head, :], k[:, kvh, :], scale)
    la, ca, info = encode_from_probabilities(p, tile, gran, alpha, beta, gamma)
    info["p"] = p
    return la, ca, info
