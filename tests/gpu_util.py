"""Helpers for the -m gpu parity tests: run the CUDA path through the C-ABI binding, run the oracle on the same
seeded inputs, compare.  Tolerances are BASELINE.json's north_star: attention max-abs 2e-2 / mean-abs 2e-3,
row log-sum-exp 1e-3 (bf16 in, fp32 accumulate); metadata bit-exact."""
import numpy as np
import torch

from oracle import sift_oracle as so
from paper_2606_09441_b200 import api

TOL_MAX, TOL_MEAN, TOL_LSE = 2e-2, 2e-3, 1e-3


def decode_on_gpu(w):
    shape = api.Shape.from_prompt(w.shape)
    la = torch.from_numpy(w.la_blob).cuda()
    ca = torch.from_numpy(w.ca_blob).cuda()
    md = api.sift_decode_metadata(shape, la, w.la_doc_off, ca, w.ca_doc_off)
    torch.cuda.synchronize()
    return shape, md


def oracle_md(w, layers=None):
    sh = w.shape
    return so.decode_metadata(sh.doc_offsets, sh.query_len, sh.tile, sh.cross_gran, sh.n_layers, sh.n_q_heads,
                              w.la_vec, w.ca_vec, layers=layers)


def assert_metadata_equal(w, shape, md, layers=None):
    v = {k: t.cpu().numpy() for k, t in api.metadata_views(shape, md).items()}
    ref = oracle_md(w, layers)
    for k in ("tile_base", "tile_seg", "tile_row0", "tile_rows"):
        assert np.array_equal(v[k], ref[k]), k
    lay = range(w.shape.n_layers) if layers is None else layers
    for l in lay:
        for k in ("cross_ptr", "local_cnt", "local_ptr"):
            assert np.array_equal(v[k][l], ref[k][l]), (k, l)
        for h in range(w.shape.n_q_heads):
            nc = int(ref["cross_ptr"][l, h, -1])
            assert np.array_equal(v["cross_idx"][l, h, :nc], ref["cross_idx"][l, h, :nc]), ("cross_idx", l, h)
            pad = v["cross_idx"][l, h, nc:-(-nc // 128) * 128]
            assert np.all((pad >= 0) & (pad < w.shape.n_tokens)), "pad entries must be valid rows"
            nl = int(ref["local_ptr"][l, h, -1])
            assert np.array_equal(v["local_idx"][l, h, :nl], ref["local_idx"][l, h, :nl]), ("local_idx", l, h)
    # scheduler (private): a permutation of all (head, M-block) items ...
    lay_c = api.sift_metadata_layout(shape)
    for l in lay:
        s = np.sort(v["sched"][l])
        exp = np.sort(np.array([(h << 20) | mb for h in range(w.shape.n_q_heads) for mb in range(lay_c.n_mblocks)]))
        assert np.array_equal(s, exp)
        assert_schedule_order(w, v["sched"][l], ref, l)
    return v, ref


def assert_schedule_order(w, sched, ref, layer):
    """... in the order the persistent attention grid relies on: groups of kv
    heads one after the other (their K/V fit the L2), and inside a group the cost of the items never increases.  The cost
    is recomputed here from the ORACLE's counts: steps of an M-block (2 consecutive tiles of one segment) = per document
    tile ceil(cross entries of its document / 128) (G = 1) or the number of listed pages (G = tile), plus its local
    count; per user-query tile ceil((row0 + rows) / 128)."""
    sh = w.shape
    D, T, G, Hq, Hkv = sh.n_docs, sh.tile, sh.cross_gran, sh.n_q_heads, sh.n_kv_heads
    base, seg, row0, rows = ref["tile_base"], ref["tile_seg"], ref["tile_row0"], ref["tile_rows"]
    mb_tiles = []                                     # M-block -> its tiles
    for d in range(D + 1):
        for t0 in range(int(base[d]), int(base[d + 1]), 2):
            mb_tiles.append(list(range(t0, min(t0 + 2, int(base[d + 1])))))
    per_head = sh.n_tokens * sh.head_dim * 2 * 2
    kv_per_group = int(min(max((72 << 20) // max(per_head, 1), 1), Hkv))
    groups = -(-Hkv // kv_per_group)
    cap = 4096 // groups - 1                          # costs are bucketed up to this value
    last_g, last_c = -1, None
    for code in sched:
        h, mb = int(code) >> 20, int(code) & 0xFFFFF
        c = 0
        for t in mb_tiles[mb]:
            d = int(seg[t])
            if d < D:
                cp = int(ref["cross_ptr"][layer, h, d])
                c += (-(-cp // 128) if G == 1 else cp) + int(ref["local_cnt"][layer, h, t])
            else:
                c += -(-(int(row0[t]) + int(rows[t])) // 128)
        c = min(c, cap)
        g = (h // (Hq // Hkv)) // kv_per_group
        assert g >= last_g, ("kv-head groups out of order", h, mb)
        if g != last_g:
            last_g, last_c = g, None
        assert last_c is None or c <= last_c, ("cost increases inside a kv-head group", h, mb, c, last_c)
        last_c = c


def attention_errors(w, layer, o_gpu, lse_gpu, heads, rows, dense=False):
    """Compare sampled (head, row) outputs with the oracle. Returns (max_abs, mean_abs, lse_err)."""
    sh = w.shape
    q, k, v = w.qkv(layer)
    o_gpu = o_gpu.float().cpu()
    lse_gpu = lse_gpu.cpu()
    mx, sm, cnt, le = 0.0, 0.0, 0, 0.0
    rows = [int(r) for r in rows]
    for h in heads:
        if dense:
            o, lse = so.dense_causal_rows(q, k, v, h, rows)
        else:
            la, ca = so.head_vectors(w, layer, h)
            o, lse = so.sift_attention_rows(q, k, v, h, sh.doc_offsets, sh.query_len, sh.tile, sh.cross_gran, la, ca, rows)
        d = (o_gpu[rows, h, :] - o).abs()
        mx = max(mx, float(d.max()))
        sm += float(d.sum())
        cnt += d.numel()
        lg = lse_gpu[h, rows]
        both_inf = torch.isinf(lse) & torch.isinf(lg) & (lse < 0) & (lg < 0)
        ld = torch.where(both_inf, torch.zeros_like(lse), (lg - lse).abs())
        le = max(le, float(ld.max()))
    return mx, sm / max(cnt, 1), le


def run_sift(w, layer=0):
    shape, md = decode_on_gpu(w)
    q, k, v = (t.cuda() for t in w.qkv(layer))
    o, lse = api.sift_prefill_attention(shape, layer, q, k, v, md)
    torch.cuda.synchronize()
    return shape, md, o, lse


def sample_rows(w, n_per_seg=6, seed=0):
    """Rows that hit: first/last rows of tiles, ragged tails, doc boundaries, query rows."""
    sh = w.shape
    off = [int(x) for x in sh.doc_offsets]
    n = sh.n_tokens
    r = np.random.default_rng(seed)
    rows = {0, n - 1, off[-1], max(off[-1] - 1, 0)}
    for d in range(sh.n_docs):
        a, b = off[d], off[d + 1]
        rows |= {a, b - 1, min(a + sh.tile, b - 1), min(a + sh.tile - 1, b - 1)}
        rows |= {int(x) for x in r.integers(a, b, n_per_seg)}
    if sh.query_len:
        rows |= {int(x) for x in r.integers(off[-1], n, n_per_seg)}
    return sorted(x for x in rows if 0 <= x < n)
