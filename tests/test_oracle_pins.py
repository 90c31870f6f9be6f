"""Pins for oracle/sift_oracle.py against what the paper and the mathematics fix (no GPU).

Each test names the passage of /root/reference/PAPER.md (cited as PAPER.md:L<line>) it pins.
"""
import math
import os

import numpy as np
import pytest
import torch

from oracle import sift_oracle as so
from paper_2606_09441_b200 import workload as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- bit order / sizes

def test_la_enumeration_order_L203():
    # PAPER.md:L203 prints the order (0,0),(1,0),(1,1),(2,0)...
    printed = [(0, 0), (1, 0), (1, 1), (2, 0)]
    assert [so.la_bit_index(i, j) for (i, j) in printed] == [0, 1, 2, 3]
    # row-major over the whole lower triangle is a bijection onto 0..P(P+1)/2-1
    p = 7
    seen = [so.la_bit_index(i, j) for i in range(p) for j in range(i + 1)]
    assert seen == list(range(so.la_vector_bits(p)))


def test_la_msb_first_hand_bytes_L203():
    # P=3, diagonal tiles only: bits (0,0)=1,(1,0)=0,(1,1)=1,(2,0)=0,(2,1)=0,(2,2)=1 -> 1010 01xx, MSB first
    vec = np.array([0xA4], np.uint8)
    got = [[so.la_tile_bit(vec, i, j) for j in range(i + 1)] for i in range(3)]
    assert got == [[1], [0, 1], [0, 0, 1]]
    # P=8 all ones: 36 bits -> FF FF FF FF F0 (padded to the byte boundary, L203)
    vec = np.array([0xFF, 0xFF, 0xFF, 0xFF, 0xF0], np.uint8)
    assert all(so.la_tile_bit(vec, i, j) == 1 for i in range(8) for j in range(i + 1))
    assert so.la_vector_bytes(8) == 5
    # first bit of the stream is the MSB of byte 0
    assert so.get_bit(np.array([0x80], np.uint8), 0) == 1 and so.get_bit(np.array([0x01], np.uint8), 7) == 1
    assert so.get_bit(np.array([0x00, 0x40], np.uint8), 9) == 1


def test_size_example_L213():
    # "assuming P ~ 8 pages per document, the LA bit vector stores 36 bits and the CA bit vector stores 8 bits"
    assert so.la_vector_bits(8) == 36
    assert so.ca_vector_bits(1024, 128, 128) == 8
    for p in range(1, 40):
        assert so.la_vector_bytes(p) == math.ceil(p * (p + 1) / 16)
        assert so.ca_vector_bytes(p * 128, 128, 128) == math.ceil(p / 8)
    assert so.pages(2000, 128) == 16 and so.pages(2048, 128) == 16 and so.pages(2049, 128) == 17


def _fmt(nbytes, unit):
    return nbytes / 1024.0 if unit == "KB" else nbytes / (1024.0 * 1024.0)


def test_table1_all_cells_L311():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "table1.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 9
    for model, layers, heads, ctx, printed, unit in rows:
        n_docs = int(ctx) // 1024
        nbytes = so.sift_storage_bits(int(layers), int(heads), n_docs, 8) / 8.0
        val = _fmt(nbytes, unit)
        digits = 1 if "." in printed else 0
        # the table prints truncated-or-rounded values; accept either
        assert (round(val, digits) == float(printed)) or (math.floor(val * 10 ** digits) / 10 ** digits == float(printed)), \
            (model, ctx, val, printed)


def test_table1_ratios_and_breakeven_L307():
    # KV bytes per token = layers * kv_heads * head_dim * 2 (K,V) * 2 B
    kv = {"llama": 32 * 8 * 128 * 4, "qwen": 94 * 4 * 128 * 4, "minimax": 62 * 8 * 128 * 4}
    sift_per_doc = {"llama": 32 * 32 * 44 / 8, "qwen": 94 * 64 * 44 / 8, "minimax": 62 * 48 * 44 / 8}
    printed = {"llama": 23831, "qwen": 5958, "minimax": 15888}
    for m in kv:
        ratio = kv[m] * 1024 / sift_per_doc[m]
        assert int(ratio) == printed[m] or round(ratio) == printed[m], (m, ratio)
    # L307: sizes become equal at 33.6M tokens per doc (Llama 8B): P(P+1)/2 + P bits * 32*32 = 131072 B * 128 P
    p = 2 * 131072 * 8 * 128 // (32 * 32)  # ~ solve P/2 * heads*layers = 8*kv*T
    assert abs(p * 128 / 1e6 - 33.6) < 0.1
    lhs = so.sift_storage_bits(32, 32, 1, p) / 8
    rhs = kv["llama"] * p * 128
    assert abs(lhs / rhs - 1.0) < 1e-3


# ---------------------------------------------------------------- mask invariants

def _vecs(w, layer=0, head=0):
    return so.head_vectors(w, layer, head)


def _mask(w, layer=0, head=0, rows=None):
    sh = w.shape
    la, ca = _vecs(w, layer, head)
    rows = list(range(sh.n_tokens)) if rows is None else rows
    return so.expand_mask_rows(sh.doc_offsets, sh.query_len, sh.tile, sh.cross_gran, la, ca, rows)


@pytest.mark.parametrize("gran", [1, 32])
def test_all_ones_is_dense_causal(gran):
    # north_star; PAPER.md:L201-209 by construction
    w = wl.custom("ones", doc_lens=(100, 64, 33), query_len=17, tile=32, cross_gran=gran, p_loc=1.1, p_cross=1.1)
    n = w.shape.n_tokens
    m = _mask(w)
    assert np.array_equal(m, np.tril(np.ones((n, n), bool)))


def test_cross_cleared_is_block_diagonal_plus_query():
    # PAPER.md:L103 Fig 4a pattern; L147-149
    w = wl.custom("nocross", doc_lens=(100, 64, 33), query_len=17, tile=32, p_loc=0.5, p_cross=-1.0,
                  garbage_padding=True)
    sh = w.shape
    off = sh.doc_offsets
    m = _mask(w)
    for d in range(sh.n_docs):
        blk = m[off[d]:off[d + 1]]
        assert not blk[:, :off[d]].any() and not blk[:, off[d + 1]:].any()
        assert np.array_equal(np.diag(blk[:, off[d]:off[d + 1]]), np.ones(off[d + 1] - off[d], bool))  # diag tiles set
    qrows = m[off[-1]:]
    n = sh.n_tokens
    assert np.array_equal(qrows, np.tril(np.ones((n, n), bool))[off[-1]:])


def test_mask_brute_force_definition():
    # independent per-element restatement of SURVEY 8(c) Part 1 with explicit bit arithmetic
    w = wl.custom("bf", n_q_heads=2, doc_lens=(70, 129, 40), query_len=9, tile=32, p_loc=0.4, p_cross=0.3, seed=5)
    sh = w.shape
    off = [int(x) for x in sh.doc_offsets]
    for head in range(2):
        la, ca = _vecs(w, 0, head)
        m = _mask(w, 0, head)
        n = sh.n_tokens
        for q in range(0, n, 3):
            for k in range(n):
                if k > q:
                    exp = False
                elif q >= off[-1]:
                    exp = True
                else:
                    d = max(i for i in range(sh.n_docs) if off[i] <= q)
                    if k >= off[d]:
                        i, j = (q - off[d]) // 32, (k - off[d]) // 32
                        nbit = i * (i + 1) // 2 + j
                        exp = bool(la[d][nbit // 8] & (0x80 >> (nbit % 8)))
                    else:
                        dp = max(i for i in range(sh.n_docs) if off[i] <= k)
                        c = k - off[dp]
                        exp = bool(ca[dp][c // 8] & (0x80 >> (c % 8)))
                assert m[q, k] == exp, (q, k)


def test_padding_bits_ignored_A6():
    a = wl.custom("pad", doc_lens=(70, 45), query_len=5, tile=32, seed=3, garbage_padding=True)
    b = wl.custom("pad", doc_lens=(70, 45), query_len=5, tile=32, seed=3, garbage_padding=False)
    assert not np.array_equal(a.ca_blob, b.ca_blob) or not np.array_equal(a.la_blob, b.la_blob)
    assert np.array_equal(_mask(a), _mask(b))


def test_doc0_ignores_ca_and_query_ignores_both():
    w = wl.custom("q", doc_lens=(64, 64), query_len=16, tile=32, p_loc=0.3, p_cross=0.5, seed=11)
    m1 = _mask(w)
    w2 = wl.custom("q", doc_lens=(64, 64), query_len=16, tile=32, p_loc=0.9, p_cross=0.1, seed=12)
    m2 = _mask(w2)
    assert np.array_equal(m1[128:], m2[128:])          # query rows: dense causal regardless of vectors
    assert not m1[:64, 64:].any()


def test_reorder_translates_local_blocks_L159():
    w = wl.custom("ro", doc_lens=(96, 64, 40), query_len=8, tile=32, p_loc=0.4, p_cross=0.3, seed=21)
    perm = [2, 0, 1]
    w2 = w.reorder(perm)
    m, m2 = _mask(w), _mask(w2)
    off, off2 = w.shape.doc_offsets, w2.shape.doc_offsets
    for p2, p1 in enumerate(perm):
        a = m[off[p1]:off[p1 + 1], off[p1]:off[p1 + 1]]
        b = m2[off2[p2]:off2[p2 + 1], off2[p2]:off2[p2 + 1]]
        assert np.array_equal(a, b)
    # cross columns of a doc are the same key set wherever it stands (seen from the last doc)
    last_row_new = off2[3] - 1      # a row of doc at position 2 (old doc 1)
    last_row_old_doc2_cols = m2[last_row_new, off2[0]:off2[1]]   # keys of old doc 2 seen from old doc 1
    assert np.array_equal(last_row_old_doc2_cols, so.read_bits(w.ca_vec(0, 0, 2), 40))


# ---------------------------------------------------------------- attention numerics

def _attn(w, head, rows, dtype=torch.float64, layer=0):
    sh = w.shape
    q, k, v = w.qkv(layer)
    la, ca = _vecs(w, layer, head)
    return so.sift_attention_rows(q, k, v, head, sh.doc_offsets, sh.query_len, sh.tile, sh.cross_gran,
                                  la, ca, rows, dtype=dtype), (q, k, v)


def test_attention_brute_force_fp64_tiny():
    w = wl.custom("bfa", n_q_heads=4, n_kv_heads=2, head_dim=16, doc_lens=(24, 19), query_len=6, tile=8,
                  p_loc=0.4, p_cross=0.3, seed=7)
    sh = w.shape
    n = sh.n_tokens
    for head in (0, 3):
        (o, lse), (q, k, v) = _attn(w, head, list(range(n)))
        m = _mask(w, 0, head)
        kvh = head // 2                                  # A8 contiguous GQA groups
        qn, kn, vn = q[:, head].double().numpy(), k[:, kvh].double().numpy(), v[:, kvh].double().numpy()
        for r in range(n):
            allowed = [int(x) for x in np.nonzero(m[r])[0]]
            ob, lb = so.brute_force_row(qn[r], kn, vn, allowed, 1.0 / math.sqrt(16))
            assert np.allclose(o[r].numpy(), ob, atol=1e-12)
            assert abs(float(lse[r]) - lb) < 1e-12


def test_all_ones_equals_torch_sdpa_causal():
    # library special case: dense causal attention
    w = wl.custom("sdpa", n_q_heads=2, n_kv_heads=1, head_dim=32, doc_lens=(40, 33), query_len=11, tile=16,
                  p_loc=1.1, p_cross=1.1, seed=9)
    n = w.shape.n_tokens
    (o, lse), (q, k, v) = _attn(w, 1, list(range(n)), dtype=torch.float32)
    ref = torch.nn.functional.scaled_dot_product_attention(
        q[:, 1].float()[None, None], k[:, 0].float()[None, None], v[:, 0].float()[None, None], is_causal=True)[0, 0]
    assert torch.allclose(o, ref, atol=2e-6)
    od, lsed = so.dense_causal_rows(q, k, v, 1, list(range(n)), dtype=torch.float32)
    assert torch.allclose(o, od, atol=1e-6) and torch.allclose(lse, lsed, atol=1e-6)


def test_doc0_rows_equal_standalone_doc0_and_prefix_stability():
    w = wl.custom("pre", n_q_heads=2, head_dim=16, doc_lens=(48, 40, 24), query_len=8, tile=16, seed=13)
    (o, lse), (q, k, v) = _attn(w, 0, list(range(w.shape.n_tokens)))
    # a prompt holding only doc 0 (+ query) gives the same doc-0 rows: appending docs leaves earlier rows unchanged
    w0 = wl.custom("pre", n_q_heads=2, head_dim=16, doc_lens=(48,), query_len=8, tile=16, seed=13)
    assert np.array_equal(w0.la_vec(0, 0, 0), w.la_vec(0, 0, 0))
    (o0, lse0), _ = _attn(w0, 0, list(range(48)))
    assert torch.allclose(o[:48], o0, atol=1e-13) and torch.allclose(lse[:48], lse0, atol=1e-13)


def test_lse_merge_identity_and_weights_sum_to_one():
    w = wl.custom("lse", n_q_heads=1, head_dim=16, doc_lens=(32, 32), query_len=4, tile=16, p_cross=0.5, seed=17)
    sh = w.shape
    q, k, v = w.qkv(0)
    rows = list(range(32, 64))
    m = _mask(w, rows=rows)
    sc = 0.25
    o, lse = so.attention_rows(q[rows, 0], k[:, 0], v[:, 0], m, sc, torch.float64)
    mc, ml = m.copy(), m.copy()
    mc[:, 32:] = False
    ml[:, :32] = False
    oc, lc = so.attention_rows(q[rows, 0], k[:, 0], v[:, 0], mc, sc, torch.float64)
    ol, ll = so.attention_rows(q[rows, 0], k[:, 0], v[:, 0], ml, sc, torch.float64)
    assert torch.allclose(lse, torch.logaddexp(lc, ll), atol=1e-12)
    wc, wl_ = torch.exp(lc - lse), torch.exp(ll - lse)
    assert torch.allclose(wc + wl_, torch.ones_like(wc), atol=1e-12)
    assert torch.allclose(o, wc[:, None] * oc + wl_[:, None] * ol, atol=1e-12)
    # V = ones -> O = ones (softmax weights sum to 1)
    o1, _ = so.attention_rows(q[rows, 0], k[:, 0], torch.ones_like(v[:, 0]), m, sc, torch.float64)
    assert torch.allclose(o1, torch.ones_like(o1), atol=1e-12)


def test_empty_row_convention_A13():
    w = wl.custom("empty", n_q_heads=1, head_dim=16, doc_lens=(32,), query_len=4, tile=16, p_loc=-1.0,
                  p_cross=-1.0, diag_set=False, garbage_padding=False)
    (o, lse), _ = _attn(w, 0, [0, 5, 31, 33])
    assert torch.all(o[:3] == 0) and torch.all(torch.isinf(lse[:3])) and torch.all(lse[:3] < 0)
    assert torch.isfinite(lse[3])


# ---------------------------------------------------------------- metadata (MD-v1)

def _md(w, **kw):
    sh = w.shape
    return so.decode_metadata(sh.doc_offsets, sh.query_len, sh.tile, sh.cross_gran, sh.n_layers, sh.n_q_heads,
                              w.la_vec, w.ca_vec, **kw)


@pytest.mark.parametrize("gran", [1, 16])
def test_metadata_round_trip_reproduces_mask(gran):
    w = wl.custom("rt", n_layers=2, n_q_heads=3, n_kv_heads=1, doc_lens=(70, 33, 64, 17), query_len=21, tile=16,
                  cross_gran=gran, p_loc=0.35, p_cross=0.3, seed=23)
    sh = w.shape
    md = _md(w)
    rows = list(range(sh.n_tokens))
    for l in range(2):
        for h in range(3):
            la, ca = so.head_vectors(w, l, h)
            m = so.expand_mask_rows(sh.doc_offsets, sh.query_len, sh.tile, gran, la, ca, rows)
            m2 = so.metadata_to_mask_rows(md, sh.doc_offsets, sh.query_len, sh.tile, gran, l, h, rows)
            assert np.array_equal(m, m2)


def test_metadata_structure_L243_L245():
    w = wl.custom("st", n_q_heads=2, doc_lens=(100, 64, 50), query_len=40, tile=32, p_loc=0.4, p_cross=0.25, seed=29)
    sh = w.shape
    md = _md(w)
    off = sh.doc_offsets
    nt, base = md["NT"], md["tile_base"]
    assert list(md["P"]) == [4, 2, 2, 2] and nt == 10
    for h in range(2):
        cp, lp, cnt = md["cross_ptr"][0, h], md["local_ptr"][0, h], md["local_cnt"][0, h]
        assert cp[0] == 0 and np.all(np.diff(cp) >= 0)
        for d in range(3):                               # counts = number of valid set bits
            assert cp[d + 1] - cp[d] == so.read_bits(w.ca_vec(0, h, d), sh.doc_lens[d]).sum()
            seg = md["cross_idx"][0, h, cp[d]:cp[d + 1]]
            assert np.all(np.diff(seg) > 0) and (len(seg) == 0 or (seg[0] >= off[d] and seg[-1] < off[d + 1]))
        assert np.array_equal(np.diff(lp), cnt) and lp[0] == 0
        for t in range(nt):
            lst = md["local_idx"][0, h, lp[t]:lp[t + 1]]
            assert np.all(np.diff(lst) > 0)
            if t >= base[3]:                             # query M-block: all causal N-blocks (L243)
                assert cnt[t] == t + 1 and np.array_equal(lst, np.arange(t + 1))
            else:
                d = md["tile_seg"][t]
                assert np.all(lst >= base[d]) and np.all(lst <= t) and lst[-1] == t   # diagonal set
        # paper-faithful list: CA entries then LA entries (L245)
        t = int(base[2]) + 1
        pv = so.paper_view(md, 0, h, t)
        assert np.array_equal(pv[:cp[2]], md["cross_idx"][0, h, :cp[2]])
        assert np.array_equal(pv[cp[2]:], md["local_idx"][0, h, lp[t]:lp[t + 1]])


def test_metadata_hand_example():
    # one doc of 3 tiles with LA = 0xA4 (diag only), second doc 2 tiles all ones; CA doc0 = 0b10010000 over 5 keys... G=1
    sh = wl.PromptShape(1, 1, 1, 16, (12, 8), 4, tile=4, cross_gran=1)
    la = [np.array([0xA4], np.uint8), np.array([0xE0], np.uint8)]
    ca = [np.array([0x90, 0x10], np.uint8), np.array([0xFF], np.uint8)]
    md = so.decode_metadata(sh.doc_offsets, 4, 4, 1, 1, 1, lambda l, h, d: la[d], lambda l, h, d: ca[d])
    assert list(md["cross_ptr"][0, 0]) == [0, 3, 11]
    assert list(md["cross_idx"][0, 0, :11]) == [0, 3, 11, 12, 13, 14, 15, 16, 17, 18, 19]
    assert list(md["local_cnt"][0, 0]) == [1, 1, 1, 1, 2, 6]
    assert list(md["local_idx"][0, 0, :12]) == [0, 1, 2, 3, 3, 4, 0, 1, 2, 3, 4, 5]


def test_metadata_local_lists_invariant_under_reorder():
    w = wl.custom("ro2", doc_lens=(96, 64, 40), query_len=8, tile=32, p_loc=0.4, p_cross=0.3, seed=31)
    perm = [1, 2, 0]
    w2 = w.reorder(perm)
    a, b = _md(w), _md(w2)
    for p2, p1 in enumerate(perm):
        for i in range(int(a["P"][p1])):
            t1, t2 = int(a["tile_base"][p1]) + i, int(b["tile_base"][p2]) + i
            l1 = a["local_idx"][0, 0, a["local_ptr"][0, 0, t1]:a["local_ptr"][0, 0, t1 + 1]] - a["tile_base"][p1]
            l2 = b["local_idx"][0, 0, b["local_ptr"][0, 0, t2]:b["local_ptr"][0, 0, t2 + 1]] - b["tile_base"][p2]
            assert np.array_equal(l1, l2)


def test_marked_pairs_counts():
    w = wl.custom("mp", doc_lens=(50, 30), query_len=10, tile=16, p_loc=1.1, p_cross=1.1)
    la, ca = so.head_vectors(w, 0, 0)
    n = 90
    assert so.marked_pairs(w.shape.doc_offsets, 10, 16, 1, la, ca) == n * (n + 1) // 2


# ------------------------------------------------------------------ Part 4: offline metadata generation (encoder)

def test_encoder_uniform_attention_closed_form():
    """q = 0 => p[q, k] = 1/(q+1) for k <= q.  LA tile (i, j) holds max p = 1/(i*T+1), so it is marked iff
    i*T + 1 <= 1/alpha; key k is hit by rows k .. floor(1/beta)-1, so hits(k) = max(0, min(L, floor(1/beta)) - k)
    and its bit is hits > gamma * (L - k)."""
    n, t, d = 40, 8, 16
    q = torch.zeros((n, 1, d), dtype=torch.bfloat16)
    k = torch.randn((n, 1, d), generator=torch.Generator().manual_seed(1)).to(torch.bfloat16)
    alpha, beta, gamma = 1.0 / 17.5, 1.0 / 12.5, 0.25
    la, ca, info = so.encode_document(q, k, 0, t, 1, alpha, beta, gamma)
    pt = 5
    exp_la = [1 if i * t + 1 <= 17 else 0 for i in range(pt) for j in range(i + 1)]
    assert list(info["la_bits"]) == exp_la
    assert np.array_equal(la, so.pack_bits_msb(exp_la)) and len(la) == so.la_vector_bytes(pt)
    exp_hits = [max(0, 12 - kk) for kk in range(n)]
    assert list(info["hits"]) == exp_hits
    exp_ca = [1 if exp_hits[kk] > 0.25 * (n - kk) else 0 for kk in range(n)]
    assert list(info["ca_bits"]) == exp_ca and np.array_equal(ca, so.pack_bits_msb(exp_ca))
    # page-granular: the same hits and cells summed over the T keys of a page
    la2, ca2, info2 = so.encode_document(q, k, 0, t, t, alpha, beta, gamma)
    exp_pg = []
    for g in range(pt):
        hits = sum(exp_hits[g * t:(g + 1) * t]); cells = sum(n - kk for kk in range(g * t, (g + 1) * t))
        exp_pg.append(1 if hits > 0.25 * cells else 0)
    assert list(info2["ca_bits"]) == exp_pg and len(ca2) == so.ca_vector_bytes(n, t, t) and np.array_equal(la2, la)


def test_encoder_one_hot_attention_gives_diagonal_A4():
    """Every row attends (almost) only to itself: only diagonal tiles hold a probability >= alpha, which for P = 3 is
    the byte 0xA4 of the enumeration printed at PAPER.md:L203; each key is hit by exactly one row (itself)."""
    n, t, d = 12, 4, 16
    e = torch.eye(n, d) * 40.0                 # logits 40*40/4 = 400 on the diagonal, 0 elsewhere
    q = e.reshape(n, 1, d).to(torch.bfloat16)
    k = e.reshape(n, 1, d).to(torch.bfloat16)
    la, ca, info = so.encode_document(q, k, 0, t, 1, 1e-3, 1e-2, 0.1)
    assert bytes(la) == bytes([0xA4])
    assert list(info["hits"]) == [1] * n
    assert list(info["ca_bits"]) == [1 if 1 > float(np.float32(0.1)) * (n - kk) else 0 for kk in range(n)]   # the last 9 keys


def test_encoder_thresholds_monotone_and_extremes():
    """alpha below every causal probability marks all tiles (FF..-style all-ones vector); alpha > 1 marks none; raising
    alpha / beta never sets a bit that was clear."""
    n, t, d = 50, 16, 32
    g = torch.Generator().manual_seed(3)
    q = torch.randn((n, 2, d), generator=g).to(torch.bfloat16)
    k = torch.randn((n, 1, d), generator=g).to(torch.bfloat16)
    _, _, info = so.encode_document(q, k, 1, t, 1, 1e-30, 1e-30, 0.0)
    assert info["la_bits"].all() and info["ca_bits"].all()
    _, _, info = so.encode_document(q, k, 1, t, 1, 1.5, 1.5, 0.0)
    assert not info["la_bits"].any() and not info["ca_bits"].any()
    prev_la, prev_ca = None, None
    for a in (1e-4, 1e-3, 1e-2, 1e-1):
        _, _, info = so.encode_document(q, k, 1, t, 1, a, a, 0.1)
        if prev_la is not None:
            assert (info["la_bits"] <= prev_la).all() and (info["ca_bits"] <= prev_ca).all()
        prev_la, prev_ca = info["la_bits"], info["ca_bits"]
    # rows sum to one and the first row is the single cell p[0, 0] = 1
    assert np.allclose(info["p"].sum(axis=1), 1.0) and info["p"][0, 0] == 1.0


# ---------------------------------------------------------------- several prompts in one call

def _small_batch(gran=1, tile=64):
    kw = dict(n_layers=1, n_q_heads=2, n_kv_heads=1, head_dim=64, tile=tile, cross_gran=gran)
    a = wl.custom("ba", doc_lens=(130, 70, 200), query_len=40, p_loc=0.5, p_cross=0.3, seed=11, **kw)
    b = wl.custom("bb", doc_lens=(), query_len=90, seed=12, **kw)                      # a prompt without documents
    c = wl.custom("bc", doc_lens=(64, 333), query_len=1, p_loc=0.4, p_cross=0.5, seed=13, **kw)
    return wl.make_batch("b3", [a, b, c])


def test_batch_of_one_is_md_v1():
    """PAPER.md:L267 (single-request TTFT) is the one-prompt case: MD-v1b of one prompt IS MD-v1."""
    w = wl.custom("one", n_layers=2, n_q_heads=2, doc_lens=(100, 260, 64), query_len=70, tile=64, seed=5)
    sh = w.shape
    single = so.decode_metadata(sh.doc_offsets, sh.query_len, sh.tile, sh.cross_gran, sh.n_layers, sh.n_q_heads, w.la_vec, w.ca_vec)
    b = wl.make_batch("one-b", [w])
    batch = so.decode_metadata_batch(b.prompts, sh.tile, sh.cross_gran, sh.n_layers, sh.n_q_heads, b.la_vec, b.ca_vec)
    for k in ("tile_base", "tile_seg", "tile_row0", "tile_rows", "cross_ptr", "local_cnt", "local_ptr"):
        assert np.array_equal(single[k], batch[k]), k
    assert batch["cross_cap"] == single["cross_cap"] and batch["local_cap"] == single["local_cap"]
    for l in range(sh.n_layers):
        for h in range(sh.n_q_heads):
            nc, nl = int(single["cross_ptr"][l, h, -1]), int(single["local_ptr"][l, h, -1])
            assert np.array_equal(single["cross_idx"][l, h, :nc], batch["cross_idx"][l, h, :nc])
            assert np.array_equal(single["local_idx"][l, h, :nl], batch["local_idx"][l, h, :nl])
    assert list(batch["seg_doc"]) == [0, 1, 2, -1] and list(batch["seg_first"]) == [0, 0, 0, 0]


@pytest.mark.parametrize("gran", [1, 64])
def test_batch_mask_is_block_diagonal_and_round_trips(gran):
    """A row of prompt p sees keys of prompt p only, by the single-prompt rule (L147-149 per request); the MD-v1b
    container, read back by its own rules, reproduces that mask (the round-trip pin of the container)."""
    b = _small_batch(gran)
    sh = b.head_shape
    rows = list(range(0, b.n_tokens, 7)) + [int(x) for x in b.row_base[1:] - 1] + [int(x) for x in b.row_base[:-1]]
    md = so.decode_metadata_batch(b.prompts, sh.tile, gran, 1, sh.n_q_heads, b.la_vec, b.ca_vec)
    n_docs = len(b.doc_lens)
    for h in range(sh.n_q_heads):
        la = [b.la_vec(0, h, d) for d in range(n_docs)]
        ca = [b.ca_vec(0, h, d) for d in range(n_docs)]
        mask = so.expand_mask_rows_batch(b.prompts, sh.tile, gran, la, ca, rows)
        for ri, q in enumerate(rows):
            p = so.prompt_of_row(q, b.row_base)
            lo, hi = int(b.row_base[p]), int(b.row_base[p + 1])
            assert not mask[ri, :lo].any() and not mask[ri, hi:].any()
            # inside its prompt the row is the single-prompt row
            m = b.members[p]
            la_p, ca_p = so.head_vectors(m, 0, h)
            ref = so.expand_mask_rows(m.shape.doc_offsets, m.shape.query_len, sh.tile, gran, la_p, ca_p, [q - lo])
            assert np.array_equal(mask[ri, lo:hi], ref[0])
        back = so.metadata_batch_to_mask_rows(md, b.prompts, sh.tile, gran, 0, h, rows)
        assert np.array_equal(back, mask)


def test_batch_container_rules():
    b = _small_batch()
    sh = b.head_shape
    md = so.decode_metadata_batch(b.prompts, sh.tile, 1, 1, sh.n_q_heads, b.la_vec, b.ca_vec)
    assert list(md["seg_doc"]) == [0, 1, 2, -1, -1, 3, 4, -1]
    assert list(md["seg_first"]) == [0, 0, 0, 0, 4, 5, 5, 5]
    cp = md["cross_ptr"][0]
    for h in range(sh.n_q_heads):
        assert cp[h, 0] == 0 and cp[h, 3] % 128 == 0          # every prompt's cross list starts at a multiple of 128
        assert np.all(np.diff(cp[h, :3]) >= 0) and np.all(np.diff(cp[h, 3:]) >= 0)
        # counts inside a prompt are plain popcounts of its documents' valid CA bits
        for d in (0, 1, 3):
            bits = so.read_bits(b.ca_vec(0, h, d), so.ca_vector_bits(b.doc_lens[d], sh.tile, 1))
            assert cp[h, d + 1] - cp[h, d] == int(bits.sum())
        # a query tile lists the tiles of its own prompt, first to itself (L243, per request)
        for p in range(3):
            seg_q = int(np.nonzero(md["seg_first"] == md["seg_first"][[3, 4, 7][p]])[0][-1])
            f = int(md["tile_base"][int(md["seg_first"][seg_q])])
            for t in range(int(md["tile_base"][seg_q]), int(md["tile_base"][seg_q + 1])):
                lo, hi = int(md["local_ptr"][0, h, t]), int(md["local_ptr"][0, h, t + 1])
                assert list(md["local_idx"][0, h, lo:hi]) == list(range(f, t + 1))


def test_batch_attention_rows_against_brute_force():
    """Slicing check: a row of the packed batch, brute-forced in fp64 over the GLOBAL K/V with the keys the batch
    mask allows, equals the oracle's per-prompt computation."""
    b = _small_batch()
    sh = b.head_shape
    q, k, v = b.qkv(0)
    n_docs = len(b.doc_lens)
    rows = [5, 399, 439, 440, 529, 530, 600, 926, 927]
    for h in range(sh.n_q_heads):
        la = [b.la_vec(0, h, d) for d in range(n_docs)]
        ca = [b.ca_vec(0, h, d) for d in range(n_docs)]
        o, lse = so.sift_attention_rows_batch(q, k, v, h, b.prompts, sh.tile, 1, la, ca, rows, dtype=torch.float64)
        mask = so.expand_mask_rows_batch(b.prompts, sh.tile, 1, la, ca, rows)
        kvh = so.kv_head_of(h, sh.n_q_heads, sh.n_kv_heads)
        for ri, r in enumerate(rows):
            allowed = np.nonzero(mask[ri])[0]
            ob, lb = so.brute_force_row(q[r, h].double().numpy(), k[:, kvh].double().numpy(), v[:, kvh].double().numpy(),
                                        allowed, 1.0 / math.sqrt(sh.head_dim))
            assert np.allclose(o[ri].numpy(), ob, atol=1e-9) and abs(float(lse[ri]) - lb) < 1e-9


# ---------------------------------------------------------------- FP8 (e4m3) inputs

def test_e4m3_decode_format_values():
    """OCP FP8 E4M3 by hand: 0x38 = 1.0, 0x7E = 448 (largest finite), 0x01 = 2^-9 (smallest subnormal), 0x08 = 2^-6
    (smallest normal), 0x3C = 1.5, 0xC0 = -2, 0x00 / 0x80 = +-0, 0x7F = NaN; and the whole table against torch."""
    got = so.e4m3_decode(np.array([0x38, 0x7E, 0x01, 0x08, 0x3C, 0xC0, 0x00, 0x80], np.uint8))
    assert list(got) == [1.0, 448.0, 2.0 ** -9, 2.0 ** -6, 1.5, -2.0, 0.0, -0.0]
    assert np.isnan(so.e4m3_decode(np.array([0x7F, 0xFF], np.uint8))).all()
    allb = np.arange(256, dtype=np.uint8)
    ref = torch.from_numpy(allb).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    ok = ~np.isnan(ref)
    assert np.array_equal(so.e4m3_decode(allb)[ok], ref[ok]) and np.isnan(so.e4m3_decode(allb)[~ok]).all()
    # strictly increasing over the positive finite codes: 127 distinct magnitudes
    assert np.all(np.diff(so.e4m3_decode(np.arange(0, 0x7F, dtype=np.uint8))) > 0)


def test_fp8_attention_is_attention_of_the_dequantised_values_and_scales_fold():
    w = wl.custom("f8", n_layers=1, n_q_heads=2, n_kv_heads=1, head_dim=64, doc_lens=(100, 70), query_len=30, tile=64, seed=9)
    sh = w.shape
    q, k, v = w.qkv(0)
    q8, qs = wl.quantize_e4m3(q)
    k8, ks = wl.quantize_e4m3(k)
    v8, vs = wl.quantize_e4m3(v)
    rows = [0, 63, 64, 99, 100, 169, 170, 199]
    for h in range(2):
        la, ca = so.head_vectors(w, 0, h)
        o, lse = so.sift_attention_rows_fp8(q8.numpy(), k8.numpy(), v8.numpy(), qs, ks, vs, h, sh.doc_offsets, sh.query_len,
                                            sh.tile, 1, la, ca, rows, dtype=torch.float64)
        # (a) the same rows from explicitly dequantised tensors through Part 2
        qd = q8.view(torch.float8_e4m3fn).double() * torch.from_numpy(qs.astype(np.float64))[None, :, None]
        kd = k8.view(torch.float8_e4m3fn).double() * torch.from_numpy(ks.astype(np.float64))[None, :, None]
        vd = v8.view(torch.float8_e4m3fn).double() * torch.from_numpy(vs.astype(np.float64))[None, :, None]
        o2, lse2 = so.sift_attention_rows(qd, kd, vd, h, sh.doc_offsets, sh.query_len, sh.tile, 1, la, ca, rows, dtype=torch.float64)
        assert torch.allclose(o, o2, atol=1e-12) and torch.allclose(lse, lse2, atol=1e-12)
        # (b) a factor moved from q_scale to the softmax scale changes nothing; v_scale is linear in O
        o3, lse3 = so.sift_attention_rows_fp8(q8.numpy(), k8.numpy(), v8.numpy(), qs * 2, ks, vs * 3, h, sh.doc_offsets, sh.query_len,
                                              sh.tile, 1, la, ca, rows, scale=0.5 / math.sqrt(64), dtype=torch.float64)
        assert torch.allclose(o3, 3 * o, atol=1e-9) and torch.allclose(lse3, lse, atol=1e-9)
        # (c) quantisation is the only difference from the bf16 path: close to the unquantised result (e4m3: 2^-4 relative)
        o4, _ = so.sift_attention_rows(q.double(), k.double(), v.double(), h, sh.doc_offsets, sh.query_len, sh.tile, 1, la, ca, rows,
                                       dtype=torch.float64)
        assert float((o - o4).abs().max()) < 0.5
