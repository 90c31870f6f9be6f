"""-m gpu: e4m3 Q/K/V (reading R7) through the C ABI against the oracle on the same bytes.
Tolerance (derived in DESIGN.md before the kernel existed: P is rounded to e4m3, 3 mantissa bits): max-abs 0.15,
mean-abs 2e-2 on O; |dLSE| <= 1e-3 (the row sum is not quantised)."""
import numpy as np
import pytest
import torch

from oracle import sift_oracle as so
from paper_2606_09441_b200 import api, workload as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu

TOL8_MAX, TOL8_MEAN = 0.15, 2e-2


def _run(w, layer=0, softmax_scale=0.0):
    sh = w.shape
    shape, md = gu.decode_on_gpu(w)
    q, k, v = w.qkv(layer)
    (q8, qs), (k8, ks), (v8, vs) = wl.quantize_e4m3(q), wl.quantize_e4m3(k), wl.quantize_e4m3(v)
    o, lse = api.sift_prefill_attention_fp8(shape, layer, q8.cuda(), k8.cuda(), v8.cuda(), qs, ks, vs, md, softmax_scale=softmax_scale)
    torch.cuda.synchronize()
    return (q8, qs, k8, ks, v8, vs), o.float().cpu(), lse.cpu()


def _errors(w, layer, packed, o, lse, heads, rows, scale=None):
    q8, qs, k8, ks, v8, vs = packed
    sh = w.shape
    mx = mean = le = 0.0
    for h in heads:
        la, ca = so.head_vectors(w, layer, h)
        ro, rl = so.sift_attention_rows_fp8(q8.numpy(), k8.numpy(), v8.numpy(), qs, ks, vs, h, sh.doc_offsets, sh.query_len,
                                            sh.tile, sh.cross_gran, la, ca, rows, scale=scale)
        d = (o[rows, h] - ro).abs()
        mx, mean = max(mx, float(d.max())), max(mean, float(d.mean()))
        both_inf = torch.isinf(rl) & torch.isinf(lse[h, rows])
        le = max(le, float(torch.where(both_inf, torch.zeros_like(rl), (lse[h, rows] - rl).abs()).max()))
    return mx, mean, le


@pytest.mark.parametrize("gran,docs,qlen", [(1, (300, 128, 517), 70), (128, (260, 1, 1000), 129), (1, (), 300)])
def test_fp8_small_all_rows(gran, docs, qlen):
    w = wl.custom("f8s", n_layers=2, n_q_heads=4, n_kv_heads=2, head_dim=128, doc_lens=docs, query_len=qlen, tile=128,
                  cross_gran=gran, p_loc=0.5, p_cross=0.3, seed=61)
    packed, o, lse = _run(w, layer=1)
    assert torch.isfinite(o).all()
    mx, mean, le = _errors(w, 1, packed, o, lse, range(4), list(range(w.shape.n_tokens)))
    assert mx <= TOL8_MAX and mean <= TOL8_MEAN and le <= gu.TOL_LSE, (mx, mean, le)


def test_fp8_explicit_scale_and_logit_range():
    """a wide logit range (Q scaled up) exercises the lazy rescale at the e4m3 threshold of 2 log2 units"""
    w = wl.custom("f8r", n_layers=1, n_q_heads=2, n_kv_heads=1, head_dim=128, doc_lens=(400, 333), query_len=100, tile=128,
                  p_loc=0.6, p_cross=0.4, seed=62)
    packed, o, lse = _run(w, softmax_scale=0.35)
    mx, mean, le = _errors(w, 0, packed, o, lse, range(2), list(range(0, w.shape.n_tokens, 3)), scale=0.35)
    assert mx <= TOL8_MAX and mean <= TOL8_MEAN and le <= gu.TOL_LSE, (mx, mean, le)


def test_fp8_c2_sampled_rows():
    w = wl.config_8b_10k()
    packed, o, lse = _run(w)
    assert torch.isfinite(o).all()
    rows = gu.sample_rows(w, n_per_seg=3, seed=5)
    mx, mean, le = _errors(w, 0, packed, o, lse, [0, 13, 31], rows)
    assert mx <= TOL8_MAX and mean <= TOL8_MEAN and le <= gu.TOL_LSE, (mx, mean, le)


def test_fp8_rejects_head_dim_64():
    w = wl.custom("f8x", head_dim=64, tile=64)
    shape, md = gu.decode_on_gpu(w)
    q8 = torch.zeros((w.shape.n_tokens, 2, 64), dtype=torch.uint8, device="cuda")
    k8 = torch.zeros((w.shape.n_tokens, 1, 64), dtype=torch.uint8, device="cuda")
    with pytest.raises(api.SiftError):
        api.sift_prefill_attention_fp8(shape, 0, q8, k8, k8, [1, 1], [1], [1], md)


def test_fp8_on_a_batch_of_prompts():
    """e4m3 Q/K/V and several prompts in one call go through the same kernel body: sampled rows against the oracle (Part 5
    on the values Part 6 decodes)."""
    kw = dict(n_layers=1, n_q_heads=4, n_kv_heads=2, head_dim=128, tile=128, cross_gran=1)
    b = wl.make_batch("f8b", [wl.custom("a", doc_lens=(300, 260), query_len=50, p_loc=0.5, p_cross=0.4, seed=71, **kw),
                              wl.custom("b", doc_lens=(129, 500, 64), query_len=130, p_loc=0.5, p_cross=0.3, seed=72, **kw)])
    sh = b.head_shape
    shape = api.Shape.from_batch(b)
    la, ca = torch.from_numpy(b.la_blob).cuda(), torch.from_numpy(b.ca_blob).cuda()
    md = api.sift_decode_metadata(shape, la, b.la_doc_off, ca, b.ca_doc_off)
    q, k, v = b.qkv(0)
    (q8, qs), (k8, ks), (v8, vs) = wl.quantize_e4m3(q), wl.quantize_e4m3(k), wl.quantize_e4m3(v)
    o, lse = api.sift_prefill_attention_fp8(shape, 0, q8.cuda(), k8.cuda(), v8.cuda(), qs, ks, vs, md)
    torch.cuda.synchronize()
    o, lse = o.float().cpu(), lse.cpu()
    deq = lambda x8, s: torch.from_numpy(so.e4m3_decode(x8.numpy()) * s.astype(np.float64)[None, :, None]).float()
    qd, kd, vd = deq(q8, qs), deq(k8, ks), deq(v8, vs)
    rows = list(range(0, b.n_tokens, 7)) + [b.n_tokens - 1]
    n_docs = len(b.doc_lens)
    for h in range(sh.n_q_heads):
        lav = [b.la_vec(0, h, d) for d in range(n_docs)]
        cav = [b.ca_vec(0, h, d) for d in range(n_docs)]
        ro, rl = so.sift_attention_rows_batch(qd, kd, vd, h, b.prompts, sh.tile, 1, lav, cav, rows)
        d = (o[rows, h] - ro).abs()
        assert float(d.max()) <= TOL8_MAX and float(d.mean()) <= TOL8_MEAN and float((lse[h, rows] - rl).abs().max()) <= gu.TOL_LSE
