"""-m gpu parity tests: CUDA path (through the C ABI) vs the oracle on the same seeded inputs."""
import numpy as np
import pytest
import torch

from paper_2606_09441_b200 import api, workload as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu


def _report(name, errs):
    print(f"[parity] {name}: max_abs={errs[0]:.3e} mean_abs={errs[1]:.3e} lse={errs[2]:.3e}")
    assert errs[0] <= gu.TOL_MAX and errs[1] <= gu.TOL_MEAN and errs[2] <= gu.TOL_LSE, (name, errs)


# ------------------------------------------------------------------ decode: bit-exact

@pytest.mark.parametrize("cfg", ["tiny", "8b-10k", "32k", "64k-ragged"])
def test_decode_bit_exact_configs(cfg):
    w = wl.CONFIGS[cfg]()
    shape, md = gu.decode_on_gpu(w)
    gu.assert_metadata_equal(w, shape, md)


@pytest.mark.parametrize("case", [
    dict(doc_lens=(1,), query_len=0, tile=64),
    dict(doc_lens=(63, 64, 65, 1, 129), query_len=1, tile=64),
    dict(doc_lens=(500, 77), query_len=300, tile=128, n_layers=3, n_q_heads=5, n_kv_heads=5),
    dict(doc_lens=(300,), query_len=0, tile=128, p_loc=1.1, p_cross=1.1),
    dict(doc_lens=(300, 200), query_len=70, tile=128, p_loc=-1.0, p_cross=-1.0, diag_set=False),
    dict(doc_lens=tuple([37] * 300), query_len=5, tile=64, n_q_heads=1),
    dict(doc_lens=(9000,), query_len=100, tile=64, n_q_heads=1),
    # page-granular CA (G = tile): entries are global tile ids
    dict(doc_lens=(63, 64, 65, 1, 129), query_len=1, tile=64, cross_gran=64),
    dict(doc_lens=(2000, 1500, 700), query_len=100, tile=128, cross_gran=128, n_layers=2, n_q_heads=4, n_kv_heads=2),
    dict(doc_lens=tuple([37] * 300), query_len=5, tile=64, n_q_heads=1, cross_gran=64, p_cross=0.6),
])
def test_decode_bit_exact_edge_cases(case):
    w = wl.custom("edge", seed=41, **case)
    shape, md = gu.decode_on_gpu(w)
    gu.assert_metadata_equal(w, shape, md)


def test_decode_no_docs():
    w = wl.custom("nodocs", doc_lens=(), query_len=200, tile=64)
    shape, md = gu.decode_on_gpu(w)
    gu.assert_metadata_equal(w, shape, md)


def test_decode_full_stack_sampled_layers_and_reorder():
    w = wl.config_full_stack(n_layers=4)
    for perm in wl.stack_orderings(w, 2):
        wp = w.reorder(perm)
        shape, md = gu.decode_on_gpu(wp)
        gu.assert_metadata_equal(wp, shape, md, layers=[0, 3])


# ------------------------------------------------------------------ attention: building blocks first

@pytest.mark.parametrize("n,hd", [(128, 128), (256, 128), (200, 64), (1000, 128), (333, 64)])
def test_dense_comparator_small(n, hd):
    w = wl.custom("dense", n_q_heads=2, n_kv_heads=1, head_dim=hd, doc_lens=(), query_len=n, tile=128, seed=n)
    q, k, v = (t.cuda() for t in w.qkv(0))
    o, lse = api.sift_dense_causal_attention(q, k, v)
    torch.cuda.synchronize()
    _report(f"dense n={n} hd={hd}", gu.attention_errors(w, 0, o, lse, [0, 1], range(n), dense=True))


def test_local_only_cross_cleared():
    w = wl.custom("loc", n_q_heads=2, n_kv_heads=1, head_dim=128, doc_lens=(512, 300), query_len=0, tile=128,
                  p_loc=0.5, p_cross=-1.0, seed=3)
    _, _, o, lse = gu.run_sift(w)
    _report("local-only", gu.attention_errors(w, 0, o, lse, [0, 1], range(w.shape.n_tokens)))


def test_cross_gather_only():
    w = wl.custom("cross", n_q_heads=2, n_kv_heads=2, head_dim=128, doc_lens=(384, 256), query_len=0, tile=128,
                  p_loc=-1.0, p_cross=0.4, seed=4)
    _, _, o, lse = gu.run_sift(w)
    _report("cross+diag", gu.attention_errors(w, 0, o, lse, [0, 1], range(w.shape.n_tokens)))


@pytest.mark.parametrize("case", [
    dict(n_q_heads=2, n_kv_heads=2, head_dim=128, doc_lens=(384, 256, 700), query_len=40, tile=128, p_cross=0.4),
    dict(n_q_heads=2, n_kv_heads=1, head_dim=64, doc_lens=(256, 300, 129), query_len=0, tile=64, p_cross=0.7),
])
def test_cross_gather_cp_async_mode(case, monkeypatch):
    """The alternative row-gather path (SIFT_GATHER_MODE=1: swizzled cp.async instead of TMA gather4)."""
    monkeypatch.setenv("SIFT_GATHER_MODE", "1")
    w = wl.custom("cross-cpasync", seed=23, **case)
    _, _, o, lse = gu.run_sift(w)
    _report(f"cp.async gather {case}", gu.attention_errors(w, 0, o, lse, range(w.shape.n_q_heads), range(w.shape.n_tokens)))


@pytest.mark.parametrize("case", [
    dict(n_q_heads=4, n_kv_heads=2, head_dim=128, doc_lens=(384, 300, 700, 130), query_len=140, tile=128, cross_gran=128, p_cross=0.5),
    dict(n_q_heads=2, n_kv_heads=1, head_dim=64, doc_lens=(256, 300, 129, 64), query_len=33, tile=64, cross_gran=64, p_cross=0.4),
])
def test_paged_cross_all_rows(case):
    """page-granular CA (one bit per tile of keys), cross pages loaded as tiled TMA boxes."""
    w = wl.custom("paged", seed=29, **case)
    shape, md, o, lse = gu.run_sift(w)
    gu.assert_metadata_equal(w, shape, md)
    _report(f"paged {case}", gu.attention_errors(w, 0, o, lse, range(w.shape.n_q_heads), range(w.shape.n_tokens)))


def test_paged_32k_sampled_rows():
    w = wl.CONFIGS["32k-paged"]()
    _, _, o, lse = gu.run_sift(w)
    assert torch.isfinite(o.float()).all()
    _report("32k-paged", gu.attention_errors(w, 0, o, lse, [3, 30], gu.sample_rows(w)))


def test_empty_rows_A13():
    w = wl.custom("empty", n_q_heads=1, head_dim=64, doc_lens=(200, 100), query_len=30, tile=64, p_loc=-1.0,
                  p_cross=-1.0, diag_set=False, seed=5)
    _, _, o, lse = gu.run_sift(w)
    assert torch.all(o[:300] == 0) and torch.all(torch.isinf(lse[:, :300]) & (lse[:, :300] < 0))
    _report("empty rows", gu.attention_errors(w, 0, o, lse, [0], range(w.shape.n_tokens)))


@pytest.mark.parametrize("case", [
    dict(head_dim=64, doc_lens=(256, 256, 256, 256), query_len=64, tile=64),
    dict(head_dim=128, doc_lens=(130, 127, 385, 1), query_len=129, tile=128, n_q_heads=4, n_kv_heads=2),
    dict(head_dim=128, doc_lens=(700, 900), query_len=300, tile=64, n_q_heads=4, n_kv_heads=1),
    dict(head_dim=64, doc_lens=(1000, 333, 64), query_len=7, tile=128, n_q_heads=3, n_kv_heads=3, p_cross=0.9),
])
def test_sift_small_all_rows(case):
    w = wl.custom("small", seed=17, **case)
    _, _, o, lse = gu.run_sift(w)
    _report(f"small {case}", gu.attention_errors(w, 0, o, lse, range(w.shape.n_q_heads), range(w.shape.n_tokens)))


def test_sift_all_ones_equals_dense_kernel_and_oracle():
    w = wl.custom("ones", n_q_heads=2, n_kv_heads=1, head_dim=128, doc_lens=(300, 212), query_len=100, tile=128,
                  p_loc=1.1, p_cross=1.1, seed=19)
    _, _, o, lse = gu.run_sift(w)
    _report("all-ones", gu.attention_errors(w, 0, o, lse, [0, 1], range(w.shape.n_tokens)))
    q, k, v = (t.cuda() for t in w.qkv(0))
    od, lsed = api.sift_dense_causal_attention(q, k, v)
    assert (o.float() - od.float()).abs().max() <= 2e-2 and (lse - lsed).abs().max() <= 1e-3


# ------------------------------------------------------------------ BASELINE.json configs

def test_config_tiny_all_rows():
    w = wl.config_tiny()
    _, _, o, lse = gu.run_sift(w)
    _report("C1 tiny", gu.attention_errors(w, 0, o, lse, [0, 1], range(w.shape.n_tokens)))


@pytest.mark.parametrize("cfg,heads", [("8b-10k", [0, 5, 17, 31]), ("32k", [3, 30]), ("64k-ragged", [9, 28])])
def test_config_sampled_rows(cfg, heads):
    w = wl.CONFIGS[cfg]()
    _, _, o, lse = gu.run_sift(w)
    assert torch.isfinite(o.float()).all()
    _report(cfg, gu.attention_errors(w, 0, o, lse, heads, gu.sample_rows(w)))


def test_full_stack_layers_and_reorder_sampled():
    """C5 shape (4 of its 32 layers to bound host memory): one decode call for all layers, then per-layer attention;
    a re-ordered prompt (vectors travel with their document) is checked against the oracle on the permuted inputs."""
    w = wl.config_full_stack(n_layers=4)
    shape, md = gu.decode_on_gpu(w)
    for layer in (0, 3):
        q, k, v = (t.cuda() for t in w.qkv(layer))
        o, lse = api.sift_prefill_attention(shape, layer, q, k, v, md)
        torch.cuda.synchronize()
        _report(f"C5 layer {layer}", gu.attention_errors(w, layer, o, lse, [1, 22], gu.sample_rows(w, n_per_seg=2)))
    w2 = w.reorder(wl.stack_orderings(w)[1])
    shape2, md2 = gu.decode_on_gpu(w2)
    q, k, v = (t.cuda() for t in w2.qkv(2))
    o, lse = api.sift_prefill_attention(shape2, 2, q, k, v, md2)
    torch.cuda.synchronize()
    _report("C5 reordered layer 2", gu.attention_errors(w2, 2, o, lse, [7], gu.sample_rows(w2, n_per_seg=2)))


def test_repeat_calls_share_metadata():
    w = wl.config_tiny()
    shape, md = gu.decode_on_gpu(w)
    q, k, v = (t.cuda() for t in w.qkv(0))
    o1, l1 = api.sift_prefill_attention(shape, 0, q, k, v, md)
    o2, l2 = api.sift_prefill_attention(shape, 0, q, k, v, md)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2) and torch.equal(l1, l2)
