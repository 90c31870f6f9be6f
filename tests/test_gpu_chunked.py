"""sift_prefill_attention_rows (chunked prefill): rows [r0, r1) of a prompt against the
same metadata.  What is unique is checked exactly: every row of a range is bit-identical to the whole-prompt call, rows
outside the range are not written, and the assembled chunks agree with the CPU oracle within north_star's tolerance."""
import pytest
import torch

from paper_2606_09441_b200 import api, workload as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu


def _prompt(name, **kw):
    w = wl.custom(name, **kw)
    shape, md = gu.decode_on_gpu(w)
    q, k, v = (t.cuda() for t in w.qkv(0))
    return w, shape, md, q, k, v


def _chunks_equal_whole(w, shape, md, q, k, v, cuts):
    o_ref, lse_ref = api.sift_prefill_attention(shape, 0, q, k, v, md)
    n = q.shape[0]
    o = torch.full_like(o_ref, -7.0)
    lse = torch.full_like(lse_ref, -7.0)
    bounds = [0] + list(cuts) + [n]
    for a, b in zip(bounds[:-1], bounds[1:]):
        before_o, before_l = o.clone(), lse.clone()
        api.sift_prefill_attention_rows(shape, 0, a, b, q, k, v, md, o, lse)
        torch.cuda.synchronize()
        assert torch.equal(o[a:b], o_ref[a:b]) and torch.equal(lse[:, a:b], lse_ref[:, a:b]), (a, b)
        keep = torch.ones(n, dtype=torch.bool, device="cuda")
        keep[a:b] = False
        assert torch.equal(o[keep], before_o[keep]) and torch.equal(lse[:, keep], before_l[:, keep]), ("wrote outside", a, b)
    assert torch.equal(o, o_ref) and torch.equal(lse, lse_ref)
    return o, lse


@pytest.mark.parametrize("gran", [1, 128])
def test_chunks_are_bit_identical_and_match_the_oracle(gran):
    """Ragged documents, cuts inside a tile, at a tile edge, at a document edge and inside the query; then the
    assembled output against the oracle on every row of two heads."""
    w, shape, md, q, k, v = _prompt("chunked", n_q_heads=4, n_kv_heads=2, head_dim=128, doc_lens=(300, 515, 128, 77, 640),
                                    query_len=190, tile=128, cross_gran=gran, p_cross=0.4, seed=91)
    n = q.shape[0]
    o, lse = _chunks_equal_whole(w, shape, md, q, k, v, cuts=(1, 128, 300, 301, 815, 1000, 1660, n - 1))
    mx, mean, le = gu.attention_errors(w, 0, o, lse, heads=range(4), rows=range(n))
    assert mx <= gu.TOL_MAX and mean <= gu.TOL_MEAN and le <= gu.TOL_LSE, (mx, mean, le)


def test_chunk_needs_no_keys_past_its_last_tile():
    """Chunked prefill proper: when a chunk runs, K / V / Q of later rows do not exist yet.  Rows from E = (end of the
    chunk's last tile) + 127 (the reach of the copy engine's last 128-row box; include/sift.h) are NaN here, K and Q
    already from row_end, and the chunk still equals the whole-prompt result."""
    w, shape, md, q, k, v = _prompt("chunked-nan", n_q_heads=4, n_kv_heads=2, head_dim=128, doc_lens=(700, 900), query_len=333,
                                    tile=128, p_cross=0.5, seed=92)
    o_ref, lse_ref = api.sift_prefill_attention(shape, 0, q, k, v, md)
    n = q.shape[0]
    for a, b, e in ((0, 600, 640 + 127), (600, 700, 700 + 127), (700, 1000, 1084 + 127), (1600, 1700, 1728 + 127)):
        q2, k2, v2 = q.clone(), k.clone(), v.clone()
        for t in (q2, k2):
            t[b:] = float("nan")
        v2[b:e] = 0.0
        v2[e:] = float("nan")
        o = torch.zeros_like(o_ref)
        lse = torch.zeros_like(lse_ref)
        api.sift_prefill_attention_rows(shape, 0, a, b, q2, k2, v2, md, o, lse)
        torch.cuda.synchronize()
        assert torch.equal(o[a:b], o_ref[a:b]) and torch.equal(lse[:, a:b], lse_ref[:, a:b]), (a, b)


def test_chunked_batch_of_prompts_and_head_dim_64():
    """Two prompts in one call (MD-v1b) cut across the prompt boundary, and the d = 64 / T = 64 instance."""
    b = wl.make_batch("chunk-batch", [wl.custom(f"cb{i}", n_q_heads=4, n_kv_heads=2, head_dim=128, doc_lens=dl, query_len=ql,
                                                tile=128, p_cross=0.5, seed=93 + i)
                                      for i, (dl, ql) in enumerate((((260, 400), 100), ((129,), 64)))])
    shape = api.Shape.from_batch(b)
    md = api.sift_decode_metadata(shape, torch.from_numpy(b.la_blob).cuda(), b.la_doc_off, torch.from_numpy(b.ca_blob).cuda(),
                                  b.ca_doc_off)
    q, k, v = (t.cuda() for t in b.qkv(0))
    _chunks_equal_whole(b, shape, md, q, k, v, cuts=(500, 760, 800))
    w, shape, md, q, k, v = _prompt("chunked-64", n_q_heads=4, n_kv_heads=4, head_dim=64, doc_lens=(200, 333), query_len=70,
                                    tile=64, p_cross=0.5, seed=95)
    _chunks_equal_whole(w, shape, md, q, k, v, cuts=(64, 100, 533))


def test_range_arguments():
    w, shape, md, q, k, v = _prompt("chunked-args", n_q_heads=2, n_kv_heads=1, head_dim=128, doc_lens=(200,), query_len=56,
                                    tile=128, p_cross=0.5, seed=96)
    o = torch.full_like(q, 3.0)
    n0 = api.sift_launch_count()
    api.sift_prefill_attention_rows(shape, 0, 100, 100, q, k, v, md, o)        # empty: no launch, nothing written
    torch.cuda.synchronize()
    assert api.sift_launch_count() == n0 and bool((o == 3.0).all())
    for a, b in ((-1, 10), (10, 5), (0, 257)):
        with pytest.raises(api.SiftError):
            api.sift_prefill_attention_rows(shape, 0, a, b, q, k, v, md, o)
    # the whole range is the plain call
    o_ref, _ = api.sift_prefill_attention(shape, 0, q, k, v, md)
    api.sift_prefill_attention_rows(shape, 0, 0, 256, q, k, v, md, o)
    torch.cuda.synchronize()
    assert torch.equal(o, o_ref)
