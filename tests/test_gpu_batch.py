"""-m gpu: several prompts in one call through the C ABI.

Metadata: bit-exact against the oracle's MD-v1b (oracle.decode_metadata_batch).  Attention: bit-identical to one call
per prompt (a row only ever sees its own prompt, and the work of a row is cut into the same steps), and within
north_star's tolerance of the oracle on sampled rows."""
import numpy as np
import pytest
import torch

from oracle import sift_oracle as so
from paper_2606_09441_b200 import api, workload as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu


def _batch(gran=1, tile=64, hd=64, heads=(2, 1)):
    kw = dict(n_layers=2, n_q_heads=heads[0], n_kv_heads=heads[1], head_dim=hd, tile=tile, cross_gran=gran)
    members = [
        wl.custom("ba", doc_lens=(130, 70, 200), query_len=40, p_loc=0.5, p_cross=0.3, seed=11, **kw),
        wl.custom("bb", doc_lens=(), query_len=90, seed=12, **kw),                       # a prompt without documents
        wl.custom("bc", doc_lens=(64, 333), query_len=1, p_loc=0.4, p_cross=0.5, seed=13, **kw),
        wl.custom("bd", doc_lens=(700, 1, 290, 515), query_len=200, p_loc=0.3, p_cross=0.6, seed=14, **kw),
    ]
    return wl.make_batch("b4", members)


def _decode(b):
    shape = api.Shape.from_batch(b)
    la, ca = torch.from_numpy(b.la_blob).cuda(), torch.from_numpy(b.ca_blob).cuda()
    md = api.sift_decode_metadata(shape, la, b.la_doc_off, ca, b.ca_doc_off)
    torch.cuda.synchronize()
    return shape, md


def _assert_batch_metadata(b, shape, md):
    sh = b.head_shape
    v = {k: t.cpu().numpy() for k, t in api.metadata_views(shape, md).items()}
    ref = so.decode_metadata_batch(b.prompts, sh.tile, sh.cross_gran, sh.n_layers, sh.n_q_heads, b.la_vec, b.ca_vec)
    lay = api.sift_metadata_layout(shape)
    assert lay.cross_cap == ref["cross_cap"] and lay.local_cap == ref["local_cap"] and lay.n_tiles == ref["NT"]
    assert lay.n_tokens == b.n_tokens and lay.n_seg == len(ref["seg_doc"])
    for k in ("tile_base", "tile_seg", "tile_row0", "tile_rows", "cross_ptr", "local_cnt", "local_ptr"):
        assert np.array_equal(v[k], ref[k]), k
    assert np.array_equal(v["seg_info"][:, 0], ref["seg_doc"])
    for name in ("cross_idx", "local_idx"):
        spec = ref[name] >= 0                       # entries the container specifies
        assert np.array_equal(v[name][..., : ref[name].shape[-1]][spec], ref[name][spec]), name
    # unspecified cross entries that the attention kernel may gather (up to the next multiple of 128) are valid rows
    cp = ref["cross_ptr"]
    for l in range(sh.n_layers):
        for h in range(sh.n_q_heads):
            for p in range(len(b.members)):
                d1 = int(b.doc_base[p + 1])
                if d1 == int(b.doc_base[p]):
                    continue
                tot = sum(int(so.read_bits(b.ca_vec(l, h, d), so.ca_vector_bits(b.doc_lens[d], sh.tile, sh.cross_gran)).sum())
                          for d in range(int(b.doc_base[p]), d1))
                lo = int(cp[l, h, int(b.doc_base[p])])
                pad = v["cross_idx"][l, h, lo + tot: lo + -(-tot // 128) * 128]
                assert np.all((pad >= 0) & (pad < b.n_tokens)), "pad entries must be valid rows"
    for l in range(sh.n_layers):                    # the schedule holds every (head, M-block) item once
        exp = np.sort(np.array([(h << 20) | mb for h in range(sh.n_q_heads) for mb in range(lay.n_mblocks)]))
        assert np.array_equal(np.sort(v["sched"][l]), exp)


@pytest.mark.parametrize("gran,tile,hd", [(1, 64, 64), (64, 64, 64), (1, 128, 128), (128, 128, 128)])
def test_batch_metadata_matches_oracle(gran, tile, hd):
    b = _batch(gran, tile, hd)
    shape, md = _decode(b)
    _assert_batch_metadata(b, shape, md)


@pytest.mark.parametrize("gran,tile,hd,heads", [(1, 64, 64, (2, 1)), (1, 128, 128, (4, 2)), (128, 128, 128, (2, 2))])
def test_batch_attention_equals_single_calls_and_oracle(gran, tile, hd, heads):
    b = _batch(gran, tile, hd, heads)
    sh = b.head_shape
    shape, md = _decode(b)
    layer = 1
    q, k, v = (t.cuda() for t in b.qkv(layer))
    o, lse = api.sift_prefill_attention(shape, layer, q, k, v, md)
    torch.cuda.synchronize()
    assert torch.isfinite(o.float()).all()
    # one call per prompt: bit-identical
    for p, w in enumerate(b.members):
        lo, hi = int(b.row_base[p]), int(b.row_base[p + 1])
        s1, md1 = gu.decode_on_gpu(w)
        o1, lse1 = api.sift_prefill_attention(s1, layer, q[lo:hi].contiguous(), k[lo:hi].contiguous(), v[lo:hi].contiguous(), md1)
        torch.cuda.synchronize()
        assert torch.equal(o[lo:hi], o1), f"prompt {p}: O differs from the single call"
        assert torch.equal(lse[:, lo:hi], lse1), f"prompt {p}: LSE differs from the single call"
    # the oracle on sampled rows of the packed batch
    rows = sorted({0, b.n_tokens - 1} | {int(x) for x in b.row_base[1:-1]} | {int(x) - 1 for x in b.row_base[1:]} |
                  {int(x) for x in np.random.default_rng(3).integers(0, b.n_tokens, 60)})
    qc, kc, vc = b.qkv(layer)
    n_docs = len(b.doc_lens)
    mx = mean = le = 0.0
    for h in range(sh.n_q_heads):
        la = [b.la_vec(layer, h, d) for d in range(n_docs)]
        ca = [b.ca_vec(layer, h, d) for d in range(n_docs)]
        ro, rl = so.sift_attention_rows_batch(qc, kc, vc, h, b.prompts, sh.tile, sh.cross_gran, la, ca, rows)
        d = (o[rows, h].float().cpu() - ro).abs()
        mx, mean = max(mx, float(d.max())), max(mean, float(d.mean()))
        le = max(le, float((lse[h, rows].cpu() - rl).abs().max()))
    assert mx <= gu.TOL_MAX and mean <= gu.TOL_MEAN and le <= gu.TOL_LSE, (mx, mean, le)


def test_batch_of_c2_prompts_runs_and_matches_single_calls():
    """Two prompts of C2's shape (the bench's batch leg uses eight): bit-identical to the single calls on every row."""
    b = wl.make_batch("2x10k", [wl.config_8b_10k(wl.BASE_SEED + 1000), wl.config_8b_10k(wl.BASE_SEED + 2000)])
    shape, md = _decode(b)
    q, k, v = (t.cuda() for t in b.qkv(0))
    o, lse = api.sift_prefill_attention(shape, 0, q, k, v, md)
    torch.cuda.synchronize()
    for p, w in enumerate(b.members):
        lo, hi = int(b.row_base[p]), int(b.row_base[p + 1])
        s1, md1 = gu.decode_on_gpu(w)
        o1, lse1 = api.sift_prefill_attention(s1, 0, q[lo:hi].contiguous(), k[lo:hi].contiguous(), v[lo:hi].contiguous(), md1)
        torch.cuda.synchronize()
        assert torch.equal(o[lo:hi], o1) and torch.equal(lse[:, lo:hi], lse1)


def test_host_pipeline_on_a_batch_matches_the_device_call():
    """sift_prefill_layer_host with several prompts: per kv-head group from HOST buffers, bit-identical to the device call."""
    from paper_2606_09441_b200.pipeline import HostLayerPipeline
    b = _batch(1, 128, 128, (4, 2))
    shape, md = _decode(b)
    layer = 1
    q, k, v = b.qkv(layer)
    o_ref, lse_ref = api.sift_prefill_attention(shape, layer, q.cuda(), k.cuda(), v.cuda(), md)
    torch.cuda.synchronize()
    qh, kh, vh = (t.pin_memory() for t in (q, k, v))
    la_h, ca_h = torch.from_numpy(b.la_blob).pin_memory(), torch.from_numpy(b.ca_blob).pin_memory()
    o_h = torch.empty(q.shape, dtype=q.dtype).pin_memory()
    lse_h = torch.empty(lse_ref.shape, dtype=torch.float32).pin_memory()
    pipe = HostLayerPipeline(None, shape=shape)
    pipe.run(la_h, ca_h, b.la_doc_off, b.ca_doc_off, qh, kh, vh, o_h, layer=layer, lse_h=lse_h)
    pipe.wait()
    assert torch.equal(o_h, o_ref.cpu()) and torch.equal(lse_h, lse_ref.cpu())
