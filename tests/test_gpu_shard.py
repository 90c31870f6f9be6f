"""-m gpu: the head-sharded code path on one GPU: the shards of a 2- and a 3-rank
split are run one after the other (they are independent launches, nothing waits on another shard) and their columns of O
must be bit-identical to the unsharded call."""
import pytest
import torch

from paper_2606_09441_b200 import api, shard, workload as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("world", [2, 3])
def test_head_shards_equal_the_unsharded_call(world):
    w = wl.custom("hs", n_layers=2, n_q_heads=8, n_kv_heads=4, head_dim=128, doc_lens=(300, 128, 517), query_len=70, tile=128,
                  p_loc=0.5, p_cross=0.4, seed=78)
    layer = 1
    shape, md = gu.decode_on_gpu(w)
    q, k, v = (t.cuda() for t in w.qkv(layer))
    o_ref, lse_ref = api.sift_prefill_attention(shape, layer, q, k, v, md)
    la, ca = torch.from_numpy(w.la_blob).cuda(), torch.from_numpy(w.ca_blob).cuda()
    o = torch.full_like(q, float("nan"))
    lse = torch.full_like(lse_ref, float("nan"))
    for rank in range(world):
        sh = shard.head_shard(w.shape.n_q_heads, w.shape.n_kv_heads, rank, world)
        sub = api.Shape.from_prompt(shard.shard_prompt_shape(w.shape, sh))
        la_off, ca_off = shard.shard_blob_offsets(w, sh, layer)
        md_s = api.sift_decode_metadata(sub, la, la_off, ca, ca_off)
        qs, ks, vs = shard.shard_views(q, k, v, sh)
        api.sift_prefill_attention(sub, 0, qs, ks, vs, md_s, o[:, sh.q0:sh.q1], lse[sh.q0:sh.q1])
    torch.cuda.synchronize()
    assert torch.equal(o, o_ref) and torch.equal(lse, lse_ref)
