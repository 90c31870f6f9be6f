"""-m gpu parity at full size for the widened rows of SURVEY.md 8(f), at the sizes bench.py times them (VERDICT r2,
weak 8): page-granular CA on C3 and C4 (every head, a row in every query tile + tails + boundaries), e4m3 Q/K/V on C3
and C4 (the same rows on a subset of heads that covers every kv head -- the e4m3 oracle is slow: all 32 heads of both took
12 of the suite's 19 minutes in the r3 builder run, where they measured max-abs 4.4e-2 / mean-abs 2.3e-3; the measured
errors are printed beside the bound, which is 2x those figures for this test), the encoder on the benched 2000-token document
and on 4096 tokens, and the TP = 8 head split of C2 bit-identical to the unsharded call."""
import numpy as np
import pytest
import torch

from paper_2606_09441_b200 import api, shard, workload as wl
from tests import gpu_util as gu
from tests.test_gpu_full_size import _check, rows_one_per_tile
from tests.test_gpu_fp8 import TOL8_MAX, TOL8_MEAN, _errors as fp8_errors, _run as fp8_run
from tests.test_gpu_parity import _encode_case

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg", ["32k-paged", "64k-paged"])
def test_paged_every_head_every_tile(cfg):
    w = wl.CONFIGS["32k-paged"]() if cfg == "32k-paged" else wl.config_64k_ragged(cross_gran=128)
    shape, md, o, lse = gu.run_sift(w)
    assert torch.isfinite(o.float()).all()
    if cfg == "64k-paged":
        gu.assert_metadata_equal(w, shape, md)          # 24 ragged documents, one CA bit per page
    _check(cfg + " all heads x (row per tile + tails + boundaries)",
           gu.attention_errors(w, 0, o, lse, range(w.shape.n_q_heads), rows_one_per_tile(w)))


# 2x the worst error measured on all 32 heads of C3 and C4 (r3 builder run: 4.38e-2 / 2.28e-3); DESIGN.md's derivation
# (TOL8_MAX, TOL8_MEAN) stays the upper bound for the small cases
FULL8_MAX, FULL8_MEAN = 0.09, 5e-3
assert FULL8_MAX <= TOL8_MAX and FULL8_MEAN <= TOL8_MEAN


@pytest.mark.parametrize("cfg,heads", [("32k", range(0, 32, 2)), ("64k-ragged", range(1, 32, 4))])
def test_fp8_every_kv_head_every_tile(cfg, heads):
    w = wl.CONFIGS[cfg]()
    packed, o, lse = fp8_run(w)
    assert torch.isfinite(o).all()
    mx, mean, le = fp8_errors(w, 0, packed, o, lse, heads, rows_one_per_tile(w))
    print(f"[parity-full] fp8 {cfg} heads {list(heads)}: max_abs={mx:.3e} (bound {FULL8_MAX}) mean_abs={mean:.3e} (bound {FULL8_MEAN}) lse={le:.3e}")
    assert mx <= FULL8_MAX and mean <= FULL8_MEAN and le <= gu.TOL_LSE, (mx, mean, le)


@pytest.mark.parametrize("case", [
    dict(n=2000, hq=4, hkv=1, d=128, tile=128, gran=1, seed=11, q_gain=2.0),      # the document bench.py's encode leg times: 16 ragged row blocks
    dict(n=4096, hq=2, hkv=1, d=128, tile=128, gran=128, seed=12, q_gain=2.0),    # the longest document of C4's recipe, page-granular
])
def test_encode_benched_sizes(case):
    assert _encode_case(**case) > 0


def test_c2_eight_way_head_shards_equal_the_unsharded_call():
    w = wl.config_8b_10k()
    world = 8
    shape, md = gu.decode_on_gpu(w)
    q, k, v = (t.cuda() for t in w.qkv(0))
    o_ref, lse_ref = api.sift_prefill_attention(shape, 0, q, k, v, md)
    la, ca = torch.from_numpy(w.la_blob).cuda(), torch.from_numpy(w.ca_blob).cuda()
    o = torch.full_like(q, float("nan"))
    lse = torch.full_like(lse_ref, float("nan"))
    for rank in range(world):
        sh = shard.head_shard(w.shape.n_q_heads, w.shape.n_kv_heads, rank, world)
        assert sh.n_kv == 1 and sh.n_q == 4
        sub = api.Shape.from_prompt(shard.shard_prompt_shape(w.shape, sh))
        la_off, ca_off = shard.shard_blob_offsets(w, sh, 0)
        md_s = api.sift_decode_metadata(sub, la, la_off, ca, ca_off)
        qs, ks, vs = shard.shard_views(q, k, v, sh)
        api.sift_prefill_attention(sub, 0, qs, ks, vs, md_s, o[:, sh.q0:sh.q1], lse[sh.q0:sh.q1])
    torch.cuda.synchronize()
    assert torch.equal(o, o_ref) and torch.equal(lse, lse_ref)
