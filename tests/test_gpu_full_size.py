"""-m gpu parity at BASELINE.json's full sizes, in the launch configuration bench.py times:
C2 and C3 on every head and every row; C4 on every head with a row in every query tile (so that all four kv-head
groups of its schedule are compared) plus ragged tails and document boundaries; C5 on the real 32-layer stack with the
survey's sample plan: all heads of layers {0, 15, 31} for ordering 0, and 8 seeded (head, tile) pairs incl. a query
tile for every (layer, ordering).  Q/K/V are generated one layer at a time."""
import numpy as np
import pytest
import torch

from paper_2606_09441_b200 import api, workload as wl
from oracle import sift_oracle as so
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu


def _check(name, errs):
    print(f"[parity-full] {name}: max_abs={errs[0]:.3e} mean_abs={errs[1]:.3e} lse={errs[2]:.3e}")
    assert errs[0] <= gu.TOL_MAX and errs[1] <= gu.TOL_MEAN and errs[2] <= gu.TOL_LSE, (name, errs)


@pytest.mark.parametrize("cfg", ["8b-10k", "32k"])
def test_every_head_every_row(cfg):
    w = wl.CONFIGS[cfg]()
    _, _, o, lse = gu.run_sift(w)
    assert torch.isfinite(o.float()).all()
    _check(cfg + " all heads x all rows", gu.attention_errors(w, 0, o, lse, range(w.shape.n_q_heads), range(w.shape.n_tokens)))


def rows_one_per_tile(w, seed=0):
    """One seeded row inside every query tile, the last row of every tile (ragged tails), document boundaries."""
    sh = w.shape
    tt = so.tile_tables(sh.doc_offsets, sh.query_len, sh.tile)
    r = np.random.default_rng(seed)
    rows = set(gu.sample_rows(w, n_per_seg=2, seed=seed))
    for r0, nr in zip(tt["tile_row0"], tt["tile_rows"]):
        rows.add(int(r0) + int(r.integers(0, int(nr))))
        rows.add(int(r0) + int(nr) - 1)
    return sorted(rows)


def test_64k_every_head_every_tile():
    w = wl.config_64k_ragged()
    _, _, o, lse = gu.run_sift(w)
    assert torch.isfinite(o.float()).all()
    _check("64k-ragged all heads x (row per tile + tails + boundaries)",
           gu.attention_errors(w, 0, o, lse, range(w.shape.n_q_heads), rows_one_per_tile(w)))


def test_full_stack_32_layers_sample_plan():
    L = 32
    w0 = wl.config_full_stack(n_layers=L)
    orders = wl.stack_orderings(w0, 4)
    off0 = [int(x) for x in w0.shape.doc_offsets]
    la, ca = torch.from_numpy(w0.la_blob).cuda(), torch.from_numpy(w0.ca_blob).cuda()
    cases = []
    for perm in orders:
        w = w0.reorder(perm)
        shape = api.Shape.from_prompt(w.shape)
        md = api.sift_decode_metadata(shape, la, w.la_doc_off, ca, w.ca_doc_off)   # ONE decode call for all 32 layers
        rows = torch.cat([torch.arange(off0[d], off0[d + 1]) for d in perm] + [torch.arange(off0[-1], w0.shape.n_tokens)])
        tt = so.tile_tables(w.shape.doc_offsets, w.shape.query_len, w.shape.tile)
        cases.append((w, shape, md, rows, tt))
    torch.cuda.synchronize()
    rng = np.random.default_rng(20260609)
    sh = w0.shape
    worst = [0.0, 0.0, 0.0]
    for layer in range(L):
        q0, k0, v0 = w0.qkv(layer)                       # identity ordering; a re-ordered prompt permutes row blocks
        for oi, (w, shape, md, rows, tt) in enumerate(cases):
            q, k, v = (t.index_select(0, rows) for t in (q0, k0, v0)) if oi else (q0, k0, v0)
            o, lse = api.sift_prefill_attention(shape, layer, q.cuda(), k.cuda(), v.cuda(), md)
            torch.cuda.synchronize()
            o_c, lse_c = o.float().cpu(), lse.cpu()
            nt = int(tt["NT"])
            first_q = int(tt["tile_base"][sh.n_docs])
            tiles = [int(x) for x in rng.integers(0, first_q, 7)] + [int(rng.integers(first_q, nt))]   # 7 doc tiles + a query tile
            heads = [int(x) for x in rng.integers(0, sh.n_q_heads, 8)]
            for h, t in zip(heads, tiles):
                rws = list(range(int(tt["tile_row0"][t]), int(tt["tile_row0"][t]) + int(tt["tile_rows"][t])))
                la_v, ca_v = so.head_vectors(w, layer, h)
                oo, ll = so.sift_attention_rows(q, k, v, h, w.shape.doc_offsets, sh.query_len, sh.tile, sh.cross_gran, la_v, ca_v, rws)
                d = (o_c[rws, h, :] - oo).abs()
                worst = [max(worst[0], float(d.max())), max(worst[1], float(d.mean())), max(worst[2], float((lse_c[h, rws] - ll).abs().max()))]
            if oi == 0 and layer in (0, 15, 31):
                _check(f"C5 layer {layer} ordering 0, all heads x all rows",
                       gu.attention_errors(w, layer, o, lse, range(sh.n_q_heads), range(sh.n_tokens)))
    _check("C5 32 layers x 4 orderings x 8 (head, tile) pairs (worst tile)", worst)
