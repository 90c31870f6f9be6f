"""The seeded input generator: shapes of BASELINE.json's configs, and that the only format knowledge it
uses (diagonal tile positions) agrees with the oracle's independent reader."""
import numpy as np

from oracle import sift_oracle as so
from paper_2606_09441_b200 import workload as wl


def test_config_shapes():
    c1, c2, c3 = wl.config_tiny(), wl.config_8b_10k(), wl.config_32k()
    assert c1.shape.n_tokens == 1088 and c1.shape.tile == 64 and c1.shape.head_dim == 64
    assert c2.shape.n_tokens == 10368 and (c2.shape.n_q_heads, c2.shape.n_kv_heads) == (32, 8)
    assert c3.shape.n_tokens == 32256 and c3.shape.pages(0) == 16
    lens = wl.ragged_doc_lens(wl.BASE_SEED)
    assert all(1024 <= x <= 4096 for x in lens) and sum(lens) + 512 <= 65536 and len(lens) <= 24
    assert c3.shape.la_bytes(0) == so.la_vector_bytes(16) and c3.shape.ca_bytes(0) == 250


def test_diagonal_tiles_set_and_densities():
    w = wl.config_8b_10k()
    sh = w.shape
    for h in (0, 7, 31):
        for d in (0, 9):
            lv = w.la_vec(0, h, d)
            assert all(so.la_tile_bit(lv, i, i) == 1 for i in range(8))
            off = [so.la_tile_bit(lv, i, j) for i in range(8) for j in range(i)]
        ca = np.concatenate([so.read_bits(w.ca_vec(0, h, d), 1024) for d in range(10)])
        assert abs(ca.mean() - w.p_cross[0, h]) < 0.03
    assert 0.2 <= w.p_loc.min() and w.p_loc.max() <= 0.4 and 0.1 <= w.p_cross.min() and w.p_cross.max() <= 0.3


def test_determinism_and_reorder_views():
    a, b = wl.config_tiny(), wl.config_tiny()
    assert np.array_equal(a.la_blob, b.la_blob) and np.array_equal(a.ca_blob, b.ca_blob)
    qa, ka, va = a.qkv(0)
    qb, kb, vb = b.qkv(0)
    assert qa.equal(qb) and ka.equal(kb) and va.equal(vb)
    r = a.reorder([3, 1, 0, 2])
    assert np.array_equal(r.la_vec(0, 1, 0), a.la_vec(0, 1, 3)) and np.array_equal(r.ca_vec(0, 0, 2), a.ca_vec(0, 0, 0))
    qr, kr, vr = r.qkv(0)
    assert qr[0:256].equal(qa[768:1024]) and kr[512:768].equal(ka[0:256]) and qr[1024:].equal(qa[1024:])


def test_marked_pairs_metric_matches_oracle_mask_count():
    """bench.py's pair count (integer arithmetic over MD-v1 arrays) against the oracle's explicit mask, G = 1 and G = tile."""
    import pytest
    from oracle import sift_oracle as so
    from paper_2606_09441_b200 import metrics
    for gran in (1, 16):
        w = wl.custom("pairs", doc_lens=(50, 33, 16, 70), query_len=21, tile=16, cross_gran=gran, p_loc=0.4, p_cross=0.35,
                      n_q_heads=2, seed=5)
        sh = w.shape
        md = so.decode_metadata(sh.doc_offsets, sh.query_len, sh.tile, gran, 1, 2, w.la_vec, w.ca_vec)
        got = metrics.marked_pairs_per_head(md, 0, sh.n_docs, gran)
        for h in range(2):
            la, ca = so.head_vectors(w, 0, h)
            assert int(got[h]) == so.marked_pairs(sh.doc_offsets, sh.query_len, sh.tile, gran, la, ca)
