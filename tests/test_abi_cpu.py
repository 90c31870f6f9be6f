"""No-GPU checks of the C-ABI library: it builds, loads, exports every symbol include/sift.h declares, its host-side
layout arithmetic agrees with the oracle's capacities, and bad arguments are rejected without touching a device."""
import ctypes as C
import re

import numpy as np
import pytest

from oracle import sift_oracle as so
from paper_2606_09441_b200 import api, build, workload as wl


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build_library()


def test_exports_match_header():
    hdr = open(build.ROOT + "/include/sift.h").read()
    declared = set(re.findall(r"\b(sift_[a-z0-9_]+)\s*\(", hdr))
    declared -= {"sift_status"}
    assert declared == set(api.EXPORTS), declared ^ set(api.EXPORTS)
    L = C.CDLL(build.LIB)
    for name in declared:
        assert hasattr(L, name), name
    assert "sift-b200" in api.sift_version()


@pytest.mark.parametrize("cfg", ["tiny", "8b-10k", "32k", "64k-ragged", "32k-paged"])
def test_layout_matches_oracle_capacities(cfg):
    w = wl.CONFIGS[cfg]()
    sh = w.shape
    lay = api.sift_metadata_layout(api.Shape.from_prompt(sh))
    tt = so.tile_tables(sh.doc_offsets, sh.query_len, sh.tile)
    assert lay.n_tiles == tt["NT"]
    assert lay.cross_cap == so.cross_capacity(sh.doc_offsets, sh.cross_gran)
    assert lay.local_cap == so.local_capacity(tt)
    assert lay.total_bytes == api.sift_metadata_size(api.Shape.from_prompt(sh))
    offs = [lay.tile_base, lay.tile_seg, lay.tile_row0, lay.tile_rows, lay.cross_ptr, lay.cross_idx, lay.local_cnt,
            lay.local_ptr, lay.local_idx, lay.mblock_tile0, lay.sched, lay.counters, lay.total_bytes]
    assert offs == sorted(offs) and all(o % 128 == 0 for o in offs)


def test_bad_arguments_rejected():
    good = dict(n_layers=1, n_q_heads=4, n_kv_heads=2, head_dim=64, doc_offsets=np.array([0, 100, 200]), query_len=10,
                tile=64)
    api.sift_metadata_size(api.Shape(**good))
    api.sift_metadata_size(api.Shape(**{**good, "cross_gran": 64}))    # page-granular CA: G = tile
    api.sift_metadata_size(api.Shape(**{**good, "doc_offsets": np.arange(0, 513 * 8, 8)}))   # SIFT_MAX_DOCS = 512 documents
    for bad in (dict(head_dim=96), dict(tile=32), dict(cross_gran=32), dict(n_kv_heads=3),
                dict(doc_offsets=np.array([0, 100, 100])), dict(doc_offsets=np.array([1, 100])),
                dict(doc_offsets=np.arange(0, 64 * 600, 64)), dict(doc_offsets=np.arange(0, 514 * 8, 8))):   # > SIFT_MAX_DOCS
        with pytest.raises(api.SiftError):
            api.sift_metadata_size(api.Shape(**{**good, **bad}))
    # NULL device pointers are refused before any launch
    sh = api.Shape(**good)
    rc = api.lib().sift_decode_metadata(C.byref(sh.c), None, None, None, None, None, 0, None)
    assert rc == -1 and b"NULL" in api.lib().sift_last_error()
    rc = api.lib().sift_prefill_attention(C.byref(sh.c), 0, None, None, None, 0, 0, 0, None, None, 0, None, 0.0, None)
    assert rc == -1
    rc = api.lib().sift_dense_causal_attention(128, 4, 2, 80, None, None, None, 0, 0, 0, None, 0, None, 0.0, None)
    assert rc == -2
