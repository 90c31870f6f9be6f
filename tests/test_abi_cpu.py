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


def test_v1_sized_structs_are_neither_over_read_nor_over_written():
    """A caller built against the header before the prompt fields passes struct_size = SIFT_SHAPE_SIZE_V1 and owns a
    sift_md_layout that ends before n_seg (include/sift.h: SIFT_MD_LAYOUT_SIZE_V1).  The bytes behind both structs are
    poisoned here: the library must ignore the ones behind the shape and leave the ones behind the layout alone."""
    shape_v1, lay_v1 = api.SiftShape.n_prompts.offset, api.SiftMdLayout.n_seg.offset
    full = api.Shape(2, 8, 4, 128, np.array([0, 300, 1000, 1130]), 77, 128, 1)
    want = api.sift_metadata_layout(full)
    assert want.struct_size == C.sizeof(api.SiftMdLayout)
    sbuf = (C.c_uint8 * (shape_v1 + 64))(*([0xCD] * (shape_v1 + 64)))     # garbage n_prompts / prompt pointers
    C.memmove(sbuf, C.byref(full.c), shape_v1)
    C.cast(sbuf, C.POINTER(C.c_uint32))[0] = shape_v1
    obuf = (C.c_uint8 * (lay_v1 + 64))(*([0xAB] * (lay_v1 + 64)))
    L = api.lib()
    rc = L.sift_metadata_layout(C.cast(sbuf, C.POINTER(api.SiftShape)), C.cast(obuf, C.POINTER(api.SiftMdLayout)))
    assert rc == 0, api.lib().sift_last_error()
    assert bytes(obuf[lay_v1:]) == b"\xab" * 64
    got = api.SiftMdLayout()
    C.memmove(C.byref(got), obuf, lay_v1)
    assert got.struct_size == lay_v1
    for name, _ in api.SiftMdLayout._fields_[1:]:
        if getattr(api.SiftMdLayout, name).offset < lay_v1:
            assert getattr(got, name) == getattr(want, name), name
    n = C.c_size_t(0)
    assert L.sift_metadata_size(C.cast(sbuf, C.POINTER(api.SiftShape)), C.byref(n)) == 0 and n.value == want.total_bytes
    ws = C.c_size_t(0)      # the host-buffer entry copies the shape: it must stop at struct_size too
    assert L.sift_prefill_layer_host_workspace_size(C.cast(sbuf, C.POINTER(api.SiftShape)), 1000, 1000, C.byref(ws)) == 0
    assert ws.value == api.sift_prefill_layer_host_workspace_size(full, 1000, 1000)


def test_one_prompt_given_as_arrays_is_the_single_prompt_shape():
    """api.Shape built by hand with prompt_* arrays of one prompt: the library takes n_prompts <= 1 as one prompt and
    reads query_len, so the binding folds the arrays into query_len and both sides size Q / O / LSE alike."""
    off = np.array([0, 300, 1000])
    a = api.Shape(1, 4, 2, 128, off, 0, 128, 1, prompt_doc_start=np.array([0, 2]), prompt_query_len=np.array([55]))
    b = api.Shape(1, 4, 2, 128, off, 55, 128, 1)
    assert a.query_len == 55 and a.c.n_prompts == 0 and a.n_tokens == b.n_tokens == 1055
    la, lb = api.sift_metadata_layout(a), api.sift_metadata_layout(b)
    assert la.n_tokens == lb.n_tokens == 1055 and la.total_bytes == lb.total_bytes
