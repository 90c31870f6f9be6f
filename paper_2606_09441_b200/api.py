"""ctypes binding of libsift_b200.so (include/sift.h).  Argument marshalling only: every step of the hot
path runs in the library's CUDA kernels.  There is no CPU fallback: a missing library raises."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Dict, Optional, Tuple

import numpy as np
import torch

from .build import LIB

SIFT_OK = 0
EXPORTS = ("sift_version", "sift_last_error", "sift_metadata_size", "sift_metadata_layout",
           "sift_decode_metadata", "sift_prefill_attention", "sift_dense_causal_attention", "sift_launch_count",
           "sift_encode_workspace_size", "sift_encode_output_sizes", "sift_encode_document",
           "sift_host_ctx_create", "sift_host_ctx_destroy", "sift_prefill_layer_host_workspace_size",
           "sift_prefill_layer_host", "sift_paper_index_offsets", "sift_export_paper_indices",
           "sift_prefill_attention_fp8", "sift_encode_document_static", "sift_encode_static_scratch_bytes",
           "sift_prefill_attention_rows")


class SiftShape(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_layers", C.c_int32), ("n_q_heads", C.c_int32),
                ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32), ("n_docs", C.c_int32),
                ("query_len", C.c_int32), ("tile", C.c_int32), ("cross_gran", C.c_int32),
                ("doc_offsets", C.POINTER(C.c_int32)),
                ("n_prompts", C.c_int32), ("prompt_doc_start", C.POINTER(C.c_int32)),
                ("prompt_query_len", C.POINTER(C.c_int32))]


class SiftMdLayout(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_tiles", C.c_int32), ("cross_cap", C.c_int32),
                ("local_cap", C.c_int32), ("n_mblocks", C.c_int32), ("n_items", C.c_int32)] + \
               [(n, C.c_size_t) for n in ("tile_base", "tile_seg", "tile_row0", "tile_rows", "cross_ptr", "cross_idx",
                                          "local_cnt", "local_ptr", "local_idx", "mblock_tile0", "sched", "counters",
                                          "total_bytes")] + \
               [("n_seg", C.c_int32), ("n_tokens", C.c_int32), ("seg_info", C.c_size_t)]


class SiftError(RuntimeError):
    pass


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB):
            raise SiftError(f"{LIB} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                            "(there is no CPU fallback)")
        L = C.CDLL(LIB)
        L.sift_version.restype = C.c_char_p
        L.sift_last_error.restype = C.c_char_p
        L.sift_launch_count.restype = C.c_int64
        L.sift_metadata_size.argtypes = [C.POINTER(SiftShape), C.POINTER(C.c_size_t)]
        L.sift_metadata_layout.argtypes = [C.POINTER(SiftShape), C.POINTER(SiftMdLayout)]
        L.sift_decode_metadata.argtypes = [C.POINTER(SiftShape), C.c_void_p, C.POINTER(C.c_int64), C.c_void_p,
                                           C.POINTER(C.c_int64), C.c_void_p, C.c_size_t, C.c_void_p]
        L.sift_prefill_attention.argtypes = [C.POINTER(SiftShape), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                             C.c_int64, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_int64,
                                             C.c_void_p, C.c_float, C.c_void_p]
        a = L.sift_prefill_attention.argtypes
        L.sift_prefill_attention_rows.argtypes = a[:2] + [C.c_int32, C.c_int32] + a[2:]
        L.sift_dense_causal_attention.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p,
                                                  C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_void_p, C.c_int64,
                                                  C.c_void_p, C.c_float, C.c_void_p]
        L.sift_encode_workspace_size.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]
        L.sift_encode_document.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p,
                                           C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_float, C.c_float, C.c_float,
                                           C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        L.sift_encode_output_sizes.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
        L.sift_encode_static_scratch_bytes.restype = C.c_size_t
        L.sift_encode_document_static.argtypes = L.sift_encode_document.argtypes[:-3] + [C.c_void_p]
        L.sift_host_ctx_create.argtypes = [C.POINTER(C.c_void_p)]
        L.sift_host_ctx_destroy.argtypes = [C.c_void_p]
        L.sift_prefill_layer_host_workspace_size.argtypes = [C.POINTER(SiftShape), C.c_size_t, C.c_size_t, C.POINTER(C.c_size_t)]
        L.sift_prefill_layer_host.argtypes = [C.c_void_p, C.POINTER(SiftShape), C.c_int32,
                                              C.c_void_p, C.c_size_t, C.POINTER(C.c_int64),
                                              C.c_void_p, C.c_size_t, C.POINTER(C.c_int64),
                                              C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64,
                                              C.c_void_p, C.c_int64, C.c_void_p, C.c_float, C.c_void_p, C.c_size_t, C.c_void_p]
        L.sift_paper_index_offsets.argtypes = [C.POINTER(SiftShape), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.sift_export_paper_indices.argtypes = [C.POINTER(SiftShape), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                                C.c_int64, C.c_void_p]
        L.sift_prefill_attention_fp8.argtypes = [C.POINTER(SiftShape), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                                 C.c_int64, C.c_int64, C.c_int64, C.POINTER(C.c_float), C.POINTER(C.c_float),
                                                 C.POINTER(C.c_float), C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p,
                                                 C.c_float, C.c_void_p]
        _lib = L
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != SIFT_OK:
        raise SiftError(f"{what} failed ({rc}): {lib().sift_last_error().decode()}")


def sift_version() -> str:
    return lib().sift_version().decode()


def sift_launch_count() -> int:
    return int(lib().sift_launch_count())


@dataclass
class Shape:
    """Python mirror of sift_shape; keeps the host offset array alive."""
    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    doc_offsets: np.ndarray
    query_len: int
    tile: int
    cross_gran: int = 1
    # several prompts in one call (sift.h): documents [prompt_doc_start[p], prompt_doc_start[p+1]) + a query each
    prompt_doc_start: Optional[np.ndarray] = None
    prompt_query_len: Optional[np.ndarray] = None

    def __post_init__(self):
        self.doc_offsets = np.ascontiguousarray(self.doc_offsets, dtype=np.int32)
        ip = C.POINTER(C.c_int32)
        n_prompts, pds, pql = 0, ip(), ip()
        if self.prompt_query_len is not None and len(self.prompt_query_len) == 1:
            # the library reads n_prompts <= 1 as "one prompt" and takes query_len: say it that way here too
            self.query_len = int(np.asarray(self.prompt_query_len)[0])
            self.prompt_doc_start = self.prompt_query_len = None
        if self.prompt_doc_start is not None:
            self.prompt_doc_start = np.ascontiguousarray(self.prompt_doc_start, dtype=np.int32)
            self.prompt_query_len = np.ascontiguousarray(self.prompt_query_len, dtype=np.int32)
            n_prompts = len(self.prompt_query_len)
            pds, pql = self.prompt_doc_start.ctypes.data_as(ip), self.prompt_query_len.ctypes.data_as(ip)
        self._c = SiftShape(C.sizeof(SiftShape), self.n_layers, self.n_q_heads, self.n_kv_heads, self.head_dim,
                            len(self.doc_offsets) - 1, self.query_len, self.tile, self.cross_gran,
                            self.doc_offsets.ctypes.data_as(ip), n_prompts, pds, pql)

    @classmethod
    def from_prompt(cls, ps) -> "Shape":
        return cls(ps.n_layers, ps.n_q_heads, ps.n_kv_heads, ps.head_dim, ps.doc_offsets, ps.query_len, ps.tile,
                   ps.cross_gran)

    @classmethod
    def from_batch(cls, b) -> "Shape":
        """b: workload.BatchWorkload (prompts packed back to back on the token axis)."""
        if len(b.members) == 1:
            return cls.from_prompt(b.members[0].shape)
        hs = b.head_shape
        off = np.concatenate([[0], np.cumsum(np.asarray(b.doc_lens, dtype=np.int64))])
        return cls(hs.n_layers, hs.n_q_heads, hs.n_kv_heads, hs.head_dim, off, 0, hs.tile, hs.cross_gran,
                   b.prompt_doc_start, b.prompt_query_len)

    @property
    def n_tokens(self) -> int:
        if self.prompt_query_len is not None:   # two or more prompts (__post_init__ folds one prompt into query_len)
            return int(self.doc_offsets[-1]) + int(self.prompt_query_len.sum())
        return int(self.doc_offsets[-1]) + self.query_len

    @property
    def c(self) -> SiftShape:
        return self._c


def sift_metadata_layout(shape: Shape) -> SiftMdLayout:
    lay = SiftMdLayout()
    _check(lib().sift_metadata_layout(C.byref(shape.c), C.byref(lay)), "sift_metadata_layout")
    return lay


def sift_metadata_size(shape: Shape) -> int:
    n = C.c_size_t(0)
    _check(lib().sift_metadata_size(C.byref(shape.c), C.byref(n)), "sift_metadata_size")
    return int(n.value)


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _i64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int64)


def sift_decode_metadata(shape: Shape, la_base: torch.Tensor, la_doc_off, ca_base: torch.Tensor, ca_doc_off,
                         metadata: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """la_base/ca_base: uint8 CUDA tensors; returns the metadata buffer (uint8 CUDA tensor)."""
    assert la_base.is_cuda and ca_base.is_cuda and la_base.dtype == torch.uint8 and ca_base.dtype == torch.uint8
    if metadata is None:
        metadata = torch.empty(sift_metadata_size(shape), dtype=torch.uint8, device=la_base.device)
    lo, co = _i64(la_doc_off), _i64(ca_doc_off)
    rc = lib().sift_decode_metadata(C.byref(shape.c), la_base.data_ptr(), lo.ctypes.data_as(C.POINTER(C.c_int64)),
                                    ca_base.data_ptr(), co.ctypes.data_as(C.POINTER(C.c_int64)),
                                    metadata.data_ptr(), metadata.numel(), _stream(stream))
    _check(rc, "sift_decode_metadata")
    return metadata


def _check_qkv(q, k, v):
    for t in (q, k, v):
        assert t.is_cuda and t.dtype == torch.bfloat16 and t.dim() == 3 and t.stride(2) == 1 and t.stride(1) == t.shape[2]


def sift_prefill_attention(shape: Shape, layer: int, q: torch.Tensor, k: torch.Tensor, v: torch.Tensor,
                           metadata: torch.Tensor, out: Optional[torch.Tensor] = None,
                           lse: Optional[torch.Tensor] = None, softmax_scale: float = 0.0, return_lse: bool = True,
                           stream=None) -> Tuple[torch.Tensor, Optional[torch.Tensor]]:
    _check_qkv(q, k, v)
    if out is None:
        out = torch.empty_like(q)
    if lse is None and return_lse:
        lse = torch.empty((q.shape[1], q.shape[0]), dtype=torch.float32, device=q.device)
    rc = lib().sift_prefill_attention(C.byref(shape.c), layer, q.data_ptr(), k.data_ptr(), v.data_ptr(),
                                      q.stride(0), k.stride(0), v.stride(0), metadata.data_ptr(), out.data_ptr(),
                                      out.stride(0), lse.data_ptr() if lse is not None else None,
                                      float(softmax_scale), _stream(stream))
    _check(rc, "sift_prefill_attention")
    return out, lse


def sift_prefill_attention_rows(shape: Shape, layer: int, row_begin: int, row_end: int, q: torch.Tensor, k: torch.Tensor,
                                v: torch.Tensor, metadata: torch.Tensor, out: torch.Tensor,
                                lse: Optional[torch.Tensor] = None, softmax_scale: float = 0.0, stream=None) -> None:
    """Rows [row_begin, row_end) of sift_prefill_attention (chunked prefill): `out` [N, Hq, d] and `lse` [Hq, N] are the
    full-size arrays, only the rows of the range are written."""
    _check_qkv(q, k, v)
    rc = lib().sift_prefill_attention_rows(C.byref(shape.c), layer, int(row_begin), int(row_end), q.data_ptr(), k.data_ptr(),
                                           v.data_ptr(), q.stride(0), k.stride(0), v.stride(0), metadata.data_ptr(),
                                           out.data_ptr(), out.stride(0), lse.data_ptr() if lse is not None else None,
                                           float(softmax_scale), _stream(stream))
    _check(rc, "sift_prefill_attention_rows")


def sift_dense_causal_attention(q: torch.Tensor, k: torch.Tensor, v: torch.Tensor, out: Optional[torch.Tensor] = None,
                                lse: Optional[torch.Tensor] = None, softmax_scale: float = 0.0,
                                return_lse: bool = True, stream=None) -> Tuple[torch.Tensor, Optional[torch.Tensor]]:
    _check_qkv(q, k, v)
    if out is None:
        out = torch.empty_like(q)
    if lse is None and return_lse:
        lse = torch.empty((q.shape[1], q.shape[0]), dtype=torch.float32, device=q.device)
    rc = lib().sift_dense_causal_attention(q.shape[0], q.shape[1], k.shape[1], q.shape[2], q.data_ptr(), k.data_ptr(),
                                           v.data_ptr(), q.stride(0), k.stride(0), v.stride(0), out.data_ptr(),
                                           out.stride(0), lse.data_ptr() if lse is not None else None,
                                           float(softmax_scale), _stream(stream))
    _check(rc, "sift_dense_causal_attention")
    return out, lse


def metadata_views(shape: Shape, metadata: torch.Tensor) -> Dict[str, torch.Tensor]:
    """int32 views of the MD-v1 arrays inside the buffer (no copies)."""
    lay = sift_metadata_layout(shape)
    m32 = metadata.view(torch.int32)
    L, H, D, NT = shape.n_layers, shape.n_q_heads, len(shape.doc_offsets) - 1, lay.n_tiles

    def v(off, *dims):
        n = int(np.prod(dims))
        return m32[off // 4: off // 4 + n].view(*dims)
    return {
        "tile_base": v(lay.tile_base, lay.n_seg + 1), "tile_seg": v(lay.tile_seg, NT), "tile_row0": v(lay.tile_row0, NT),
        "tile_rows": v(lay.tile_rows, NT), "cross_ptr": v(lay.cross_ptr, L, H, D + 1),
        "cross_idx": v(lay.cross_idx, L, H, lay.cross_cap), "local_cnt": v(lay.local_cnt, L, H, NT),
        "local_ptr": v(lay.local_ptr, L, H, NT + 1), "local_idx": v(lay.local_idx, L, H, lay.local_cap),
        "mblock_tile0": v(lay.mblock_tile0, lay.n_mblocks + 1), "sched": v(lay.sched, L, lay.n_items),
        "counters": v(lay.counters, L, 2), "seg_info": v(lay.seg_info, lay.n_seg, 4),
    }


def sift_encode_document(q: torch.Tensor, k: torch.Tensor, lse: torch.Tensor, tile: int, cross_gran: int = 1,
                         alpha: float = 1e-3, beta: float = 1e-2, gamma: float = 0.1, softmax_scale: float = 0.0,
                         stream=None) -> Tuple[torch.Tensor, torch.Tensor]:
    """Offline metadata generation for one document and layer (include/sift.h).  q [L,Hq,d], k [L,Hkv,d] bf16 CUDA,
    lse [Hq,L] fp32 CUDA (from sift_dense_causal_attention on the document).  Returns (la [Hq, la_bytes], ca [Hq, ca_bytes])."""
    assert q.is_cuda and k.is_cuda and lse.is_cuda and q.dtype == torch.bfloat16 and k.dtype == torch.bfloat16
    assert lse.dtype == torch.float32 and lse.is_contiguous() and q.stride(2) == 1 and k.stride(2) == 1
    assert q.stride(1) == q.shape[2] and k.stride(1) == k.shape[2]
    n, hq, d = q.shape
    hkv = k.shape[1]
    lb, cb, nb = C.c_size_t(), C.c_size_t(), C.c_size_t()
    _check(lib().sift_encode_output_sizes(n, tile, cross_gran, C.byref(lb), C.byref(cb)), "sift_encode_output_sizes")
    la_bytes, ca_bytes = int(lb.value), int(cb.value)
    _check(lib().sift_encode_workspace_size(n, hq, tile, C.byref(nb)), "sift_encode_workspace_size")
    ws = torch.empty(nb.value, dtype=torch.uint8, device=q.device)
    la = torch.empty((hq, la_bytes), dtype=torch.uint8, device=q.device)
    ca = torch.empty((hq, ca_bytes), dtype=torch.uint8, device=q.device)
    _check(lib().sift_encode_document(n, hq, hkv, d, tile, cross_gran, q.data_ptr(), k.data_ptr(), q.stride(0), k.stride(0),
                                      lse.data_ptr(), alpha, beta, gamma, softmax_scale, la.data_ptr(), ca.data_ptr(),
                                      ws.data_ptr(), nb.value, _stream(stream)), "sift_encode_document")
    return la, ca


def sift_encode_static_scratch_bytes() -> int:
    """Size of the encoder's built-in scratch array (include/sift.h: SIFT_ENCODE_STATIC_SCRATCH_BYTES)."""
    return int(lib().sift_encode_static_scratch_bytes())


def sift_encode_document_static(q: torch.Tensor, k: torch.Tensor, lse: torch.Tensor, la: torch.Tensor, ca: torch.Tensor,
                                tile: int, cross_gran: int = 1, alpha: float = 1e-3, beta: float = 1e-2,
                                gamma: float = 0.1, softmax_scale: float = 0.0, stream=None) -> None:
    """sift_encode_document for a caller that may not allocate device memory (include/sift.h): the scratch is an array
    inside the library, so this wrapper allocates nothing either and the caller hands in the outputs, la [Hq, la_bytes]
    and ca [Hq, ca_bytes] uint8 CUDA (sizes from sift_encode_output_sizes).  Documents whose scratch exceeds
    sift_encode_static_scratch_bytes() raise SiftError.  All calls on one GPU share that one array: keep them ordered."""
    assert q.is_cuda and k.is_cuda and lse.is_cuda and q.dtype == torch.bfloat16 and k.dtype == torch.bfloat16
    assert lse.dtype == torch.float32 and lse.is_contiguous() and q.stride(2) == 1 and k.stride(2) == 1
    assert q.stride(1) == q.shape[2] and k.stride(1) == k.shape[2]
    n, hq, d = q.shape
    la_bytes, ca_bytes = sift_encode_output_sizes(n, tile, cross_gran)
    for t, nb in ((la, la_bytes), (ca, ca_bytes)):
        assert t.is_cuda and t.dtype == torch.uint8 and t.is_contiguous() and tuple(t.shape) == (hq, nb), (t.shape, (hq, nb))
    _check(lib().sift_encode_document_static(n, hq, k.shape[1], d, tile, cross_gran, q.data_ptr(), k.data_ptr(), q.stride(0),
                                             k.stride(0), lse.data_ptr(), alpha, beta, gamma, softmax_scale, la.data_ptr(),
                                             ca.data_ptr(), _stream(stream)), "sift_encode_document_static")


def sift_encode_output_sizes(doc_len: int, tile: int, cross_gran: int) -> Tuple[int, int]:
    """Bytes of one q-head's LA / CA vector of a document (include/sift.h)."""
    lb, cb = C.c_size_t(), C.c_size_t()
    _check(lib().sift_encode_output_sizes(doc_len, tile, cross_gran, C.byref(lb), C.byref(cb)), "sift_encode_output_sizes")
    return int(lb.value), int(cb.value)


class HostContext:
    """sift_host_ctx (include/sift.h): the three internal streams + events of sift_prefill_layer_host."""

    def __init__(self):
        self._h = C.c_void_p()
        _check(lib().sift_host_ctx_create(C.byref(self._h)), "sift_host_ctx_create")

    def close(self):
        if self._h:
            lib().sift_host_ctx_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def sift_prefill_layer_host_workspace_size(shape: Shape, la_blob_bytes: int, ca_blob_bytes: int) -> int:
    n = C.c_size_t(0)
    _check(lib().sift_prefill_layer_host_workspace_size(C.byref(shape.c), la_blob_bytes, ca_blob_bytes, C.byref(n)),
           "sift_prefill_layer_host_workspace_size")
    return int(n.value)


def sift_prefill_layer_host(ctx: HostContext, shape: Shape, layer: int, la_h: torch.Tensor, la_doc_off,
                            ca_h: torch.Tensor, ca_doc_off, q_h: torch.Tensor, k_h: torch.Tensor, v_h: torch.Tensor,
                            o_h: torch.Tensor, workspace: torch.Tensor, lse_h: Optional[torch.Tensor] = None,
                            softmax_scale: float = 0.0, stream=None) -> None:
    """All *_h tensors are HOST tensors (pinned for asynchronous copies); workspace is a uint8 CUDA tensor of at least
    sift_prefill_layer_host_workspace_size bytes.  Enqueues only: synchronise `stream` before reading o_h."""
    for t in (la_h, ca_h, q_h, k_h, v_h, o_h):
        assert not t.is_cuda
    assert workspace.is_cuda and workspace.dtype == torch.uint8
    for t in (q_h, k_h, v_h, o_h):
        assert t.dtype == torch.bfloat16 and t.dim() == 3 and t.stride(2) == 1 and t.stride(1) == t.shape[2]
    lo, co = _i64(la_doc_off), _i64(ca_doc_off)
    rc = lib().sift_prefill_layer_host(ctx._h, C.byref(shape.c), layer,
                                       la_h.data_ptr(), la_h.numel(), lo.ctypes.data_as(C.POINTER(C.c_int64)),
                                       ca_h.data_ptr(), ca_h.numel(), co.ctypes.data_as(C.POINTER(C.c_int64)),
                                       q_h.data_ptr(), k_h.data_ptr(), v_h.data_ptr(), q_h.stride(0), k_h.stride(0),
                                       v_h.stride(0), o_h.data_ptr(), o_h.stride(0),
                                       lse_h.data_ptr() if lse_h is not None else None, float(softmax_scale),
                                       workspace.data_ptr(), workspace.numel(), _stream(stream))
    _check(rc, "sift_prefill_layer_host")


def sift_paper_index_offsets(shape: Shape, layer: int, metadata: torch.Tensor, stream=None) -> torch.Tensor:
    """int64 CUDA tensor [n_q_heads, NT + 1] (include/sift.h: the paper's per-(head, M-block) list offsets)."""
    nt = sift_metadata_layout(shape).n_tiles
    ptr = torch.empty((shape.n_q_heads, nt + 1), dtype=torch.int64, device=metadata.device)
    _check(lib().sift_paper_index_offsets(C.byref(shape.c), layer, metadata.data_ptr(), ptr.data_ptr(), _stream(stream)),
           "sift_paper_index_offsets")
    return ptr


def sift_export_paper_indices(shape: Shape, layer: int, metadata: torch.Tensor, ptr: torch.Tensor, idx: torch.Tensor,
                              stream=None) -> torch.Tensor:
    """idx: int32 CUDA tensor [n_q_heads, head_stride], sized by the caller from ptr[:, -1]."""
    assert idx.is_cuda and idx.dtype == torch.int32 and idx.dim() == 2 and idx.stride(1) == 1
    _check(lib().sift_export_paper_indices(C.byref(shape.c), layer, metadata.data_ptr(), ptr.data_ptr(), idx.data_ptr(),
                                           idx.stride(0), _stream(stream)), "sift_export_paper_indices")
    return idx


def sift_prefill_attention_fp8(shape: Shape, layer: int, q8: torch.Tensor, k8: torch.Tensor, v8: torch.Tensor,
                               q_scale, k_scale, v_scale, metadata: torch.Tensor, out: Optional[torch.Tensor] = None,
                               lse: Optional[torch.Tensor] = None, softmax_scale: float = 0.0, stream=None
                               ) -> Tuple[torch.Tensor, torch.Tensor]:
    """q8 [N, Hq, 128], k8, v8 [N, Hkv, 128]: uint8 CUDA tensors holding e4m3 bytes; scales: float32 host arrays."""
    for t in (q8, k8, v8):
        assert t.is_cuda and t.dtype == torch.uint8 and t.dim() == 3 and t.stride(2) == 1 and t.stride(1) == t.shape[2]
    if out is None:
        out = torch.empty(q8.shape, dtype=torch.bfloat16, device=q8.device)
    if lse is None:
        lse = torch.empty((q8.shape[1], q8.shape[0]), dtype=torch.float32, device=q8.device)
    fp = C.POINTER(C.c_float)
    qs, ks, vs = (np.ascontiguousarray(a, dtype=np.float32) for a in (q_scale, k_scale, v_scale))
    rc = lib().sift_prefill_attention_fp8(C.byref(shape.c), layer, q8.data_ptr(), k8.data_ptr(), v8.data_ptr(),
                                          q8.stride(0), k8.stride(0), v8.stride(0), qs.ctypes.data_as(fp),
                                          ks.ctypes.data_as(fp), vs.ctypes.data_as(fp), metadata.data_ptr(),
                                          out.data_ptr(), out.stride(0), lse.data_ptr(), float(softmax_scale), _stream(stream))
    _check(rc, "sift_prefill_attention_fp8")
    return out, lse
