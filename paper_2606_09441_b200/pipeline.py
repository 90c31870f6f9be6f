"""Host-buffer entry for one prefill layer: Q/K/V and the bit vectors start in pinned HOST memory, O ends there.

Stream plumbing only (every step of the path still runs in the library's kernels): the layer is cut into kv-head groups
(a kv head and its q-heads are an independent unit of the path); for each group the host->device copy
of its Q/K/V columns (cudaMemcpy2DAsync on the token-major [N][H][d] tensors), metadata decode + attention for its
q-heads, and the device->host copy of its O columns run on three streams, so that PCIe traffic in both directions
overlaps the kernels and each other instead of bracketing them.  bench.py's `e2e` leg times this.
"""
from __future__ import annotations

from typing import List

import numpy as np
import torch

from . import api

try:
    from cuda.bindings import runtime as _rt
except Exception:                       # pragma: no cover - older cuda-python layout
    from cuda import cudart as _rt


def _copy2d(dst_ptr: int, dpitch: int, src_ptr: int, spitch: int, width: int, height: int, kind, stream: torch.cuda.Stream):
    (err,) = _rt.cudaMemcpy2DAsync(dst_ptr, dpitch, src_ptr, spitch, width, height, kind, stream.cuda_stream)
    if err != _rt.cudaError_t.cudaSuccess:
        raise api.SiftError(f"cudaMemcpy2DAsync failed: {err}")


class HostLayerPipeline:
    """Reusable per-prompt-shape state: device buffers, one metadata buffer and sub-shape per kv-head group, streams."""

    def __init__(self, prompt_shape, device: str = "cuda", kv_whole: bool = True):
        # kv_whole: K and V (1/4 of the input bytes under 4:1 GQA) go up front as two contiguous copies instead of
        # per-group strided ones (rows of 256 B make poor DMA descriptors); Q and O are copied per group either way
        ps = prompt_shape
        self.ps = ps
        self.kv_whole = kv_whole
        self.n, self.hq, self.hkv, self.d = ps.n_tokens, ps.n_q_heads, ps.n_kv_heads, ps.head_dim
        self.hpg = self.hq // self.hkv
        dev = torch.device(device)
        self.q = torch.empty((self.n, self.hq, self.d), dtype=torch.bfloat16, device=dev)
        self.k = torch.empty((self.n, self.hkv, self.d), dtype=torch.bfloat16, device=dev)
        self.v = torch.empty_like(self.k)
        self.o = torch.empty_like(self.q)
        self.lse = torch.empty((self.hq, self.n), dtype=torch.float32, device=dev)
        self.sub = api.Shape(1, self.hpg, 1, self.d, ps.doc_offsets, ps.query_len, ps.tile, ps.cross_gran)
        nbytes = api.sift_metadata_size(self.sub)
        self.md: List[torch.Tensor] = [torch.empty(nbytes, dtype=torch.uint8, device=dev) for _ in range(self.hkv)]
        self.la_bytes = np.array([ps.la_bytes(p) for p in range(ps.n_docs)], dtype=np.int64)
        self.ca_bytes = np.array([ps.ca_bytes(p) for p in range(ps.n_docs)], dtype=np.int64)
        self.s_in, self.s_cmp, self.s_out = (torch.cuda.Stream(device=dev) for _ in range(3))
        self.ev_in = [torch.cuda.Event() for _ in range(self.hkv)]
        self.ev_cmp = [torch.cuda.Event() for _ in range(self.hkv)]
        self.la = self.ca = None

    def run(self, la_h: torch.Tensor, ca_h: torch.Tensor, la_doc_off, ca_doc_off, q_h: torch.Tensor, k_h: torch.Tensor,
            v_h: torch.Tensor, o_h: torch.Tensor, layer: int = 0) -> None:
        """All tensors pinned host memory; q_h/o_h [N,Hq,d], k_h/v_h [N,Hkv,d] bf16; la_h/ca_h the uint8 blobs (layout
        [layer][q_head][bytes] per document).  Returns after enqueueing; synchronise `self.s_out` (or call wait())."""
        if self.la is None or self.la.numel() != la_h.numel():
            self.la = torch.empty_like(la_h, device=self.q.device)
            self.ca = torch.empty_like(ca_h, device=self.q.device)
        H2D, D2H = _rt.cudaMemcpyKind.cudaMemcpyHostToDevice, _rt.cudaMemcpyKind.cudaMemcpyDeviceToHost
        cur = torch.cuda.current_stream()
        for s in (self.s_in, self.s_cmp, self.s_out):
            s.wait_stream(cur)
        n, d2 = self.n, self.d * 2
        qp, kp = self.hq * d2, self.hkv * d2                     # row pitches in bytes
        la_off = np.asarray(la_doc_off, dtype=np.int64)
        ca_off = np.asarray(ca_doc_off, dtype=np.int64)
        with torch.cuda.stream(self.s_in):
            self.la.copy_(la_h, non_blocking=True)
            self.ca.copy_(ca_h, non_blocking=True)
            if self.kv_whole:                                    # K, V in one contiguous copy each (see __init__)
                self.k.copy_(k_h, non_blocking=True)
                self.v.copy_(v_h, non_blocking=True)
        for g in range(self.hkv):
            h0 = g * self.hpg
            if not self.kv_whole:
                _copy2d(self.k.data_ptr() + g * d2, kp, k_h.data_ptr() + g * d2, kp, d2, n, H2D, self.s_in)
                _copy2d(self.v.data_ptr() + g * d2, kp, v_h.data_ptr() + g * d2, kp, d2, n, H2D, self.s_in)
            _copy2d(self.q.data_ptr() + h0 * d2, qp, q_h.data_ptr() + h0 * d2, qp, self.hpg * d2, n, H2D, self.s_in)
            self.ev_in[g].record(self.s_in)
            self.s_cmp.wait_event(self.ev_in[g])
            with torch.cuda.stream(self.s_cmp):
                # the q-heads of this group inside each document's [layer][q_head][bytes] blob
                lo = la_off + (layer * self.hq + h0) * self.la_bytes
                co = ca_off + (layer * self.hq + h0) * self.ca_bytes
                api.sift_decode_metadata(self.sub, self.la, lo, self.ca, co, self.md[g])
                api.sift_prefill_attention(self.sub, 0, self.q[:, h0:h0 + self.hpg], self.k[:, g:g + 1], self.v[:, g:g + 1],
                                           self.md[g], self.o[:, h0:h0 + self.hpg], self.lse[h0:h0 + self.hpg])
            self.ev_cmp[g].record(self.s_cmp)
            self.s_out.wait_event(self.ev_cmp[g])
            _copy2d(o_h.data_ptr() + h0 * d2, qp, self.o.data_ptr() + h0 * d2, qp, self.hpg * d2, n, D2H, self.s_out)
        cur.wait_stream(self.s_out)

    def wait(self) -> None:
        self.s_out.synchronize()
