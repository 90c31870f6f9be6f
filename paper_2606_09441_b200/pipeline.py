"""Host-buffer entry for one prefill layer: a thin holder around the C-ABI call ``sift_prefill_layer_host``
(include/sift.h; paper_2606_09441_b200/csrc/sift_pipeline.cu).  Q/K/V and the bit vectors start in pinned HOST memory,
O ends there; the per-kv-head-group H2D / decode + attention / D2H overlap on three streams happens inside the
library.  This class only keeps the device workspace and the context alive between calls (argument marshalling)."""
from __future__ import annotations

import torch

from . import api


class HostLayerPipeline:
    def __init__(self, prompt_shape, device: str = "cuda", shape: "api.Shape" = None):
        """prompt_shape: workload.PromptShape of one prompt; or shape: an api.Shape (e.g. Shape.from_batch)."""
        self.ps = prompt_shape
        self.shape = shape if shape is not None else api.Shape.from_prompt(prompt_shape)
        self.device = torch.device(device)
        self.ctx = api.HostContext()
        self.ws = None
        self._stream = None

    def run(self, la_h: torch.Tensor, ca_h: torch.Tensor, la_doc_off, ca_doc_off, q_h: torch.Tensor, k_h: torch.Tensor,
            v_h: torch.Tensor, o_h: torch.Tensor, layer: int = 0, lse_h: torch.Tensor = None, softmax_scale: float = 0.0) -> None:
        """Enqueues one layer on the current stream (which then waits for the whole pipeline); call wait() or
        synchronise that stream before reading o_h."""
        need = api.sift_prefill_layer_host_workspace_size(self.shape, la_h.numel(), ca_h.numel())
        if self.ws is None or self.ws.numel() < need:
            self.ws = torch.empty(need, dtype=torch.uint8, device=self.device)
        self._stream = torch.cuda.current_stream()
        api.sift_prefill_layer_host(self.ctx, self.shape, layer, la_h, la_doc_off, ca_h, ca_doc_off, q_h, k_h, v_h, o_h,
                                    self.ws, lse_h, softmax_scale, self._stream)

    def wait(self) -> None:
        if self._stream is not None:
            self._stream.synchronize()
