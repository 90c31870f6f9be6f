"""Seeded synthetic RAG-prompt inputs (bit vectors + Q/K/V) for the SIFT hot path.

This module is INPUT GENERATION ONLY.  It holds none of the method's arithmetic
(no mask expansion, no decode, no attention); the oracle (``oracle/``) and the
CUDA path (``paper_2606_09441_b200/csrc``) both consume the arrays it returns and
neither imports the other.  The only format knowledge used here is the position
of the diagonal tiles inside an LA vector (row-major lower
triangle, MSB-first) because BASELINE.json's configs say "diagonal tiles always
set"; ``tests/test_workload.py`` checks that claim with the oracle's own reader.

Stand-in statement: the paper measures on
LongBench-derived RAG prompts.  Those items are not in this
repository and are not reconstructed; only shapes (Llama-8B-class GQA 32/8x128,
PAPER.md:L261), document lengths and mark densities
are borrowed, as fixed by BASELINE.json ``configs``.

Layout of the bit-vector blobs: one blob per document,
``[layer][q_head][bytes]`` contiguous; ``la_doc_off[pos]``/``ca_doc_off[pos]``
give the byte offset of the blob of the document standing at prompt position
``pos``.  Re-ordering a prompt permutes those offsets ("vectors travel with
their doc", BASELINE.json config 5).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Callable, Dict, List, Optional, Sequence, Tuple

import numpy as np
import torch

BASE_SEED = 20260609
# stream ids
_S_Q, _S_K, _S_V, _S_LA, _S_CA, _S_DENS, _S_LEN, _S_SCALE, _S_ORDER = 1, 2, 3, 4, 5, 6, 7, 8, 9


def _rng(*key: int) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([int(k) & 0xFFFFFFFF for k in key]))


def _torch_gen(*key: int) -> torch.Generator:
    s = np.random.SeedSequence([int(k) & 0xFFFFFFFF for k in key]).generate_state(1, dtype=np.uint64)[0]
    g = torch.Generator(device="cpu")
    g.manual_seed(int(s >> np.uint64(1)))
    return g


def ceil_div(a: int, b: int) -> int:
    return -(-a // b)


@dataclass(frozen=True)
class PromptShape:
    """Static description of one prompt (documents in prompt order, then the query)."""

    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    doc_lens: Tuple[int, ...]
    query_len: int
    tile: int
    cross_gran: int = 1

    @property
    def n_docs(self) -> int:
        return len(self.doc_lens)

    @property
    def doc_offsets(self) -> np.ndarray:
        off = np.zeros(self.n_docs + 1, dtype=np.int32)
        off[1:] = np.cumsum(np.asarray(self.doc_lens, dtype=np.int64))
        return off

    @property
    def n_tokens(self) -> int:
        return int(sum(self.doc_lens)) + self.query_len

    def pages(self, d: int) -> int:
        return ceil_div(self.doc_lens[d], self.tile)

    def la_bits(self, d: int) -> int:
        p = self.pages(d)
        return p * (p + 1) // 2

    def ca_bits(self, d: int) -> int:
        return ceil_div(self.doc_lens[d], self.cross_gran)

    def la_bytes(self, d: int) -> int:
        return ceil_div(self.la_bits(d), 8)

    def ca_bytes(self, d: int) -> int:
        return ceil_div(self.ca_bits(d), 8)


@dataclass
class Workload:
    name: str
    shape: PromptShape
    seed: int
    doc_ids: Tuple[int, ...]            # identity of the document at each prompt position
    la_blob: np.ndarray                  # uint8, all documents
    ca_blob: np.ndarray                  # uint8, all documents
    la_doc_off: np.ndarray               # int64 [n_docs], by prompt position
    ca_doc_off: np.ndarray               # int64 [n_docs], by prompt position
    p_loc: np.ndarray                    # [n_layers, n_q_heads]
    p_cross: np.ndarray                  # [n_layers, n_q_heads]
    q_scale: Optional[np.ndarray] = None  # [n_layers, n_q_heads] or None
    k_scale: Optional[np.ndarray] = None  # [n_layers, n_kv_heads] or None
    recipe: str = ""

    # -- per-(layer, head, position) views of the packed vectors -------------------
    def la_vec(self, layer: int, head: int, pos: int) -> np.ndarray:
        nb = self.shape.la_bytes(pos)
        o = int(self.la_doc_off[pos]) + (layer * self.shape.n_q_heads + head) * nb
        return self.la_blob[o:o + nb]

    def ca_vec(self, layer: int, head: int, pos: int) -> np.ndarray:
        nb = self.shape.ca_bytes(pos)
        o = int(self.ca_doc_off[pos]) + (layer * self.shape.n_q_heads + head) * nb
        return self.ca_blob[o:o + nb]

    # -- Q/K/V ------------------------------------------------------------------------
    def qkv(self, layer: int) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
        """bf16 CPU tensors Q [N,Hq,d], K,V [N,Hkv,d]; generated per document id so a
        document's block is the same wherever it stands in the prompt."""
        sh = self.shape
        n = sh.n_tokens
        q = torch.empty((n, sh.n_q_heads, sh.head_dim), dtype=torch.bfloat16)
        k = torch.empty((n, sh.n_kv_heads, sh.head_dim), dtype=torch.bfloat16)
        v = torch.empty((n, sh.n_kv_heads, sh.head_dim), dtype=torch.bfloat16)
        off = sh.doc_offsets
        segs = [(int(off[p]), int(off[p + 1]), self.doc_ids[p]) for p in range(sh.n_docs)]
        segs.append((int(off[-1]), n, 1 << 20))  # the user query is its own segment
        qs = None if self.q_scale is None else torch.from_numpy(self.q_scale[layer].astype(np.float32))
        ks = None if self.k_scale is None else torch.from_numpy(self.k_scale[layer].astype(np.float32))
        for (a, b, did) in segs:
            if b <= a:
                continue
            xq = torch.randn((b - a, sh.n_q_heads, sh.head_dim), generator=_torch_gen(self.seed, _S_Q, layer, did))
            xk = torch.randn((b - a, sh.n_kv_heads, sh.head_dim), generator=_torch_gen(self.seed, _S_K, layer, did))
            xv = torch.randn((b - a, sh.n_kv_heads, sh.head_dim), generator=_torch_gen(self.seed, _S_V, layer, did))
            if qs is not None:
                xq = xq * qs[None, :, None]
            if ks is not None:
                xk = xk * ks[None, :, None]
            q[a:b] = xq.to(torch.bfloat16)
            k[a:b] = xk.to(torch.bfloat16)
            v[a:b] = xv.to(torch.bfloat16)
        return q, k, v

    def qkv_on_device(self, layer: int, device: str = "cuda") -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
        """Same recipe as ``qkv`` (N(0,1) per (layer, document id), optional per-head scales, rounded to bf16) drawn by
        the DEVICE generator: a different random stream, so NOT the arrays the oracle sees.  For timing legs that need
        many layers resident (bench.py full-stack: 32 layers would take minutes on the host generator); every parity
        test uses ``qkv``."""
        sh = self.shape
        n = sh.n_tokens
        dev = torch.device(device)
        q = torch.empty((n, sh.n_q_heads, sh.head_dim), dtype=torch.bfloat16, device=dev)
        k = torch.empty((n, sh.n_kv_heads, sh.head_dim), dtype=torch.bfloat16, device=dev)
        v = torch.empty((n, sh.n_kv_heads, sh.head_dim), dtype=torch.bfloat16, device=dev)
        off = sh.doc_offsets
        segs = [(int(off[p]), int(off[p + 1]), self.doc_ids[p]) for p in range(sh.n_docs)] + [(int(off[-1]), n, 1 << 20)]
        qs = None if self.q_scale is None else torch.from_numpy(self.q_scale[layer].astype(np.float32)).to(dev)
        ks = None if self.k_scale is None else torch.from_numpy(self.k_scale[layer].astype(np.float32)).to(dev)
        g = torch.Generator(device=dev)
        for (a, b, did) in segs:
            if b <= a:
                continue
            for t, sid, heads, sc in ((q, _S_Q, sh.n_q_heads, qs), (k, _S_K, sh.n_kv_heads, ks), (v, _S_V, sh.n_kv_heads, None)):
                g.manual_seed(int(_torch_gen(self.seed, sid, layer, did).initial_seed()))
                x = torch.randn((b - a, heads, sh.head_dim), generator=g, device=dev)
                if sc is not None:
                    x = x * sc[None, :, None]
                t[a:b] = x.to(torch.bfloat16)
        return q, k, v

    # -- re-ordering ------------------------------------------------------------------
    def reorder(self, perm: Sequence[int], name: Optional[str] = None) -> "Workload":
        """Prompt whose position p holds the document that stood at position perm[p]."""
        perm = list(perm)
        assert sorted(perm) == list(range(self.shape.n_docs))
        sh = replace(self.shape, doc_lens=tuple(self.shape.doc_lens[i] for i in perm))
        return replace(
            self,
            name=name or (self.name + "-perm"),
            shape=sh,
            doc_ids=tuple(self.doc_ids[i] for i in perm),
            la_doc_off=self.la_doc_off[perm].copy(),
            ca_doc_off=self.ca_doc_off[perm].copy(),
        )


def _diag_bit_positions(p: int) -> np.ndarray:
    # lower triangle enumerated row-major (0,0),(1,0),(1,1),(2,0)...
    i = np.arange(p, dtype=np.int64)
    return i * (i + 1) // 2 + i


def build_workload(
    name: str,
    shape: PromptShape,
    seed: int,
    p_loc: np.ndarray,
    p_cross: np.ndarray,
    *,
    diag_set: bool = True,
    garbage_padding: bool = True,
    q_scale: Optional[np.ndarray] = None,
    k_scale: Optional[np.ndarray] = None,
    recipe: str = "",
) -> Workload:
    """Draw i.i.d. Bernoulli marks per (layer, head, doc, tile / key group) and pack them MSB-first."""
    L, H = shape.n_layers, shape.n_q_heads
    p_loc = np.broadcast_to(np.asarray(p_loc, dtype=np.float64), (L, H))
    p_cross = np.broadcast_to(np.asarray(p_cross, dtype=np.float64), (L, H))
    la_parts: List[np.ndarray] = []
    ca_parts: List[np.ndarray] = []
    la_off = np.zeros(shape.n_docs, dtype=np.int64)
    ca_off = np.zeros(shape.n_docs, dtype=np.int64)
    la_pos = 0
    ca_pos = 0
    for d in range(shape.n_docs):
        nla, nca = shape.la_bits(d), shape.ca_bits(d)
        bla, bca = shape.la_bytes(d), shape.ca_bytes(d)
        r = _rng(seed, _S_LA, d)
        bits = r.random((L, H, bla * 8)) < p_loc[:, :, None]
        if diag_set:
            bits[:, :, _diag_bit_positions(shape.pages(d))] = True
        if garbage_padding:
            bits[:, :, nla:] = r.random((L, H, bla * 8 - nla)) < 0.5
        else:
            bits[:, :, nla:] = False
        la_parts.append(np.packbits(bits, axis=-1, bitorder="big").reshape(-1))
        r = _rng(seed, _S_CA, d)
        bits = r.random((L, H, bca * 8)) < p_cross[:, :, None]
        if garbage_padding:
            bits[:, :, nca:] = r.random((L, H, bca * 8 - nca)) < 0.5
        else:
            bits[:, :, nca:] = False
        ca_parts.append(np.packbits(bits, axis=-1, bitorder="big").reshape(-1))
        la_off[d], ca_off[d] = la_pos, ca_pos
        la_pos += la_parts[-1].size
        ca_pos += ca_parts[-1].size
    # 16 spare bytes so that an aligned 4-byte read of the last word stays inside the allocation
    la_blob = np.concatenate(la_parts + [np.zeros(16, np.uint8)]) if la_parts else np.zeros(16, np.uint8)
    ca_blob = np.concatenate(ca_parts + [np.zeros(16, np.uint8)]) if ca_parts else np.zeros(16, np.uint8)
    return Workload(
        name=name, shape=shape, seed=seed, doc_ids=tuple(range(shape.n_docs)),
        la_blob=la_blob, ca_blob=ca_blob, la_doc_off=la_off, ca_doc_off=ca_off,
        p_loc=np.array(p_loc), p_cross=np.array(p_cross), q_scale=q_scale, k_scale=k_scale, recipe=recipe,
    )


# ---------------------------------------------------------------------------------------
# BASELINE.json configs (C1..C5).  SURVEY.md 8(d) table; readings A1, A23, A24.
# ---------------------------------------------------------------------------------------

def config_tiny(seed: int = BASE_SEED) -> Workload:
    sh = PromptShape(1, 2, 1, 64, (256,) * 4, 64, tile=64, cross_gran=1)
    return build_workload("C1-tiny", sh, seed, 0.3, 0.2,
                          recipe="4x256+64, T=64, LA Bernoulli(0.3) diag set, CA Bernoulli(0.2) per key")


def _uniform_dens(seed: int, L: int, H: int, lo_l, hi_l, lo_c, hi_c):
    r = _rng(seed, _S_DENS)
    return r.uniform(lo_l, hi_l, (L, H)), r.uniform(lo_c, hi_c, (L, H))


def _beta_dens(seed: int, L: int, H: int):
    r = _rng(seed, _S_DENS)
    return r.beta(2.0, 6.0, (L, H)), r.beta(2.0, 8.0, (L, H))


def config_8b_10k(seed: int = BASE_SEED) -> Workload:
    sh = PromptShape(1, 32, 8, 128, (1024,) * 10, 128, tile=128, cross_gran=1)
    pl, pc = _uniform_dens(seed, 1, 32, 0.2, 0.4, 0.1, 0.3)
    return build_workload("C2-8b-10k", sh, seed, pl, pc,
                          recipe="10x1024+128, T=128, p_loc~U(.2,.4), p_cross~U(.1,.3) per head")


def config_32k(seed: int = BASE_SEED, n_layers: int = 1, cross_gran: int = 1) -> Workload:
    sh = PromptShape(n_layers, 32, 8, 128, (2000,) * 16, 256, tile=128, cross_gran=cross_gran)
    pl, pc = _beta_dens(seed, n_layers, 32)
    name = ("C3-32k" if n_layers == 1 else f"C5-stack{n_layers}") + ("" if cross_gran == 1 else "-paged")
    return build_workload(name, sh, seed, pl, pc,
                          recipe="16x2000+256, T=128, p_loc~Beta(2,6), p_cross~Beta(2,8) per (layer, head)")


def ragged_doc_lens(seed: int, n_docs: int = 24, lo: int = 1024, hi: int = 4096,
                    query_len: int = 512, max_total: int = 65536) -> Tuple[int, ...]:
    """Reading A23: draw n_docs lengths, walk in order, clip the doc that would overflow to the
    remainder (dropping it and the rest if the remainder is < lo)."""
    r = _rng(seed, _S_LEN)
    lens = r.integers(lo, hi + 1, n_docs)
    out: List[int] = []
    tot = 0
    for x in lens:
        room = max_total - query_len - tot
        if room < lo:
            break
        x = int(min(int(x), room))
        out.append(x)
        tot += x
    return tuple(out)


def config_64k_ragged(seed: int = BASE_SEED, cross_gran: int = 1) -> Workload:
    lens = ragged_doc_lens(seed)
    sh = PromptShape(1, 32, 8, 128, lens, 512, tile=128, cross_gran=cross_gran)
    pl, pc = _beta_dens(seed, 1, 32)
    r = _rng(seed, _S_SCALE)
    qs = r.lognormal(0.0, 0.5, (1, 32))
    ks = r.lognormal(0.0, 0.5, (1, 8))
    return build_workload("C4-64k-ragged" + ("" if cross_gran == 1 else "-paged"), sh, seed, pl, pc, q_scale=qs, k_scale=ks,
                          recipe="24 docs U[1024,4096] clipped to <=65536 incl. 512 query; Beta densities; "
                                 "Q/K scaled per head by LogNormal(0,.5)")


def config_full_stack(seed: int = BASE_SEED, n_layers: int = 32) -> Workload:
    return config_32k(seed, n_layers=n_layers)


def stack_orderings(w: Workload, n: int = 4) -> List[List[int]]:
    """identity + (n-1) seeded permutations of the documents (query stays last)."""
    r = _rng(w.seed, _S_ORDER)
    out = [list(range(w.shape.n_docs))]
    for _ in range(n - 1):
        out.append([int(x) for x in r.permutation(w.shape.n_docs)])
    return out


def quantize_e4m3(x: torch.Tensor, per_head_amax: float = 448.0) -> Tuple[torch.Tensor, np.ndarray]:
    """Input plumbing for the FP8 variant: x [N, H, d] float -> (uint8 e4m3 bytes [N, H, d], fp32
    scale per head) with scale[h] = max|x[:, h]| / per_head_amax, so that x ~ scale[h] * decode(bytes).  Rounding is the
    library conversion of torch (round to nearest even); values are clamped to the format's range first."""
    xf = x.float()
    amax = xf.abs().amax(dim=(0, 2)).clamp_min(1e-12)
    scale = (amax / per_head_amax)
    y = (xf / scale[None, :, None]).clamp(-448.0, 448.0).to(torch.float8_e4m3fn)
    return y.view(torch.uint8), scale.numpy().astype(np.float32)


@dataclass
class BatchWorkload:
    """Several prompts packed back to back on the token axis: prompt p = its documents, then its
    query.  Input plumbing only: the members' blobs are concatenated and their byte offsets shifted."""
    name: str
    members: Tuple[Workload, ...]

    def __post_init__(self):
        m0 = self.members[0].shape
        for w in self.members:
            sh = w.shape
            assert (sh.n_layers, sh.n_q_heads, sh.n_kv_heads, sh.head_dim, sh.tile, sh.cross_gran) == \
                   (m0.n_layers, m0.n_q_heads, m0.n_kv_heads, m0.head_dim, m0.tile, m0.cross_gran)
        la_base = np.cumsum([0] + [len(w.la_blob) for w in self.members])
        ca_base = np.cumsum([0] + [len(w.ca_blob) for w in self.members])
        self.la_blob = np.concatenate([w.la_blob for w in self.members] + [np.zeros(4, np.uint8)])
        self.ca_blob = np.concatenate([w.ca_blob for w in self.members] + [np.zeros(4, np.uint8)])
        self.la_doc_off = np.concatenate([w.la_doc_off + la_base[i] for i, w in enumerate(self.members)]).astype(np.int64)
        self.ca_doc_off = np.concatenate([w.ca_doc_off + ca_base[i] for i, w in enumerate(self.members)]).astype(np.int64)
        self.doc_base = np.cumsum([0] + [w.shape.n_docs for w in self.members]).astype(np.int64)

    # -- what the library is told ---------------------------------------------------------------
    @property
    def head_shape(self) -> PromptShape:
        return self.members[0].shape

    @property
    def doc_lens(self) -> Tuple[int, ...]:
        return tuple(x for w in self.members for x in w.shape.doc_lens)

    @property
    def prompt_doc_start(self) -> np.ndarray:
        return self.doc_base.astype(np.int32)

    @property
    def prompt_query_len(self) -> np.ndarray:
        return np.asarray([w.shape.query_len for w in self.members], np.int32)

    @property
    def n_tokens(self) -> int:
        return int(sum(w.shape.n_tokens for w in self.members))

    @property
    def row_base(self) -> np.ndarray:
        return np.cumsum([0] + [w.shape.n_tokens for w in self.members]).astype(np.int64)

    # -- what the oracle is told -------------------------------------------------------------------
    @property
    def prompts(self):
        return [([int(x) for x in w.shape.doc_offsets], w.shape.query_len) for w in self.members]

    def _member_of_doc(self, d: int):
        p = int(np.searchsorted(self.doc_base, d, side="right")) - 1
        return self.members[p], d - int(self.doc_base[p])

    def la_vec(self, layer: int, head: int, d: int) -> np.ndarray:
        w, pos = self._member_of_doc(d)
        return w.la_vec(layer, head, pos)

    def ca_vec(self, layer: int, head: int, d: int) -> np.ndarray:
        w, pos = self._member_of_doc(d)
        return w.ca_vec(layer, head, pos)

    def qkv(self, layer: int) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
        parts = [w.qkv(layer) for w in self.members]
        return tuple(torch.cat([p[i] for p in parts]) for i in range(3))


def make_batch(name: str, members: Sequence[Workload]) -> BatchWorkload:
    return BatchWorkload(name, tuple(members))


def config_batch_8x10k(seed: int = BASE_SEED) -> BatchWorkload:
    """Eight prompts of C2's shape (10 x 1024 + 128, 32/8 heads, d = 128), different seeds: the multi-request case of
    SURVEY.md 8(f)-3 (short prompts in one launch fill the GPU where one of them cannot)."""
    return make_batch("batch-8x10k", [config_8b_10k(seed + 1000 * (i + 1)) for i in range(8)])


CONFIGS: Dict[str, Callable[[], Workload]] = {
    "tiny": config_tiny,
    "8b-10k": config_8b_10k,
    "32k": config_32k,
    "64k-ragged": config_64k_ragged,
    "full-stack": config_full_stack,
    # the paper's page-granular CA (one bit per 128-key page) on C3's shape, same densities per bit
    "32k-paged": lambda seed=BASE_SEED: config_32k(seed, cross_gran=128),
}


def custom(name: str, *, n_layers=1, n_q_heads=2, n_kv_heads=1, head_dim=64, doc_lens=(256, 256),
           query_len=64, tile=64, cross_gran=1, p_loc=0.3, p_cross=0.2, seed=1, diag_set=True,
           garbage_padding=True) -> Workload:
    sh = PromptShape(n_layers, n_q_heads, n_kv_heads, head_dim, tuple(int(x) for x in doc_lens),
                     query_len, tile, cross_gran)
    return build_workload(name, sh, seed, p_loc, p_cross, diag_set=diag_set, garbage_padding=garbage_padding,
                          recipe="custom test case")
