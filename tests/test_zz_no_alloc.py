"""sift_encode_document_static: the offline encoder for callers that cannot allocate device memory.

Who that is: code that runs inside somebody else's memory regime.  A custom op or plug-in gets its input and output
buffers from the host framework and has no way to ask that framework's allocator for more; an inference server that
reserved all free HBM for its KV-cache pool at start-up cannot count on a cudaMalloc succeeding, and a cudaMalloc that
does succeed blocks the whole device while it runs.  For them the library carries the encoder's scratch (per-key hit
counters, per-tile flags) in a fixed 4 MiB array of its own device image, and the entry point takes only inputs and
outputs (include/sift.h).

What is checked: the new entry point writes exactly the bytes sift_encode_document writes with a caller-supplied
workspace (the outputs are bit vectors, so the tolerance is equality, as in the other metadata tests), on two calls in a
row.  The second call uses a different, shorter document so that it finds the first call's counters in the shared array:
if the entry point did not clear what it uses, the second comparison fails.  Oversized requests must be refused with a
message, not truncated.  The file is named to be collected last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It holds no state of its own, so it passes alone in a fresh process (where its first
call also performs the once-per-device address look-up) and after the rest of the suite.
"""
import ctypes as C

import pytest
import torch

from paper_2606_09441_b200 import api, build

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build_library()


def _document(n, hq, hkv, d, seed, q_gain=2.0):
    g = torch.Generator().manual_seed(seed)
    q = (torch.randn((n, hq, d), generator=g) * q_gain).to(torch.bfloat16).cuda()
    k = torch.randn((n, hkv, d), generator=g).to(torch.bfloat16).cuda()
    v = torch.randn((n, hkv, d), generator=g).to(torch.bfloat16).cuda()
    _, lse = api.sift_dense_causal_attention(q, k, v)      # pass 1 of the encoder: the document's row log-sum-exp
    return q, k, lse


def _both_paths(n, hq, hkv, d, tile, gran, seed):
    q, k, lse = _document(n, hq, hkv, d, seed)
    la_ref, ca_ref = api.sift_encode_document(q, k, lse, tile, gran)          # existing path: workspace from torch
    la_bytes, ca_bytes = api.sift_encode_output_sizes(n, tile, gran)
    # outputs pre-filled with a pattern: every byte must be written by the call
    la = torch.full((hq, la_bytes), 0xA5, dtype=torch.uint8, device="cuda")
    ca = torch.full((hq, ca_bytes), 0xA5, dtype=torch.uint8, device="cuda")
    api.sift_encode_document_static(q, k, lse, la, ca, tile, gran)
    torch.cuda.synchronize()
    assert torch.equal(la, la_ref), f"LA bytes differ (n={n}, T={tile}, G={gran})"
    assert torch.equal(ca, ca_ref), f"CA bytes differ (n={n}, T={tile}, G={gran})"
    return int(la_ref.count_nonzero()) + int(ca_ref.count_nonzero())


def test_static_scratch_encoder_matches_workspace_encoder_twice():
    # call 1: 1500 tokens, 8 q-heads -> the counters of 8 x 1536 keys and 8 x 78 tile flags are left in the array
    nz1 = _both_paths(n=1500, hq=8, hkv=2, d=128, tile=128, gran=1, seed=11)
    # call 2, straight after, smaller and at the other tile size / granularity: its scratch overlaps call 1's leftovers
    nz2 = _both_paths(n=700, hq=4, hkv=4, d=64, tile=64, gran=64, seed=12)
    assert nz1 > 0 and nz2 > 0      # the comparison was not between two empty results


def test_static_scratch_encoder_refuses_what_does_not_fit():
    cap = api.sift_encode_static_scratch_bytes()
    assert cap == 4 << 20
    n, hq, tile = 16384, 64, 64     # 64 heads x (16384 + 256 * 257 / 2) words = 12.6 MB of scratch
    need = C.c_size_t()
    assert api.lib().sift_encode_workspace_size(n, hq, tile, C.byref(need)) == 0 and need.value > cap
    q = torch.zeros((n, hq, 64), dtype=torch.bfloat16, device="cuda")
    k = torch.zeros((n, 1, 64), dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros((hq, n), dtype=torch.float32, device="cuda")
    la_bytes, ca_bytes = api.sift_encode_output_sizes(n, tile, 1)
    la = torch.full((hq, la_bytes), 0xA5, dtype=torch.uint8, device="cuda")
    ca = torch.full((hq, ca_bytes), 0xA5, dtype=torch.uint8, device="cuda")
    launches = api.sift_launch_count()
    with pytest.raises(api.SiftError, match="SIFT_ENCODE_STATIC_SCRATCH_BYTES"):
        api.sift_encode_document_static(q, k, lse, la, ca, tile, 1)
    torch.cuda.synchronize()
    assert api.sift_launch_count() == launches                       # nothing was enqueued
    assert bool((la == 0xA5).all()) and bool((ca == 0xA5).all())     # outputs untouched
    # the largest case the header promises (32 q-heads, 12,288 tokens, tile 64) is accepted by the size check
    assert api.lib().sift_encode_workspace_size(12288, 32, 64, C.byref(need)) == 0 and need.value <= cap
