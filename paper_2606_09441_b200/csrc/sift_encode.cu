// SIFT offline metadata generation for sm_100a (sec 4.1, L209 sec 4.2, L223 sec 4.4):
// from the standalone dense causal attention of ONE document, per q-head,
//   LA bit (i, j) = 1  iff  tile (i, j) of the document's causal triangle holds at least one probability >= alpha,
//   CA bit g      = 1  iff  the fraction of causal (query, key) cells of key group g (one key at G = 1, a page of T
//                           keys at G = tile) whose probability is >= beta exceeds gamma        (reading R6).
// Two passes, FlashAttention style: pass 1 is the row log-sum-exp of the document, which the caller gets from
// sift_dense_causal_attention on the document alone; pass 2 (here) recomputes S = Q K^T tile by tile on the tensor
// cores (tcgen05, TMEM accumulators), compares log2-domain scores against log2(alpha) / log2(beta) (no exp needed),
// and reduces: per-tile "any" flags with warp votes, per-key counts with ballots + popc.  A second small kernel packs
// the bits MSB-first.
#include <cuda.h>
#include <cuda_bf16.h>
#include <math.h>
#include <string.h>
#include <mutex>

#include "sift_common.h"
#include "sm100_ptx.cuh"

namespace sift {
using namespace ptx;

constexpr int kEncThreads = 128;   // one row of a 128-row block per thread

struct EncParams {
  int32_t doc_len, n_q_heads, n_kv_heads, tile, gran;
  const float* lse;       // [Hq][doc_len], natural log
  float sl;               // softmax_scale * log2(e)
  float log2_alpha, log2_beta;
  int32_t* col_cnt;       // [Hq][len128]
  int32_t* tile_flag;     // [Hq][PT (PT + 1) / 2]
  int32_t len128;         // doc_len rounded up to 128
  int32_t n_la_bits;      // PT (PT + 1) / 2
};

template <int HD>
struct EncSmem {
  static constexpr int kTileBytes = 128 * HD * 2;
  static constexpr int kQOff = 0, kKOff = kTileBytes, kBarOff = 3 * kTileBytes;   // Q, 2 K stages
  static constexpr int bQFull = 0, bKFull = 1, bSFull = 3;                        // 1 + 2 + 2 barriers
  static constexpr int kInfoOff = kBarOff + 64;
  static constexpr int kBytes = kInfoOff + 64;
};

__device__ __forceinline__ uint64_t enc_kdesc(uint32_t tile_addr, int k) {   // K-major, 128B swizzle, 16-element K chunk k
  return umma_desc_sw128(tile_addr + (k >> 2) * (128 * 128) + (k & 3) * 32, 16, 1024);
}

template <int HD>
__global__ void __launch_bounds__(kEncThreads)
sift_encode_scores_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k, const EncParams p) {
  using S = EncSmem<HD>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t sbase = smem_u32(smem_raw);
  if ((sbase & 1023u) != 0) __trap();
  auto bar = [&](int i) -> uint32_t { return sbase + S::kBarOff + i * 8; };
  volatile int32_t* info = reinterpret_cast<volatile int32_t*>(smem_raw + S::kInfoOff);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int i = (int)gridDim.x - 1 - (int)blockIdx.x;       // longest row blocks (most key blocks) first
  const int h = blockIdx.y, kvh = h / (p.n_q_heads / p.n_kv_heads);
  const int L = p.doc_len, T = p.tile;
  const int n_j = i + 1;                                   // key blocks 0 .. i (causal)
  constexpr uint32_t idesc = umma_idesc_bf16(128, 128, 0, 0);
  constexpr int kHalves = HD / 64;

  if (tid == 0) {
    for (int b = 0; b < 5; ++b) mbar_init(bar(b), 1);
    fence_barrier_init();
    for (int k = 1; k < 5; ++k) info[k] = 0;
  }
  if (warp == 0) {
    tmem_alloc(smem_u32(const_cast<int32_t*>(&info[0])), 256);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = (uint32_t)info[0];
  const uint32_t q_smem = sbase + S::kQOff, k_smem = sbase + S::kKOff;

  auto load_k = [&](int j) {                               // thread 0
    const int st = j & 1;
    mbar_arrive_expect_tx(bar(S::bKFull + st), S::kTileBytes);
    for (int hf = 0; hf < kHalves; ++hf)
      tma_load_2d(k_smem + st * S::kTileBytes + hf * (128 * 128), &tm_k, bar(S::bKFull + st), kvh * HD + hf * 64, j * 128);
  };
  auto issue = [&](int j) {                                // thread 0: S[j & 1] = Q K_j^T
    const int st = j & 1;
    mbar_wait(bar(S::bKFull + st), (j >> 1) & 1, 500);
    tc_fence_after();
    for (int k = 0; k < HD / 16; ++k)
      umma_ss(tmem + st * 128, enc_kdesc(q_smem, k), enc_kdesc(k_smem + st * S::kTileBytes, k), idesc, k > 0);
    umma_commit(bar(S::bSFull + st));
  };
  if (tid == 0) {
    mbar_arrive_expect_tx(bar(S::bQFull), S::kTileBytes);
    for (int hf = 0; hf < kHalves; ++hf)
      tma_load_2d(q_smem + hf * (128 * 128), &tm_q, bar(S::bQFull), h * HD + hf * 64, i * 128);
    load_k(0);
    if (n_j > 1) load_k(1);
    mbar_wait(bar(S::bQFull), 0, 501);
    issue(0);
  }
  __syncwarp();

  const int r = tid, row = i * 128 + r;
  const bool row_ok = row < L;
  const float lse2 = row_ok ? p.lse[(int64_t)h * L + row] * 1.4426950408889634f : INFINITY;
  const float thr_a = (p.log2_alpha + lse2) / p.sl, thr_b = (p.log2_beta + lse2) / p.sl;   // thresholds on the raw score
  const uint32_t lane_addr = (uint32_t)(warp * 32) << 16;
  const int rh = (T == 64) ? (warp >> 1) : 0;              // LA row sub-tile of this warp inside the 128-row block
  const int pt = (L + T - 1) / T;

  for (int j = 0; j < n_j; ++j) {
    const int st = j & 1;
    if (tid == 0 && j + 1 < n_j) issue(j + 1);             // next block's MMA runs while this one is examined
    __syncwarp();
    mbar_wait(bar(S::bSFull + st), (j >> 1) & 1, 502);
    tc_fence_after();
    if (tid == 0 && j + 2 < n_j) load_k(j + 2);            // the MMA of block j is complete: its K stage is free
    __syncwarp();
    const int key0 = j * 128;
    bool any_a[2] = {false, false};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      uint32_t raw[32];
      tmem_ld32(tmem + lane_addr + st * 128 + c * 32, raw);
      tmem_wait_ld();
      // log2 p = s * sl - lse2 >= log2(threshold)  <=>  s >= (log2(threshold) + lse2) / sl: one comparison of the raw
      // score against a per-row constant (rows beyond the document have lse2 = +inf: never true).  Off the diagonal
      // every key is causal, and "some p >= alpha" is one comparison of the row's maximum: ~2.5 instructions per score
      // instead of ~14 (the kernel is bound by these, not by the MMAs).
      uint32_t wb = 0;
      bool aa;
      if (j < i) {
        float mxs = -INFINITY;
#pragma unroll
        for (int cc = 0; cc < 32; ++cc) {
          const float sc = __uint_as_float(raw[cc]);
          mxs = fmaxf(mxs, sc);
          if (sc >= thr_b) wb |= 1u << cc;
        }
        aa = mxs >= thr_a;
      } else {                                                            // diagonal block: keys after the row are not causal
        uint32_t wa = 0;
#pragma unroll
        for (int cc = 0; cc < 32; ++cc) {
          const float sc = __uint_as_float(raw[cc]);
          if (sc >= thr_b) wb |= 1u << cc;
          if (sc >= thr_a) wa |= 1u << cc;
        }
        const int lim = row - key0 - c * 32;                              // columns 0 .. lim of this chunk are causal
        const uint32_t vm = lim >= 31 ? 0xffffffffu : (lim < 0 ? 0u : ((2u << lim) - 1u));
        wb &= vm;
        aa = (wa & vm) != 0u;
      }
      any_a[c >> 1] = any_a[c >> 1] || aa;
      // per-key counts of this warp's 32 rows: transpose the 32 x 32 bit matrix (lane = row, bit = column) with five
      // butterfly exchanges so that lane c holds column c, then popc (5 shuffles instead of 32 ballots)
      uint32_t xt = wb;
#pragma unroll
      for (int jj = 16; jj >= 1; jj >>= 1) {
        const uint32_t mk = (jj == 16) ? 0x0000ffffu : (jj == 8) ? 0x00ff00ffu : (jj == 4) ? 0x0f0f0f0fu : (jj == 2) ? 0x33333333u : 0x55555555u;
        const uint32_t y = __shfl_xor_sync(0xffffffffu, xt, jj);
        xt = (lane & jj) ? ((xt & ~mk) | ((y >> jj) & mk)) : ((xt & mk) | ((y << jj) & ~mk));
      }
      const int cnt = __popc(xt);
      if (cnt) atomicAdd(&p.col_cnt[(int64_t)h * p.len128 + key0 + c * 32 + lane], cnt);
    }
    // tile "any" flags: a warp that saw a probability >= alpha writes the flag itself (every writer stores 1)
    {
      int32_t* tf = p.tile_flag + (int64_t)h * p.n_la_bits;
      if (T == 64) {
#pragma unroll
        for (int ch = 0; ch < 2; ++ch) {
          const int ti = 2 * i + rh, tj = 2 * j + ch;
          if (__any_sync(0xffffffffu, any_a[ch]) && lane == 0 && tj <= ti && ti < pt) tf[ti * (ti + 1) / 2 + tj] = 1;
        }
      } else {
        if (__any_sync(0xffffffffu, any_a[0] || any_a[1]) && lane == 0) tf[i * (i + 1) / 2 + j] = 1;
      }
    }
    tc_fence_before();
    __syncthreads();            // every warp has read S[st]: the MMA of block j + 2 may overwrite it
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 256);
}

// Packs the flags / counts of one head into the MSB-first bit vectors.
__global__ void __launch_bounds__(256)
sift_encode_pack_kernel(const EncParams p, float gamma, uint8_t* la_out, uint8_t* ca_out, int la_bytes, int ca_bytes) {
  const int h = blockIdx.x, L = p.doc_len, G = p.gran;
  const int32_t* tf = p.tile_flag + (int64_t)h * p.n_la_bits;
  const int32_t* cc = p.col_cnt + (int64_t)h * p.len128;
  for (int b = threadIdx.x; b < la_bytes; b += blockDim.x) {
    uint32_t v = 0;
    for (int k = 0; k < 8; ++k) {
      const int n = b * 8 + k;
      if (n < p.n_la_bits && tf[n]) v |= 0x80u >> k;
    }
    la_out[(int64_t)h * la_bytes + b] = (uint8_t)v;
  }
  const int n_groups = (L + G - 1) / G;
  for (int b = threadIdx.x; b < ca_bytes; b += blockDim.x) {
    uint32_t v = 0;
    for (int k = 0; k < 8; ++k) {
      const int g = b * 8 + k;
      if (g >= n_groups) break;
      long long hits = 0, cells = 0;
      for (int key = g * G; key < min(L, (g + 1) * G); ++key) { hits += cc[key]; cells += L - key; }
      // "exceeds gamma", decided in fp64 on the fp32 value of gamma the ABI carries
      if ((double)hits > (double)gamma * (double)cells) v |= 0x80u >> k;
    }
    ca_out[(int64_t)h * ca_bytes + b] = (uint8_t)v;
  }
}

static int enc_check(int32_t doc_len, int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, int32_t tile, int32_t gran) {
  if (doc_len < 1 || doc_len > (1 << 20) || n_q_heads < 1 || n_q_heads > 255 || n_kv_heads < 1 || n_q_heads % n_kv_heads)
    return set_error(SIFT_ERR_INVALID_ARG, "bad dimensions");
  if (head_dim != 64 && head_dim != 128) return set_error(SIFT_ERR_UNSUPPORTED, "head_dim %d not in {64,128}", head_dim);
  if (tile != 64 && tile != 128) return set_error(SIFT_ERR_UNSUPPORTED, "tile %d not in {64,128}", tile);
  if (gran != 1 && gran != tile) return set_error(SIFT_ERR_UNSUPPORTED, "cross_gran %d not in {1, tile}", gran);
  return SIFT_OK;
}

template <int HD>
static int enc_launch(const EncParams& p, const void* Q, const void* K, int64_t qs, int64_t ks, cudaStream_t st) {
  CUtensorMap tq, tk;
  int rc;
  if ((rc = make_tensor_map_2d(&tq, Q, p.doc_len, (int64_t)p.n_q_heads * HD, qs, 128))) return rc;
  if ((rc = make_tensor_map_2d(&tk, K, p.doc_len, (int64_t)p.n_kv_heads * HD, ks, 128))) return rc;
  if ((rc = ensure_dynamic_smem(reinterpret_cast<const void*>(&sift_encode_scores_kernel<HD>), EncSmem<HD>::kBytes,
                                HD == 128 ? kSmemSlotEnc128 : kSmemSlotEnc64)))
    return rc;
  sift_encode_scores_kernel<HD><<<dim3(p.len128 / 128, p.n_q_heads), kEncThreads, EncSmem<HD>::kBytes, st>>>(tq, tk, p);
  return SIFT_OK;
}

}  // namespace sift

using namespace sift;

extern "C" int sift_encode_workspace_size(int32_t doc_len, int32_t n_q_heads, int32_t tile, size_t* bytes) {
  if (!bytes) return set_error(SIFT_ERR_INVALID_ARG, "bytes is NULL");
  if (doc_len < 1 || n_q_heads < 1 || (tile != 64 && tile != 128)) return set_error(SIFT_ERR_INVALID_ARG, "bad dimensions");
  const int64_t len128 = (doc_len + 127) / 128 * 128, pt = (doc_len + tile - 1) / tile;
  *bytes = (size_t)n_q_heads * (size_t)(len128 + pt * (pt + 1) / 2) * 4;
  return SIFT_OK;
}

extern "C" int sift_encode_output_sizes(int32_t doc_len, int32_t tile, int32_t cross_gran, size_t* la_bytes, size_t* ca_bytes) {
  if (!la_bytes || !ca_bytes) return set_error(SIFT_ERR_INVALID_ARG, "NULL pointer");
  if (doc_len < 1 || (tile != 64 && tile != 128) || (cross_gran != 1 && cross_gran != tile))
    return set_error(SIFT_ERR_INVALID_ARG, "bad dimensions");
  const int64_t pt = (doc_len + tile - 1) / tile, nb = (doc_len + cross_gran - 1) / cross_gran;
  *la_bytes = (size_t)((pt * (pt + 1) / 2 + 7) / 8);
  *ca_bytes = (size_t)((nb + 7) / 8);
  return SIFT_OK;
}

extern "C" int sift_encode_document(int32_t doc_len, int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, int32_t tile,
                                    int32_t cross_gran, const void* Q, const void* K, int64_t q_row_stride,
                                    int64_t k_row_stride, const float* lse, float alpha, float beta, float gamma,
                                    float softmax_scale, uint8_t* la_out, uint8_t* ca_out, void* workspace,
                                    size_t workspace_bytes, void* stream) {
  int rc = enc_check(doc_len, n_q_heads, n_kv_heads, head_dim, tile, cross_gran);
  if (rc) return rc;
  if (!Q || !K || !lse || !la_out || !ca_out || !workspace) return set_error(SIFT_ERR_INVALID_ARG, "NULL pointer");
  if (((uintptr_t)Q & 15) || ((uintptr_t)K & 15) || (q_row_stride * 2) % 16 || (k_row_stride * 2) % 16)
    return set_error(SIFT_ERR_INVALID_ARG, "Q / K base or row stride not 16-byte aligned");
  if (!(alpha > 0.f) || !(beta > 0.f) || !(gamma >= 0.f)) return set_error(SIFT_ERR_INVALID_ARG, "alpha, beta must be > 0, gamma >= 0");
  size_t need = 0;
  sift_encode_workspace_size(doc_len, n_q_heads, tile, &need);
  if (workspace_bytes < need) return set_error(SIFT_ERR_WORKSPACE, "workspace %zu < %zu bytes", workspace_bytes, need);
  EncParams p;
  memset(&p, 0, sizeof(p));
  p.doc_len = doc_len; p.n_q_heads = n_q_heads; p.n_kv_heads = n_kv_heads; p.tile = tile; p.gran = cross_gran;
  p.lse = lse;
  const float sc = softmax_scale > 0.f ? softmax_scale : 1.0f / sqrtf((float)head_dim);
  p.sl = sc * 1.4426950408889634f;
  p.log2_alpha = log2f(alpha); p.log2_beta = log2f(beta);
  p.len128 = (doc_len + 127) / 128 * 128;
  const int pt = (doc_len + tile - 1) / tile;
  p.n_la_bits = pt * (pt + 1) / 2;
  p.col_cnt = static_cast<int32_t*>(workspace);
  p.tile_flag = p.col_cnt + (int64_t)n_q_heads * p.len128;
  cudaStream_t st = (cudaStream_t)stream;
  cudaGetLastError();
  cudaMemsetAsync(workspace, 0, need, st);
  rc = head_dim == 128 ? enc_launch<128>(p, Q, K, q_row_stride, k_row_stride, st) : enc_launch<64>(p, Q, K, q_row_stride, k_row_stride, st);
  if (rc) return rc;
  const int la_bytes = (p.n_la_bits + 7) / 8, ca_bytes = ((doc_len + cross_gran - 1) / cross_gran + 7) / 8;
  sift_encode_pack_kernel<<<n_q_heads, 256, 0, st>>>(p, gamma, la_out, ca_out, la_bytes, ca_bytes);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return set_error(SIFT_ERR_CUDA, "encode launch: %s", cudaGetErrorString(e));
  count_launch(2);
  return SIFT_OK;
}

// ---- sift_encode_document_static: the encoder for callers that have no device allocator (include/sift.h) ----
// The per-key counters and per-tile flags that sift_encode_document keeps in a caller-supplied workspace live here in
// a fixed array inside the library's device image.  The CUDA runtime places it in every GPU's memory when the module is
// loaded there and releases it when the process exits: SIFT_ENCODE_STATIC_SCRATCH_BYTES per GPU, used or not.
static __device__ __align__(256) unsigned char g_encode_static_scratch[SIFT_ENCODE_STATIC_SCRATCH_BYTES];

namespace sift {
// In host code `g_encode_static_scratch` is only the host-side handle of the symbol, not a device address; the address
// a kernel can use differs per GPU and is looked up once per device, with that device current, and remembered here.
constexpr int kMaxStaticDevices = 64;
static std::mutex g_static_mu;
static void* g_static_ptr[kMaxStaticDevices];   // device address of the array on device i, NULL until its first call

static int encode_static_scratch(void** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return set_error(SIFT_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxStaticDevices) return set_error(SIFT_ERR_UNSUPPORTED, "device ordinal %d >= %d", dev, kMaxStaticDevices);
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_encode_static_scratch);
    if (e != cudaSuccess || !ptr) {
      cudaGetLastError();
      return set_error(SIFT_ERR_CUDA, "cudaGetSymbolAddress(static encoder scratch) on device %d: %s", dev, cudaGetErrorString(e));
    }
    g_static_ptr[dev] = ptr;
  }
  *out = g_static_ptr[dev];
  return SIFT_OK;
}
}  // namespace sift

extern "C" size_t sift_encode_static_scratch_bytes(void) { return (size_t)SIFT_ENCODE_STATIC_SCRATCH_BYTES; }

extern "C" int sift_encode_document_static(int32_t doc_len, int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim,
                                           int32_t tile, int32_t cross_gran, const void* Q, const void* K,
                                           int64_t q_row_stride, int64_t k_row_stride, const float* lse, float alpha,
                                           float beta, float gamma, float softmax_scale, uint8_t* la_out, uint8_t* ca_out,
                                           void* stream) {
  int rc = enc_check(doc_len, n_q_heads, n_kv_heads, head_dim, tile, cross_gran);
  if (rc) return rc;
  size_t need = 0;
  if ((rc = sift_encode_workspace_size(doc_len, n_q_heads, tile, &need))) return rc;
  if (need > (size_t)SIFT_ENCODE_STATIC_SCRATCH_BYTES)
    return set_error(SIFT_ERR_WORKSPACE,
                     "sift_encode_document_static: doc_len %d x %d q-heads at tile %d needs %zu bytes of scratch, the "
                     "built-in array holds %zu (SIFT_ENCODE_STATIC_SCRATCH_BYTES); use sift_encode_document with a "
                     "workspace of your own, or encode fewer heads per call",
                     doc_len, n_q_heads, tile, need, (size_t)SIFT_ENCODE_STATIC_SCRATCH_BYTES);
  void* scratch = nullptr;
  if ((rc = encode_static_scratch(&scratch))) return rc;
  // From here on it is the ordinary encoder on the built-in scratch: it clears the `need` bytes it uses on `stream`
  // (the array still holds the previous call's counts), runs the score and pack kernels, and allocates nothing.
  return sift_encode_document(doc_len, n_q_heads, n_kv_heads, head_dim, tile, cross_gran, Q, K, q_row_stride, k_row_stride,
                              lse, alpha, beta, gamma, softmax_scale, la_out, ca_out, scratch,
                              (size_t)SIFT_ENCODE_STATIC_SCRATCH_BYTES, stream);
}
