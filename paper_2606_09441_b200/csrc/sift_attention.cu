// SIFT block-sparse causal prefill attention for sm_100a (sec 5.2; mask per L147-149, L201-209).
//
// Paper design (FlashAttention-3 on H200: TMA + wgmma, the N-block index read from sparse_n_indices[i]) is prior art.
// This kernel keeps the idea "an index list drives which K/V tile the copy engine fetches" and is otherwise built for
// Blackwell:
//   * persistent CTAs (one per SM, 16 warps) pull (q-head, M-block) work items through an atomic counter in the order the
//     decode's scheduler fixed (kv-head groups sized to the L2, longest first inside a group);
//   * an M-block is kNQ = 2 query tiles of 128 TMEM lanes of the same document and head: they share the head's cross
//     list, so every gathered K/V tile in shared memory feeds two accumulators;
//   * warp roles: warp 13 = work-item fetch + Q tiles (TMA); warp 1 = tcgen05.mma issuer (warp-uniform operands, one
//     elected lane issues); warps 2, 3, 14 = K producers, warps 0, 12, 15 = V producers (tiled TMA boxes for local tiles,
//     pages and dense rows; TMA `tile::gather4` for the row-granular cross keys); warps 4..11 = one softmax
//     warpgroup per query tile (one row per thread, S read with tcgen05.ld, P written back to TMEM as bf16 in four key
//     ranges and used as the A operand of the P*V MMAs, lazy rescale of the TMEM-resident O accumulator);
//   * registers are re-split with setmaxnreg per sub-partition: softmax 216, MMA issuer 56, producers 40, item warp 24;
//   * S = Q K^T and O += P V are tcgen05.mma.kind::f16 (bf16 in, fp32 accumulate in TMEM).
// Work decomposition of one DOC item (document d >= 0, head h):
//   cross phase  groups of 128 entries of cross_idx[h][0 .. cross_ptr[h][d]) (G = 1; one listed page per step at G = tile)  (a6)
//   local phase  union of the tiles' local lists; the diagonal tile is causally masked  (a7)
// and of a DENSE item (user-query rows, or the dense comparator): key blocks 0,128,.. up to the last row (a8).
#include <cuda.h>
#include <cuda_bf16.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <type_traits>

#include "sift_common.h"
#include "sm100_ptx.cuh"

namespace sift {
using namespace ptx;

constexpr int kNQ = SIFT_Q_TILES_PER_ITEM;  // query tiles per work item
static_assert(kNQ == 2, "an M-block is two query tiles: two softmax warpgroups, two S and two O accumulators in TMEM");
constexpr int kBM = 128;                    // rows of one query tile = TMEM lanes
constexpr int kBN = 128;                    // keys per step
#ifndef SIFT_PV_PARTS
#define SIFT_PV_PARTS 4
#endif
constexpr int kPvParts = SIFT_PV_PARTS;     // P V is issued in this many key ranges, each as soon as its P is written
static_assert(kPvParts == 1 || kPvParts == 2 || kPvParts == 4, "P V parts");
constexpr int kNumThreads = 256 + 128 * kNQ;        // 16 warps, every one with a role: V/MMA/K/K, two softmax warpgroups, V/item/K/V
                                                   // (4 warps per SM sub-partition: registers are pooled per sub-partition)
constexpr int kFirstVWarp = 4 + 4 * kNQ;
constexpr int kProducerThreads = 96;              // per operand: K = warps 2, 3, 14; V = warps 0, 12, 15
constexpr float kRescaleThreshold = 8.0f;   // log2 units: P stays <= 2^8 with a stale max
constexpr uint32_t kTmemCols = 512;

constexpr int kRegsEntry = (kNQ == 2) ? 128 : 168;               // what __launch_bounds__(kNumThreads, 1) yields
// 4 warps per sub-partition share 512 registers per lane: 2 x 216 + 2 x 40 (measured: 208/48 -1%, 200/56 -5%, 192/64 -30%:
// the softmax loop holds a whole 128-column row of S)
constexpr int kRegsOther = 40;                                   // producer warps after setmaxnreg.dec
constexpr int kItemWarp = kFirstVWarp + 1;                       // warp 13: item fetch + Q loads; shares sub-partition 1 with
constexpr int kRegsItem = 24, kRegsMma = 56;                     // the MMA issuer (warp 1), whose loop spilled at 40 registers
constexpr int kRegsSoftmax = 216;              // softmax warps after setmaxnreg.inc

static_assert(kNQ * kRegsSoftmax + 2 * kRegsOther <= (kNumThreads / 128) * kRegsEntry &&
              kNQ * kRegsSoftmax + kRegsItem + kRegsMma <= (kNumThreads / 128) * kRegsEntry,
              "setmaxnreg budget exceeds the register pool the CTA is launched with (softmax warps would block)");

struct AttnParams {
  // metadata (null in dense mode)
  const int32_t *tile_seg, *tile_row0, *tile_rows, *mblock_tile0;
  const int32_t* seg_info;   // [n_seg][4]: document index (-1: query), first document / first row / first tile of the prompt
  const int32_t *cross_ptr, *cross_idx, *local_cnt, *local_ptr, *local_idx;  // already offset to the layer
  const int32_t* sched;                                                      // already offset to the layer
  int32_t* counters;                                                         // [2]: next item, finished CTAs
  int32_t n_items, n_docs, n_tiles, cross_cap, local_cap, n_mblocks;
  int32_t zero;   // always 0 (see the TMEM address note in the kernel)
  int32_t dense;  // 1: every M-block is a DENSE item over n_tokens rows
  int32_t n_tokens, n_q_heads, n_kv_heads, tile;
  int32_t kv_per_group;     // dense comparator: kv heads scheduled together (sched_kv_heads_per_group)
  int32_t o_vec32;          // O rows are 32-byte aligned: the epilogue may use 256-bit stores
  int32_t paged;            // cross_gran == tile: cross entries are global tile ids, one tiled step each
  int32_t row_lo, row_hi;   // only rows [row_lo, row_hi) are computed and written (sift_prefill_attention_rows; the whole
                            // prompt: 0, n_tokens)
  int32_t ranged;           // the range is a proper part: the item warp skips M-blocks outside [mb_lo, mb_hi)
  int32_t mb_lo, mb_hi;
  __nv_bfloat16* o;
  int64_t o_row_stride;
  float* lse;  // [Hq][N] or null
  float scale_log2;
};

// EB = bytes per Q/K/V element: 2 = bf16 (kind::f16), 1 = e4m3 (kind::f8f6f4, reading R7)
template <int HD, int EB = 2>
struct Smem {
  static_assert(HD * EB % 128 == 0, "a tile row is a whole number of 128-byte swizzle rows");
  static constexpr int kHalves = HD * EB / 128;            // 128-byte column blocks of a tile
  static constexpr int kHalfElems = 128 / EB;              // elements per block row
  static constexpr int kTileBytes = kBN * HD * EB;         // one K or V tile / one Q tile
  // d = 128: 5 stages of 32 KB fit beside the two Q tiles; 2 K + 3 V measured 1-3% faster than 3 K + 2 V (a V stage is
  // held from the P V of one step to the end of the next, a K stage only across its own Q K^T)
  static constexpr int kKStages = (kTileBytes == 32768 ? 2 : 4);
  static constexpr int kVStages = (kTileBytes == 32768 ? 3 : 4);
  static constexpr int kQOff = 0;
  static constexpr int kKOff = kQOff + kNQ * kTileBytes;
  static constexpr int kVOff = kKOff + kKStages * kTileBytes;
  static constexpr int kBarOff = kVOff + kVStages * kTileBytes;
  // barrier slots (8 B each)
  static constexpr int bQFull = 0, bQEmpty = 1;
  static constexpr int bKFull = 2, bKEmpty = bKFull + kKStages;
  static constexpr int bVFull = bKEmpty + kKStages, bVEmpty = bVFull + kVStages;
  static constexpr int bSFull = bVEmpty + kVStages, bPFull = bSFull + kNQ, bODone = bPFull + kNQ * kPvParts;   // bPFull + part * kNQ + q
  static constexpr int bItemFull = bODone + kNQ, bItemEmpty = bItemFull + 2;
  static constexpr int bInfoFull = bItemEmpty + 2;      // the item warp has decoded the item of this slot (for the softmax warpgroups)
  static constexpr int kNumBars = bInfoFull + 2;
  static constexpr int kInfoOff = kBarOff + ((kNumBars * 8 + 15) / 16) * 16;
  // info words: [0] tmem base, [1..2] item ring, [3] "the item has MMA steps" (item warp -> MMA issuer), [4 .. 4+kKStages) per-K-stage step info,
  // [16 .. 48) the decoded work items of the two ring slots (item warp -> softmax warpgroups, 16 words each)
  static constexpr int kBytes = kInfoOff + 64 + 2 * 64;
  static_assert(kBytes <= 227 * 1024, "shared memory budget");
};

// One work item as every role sees it.
struct Item {
  int h, kvh;
  int is_dense;            // DENSE (query rows / comparator) or DOC
  int row0[kNQ], rows[kNQ];  // global first row and valid rows of each query tile (rows <= 0: tile absent)
  int tile_id[kNQ];
  int c0, cp;              // DOC: its document attends cross entries [c0, cp) of the head's list (c0 = start of the
                           // prompt's list, a multiple of 128; 0 with one prompt)
  int kbase;               // DENSE: first key row (first row of the prompt; 0 with one prompt and in the comparator)
  int lptr[kNQ], lcnt[kNQ];  // DOC: local list of each tile
};

// what a softmax warpgroup needs of a work item, as the item warp publishes it through shared memory (16 words per ring
// slot): the dependent global loads of load_item plus the diagonal test then run once, a whole item ahead, instead of at
// the start of every item on the warpgroup's own path
struct ItemInfo {
  int h, is_dense, c0, cp, kbase, row0[kNQ], rows[kNQ], lcnt[kNQ], diag[kNQ];
};
__device__ __forceinline__ void publish_item(volatile int32_t* w, const Item& it, const int (&diag)[kNQ]) {
  w[0] = it.h; w[1] = it.is_dense; w[2] = it.c0; w[3] = it.cp; w[4] = it.kbase;
#pragma unroll
  for (int q = 0; q < kNQ; ++q) { w[5 + q] = it.row0[q]; w[7 + q] = it.rows[q]; w[9 + q] = it.lcnt[q]; w[11 + q] = diag[q]; }
}
__device__ __forceinline__ ItemInfo read_item(const volatile int32_t* w) {
  ItemInfo it;
  it.h = w[0]; it.is_dense = w[1]; it.c0 = w[2]; it.cp = w[3]; it.kbase = w[4];
#pragma unroll
  for (int q = 0; q < kNQ; ++q) { it.row0[q] = w[5 + q]; it.rows[q] = w[7 + q]; it.lcnt[q] = w[9 + q]; it.diag[q] = w[11 + q]; }
  return it;
}

__device__ __forceinline__ Item load_item(const AttnParams& p, int code) {
  Item it;
  const int h = code >> 20, mb = code & 0xFFFFF;
  it.h = h;
  it.kvh = h / (p.n_q_heads / p.n_kv_heads);
  it.c0 = 0; it.cp = 0; it.kbase = 0;
  if (p.dense) {
    it.is_dense = 1;
#pragma unroll
    for (int q = 0; q < kNQ; ++q) {
      it.row0[q] = (mb * kNQ + q) * kBM;
      it.rows[q] = min(kBM, p.n_tokens - it.row0[q]);
      it.tile_id[q] = 0; it.lptr[q] = 0; it.lcnt[q] = 0;
    }
    return it;
  }
  const int t0 = p.mblock_tile0[mb];
  const int nt = min(kNQ, p.mblock_tile0[mb + 1] - t0);
  const int seg = p.tile_seg[t0];
  const int4 si = reinterpret_cast<const int4*>(p.seg_info)[seg];
  it.is_dense = (si.x < 0);
  it.kbase = si.z;
  const int64_t lh = h;  // pointers are already offset to the layer
  if (!it.is_dense) {
    it.c0 = p.cross_ptr[lh * (p.n_docs + 1) + si.y];
    it.cp = p.cross_ptr[lh * (p.n_docs + 1) + si.x];
  }
#pragma unroll
  for (int q = 0; q < kNQ; ++q) {
    bool on = q < nt;
    if (on) {
      it.row0[q] = p.tile_row0[t0 + q];
      it.rows[q] = p.tile_rows[t0 + q];
      on = it.row0[q] < p.row_hi && it.row0[q] + it.rows[q] > p.row_lo;   // a tile outside the row range is absent
    }
    if (on) {
      it.tile_id[q] = t0 + q;
      it.lptr[q] = p.local_ptr[lh * (p.n_tiles + 1) + t0 + q];
      it.lcnt[q] = p.local_cnt[lh * p.n_tiles + t0 + q];
    } else {
      it.tile_id[q] = -1; it.row0[q] = 0; it.rows[q] = 0; it.lptr[q] = 0; it.lcnt[q] = 0;
    }
  }
  return it;
}

// number of key blocks a DENSE tile attends: keys 0 .. row0+rows-1
__device__ __forceinline__ int dense_steps(int row0, int rows) { return rows > 0 ? (row0 + rows + kBN - 1) / kBN : 0; }


// ------------------------------------------------------------------------------------------------
// descriptors
// ------------------------------------------------------------------------------------------------
// Q / K tile in smem: blocks of [128 rows x 128 B], 128-byte swizzle (what TMA writes).  K-chunk k = 32 bytes of a row
// (16 bf16 or 32 e4m3 = one MMA's K):
__device__ __forceinline__ uint64_t kmajor_desc(uint32_t tile_addr, int k) {
  return umma_desc_sw128(tile_addr + (k >> 2) * (kBN * 128) + (k & 3) * 32, 16, 1024);
}
// V tile, same smem image, used MN-major (N = head dim contiguous): K-chunk k = the key rows of one MMA (16 bf16 rows =
// 2 KB, 32 e4m3 rows = 4 KB), column blocks kBN * 128 bytes apart
template <int EB>
__device__ __forceinline__ uint64_t v_desc(uint32_t tile_addr, int k) {
  return umma_desc_sw128(tile_addr + k * (4096 / EB), kBN * 128, 1024);
}

// compile-time unrolled issue loops (the TMEM offsets must be immediates)
// (K counts MMA K-steps: 16 keys (bf16) or 32 keys (e4m3) of P = 8 TMEM columns either way)
template <int EB, int Q, int ACC, int K, int KEND>
__device__ __forceinline__ void issue_pv(uint32_t tz, uint32_t vt, uint32_t idesc) {
  if constexpr (K < KEND) {
    umma_ts_off<256 + Q * 128, Q * 128 + K * 8, EB == 1>(tz, v_desc<EB>(vt, K), idesc, (ACC) | (K > 0));
    issue_pv<EB, Q, ACC, K + 1, KEND>(tz, vt, idesc);
  }
}
template <int HD, int EB, int Q, int K = 0>
__device__ __forceinline__ void issue_qk(uint32_t tz, uint32_t qt, uint32_t kt, uint32_t idesc) {
  if constexpr (K < HD * EB / 32) {
    umma_ss_off<Q * 128, EB == 1>(tz, kmajor_desc(qt, K), kmajor_desc(kt, K), idesc, K > 0);
    issue_qk<HD, EB, Q, K + 1>(tz, qt, kt, idesc);
  }
}

// e4m3 path: per-q-head factors (kernel parameter, by value): logits scale in log2 units and the scale of V
struct F8Scales {
  float qk_log2[256];   // softmax_scale * log2(e) * q_scale[h] * k_scale[kv(h)]
  float v[256];         // v_scale[kv(h)]
};
constexpr float kP8Shift = 64.f;             // e4m3 P is stored as 2^6 P: weights down to 2^-15 stay representable
constexpr float kRescaleThresholdF8 = 2.0f;  // so that 2^6 P <= 2^8 < 448 with a stale max

// N bf16 of one row of O (packed in pairs) to global memory
template <int HD>
__device__ __forceinline__ void store_o_row(__nv_bfloat16* row, const uint32_t (&w)[HD / 2], bool vec32) {
  if (vec32) {
    // 32-byte stores: every lane fills a whole sector of its own row (a thread owns a row, so a 16-byte store touches
    // half a sector; +0.7% at 32K, +1.8% at 10K)
#pragma unroll
    for (int i = 0; i < HD / 16; ++i)
      asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(row + i * 16), "r"(w[8 * i]), "r"(w[8 * i + 1]),
                   "r"(w[8 * i + 2]), "r"(w[8 * i + 3]), "r"(w[8 * i + 4]), "r"(w[8 * i + 5]), "r"(w[8 * i + 6]),
                   "r"(w[8 * i + 7]) : "memory");
  } else {
#pragma unroll
    for (int i = 0; i < HD / 8; ++i)
      *reinterpret_cast<uint4*>(row + i * 8) = make_uint4(w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
  }
}

template <int HD, int EB>
__device__ __forceinline__ void sift_attention_body(const CUtensorMap& tm_q, const CUtensorMap& tm_k, const CUtensorMap& tm_v,
                                                    const CUtensorMap& tm_kg, const CUtensorMap& tm_vg, const AttnParams& p,
                                                    const F8Scales* f8) {
  using S = Smem<HD, EB>;
  constexpr bool kF8 = (EB == 1);
  extern __shared__ __align__(1024) uint8_t smem_raw[];    // the only shared memory of the kernel: starts 1024-aligned
  const uint32_t sbase = smem_u32(smem_raw);
  uint8_t* sgen = smem_raw;
  if ((sbase & 1023u) != 0) { if (threadIdx.x == 0) printf("sift: dynamic shared memory not 1024-byte aligned\n"); __trap(); }
  const uint32_t bar0 = sbase + S::kBarOff;
  auto bar = [&](int i) -> uint32_t { return bar0 + i * 8; };
  volatile int32_t* info = reinterpret_cast<volatile int32_t*>(sgen + S::kInfoOff);
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;   // warp-uniform role id
  constexpr uint32_t idesc_qk = kF8 ? umma_idesc_e4m3(kBM, kBN, 0, 0) : umma_idesc_bf16(kBM, kBN, 0, 0);
  constexpr uint32_t idesc_pv = kF8 ? umma_idesc_e4m3(kBM, HD, 0, 1) : umma_idesc_bf16(kBM, HD, 0, 1);
  constexpr int kPvSteps = kBN * EB / 32;     // MMA K-steps of one P V (16 bf16 keys or 32 e4m3 keys each)

  if (warp == 0 && lane == 0) {
    mbar_init(bar(S::bQFull), 1);
    mbar_init(bar(S::bQEmpty), 1);
    for (int i = 0; i < S::kKStages; ++i) { mbar_init(bar(S::bKFull + i), kProducerThreads); mbar_init(bar(S::bKEmpty + i), 1); }
    for (int i = 0; i < S::kVStages; ++i) { mbar_init(bar(S::bVFull + i), kProducerThreads); mbar_init(bar(S::bVEmpty + i), 1); }
    for (int q = 0; q < kNQ; ++q) {
      mbar_init(bar(S::bSFull + q), 1);
      for (int part = 0; part < kPvParts; ++part) mbar_init(bar(S::bPFull + part * kNQ + q), 128);   // P of one key range written
      mbar_init(bar(S::bODone + q), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar(S::bItemFull + i), 1); mbar_init(bar(S::bItemEmpty + i), 7 + 128 * kNQ); mbar_init(bar(S::bInfoFull + i), 1);
    }
    fence_barrier_init();
    prefetch_tensormap(&tm_q); prefetch_tensormap(&tm_k); prefetch_tensormap(&tm_v);
    prefetch_tensormap(&tm_kg); prefetch_tensormap(&tm_vg);
  }
  if (warp == 2) {
    tmem_alloc(smem_u32(const_cast<int32_t*>(&info[0])), kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  // The CTA owns the whole TMEM (512 columns, 1 CTA per SM), so the allocation starts at column 0, lane 0: addresses
  // below are compile-time constants (uniform registers for the MMA issuer).
  if (info[0] != 0) { if (threadIdx.x == 0) printf("sift: unexpected TMEM base %d\n", (int)info[0]); __trap(); }
  // (p.zero is a kernel parameter that is always 0: an operand ptxas must treat as a uniform run-time value, which
  // keeps the tcgen05 address operands in uniform registers instead of a vector-register constant + R2UR.)
  constexpr uint32_t tmem_base = 0;
  const uint32_t tz = (uint32_t)p.zero;

  // register budget: the four non-softmax warps give registers to the softmax warpgroups (setmaxnreg at the top of
  // every role branch so that it dominates the role's code)
  if (warp == kItemWarp) {
    // ======================================= item fetch + Q producer =======================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsItem));
    const uint32_t q_smem = sbase + S::kQOff;
    for (int it_n = 0;;) {
      const int slot = it_n & 1;
      mbar_wait(bar(S::bItemEmpty + slot), ((it_n >> 1) & 1) ^ 1, 100);
      int code = -1;
      if (lane == 0) {
        const int idx = atomicAdd(&p.counters[0], 1);
        if (idx < p.n_items) {
          if (p.dense) {   // kv-head groups one after the other, longest M-blocks first inside a group
            const int hpg = (p.n_q_heads / p.n_kv_heads) * p.kv_per_group, per_group = hpg * p.n_mblocks;   // (last group may be short)
            const int g = idx / per_group, rem = idx - g * per_group;
            const int hin = min(hpg, p.n_q_heads - g * hpg);   // q-heads in this group
            code = ((g * hpg + rem % hin) << 20) | (p.n_mblocks - 1 - rem / hin);
          } else {
            code = p.sched[idx];
          }
        }
        if (code < 0) {
          const int f = atomicAdd(&p.counters[1], 1);
          if (f == (int)gridDim.x - 1) { atomicExch(&p.counters[0], 0); atomicExch(&p.counters[1], 0); }
        }
      }
      code = __shfl_sync(0xffffffffu, code, 0);
      // row-range call: M-blocks are numbered in token order, so the ones with rows in [row_lo, row_hi) are the index
      // range [mb_lo, mb_hi) the host worked out; an item outside it is dropped here and the next one fetched into the
      // same ring slot (one atomic + one load per skipped item, on this warp only: no other role sees a skipped item)
      if (p.ranged && code >= 0 && ((code & 0xFFFFF) < p.mb_lo || (code & 0xFFFFF) >= p.mb_hi)) continue;
      if (lane == 0) {
        info[1 + slot] = code;
        mbar_arrive(bar(S::bItemFull + slot));
      }
      __syncwarp();
      if (code < 0) break;
      const Item it = load_item(p, code);
      {
        int diag[kNQ];
#pragma unroll
        for (int q = 0; q < kNQ; ++q)
          diag[q] = !it.is_dense && it.lcnt[q] > 0 &&
                    p.local_idx[(int64_t)it.h * p.local_cap + it.lptr[q] + it.lcnt[q] - 1] == it.tile_id[q];
        if (lane == 0) {
          publish_item(info + 16 + 16 * slot, it, diag);
          mbar_arrive(bar(S::bInfoFull + slot));
        }
      }
      // ---- Q tiles
      mbar_wait(bar(S::bQEmpty), (it_n & 1) ^ 1, 101);
      if (lane == 0) {
        // "this item has MMA steps", for the MMA issuer: it reads the word after its wait on bQFull (this thread's
        // arrive below releases it), so the issuer never repeats the dependent global loads of load_item, which sat on
        // its serial path at every item boundary (~3000 clk with the tensor pipe idle)
        bool hs = it.is_dense || it.cp > it.c0;
#pragma unroll
        for (int q = 0; q < kNQ; ++q) hs = hs || it.lcnt[q] > 0;
        info[3] = hs ? 1 : 0;
        mbar_arrive_expect_tx(bar(S::bQFull), kNQ * S::kTileBytes);
#pragma unroll
        for (int q = 0; q < kNQ; ++q)
#pragma unroll
          for (int hf = 0; hf < S::kHalves; ++hf)
            tma_load_2d(q_smem + q * S::kTileBytes + hf * (kBM * 128), &tm_q, bar(S::bQFull), it.h * HD + hf * S::kHalfElems,
                        it.row0[q]);
      }
      __syncwarp();
      ++it_n;
    }
  } else if (warp == 0 || warp == 2 || warp == 3 || (warp >= kFirstVWarp && warp != kItemWarp)) {
    // ======================================= K (warps 2,3) / V (last two warps) producers =======================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsOther));
    // 96 threads per operand.  Tiled steps (local tiles, pages, dense rows): one thread issues one TMA box per 64-column
    // half.  Gathered steps (row-granular cross keys): TMA `tile::gather4`, one instruction per lane and 64-column half
    // (ptxas serialises the 32 lanes of a gather4 into a loop of uniform-datapath issues, ~70 clk each from one warp,
    // which is why three warps per operand issue them: profiles/r1_gather_modes.md).
    // K: warps 2, 3, 14; V: warps 0, 12, 15 (sub-partition 1 keeps the MMA issuer and the light item warp: registers)
    const bool is_k = warp == 2 || warp == 3 || warp == kFirstVWarp + 2;
    const int pw = is_k ? (warp == 2 ? 0 : (warp == 3 ? 1 : 2)) : (warp == 0 ? 0 : (warp == kFirstVWarp ? 1 : 2));   // 0..2
    const int ptid = pw * 32 + lane;
    const int n_stages = is_k ? S::kKStages : S::kVStages;
    const int b_full = is_k ? S::bKFull : S::bVFull, b_empty = is_k ? S::bKEmpty : S::bVEmpty;
    const uint32_t ring = sbase + (is_k ? S::kKOff : S::kVOff);
    const CUtensorMap* tm_tile = is_k ? &tm_k : &tm_v;
    const CUtensorMap* tm_gath = is_k ? &tm_kg : &tm_vg;
    uint32_t st = 0, ph = 0;
    for (int it_n = 0;; ++it_n) {
      const int slot = it_n & 1;
      mbar_wait(bar(S::bItemFull + slot), (it_n >> 1) & 1, 400);
      const int code = info[1 + slot];
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(S::bItemEmpty + slot));
      if (code < 0) break;
      const Item it = load_item(p, code);
      auto emit = [&](bool gather, int src, int act, bool last) {
        // src: gather -> index of the first cross entry of the group; tiled -> first key row
        const uint32_t full = bar(b_full + st), dst = ring + st * S::kTileBytes;
        {
          // gather4 slots: 2 halves x 32 groups of 4 rows = 64 per tile, spread 22 / 22 / 20 over the three warps
          const int g = pw * 22 + lane;
          const bool g_on = gather && lane < 22 && g < 32 * S::kHalves;
          int4 r = make_int4(0, 0, 0, 0);
          if (g_on) r = *reinterpret_cast<const int4*>(p.cross_idx + (int64_t)it.h * p.cross_cap + src + (g & 31) * 4);
          mbar_wait(bar(b_empty + st), ph ^ 1, 401);
          if (ptid == 0) {
            if (is_k) info[4 + st] = act | (last ? 4 : 0);
            mbar_arrive_expect_tx(full, S::kTileBytes);
          } else {
            mbar_arrive(full);
          }
          if (gather) {
            if (g_on)
              tma_gather4(dst + (g >> 5) * (kBN * 128) + (g & 31) * 512, tm_gath, full, it.kvh * HD + (g >> 5) * S::kHalfElems, r.x, r.y, r.z, r.w);
          } else if (ptid == 0) {
#pragma unroll
            for (int hf = 0; hf < S::kHalves; ++hf)
              tma_load_2d(dst + hf * (kBN * 128), tm_tile, full, it.kvh * HD + hf * S::kHalfElems, src);
          }
        }
        if (++st == (uint32_t)n_stages) { st = 0; ph ^= 1; }
      };
      if (it.is_dense) {
        int n[kNQ], total = 0;
#pragma unroll
        for (int q = 0; q < kNQ; ++q) { n[q] = dense_steps(it.row0[q] - it.kbase, it.rows[q]); total = max(total, n[q]); }
        for (int j = 0; j < total; ++j) {
          int act = 0;
#pragma unroll
          for (int q = 0; q < kNQ; ++q) act |= (j < n[q]) << q;
          emit(false, it.kbase + j * kBN, act, j == total - 1);
        }
      } else {
        int present = 0, nloc = 0;
#pragma unroll
        for (int q = 0; q < kNQ; ++q) { present |= (it.rows[q] > 0) << q; nloc += it.lcnt[q]; }
        const int ngroups = p.paged ? 0 : (it.cp - it.c0 + kBN - 1) / kBN;
        if (p.paged) {                     // page-granular cross keys: the listed pages as tiled boxes
          const int32_t* cidx = p.cross_idx + (int64_t)it.h * p.cross_cap;
          // the page's first row is two dependent loads away (entry -> tile_row0): fetched one step ahead, so that the
          // latency runs under the wait for the stage instead of in front of every TMA issue
          int row_next = it.c0 < it.cp ? p.tile_row0[cidx[it.c0]] : 0;
          for (int e = it.c0; e < it.cp; ++e) {
            const int row = row_next;
            if (e + 1 < it.cp) row_next = p.tile_row0[cidx[e + 1]];
            emit(false, row, present, e == it.cp - 1 && nloc == 0);
          }
        }
        for (int g = 0; g < ngroups; ++g) emit(true, it.c0 + g * kBN, present, g == ngroups - 1 && nloc == 0);
        const int32_t* lidx = p.local_idx + (int64_t)it.h * p.local_cap;
        int pos[kNQ];
#pragma unroll
        for (int q = 0; q < kNQ; ++q) pos[q] = 0;
        while (true) {
          int cur[kNQ], t = 0x7fffffff;
#pragma unroll
          for (int q = 0; q < kNQ; ++q) {
            cur[q] = pos[q] < it.lcnt[q] ? lidx[it.lptr[q] + pos[q]] : 0x7fffffff;
            t = min(t, cur[q]);
          }
          if (t == 0x7fffffff) break;
          int act = 0, remaining = 0;
#pragma unroll
          for (int q = 0; q < kNQ; ++q) {
            if (cur[q] == t) { act |= 1 << q; ++pos[q]; }
            remaining += it.lcnt[q] - pos[q];
          }
          emit(false, p.tile_row0[t], act, remaining == 0);
        }
      }
    }
  } else if (warp == 1) {
    // ======================================= MMA issuer =======================================
    // The whole warp walks the loop so that every address / descriptor is warp-uniform (values read from shared
    // memory are re-broadcast with shfl so that ptxas keeps them in uniform registers); one elected lane issues.
    // With a divergent `if (lane == 0)` around the loop every tcgen05.mma operand took an R2UR round trip and the
    // issuing thread itself became the bottleneck (profiles/r1_mma_issue.md).
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsMma));
    uint32_t kst = 0, kph = 0, vst = 0, vph = 0, pph[kNQ];
#pragma unroll
    for (int q = 0; q < kNQ; ++q) pph[q] = 0;
    const uint32_t q_smem = sbase + S::kQOff, k_smem = sbase + S::kKOff, v_smem = sbase + S::kVOff;
    for (int it_n = 0;; ++it_n) {
      const int slot = it_n & 1;
      mbar_wait(bar(S::bItemFull + slot), (it_n >> 1) & 1, 200);
      const int code = __shfl_sync(0xffffffffu, (int)info[1 + slot], 0);
      if (lane == 0) mbar_arrive(bar(S::bItemEmpty + slot));
      if (code < 0) break;
      mbar_wait(bar(S::bQFull), it_n & 1, 201);
      const int has_steps = __shfl_sync(0xffffffffu, (int)info[3], 0);   // written by the item warp before its Q loads
      if (!has_steps) {
        if (lane == 0) mbar_arrive(bar(S::bQEmpty));
        continue;
      }
      tc_fence_after();
      // PV of step j-1 is issued in iteration j, right before Q K^T of step j for the same query tile (tensor-pipe
      // order PV0 QK0 PV1 QK1: the softmax of one tile overlaps the MMAs of the other).  `pending`, `act` and
      // `fresh` come from shared memory, which ptxas cannot prove warp-uniform: they only steer branches, while every
      // MMA operand is built from uniform counters (kst, vst, j) and constants.
#define SIFT_ISSUE_PV(q, ACC, K0, K1, LAST)                                                                      \
  if (elect_one()) {                                                                                             \
    issue_pv<EB, q, ACC, K0, K1>(tz, vt, idesc_pv);                                                              \
    if (LAST) umma_commit(bar(S::bODone + q));                                                                   \
  }                                                                                                              \
  __syncwarp();
  // P arrives in kPvParts key ranges: the early parts of P V run while the softmax still works on the later keys
#define SIFT_PV_PART(q, PART)                                                                                    \
  if constexpr (PART < kPvParts) {                                                                               \
    mbar_wait(bar(S::bPFull + PART * kNQ + q), pph[q], 202);                                                     \
    tc_fence_after();                                                                                            \
    if (PART == 0 && (fresh & (1 << q))) {                                                                       \
      SIFT_ISSUE_PV(q, 0, PART * (kPvSteps / kPvParts), (PART + 1) * (kPvSteps / kPvParts), PART == kPvParts - 1) \
    } else {                                                                                                     \
      SIFT_ISSUE_PV(q, 1, PART * (kPvSteps / kPvParts), (PART + 1) * (kPvSteps / kPvParts), PART == kPvParts - 1) \
    }                                                                                                            \
  }
#define SIFT_PV_STEP(q)                                                                                          \
  if (pending & (1 << q)) {                                                                                      \
    SIFT_PV_PART(q, 0) SIFT_PV_PART(q, 1) SIFT_PV_PART(q, 2) SIFT_PV_PART(q, 3)                                  \
    pph[q] ^= 1;                                                                                                 \
    fresh &= ~(1 << q);                                                                                          \
  }
#define SIFT_QK_STEP(q)                                                                                          \
  SIFT_PV_STEP(q)                                                                                                \
  if (act & (1 << q)) {                                                                                          \
    if (elect_one()) {                                                                                           \
      issue_qk<HD, EB, q>(tz, q_smem + q * S::kTileBytes, kt, idesc_qk);                                         \
      umma_commit(bar(S::bSFull + q));                                                                           \
    }                                                                                                            \
    __syncwarp();                                                                                                \
  }
      int pending = 0, fresh = (1 << kNQ) - 1;   // fresh bit q: the next P V of tile q overwrites O instead of accumulating
      // One loop body serves the steps and the drain iteration after the last step (P V of the last step only, no K
      // stage): a separate tail would duplicate all the P V issue code (the issuer's loop is ~10 KB of SASS as it is, and
      // the hot loops of the roles compete for a 32 KB instruction cache).
      bool last = false;
      for (int j = 0;; ++j) {
        const bool drain = last;                 // the previous iteration was the item's last step
        int act = 0;
        if (!drain) {
          mbar_wait(bar(S::bKFull + kst), kph, 204);
          const int inf = info[4 + kst];
          act = inf & 3;
          last = (inf & 4) != 0;
        } else {
          if (elect_one()) umma_commit(bar(S::bQEmpty));   // every Q K^T of this item has been issued
          __syncwarp();
        }
        const uint32_t kt = k_smem + kst * S::kTileBytes, vt = v_smem + vst * S::kTileBytes;
        if (j > 0) mbar_wait(bar(S::bVFull + vst), vph, 203);
        tc_fence_after();
        SIFT_QK_STEP(0)
        if constexpr (kNQ == 2) { SIFT_QK_STEP(1) }
        if (elect_one()) {
          if (j > 0) umma_commit(bar(S::bVEmpty + vst));
          if (!drain) umma_commit(bar(S::bKEmpty + kst));
        }
        __syncwarp();
        if (j > 0) { if (++vst == S::kVStages) { vst = 0; vph ^= 1; } }
        if (drain) break;
        if (++kst == S::kKStages) { kst = 0; kph ^= 1; }
        pending = act;
      }
#undef SIFT_QK_STEP
#undef SIFT_PV_STEP
#undef SIFT_ISSUE_PV
    }
  } else if (warp >= 4 && warp < kFirstVWarp) {
    // ======================================= softmax warpgroups =======================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsSoftmax));
    // One warpgroup per query tile, one row per thread.  ONE copy of the code for both warpgroups (two instantiations
    // measured 7% slower: the loop body is ~10 KB of SASS and both copies would compete for the instruction caches of
    // every sub-partition); the item fields of "my" tile are picked with selects, not indexed (no local memory).
    {
    const int q = (warp - 4) >> 2;
    const int r = (int)threadIdx.x - 128 - q * 128;        // row inside the query tile = TMEM lane
    const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t s_addr = lane_addr + q * 128;
    const uint32_t o_addr = lane_addr + 256 + q * 128;
    float sl = p.scale_log2;                 // (e4m3: per q-head, set with the item)
    const int tile_lim = min(kBN, p.tile);
    uint32_t sph = 0;
    uint32_t pv_cnt = 0;
    for (int it_n = 0;; ++it_n) {
      const int slot = it_n & 1;
      mbar_wait(bar(S::bItemFull + slot), (it_n >> 1) & 1, 300);
      const int code = info[1 + slot];
      if (code < 0) { mbar_arrive(bar(S::bItemEmpty + slot)); break; }
      int row0, rows, h, ngroups, nsteps, diag_step, lim, c0;
      bool paged_item;
      {
        mbar_wait(bar(S::bInfoFull + slot), (it_n >> 1) & 1, 304);
        const ItemInfo it = read_item(info + 16 + 16 * slot);
        mbar_arrive(bar(S::bItemEmpty + slot));
        row0 = q ? it.row0[1] : it.row0[0]; rows = q ? it.rows[1] : it.rows[0]; h = it.h;
        const int lcnt = q ? it.lcnt[1] : it.lcnt[0];
        const int diag = q ? it.diag[1] : it.diag[0];
        if (rows <= 0) continue;
        c0 = it.c0;
        ngroups = it.is_dense ? 0 : (p.paged ? it.cp - it.c0 : (it.cp - it.c0 + kBN - 1) / kBN);
        nsteps = it.is_dense ? dense_steps(row0 - it.kbase, rows) : ngroups + lcnt;
        diag_step = -1;                                   // the step (if any) that is the causally masked diagonal tile
        if (diag) diag_step = nsteps - 1;
        // columns [0, lim) of the current step are allowed for this row; lim drops by kBN per step in the cross
        // phase (ragged last group) and in DENSE items (causal frontier)
        lim = it.is_dense ? row0 - it.kbase + r + 1 : it.cp - it.c0;
        if (it.is_dense) ngroups = nsteps;                // "frontier" steps: all of them
        paged_item = p.paged && !it.is_dense;
        if constexpr (kF8) sl = f8->qk_log2[h];
      }
      float m = -INFINITY, l = 0.f;
      // page-granular cross steps: the valid rows of the page (a document's last page may be ragged) are two dependent
      // loads away; the pair for step e + 1 is issued at the top of step e, so its latency runs under this step's work
      const int32_t* pg_idx = p.cross_idx + (int64_t)h * p.cross_cap + c0;
      int pg_lim = (paged_item && ngroups > 0) ? p.tile_rows[pg_idx[0]] : kBN;
      for (int e = 0; e < nsteps; ++e, lim -= kBN) {
        int cur_lim = (e < ngroups) ? lim : (e == diag_step ? min(tile_lim, r + 1) : tile_lim);
        if (paged_item && e < ngroups) {
          cur_lim = pg_lim;
          if (e + 1 < ngroups) pg_lim = p.tile_rows[pg_idx[e + 1]];
        }
        mbar_wait(bar(S::bSFull + q), sph, 301);
        sph ^= 1;
        tc_fence_after();
        float s[kBN];
        {
          uint32_t raw0[32], raw1[32], raw2[32], raw3[32];
          tmem_ld32(s_addr + 0, raw0);
          tmem_ld32(s_addr + 32, raw1);
          tmem_ld32(s_addr + 64, raw2);
          tmem_ld32(s_addr + 96, raw3);
          tmem_wait_ld();
#pragma unroll
          for (int c = 0; c < 32; ++c) {
            s[c] = __uint_as_float(raw0[c]); s[32 + c] = __uint_as_float(raw1[c]);
            s[64 + c] = __uint_as_float(raw2[c]); s[96 + c] = __uint_as_float(raw3[c]);
          }
        }
        if (__any_sync(0xffffffffu, cur_lim < kBN)) {
#pragma unroll
          for (int c = 0; c < kBN; ++c) s[c] = (c < cur_lim) ? s[c] : -INFINITY;
        }
        // row max: four independent chains of 3-input max
        auto max32 = [&](int c0_) {
          float a0 = s[c0_], a1 = s[c0_ + 1], a2 = s[c0_ + 2], a3 = s[c0_ + 3];
#pragma unroll
          for (int c = 4; c < 32; c += 4) {
            a0 = fmaxf(a0, s[c0_ + c]); a1 = fmaxf(a1, s[c0_ + c + 1]);
            a2 = fmaxf(a2, s[c0_ + c + 2]); a3 = fmaxf(a3, s[c0_ + c + 3]);
          }
          return fmaxf(fmaxf(a0, a1), fmaxf(a2, a3));
        };
        constexpr float kThr = kF8 ? kRescaleThresholdF8 : kRescaleThreshold;
        float2 sum_a, sum_b;
        // exponentials of 32 columns -> packed P in pk (bf16: 16 words, e4m3: 8 words, stored as 2^6 P)
        auto exp_chunk = [&](int c, uint32_t* pk, float neg_m) {
          const float2 sl2 = make_float2(sl, sl), nm2 = make_float2(neg_m, neg_m);
          if constexpr (!kF8) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
              const float2 x = fma2(make_float2(s[c * 32 + 2 * i], s[c * 32 + 2 * i + 1]), sl2, nm2);
              const float2 pr = make_float2(ex2(x.x), ex2(x.y));
              if (i & 1) sum_b = add2(sum_b, pr); else sum_a = add2(sum_a, pr);
              pk[i] = pack_bf16x2(pr.x, pr.y);
            }
          } else {
            const float2 sh2 = make_float2(kP8Shift, kP8Shift), z2 = make_float2(0.f, 0.f);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const float2 xa = fma2(make_float2(s[c * 32 + 4 * i], s[c * 32 + 4 * i + 1]), sl2, nm2);
              const float2 xb = fma2(make_float2(s[c * 32 + 4 * i + 2], s[c * 32 + 4 * i + 3]), sl2, nm2);
              const float2 pa = make_float2(ex2(xa.x), ex2(xa.y)), pb = make_float2(ex2(xb.x), ex2(xb.y));
              sum_a = add2(sum_a, pa); sum_b = add2(sum_b, pb);
              const float2 qa = fma2(pa, sh2, z2), qb = fma2(pb, sh2, z2);
              pk[i] = pack_e4m3x4(qa.x, qa.y, qb.x, qb.y);
            }
          }
        };
        // P overwrites the first columns of S (bf16: 16 packed columns per 32 keys, e4m3: 8); a finished key range lets
        // its part of P V start
        auto store_chunk = [&](int c, const uint32_t* pk) {
          if constexpr (!kF8) {
            asm volatile(
                "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                ::"r"(s_addr + c * 16), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]), "r"(pk[4]), "r"(pk[5]), "r"(pk[6]),
                  "r"(pk[7]), "r"(pk[8]), "r"(pk[9]), "r"(pk[10]), "r"(pk[11]), "r"(pk[12]), "r"(pk[13]), "r"(pk[14]),
                  "r"(pk[15]) : "memory");
          } else {
            asm volatile(
                "tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                ::"r"(s_addr + c * 8), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]), "r"(pk[4]), "r"(pk[5]), "r"(pk[6]),
                  "r"(pk[7]) : "memory");
          }
          if ((c + 1) % (4 / kPvParts) == 0 && c != kBN / 32 - 1) {
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(bar(S::bPFull + ((c + 1) / (4 / kPvParts) - 1) * kNQ + q));
          }
        };
        {
          const float mx = fmaxf(fmaxf(max32(0), max32(32)), fmaxf(max32(64), max32(96)));
          const float m_new = fmaxf(m, mx);
          const bool need = (m_new - m) * sl > kThr;   // (-inf) - (-inf) = NaN -> false
          if (__any_sync(0xffffffffu, need)) {
            const float alpha = need ? ex2((m - m_new) * sl) : 1.f;
            l *= alpha;
            if (need) m = m_new;
            if (e > 0) {
              // O of this tile must hold every P*V issued so far before it is rescaled
              mbar_wait(bar(S::bODone + q), (pv_cnt - 1) & 1, 302);
              tc_fence_after();
#pragma unroll
              for (int c = 0; c < HD / 32; ++c) {
                uint32_t o[32];
                tmem_ld32(o_addr + c * 32, o);
                tmem_wait_ld();
#pragma unroll
                for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                tmem_st32(o_addr + c * 32, o);
              }
            }
          }
        }
        const float neg_m = (m == -INFINITY) ? 0.f : -m * sl;
        sum_a = make_float2(0.f, 0.f); sum_b = make_float2(0.f, 0.f);
#pragma unroll
        for (int c = 0; c < kBN / 32; ++c) {
          uint32_t pk[kF8 ? 8 : 16];
          exp_chunk(c, pk, neg_m);
          store_chunk(c, pk);
        }
        const float2 sum2 = add2(sum_a, sum_b);
        const float sum0 = sum2.x, sum1 = sum2.y;
        l += sum0 + sum1;
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(bar(S::bPFull + (kPvParts - 1) * kNQ + q));
        ++pv_cnt;
      }
      // ---- epilogue: O / l -> bf16, LSE
      const int64_t grow = (int64_t)row0 + r;
      const bool row_ok = r < rows && grow >= p.row_lo && grow < p.row_hi;
      __nv_bfloat16* orow = p.o + grow * p.o_row_stride + (int64_t)h * HD;
      if (nsteps > 0) {
        mbar_wait(bar(S::bODone + q), (pv_cnt - 1) & 1, 303);
        tc_fence_after();
        float inv = (m > -INFINITY) ? 1.f / l : 0.f;   // a row with no allowed key keeps m = -inf (A13)
        if constexpr (kF8) inv *= f8->v[h] * (1.f / kP8Shift);
#pragma unroll
        for (int c = 0; c < HD / 32; ++c) {
          uint32_t o[32];
          tmem_ld32(o_addr + c * 32, o);
          tmem_wait_ld();
          if (row_ok) {
            uint32_t w[16];
#pragma unroll
            for (int i = 0; i < 16; ++i)
              w[i] = pack_bf16x2(__uint_as_float(o[2 * i]) * inv, __uint_as_float(o[2 * i + 1]) * inv);
            store_o_row<32>(orow + c * 32, w, p.o_vec32 != 0);
          }
        }
        tc_fence_before();
      } else if (row_ok) {
#pragma unroll
        for (int i = 0; i < HD / 8; ++i) *reinterpret_cast<uint4*>(orow + i * 8) = make_uint4(0, 0, 0, 0);
      }
      if (row_ok && p.lse != nullptr)
        p.lse[(int64_t)h * p.n_tokens + grow] = (m > -INFINITY) ? (m * sl + log2f(l)) * 0.6931471805599453f : -INFINITY;
    }
    }
  } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsOther));   // (no such warp today: all 16 have a role)
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, kTmemCols);
}

template <int HD>
__global__ void __launch_bounds__(kNumThreads, 1)
sift_attention_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                      const __grid_constant__ CUtensorMap tm_v, const __grid_constant__ CUtensorMap tm_kg,
                      const __grid_constant__ CUtensorMap tm_vg, const AttnParams p) {
  sift_attention_body<HD, 2>(tm_q, tm_k, tm_v, tm_kg, tm_vg, p, nullptr);
}

// e4m3 Q/K/V (head_dim 128): the same body with kind::f8f6f4 MMAs, e4m3 P and per-head scales
__global__ void __launch_bounds__(kNumThreads, 1)
sift_attention_f8_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                         const __grid_constant__ CUtensorMap tm_v, const __grid_constant__ CUtensorMap tm_kg,
                         const __grid_constant__ CUtensorMap tm_vg, const AttnParams p, const __grid_constant__ F8Scales f8) {
  sift_attention_body<128, 1>(tm_q, tm_k, tm_v, tm_kg, tm_vg, p, &f8);
}


// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
// Work counters of the dense comparator: every call takes the next pair of a ring and clears it on its own stream
// before the launch, so dense calls in flight on different streams never share a counter (the sparse call keeps its
// counters inside the caller's metadata buffer, one pair per layer).
constexpr int kDenseCounterRing = 1024;
__device__ int32_t g_dense_counters[kDenseCounterRing][2];
static std::atomic<uint32_t> g_dense_ticket{0};

static int check_tensor(const void* ptr, int64_t stride, const char* name, int elem_bytes = 2) {
  if (!ptr) return set_error(SIFT_ERR_INVALID_ARG, "%s is NULL", name);
  if (((uintptr_t)ptr & 15) != 0 || (stride * elem_bytes) % 16 != 0)
    return set_error(SIFT_ERR_INVALID_ARG, "%s base / row stride not 16-byte aligned", name);
  return SIFT_OK;
}

template <int HD, int EB = 2>
static int launch_attention(AttnParams& p, const void* Q, const void* K, const void* V, int64_t qs, int64_t ks, int64_t vs,
                            cudaStream_t st, const F8Scales* f8 = nullptr) {
  CUtensorMap tq, tk, tv, tkg, tvg;
  int rc;
  const int64_t n = p.n_tokens;
  if ((rc = make_tensor_map_2d(&tq, Q, n, (int64_t)p.n_q_heads * HD, qs, kBM, EB))) return rc;
  if ((rc = make_tensor_map_2d(&tk, K, n, (int64_t)p.n_kv_heads * HD, ks, kBN, EB))) return rc;
  if ((rc = make_tensor_map_2d(&tv, V, n, (int64_t)p.n_kv_heads * HD, vs, kBN, EB))) return rc;
  if ((rc = make_tensor_map_2d(&tkg, K, n, (int64_t)p.n_kv_heads * HD, ks, 1, EB))) return rc;
  if ((rc = make_tensor_map_2d(&tvg, V, n, (int64_t)p.n_kv_heads * HD, vs, 1, EB))) return rc;
  int num_sms = 0;
  if ((rc = device_sm_count(&num_sms))) return rc;
  const void* fn = EB == 1 ? reinterpret_cast<const void*>(&sift_attention_f8_kernel)
                           : reinterpret_cast<const void*>(&sift_attention_kernel<HD>);
  if ((rc = ensure_dynamic_smem(fn, Smem<HD, EB>::kBytes, EB == 1 ? kSmemSlotAttnF8 : (HD == 128 ? kSmemSlotAttn128 : kSmemSlotAttn64))))
    return rc;
  const int grid = p.n_items < num_sms ? (p.n_items > 0 ? p.n_items : 1) : num_sms;
  cudaGetLastError();
  if constexpr (EB == 1) sift_attention_f8_kernel<<<grid, kNumThreads, Smem<HD, EB>::kBytes, st>>>(tq, tk, tv, tkg, tvg, p, *f8);
  else sift_attention_kernel<HD><<<grid, kNumThreads, Smem<HD>::kBytes, st>>>(tq, tk, tv, tkg, tvg, p);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return set_error(SIFT_ERR_CUDA, "attention launch: %s", cudaGetErrorString(e));
  count_launch(1);
  return SIFT_OK;
}

}  // namespace sift

using namespace sift;

// arguments common to the bf16 and the e4m3 entry: metadata pointers of the layer, output, scale
static int sparse_params(const sift_shape* shape, int32_t layer, const void* metadata, void* O, int64_t o_row_stride, float* lse,
                         float softmax_scale, AttnParams* pp) {
  sift_md_layout lay;
  int rc = compute_layout(shape, &lay);
  if (rc) return rc;
  if (layer < 0 || layer >= shape->n_layers) return set_error(SIFT_ERR_INVALID_ARG, "layer %d out of range", layer);
  if (!metadata) return set_error(SIFT_ERR_INVALID_ARG, "metadata is NULL");
  if ((rc = check_tensor(O, o_row_stride, "O"))) return rc;
  const int Hq = shape->n_q_heads, D = shape->n_docs, HD = shape->head_dim;
  if (o_row_stride < (int64_t)Hq * HD) return set_error(SIFT_ERR_INVALID_ARG, "row stride smaller than heads*head_dim");
  const char* b = static_cast<const char*>(metadata);
  auto at = [&](size_t off) { return reinterpret_cast<const int32_t*>(b + off); };
  AttnParams& p = *pp;
  memset(&p, 0, sizeof(p));
  const int64_t lh0 = (int64_t)layer * Hq;
  p.tile_seg = at(lay.tile_seg); p.tile_row0 = at(lay.tile_row0); p.tile_rows = at(lay.tile_rows);
  p.mblock_tile0 = at(lay.mblock_tile0);
  p.seg_info = at(lay.seg_info);
  p.cross_ptr = at(lay.cross_ptr) + lh0 * (D + 1);
  p.cross_idx = at(lay.cross_idx) + lh0 * lay.cross_cap;
  p.local_cnt = at(lay.local_cnt) + lh0 * lay.n_tiles;
  p.local_ptr = at(lay.local_ptr) + lh0 * (lay.n_tiles + 1);
  p.local_idx = at(lay.local_idx) + lh0 * lay.local_cap;
  p.sched = at(lay.sched) + (int64_t)layer * lay.n_items;
  p.counters = const_cast<int32_t*>(at(lay.counters)) + layer * 2;
  p.n_items = lay.n_items; p.n_docs = D; p.n_tiles = lay.n_tiles; p.cross_cap = lay.cross_cap;
  p.local_cap = lay.local_cap; p.n_mblocks = lay.n_mblocks;
  p.dense = 0;
  p.n_tokens = lay.n_tokens;
  p.n_q_heads = Hq; p.n_kv_heads = shape->n_kv_heads; p.tile = shape->tile;
  p.paged = (shape->cross_gran != 1);
  p.row_lo = 0; p.row_hi = lay.n_tokens; p.ranged = 0;
  p.o = static_cast<__nv_bfloat16*>(O); p.o_row_stride = o_row_stride; p.lse = lse;
  p.o_vec32 = (((uintptr_t)O & 31) == 0 && (o_row_stride * 2) % 32 == 0);
  const float sc = softmax_scale > 0.f ? softmax_scale : 1.0f / sqrtf((float)HD);
  p.scale_log2 = sc * 1.4426950408889634f;
  return SIFT_OK;
}

extern "C" int sift_prefill_attention(const sift_shape* shape, int32_t layer, const void* Q, const void* K, const void* V,
                                      int64_t q_row_stride, int64_t k_row_stride, int64_t v_row_stride,
                                      const void* metadata, void* O, int64_t o_row_stride, float* lse,
                                      float softmax_scale, void* stream) {
  AttnParams p;
  int rc = sparse_params(shape, layer, metadata, O, o_row_stride, lse, softmax_scale, &p);
  if (rc) return rc;
  if ((rc = check_tensor(Q, q_row_stride, "Q")) || (rc = check_tensor(K, k_row_stride, "K")) ||
      (rc = check_tensor(V, v_row_stride, "V")))
    return rc;
  const int Hq = shape->n_q_heads, HD = shape->head_dim;
  if (q_row_stride < (int64_t)Hq * HD || k_row_stride < (int64_t)shape->n_kv_heads * HD ||
      v_row_stride < (int64_t)shape->n_kv_heads * HD)
    return set_error(SIFT_ERR_INVALID_ARG, "row stride smaller than heads*head_dim");
  if (HD == 128) return launch_attention<128>(p, Q, K, V, q_row_stride, k_row_stride, v_row_stride, (cudaStream_t)stream);
  return launch_attention<64>(p, Q, K, V, q_row_stride, k_row_stride, v_row_stride, (cudaStream_t)stream);
}

extern "C" int sift_prefill_attention_rows(const sift_shape* shape, int32_t layer, int32_t row_begin, int32_t row_end,
                                           const void* Q, const void* K, const void* V, int64_t q_row_stride,
                                           int64_t k_row_stride, int64_t v_row_stride, const void* metadata, void* O,
                                           int64_t o_row_stride, float* lse, float softmax_scale, void* stream) {
  AttnParams p;
  int rc = sparse_params(shape, layer, metadata, O, o_row_stride, lse, softmax_scale, &p);
  if (rc) return rc;
  if (row_begin < 0 || row_end > p.n_tokens || row_begin > row_end)
    return set_error(SIFT_ERR_INVALID_ARG, "row range [%d, %d) not inside [0, %d)", row_begin, row_end, p.n_tokens);
  if ((rc = check_tensor(Q, q_row_stride, "Q")) || (rc = check_tensor(K, k_row_stride, "K")) ||
      (rc = check_tensor(V, v_row_stride, "V")))
    return rc;
  const int Hq = shape->n_q_heads, HD = shape->head_dim;
  if (q_row_stride < (int64_t)Hq * HD || k_row_stride < (int64_t)shape->n_kv_heads * HD ||
      v_row_stride < (int64_t)shape->n_kv_heads * HD)
    return set_error(SIFT_ERR_INVALID_ARG, "row stride smaller than heads*head_dim");
  if (row_begin == row_end) return SIFT_OK;      // nothing to compute, nothing launched
  p.row_lo = row_begin; p.row_hi = row_end;
  p.ranged = !(row_begin == 0 && row_end == p.n_tokens);
  {
    // M-blocks (kNQ tiles of one segment, numbered in token order as compute_layout counts them) that hold a row of
    // the range
    static thread_local DocTable dt;
    build_segments(shape, &dt);
    const int64_t rows_mb = (int64_t)shape->tile * kNQ;
    int64_t mb = 0;
    p.mb_lo = -1; p.mb_hi = 0;
    for (int sg = 0; sg < dt.n_seg; ++sg) {
      const int64_t a = dt.off[sg], b = dt.off[sg + 1], n_mb = (b - a + rows_mb - 1) / rows_mb;
      if (b > row_begin && a < row_end && b > a) {
        const int64_t lo = row_begin > a ? (row_begin - a) / rows_mb : 0;
        const int64_t hi = row_end < b ? (row_end - a + rows_mb - 1) / rows_mb : n_mb;   // first M-block past the range
        if (p.mb_lo < 0) p.mb_lo = (int32_t)(mb + lo);
        p.mb_hi = (int32_t)(mb + hi);
      }
      mb += n_mb;
    }
    if (p.mb_lo < 0) p.mb_lo = 0;
  }
  if (HD == 128) return launch_attention<128>(p, Q, K, V, q_row_stride, k_row_stride, v_row_stride, (cudaStream_t)stream);
  return launch_attention<64>(p, Q, K, V, q_row_stride, k_row_stride, v_row_stride, (cudaStream_t)stream);
}

extern "C" int sift_prefill_attention_fp8(const sift_shape* shape, int32_t layer, const void* Q8, const void* K8, const void* V8,
                                          int64_t q_row_stride, int64_t k_row_stride, int64_t v_row_stride,
                                          const float* q_scale, const float* k_scale, const float* v_scale,
                                          const void* metadata, void* O, int64_t o_row_stride, float* lse,
                                          float softmax_scale, void* stream) {
  AttnParams p;
  int rc = sparse_params(shape, layer, metadata, O, o_row_stride, lse, softmax_scale, &p);
  if (rc) return rc;
  if (shape->head_dim != 128) return set_error(SIFT_ERR_UNSUPPORTED, "e4m3 Q/K/V: head_dim %d (128 supported)", shape->head_dim);
  if ((rc = check_tensor(Q8, q_row_stride, "Q8", 1)) || (rc = check_tensor(K8, k_row_stride, "K8", 1)) ||
      (rc = check_tensor(V8, v_row_stride, "V8", 1)))
    return rc;
  if (!q_scale || !k_scale || !v_scale) return set_error(SIFT_ERR_INVALID_ARG, "scale array is NULL");
  const int Hq = shape->n_q_heads, Hkv = shape->n_kv_heads, HD = 128;
  if (q_row_stride < (int64_t)Hq * HD || k_row_stride < (int64_t)Hkv * HD || v_row_stride < (int64_t)Hkv * HD)
    return set_error(SIFT_ERR_INVALID_ARG, "row stride smaller than heads*head_dim");
  static thread_local F8Scales f8;
  for (int h = 0; h < Hq; ++h) {
    const int g = h / (Hq / Hkv);
    if (!(q_scale[h] > 0.f) || !(k_scale[g] > 0.f) || !(v_scale[g] > 0.f))
      return set_error(SIFT_ERR_INVALID_ARG, "scales must be positive (q-head %d)", h);
    f8.qk_log2[h] = p.scale_log2 * q_scale[h] * k_scale[g];
    f8.v[h] = v_scale[g];
  }
  return launch_attention<128, 1>(p, Q8, K8, V8, q_row_stride, k_row_stride, v_row_stride, (cudaStream_t)stream, &f8);
}

extern "C" int sift_dense_causal_attention(int32_t n_tokens, int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim,
                                           const void* Q, const void* K, const void* V, int64_t q_row_stride,
                                           int64_t k_row_stride, int64_t v_row_stride, void* O, int64_t o_row_stride,
                                           float* lse, float softmax_scale, void* stream) {
  if (n_tokens < 1 || n_tokens > (1 << 20) || n_q_heads < 1 || n_q_heads > 255 || n_kv_heads < 1 || n_q_heads % n_kv_heads)
    return set_error(SIFT_ERR_INVALID_ARG, "bad dimensions");
  if (head_dim != 64 && head_dim != 128) return set_error(SIFT_ERR_UNSUPPORTED, "head_dim %d not in {64,128}", head_dim);
  int rc;
  if ((rc = check_tensor(Q, q_row_stride, "Q")) || (rc = check_tensor(K, k_row_stride, "K")) ||
      (rc = check_tensor(V, v_row_stride, "V")) || (rc = check_tensor(O, o_row_stride, "O")))
    return rc;
  AttnParams p;
  memset(&p, 0, sizeof(p));
  p.dense = 1;
  p.n_tokens = n_tokens; p.n_q_heads = n_q_heads; p.n_kv_heads = n_kv_heads; p.tile = 128;
  p.row_lo = 0; p.row_hi = n_tokens;
  p.n_mblocks = (n_tokens + kBM * kNQ - 1) / (kBM * kNQ);
  p.kv_per_group = sched_kv_heads_per_group(n_tokens, head_dim, n_kv_heads);
  p.n_items = p.n_mblocks * n_q_heads;
  void* cptr = nullptr;
  if (cudaGetSymbolAddress(&cptr, g_dense_counters) != cudaSuccess) return set_error(SIFT_ERR_CUDA, "no device symbol");
  p.counters = static_cast<int32_t*>(cptr) + 2 * (g_dense_ticket.fetch_add(1, std::memory_order_relaxed) % kDenseCounterRing);
  if (cudaMemsetAsync(p.counters, 0, 2 * sizeof(int32_t), (cudaStream_t)stream) != cudaSuccess)
    return set_error(SIFT_ERR_CUDA, "cudaMemsetAsync(dense counters) failed");
  p.o = static_cast<__nv_bfloat16*>(O); p.o_row_stride = o_row_stride; p.lse = lse;
  p.o_vec32 = (((uintptr_t)O & 31) == 0 && (o_row_stride * 2) % 32 == 0);
  const float sc = softmax_scale > 0.f ? softmax_scale : 1.0f / sqrtf((float)head_dim);
  p.scale_log2 = sc * 1.4426950408889634f;
  if (head_dim == 128) return launch_attention<128>(p, Q, K, V, q_row_stride, k_row_stride, v_row_stride, (cudaStream_t)stream);
  return launch_attention<64>(p, Q, K, V, q_row_stride, k_row_stride, v_row_stride, (cudaStream_t)stream);
}
