// SIFT metadata decode for sm_100a (sec 5.1): bit vectors -> MD-v1 index lists.
//
// The paper launches one 128-thread CTA per (head, M-block) and replicates the CA entries into every
// M-block's list.  Here one CTA handles a whole (layer, head): the CA entries of a head form ONE ascending
// list of which document d uses the prefix [0, cross_ptr[d]), so the CA bits are scanned
// once per head instead of once per M-block.  Pass 1 (count) = popc of masked 32-bit words, offsets = block
// exclusive scan (warp shuffles), pass 2 (fill) = ffs-compaction of the same registers; the two passes of
// the paper are fused per 8192-bit chunk so the bit vectors are read from HBM once.
//
// Bit vectors are byte-aligned per (layer, head, doc), not word-aligned: the kernel reads the
// aligned 32-bit words that cover a vector and masks the lead/tail bits.
#include "sift_common.h"

namespace sift {

constexpr int kDecodeThreads = 256;
constexpr int kSchedThreads = 1024;
constexpr int kCostBuckets = 4096;

struct DecodeParams {
  const uint8_t* la;
  const uint8_t* ca;
  int32_t *tile_base, *tile_seg, *tile_row0, *tile_rows;
  int32_t *cross_ptr, *cross_idx, *local_cnt, *local_ptr, *local_idx;
  int32_t *mblock_tile0, *sched, *counters;
  int32_t n_q_heads, n_tiles, cross_cap, local_cap, n_mblocks, n_items;
};

// exclusive scan over the block; returns the exclusive prefix of v and (via total) the block sum
template <int THREADS>
__device__ __forceinline__ int block_exclusive_scan(int v, int* warp_sums /*[THREADS/32+1]*/, int& total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int n = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += n;
  }
  if (lane == 31) warp_sums[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    int s = (lane < THREADS / 32) ? warp_sums[lane] : 0;
    int si = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int n = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= o) si += n;
    }
    if (lane < THREADS / 32) warp_sums[lane] = si - s;
    if (lane == 31) warp_sums[THREADS / 32] = si;
  }
  __syncthreads();
  int res = warp_sums[wid] + inc - v;
  total = warp_sums[THREADS / 32];
  __syncthreads();
  return res;
}

// largest d in [0, n) with tab[d] <= x  (tab ascending, tab[0] <= x)
__device__ __forceinline__ int upper_seg(const int* tab, int n, int x) {
  int lo = 0, hi = n - 1;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (tab[mid] <= x) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// bit n of an MSB-first packed vector
__device__ __forceinline__ int msb_bit(const uint8_t* __restrict__ v, int n) {
  return (__ldg(v + (n >> 3)) >> (7 - (n & 7))) & 1;
}

__global__ void __launch_bounds__(kDecodeThreads)
sift_decode_lists_kernel(const __grid_constant__ DocTable dt, const DecodeParams p) {
  __shared__ int s_tile_base[SIFT_MAX_DOCS + 2];
  __shared__ int s_wstart[SIFT_MAX_DOCS + 2];
  __shared__ int s_mb_base[SIFT_MAX_DOCS + 2];
  __shared__ int s_scan[kDecodeThreads / 32 + 1];

  const int tid = threadIdx.x;
  const int h = blockIdx.x, l = blockIdx.y;
  const int D = dt.n_docs, T = dt.tile, G = dt.gran;
  const int64_t lh = (int64_t)l * p.n_q_heads + h;
  constexpr int NQ = SIFT_Q_TILES_PER_ITEM;

  // ---- step 0: per-segment tables (tiles, covering words of this head's CA vectors, M-blocks) ----------
  {
    int carry_t = 0, carry_w = 0, carry_m = 0;
    for (int d0 = 0; d0 <= D; d0 += kDecodeThreads) {
      const int d = d0 + tid;
      int pd = 0, nw = 0;
      if (d < D) {
        const int len = dt.off[d + 1] - dt.off[d];
        pd = (len + T - 1) / T;
        const int nbits = (len + G - 1) / G;
        const int64_t a = dt.ca_off[d] + lh * ((nbits + 7) >> 3);
        const int lead = (int)((reinterpret_cast<uintptr_t>(p.ca) + (uint64_t)a) & 3);
        nw = (lead * 8 + nbits + 31) >> 5;
      } else if (d == D) {
        pd = (dt.query_len + T - 1) / T;
      }
      int tot;
      int et = block_exclusive_scan<kDecodeThreads>(pd, s_scan, tot);
      if (d <= D) s_tile_base[d] = carry_t + et;
      carry_t += tot;
      int ew = block_exclusive_scan<kDecodeThreads>(nw, s_scan, tot);
      if (d <= D) s_wstart[d] = carry_w + ew;
      carry_w += tot;
      int em = block_exclusive_scan<kDecodeThreads>((pd + NQ - 1) / NQ, s_scan, tot);
      if (d <= D) s_mb_base[d] = carry_m + em;
      carry_m += tot;
    }
    if (tid == 0) {
      s_tile_base[D + 1] = carry_t;
      s_wstart[D + 1] = carry_w;   // s_wstart[D] == carry_w as well (the query has no CA words)
      s_mb_base[D + 1] = carry_m;
    }
    __syncthreads();
  }
  const int NT = s_tile_base[D + 1];
  const bool writer = (h == 0 && l == 0);
  if (writer) {
    for (int d = tid; d <= D + 1; d += kDecodeThreads) p.tile_base[d] = s_tile_base[d];
    for (int d = tid; d <= D; d += kDecodeThreads) {
      const int pd = s_tile_base[d + 1] - s_tile_base[d];
      const int nb = (pd + NQ - 1) / NQ;
      for (int k = 0; k < nb; ++k) p.mblock_tile0[s_mb_base[d] + k] = s_tile_base[d] + k * NQ;
    }
    if (tid == 0) p.mblock_tile0[s_mb_base[D + 1]] = NT;
  }

  // ---- cross list: CA bits of all documents, one virtual word sequence ---------------------------------
  int32_t* cross_ptr = p.cross_ptr + lh * (D + 1);
  int32_t* cross_idx = p.cross_idx + lh * p.cross_cap;
  const int total_words = s_wstart[D];
  int running = 0;
  if (tid == 0) cross_ptr[0] = 0;
  for (int v0 = 0; v0 < total_words; v0 += kDecodeThreads) {
    const int v = v0 + tid;
    uint32_t bits = 0;
    int key0 = 0, d = 0;
    bool last_word = false;
    if (v < total_words) {
      d = upper_seg(s_wstart, D, v);
      const int wi = v - s_wstart[d];
      const int len = dt.off[d + 1] - dt.off[d];
      const int nbits = (len + G - 1) / G;
      const uintptr_t a = reinterpret_cast<uintptr_t>(p.ca) + (uint64_t)(dt.ca_off[d] + lh * ((nbits + 7) >> 3));
      const int lead = (int)(a & 3) * 8;
      const uint32_t w = __ldg(reinterpret_cast<const uint32_t*>(a & ~(uintptr_t)3) + wi);
      // stream bit s (MSB-first within each byte, bytes ascending) -> bit s of x
      const uint32_t x = __brev(__byte_perm(w, 0, 0x0123));
      const int lo = max(0, lead - wi * 32);
      const int hi = min(32, lead + nbits - wi * 32);
      uint32_t m = (hi >= 32) ? 0xffffffffu : ((1u << hi) - 1u);
      m &= ~((lo >= 32) ? 0xffffffffu : ((1u << lo) - 1u));
      bits = x & m;
      key0 = dt.off[d] + wi * 32 - lead;   // G == 1: global key row of stream bit 0 of this word
      last_word = (v + 1 == s_wstart[d + 1]);
    }
    const int c = __popc(bits);                                   // pass 1: count
    int tot;
    int w0 = running + block_exclusive_scan<kDecodeThreads>(c, s_scan, tot);   // offsets
    running += tot;
    if (last_word) cross_ptr[d + 1] = w0 + c;
    while (bits) {                                                // pass 2: fill, global coordinates
      const int s = __ffs(bits) - 1;
      bits &= bits - 1;
      cross_idx[w0++] = key0 + s;
    }
  }
  // entries in [total, roundup128(total)) must be valid rows: the attention kernel gathers whole groups
  for (int i = running + tid; i < ((running + 127) & ~127); i += kDecodeThreads) cross_idx[i] = 0;

  // ---- local lists: LA row popcounts, offsets, fill -------------------------------------------------
  int32_t* local_cnt = p.local_cnt + lh * NT;
  int32_t* local_ptr = p.local_ptr + lh * (NT + 1);
  int32_t* local_idx = p.local_idx + lh * p.local_cap;
  running = 0;
  for (int t0 = 0; t0 < NT; t0 += kDecodeThreads) {
    const int t = t0 + tid;
    int cnt = 0, d = 0, i = 0;
    const uint8_t* lv = nullptr;
    if (t < NT) {
      d = upper_seg(s_tile_base, D + 1, t);
      i = t - s_tile_base[d];
      const int seg_len = (d < D) ? dt.off[d + 1] - dt.off[d] : dt.query_len;
      if (writer) {
        p.tile_seg[t] = d;
        p.tile_row0[t] = dt.off[d] + i * T;
        p.tile_rows[t] = min(T, seg_len - i * T);
      }
      if (d == D) {
        cnt = t + 1;                                              // query M-block: all causal N-blocks (L243)
      } else {
        const int pd = s_tile_base[d + 1] - s_tile_base[d];
        const int nbytes = (pd * (pd + 1) / 2 + 7) >> 3;
        lv = p.la + dt.la_off[d] + lh * nbytes;
        const int n0 = i * (i + 1) / 2;
        for (int j = 0; j <= i; ++j) cnt += msb_bit(lv, n0 + j);
      }
    }
    int tot;
    int w0 = running + block_exclusive_scan<kDecodeThreads>(cnt, s_scan, tot);
    running += tot;
    if (t < NT) {
      local_cnt[t] = cnt;
      local_ptr[t] = w0;
      if (d == D) {
        for (int j = 0; j <= t; ++j) local_idx[w0 + j] = j;
      } else {
        const int n0 = i * (i + 1) / 2;
        const int base = s_tile_base[d];
        for (int j = 0; j <= i; ++j)
          if (msb_bit(lv, n0 + j)) local_idx[w0++] = base + j;
      }
    }
  }
  if (tid == 0) local_ptr[NT] = running;
}

// Work items (head, M-block) of one layer sorted by descending cost (counting sort): the persistent
// attention grid pulls them through an atomic counter, longest first.
__global__ void __launch_bounds__(kSchedThreads)
sift_schedule_kernel(const DecodeParams p, int n_docs, int n_layers_unused) {
  __shared__ int s_hist[kCostBuckets];
  __shared__ int s_scan[kSchedThreads / 32 + 1];
  constexpr int NQ = SIFT_Q_TILES_PER_ITEM;
  const int l = blockIdx.x, tid = threadIdx.x;
  const int D = n_docs, NT = p.n_tiles, NMB = p.n_mblocks;
  for (int i = tid; i < kCostBuckets; i += kSchedThreads) s_hist[i] = 0;
  __syncthreads();
  auto cost_of = [&](int e) {
    const int h = e / NMB, mb = e - h * NMB;
    const int64_t lh = (int64_t)l * p.n_q_heads + h;
    const int t0 = p.mblock_tile0[mb], t1 = min(p.mblock_tile0[mb + 1], t0 + NQ);
    const int seg = p.tile_seg[t0];
    int c = 0;
    for (int t = t0; t < t1; ++t) {
      if (seg < D) c += (p.cross_ptr[lh * (D + 1) + seg] + 127) / 128 + p.local_cnt[lh * NT + t];
      else c += (p.tile_row0[t] + p.tile_rows[t] + 127) / 128;
    }
    return min(c, kCostBuckets - 1);
  };
  for (int e = tid; e < p.n_items; e += kSchedThreads) atomicAdd(&s_hist[kCostBuckets - 1 - cost_of(e)], 1);
  __syncthreads();
  {  // exclusive scan over buckets (bucket 0 = highest cost)
    constexpr int PER = kCostBuckets / kSchedThreads;
    int loc[PER], sum = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) { loc[k] = s_hist[tid * PER + k]; sum += loc[k]; }
    int tot;
    int ex = block_exclusive_scan<kSchedThreads>(sum, s_scan, tot);
#pragma unroll
    for (int k = 0; k < PER; ++k) { s_hist[tid * PER + k] = ex; ex += loc[k]; }
  }
  __syncthreads();
  int32_t* sched = p.sched + (int64_t)l * p.n_items;
  for (int e = tid; e < p.n_items; e += kSchedThreads) {
    const int h = e / NMB, mb = e - h * NMB;
    const int pos = atomicAdd(&s_hist[kCostBuckets - 1 - cost_of(e)], 1);
    sched[pos] = (h << 20) | mb;
  }
  if (tid < 2) p.counters[l * 2 + tid] = 0;
}

int launch_decode(const sift_shape* s, const sift_md_layout& lay, const DocTable& dt, const uint8_t* la_base,
                  const uint8_t* ca_base, void* md, cudaStream_t st) {
  if (lay.n_mblocks >= (1 << 20)) return set_error(SIFT_ERR_UNSUPPORTED, "too many M-blocks");
  char* b = static_cast<char*>(md);
  DecodeParams p;
  p.la = la_base;
  p.ca = ca_base;
  auto at = [&](size_t off) { return reinterpret_cast<int32_t*>(b + off); };
  p.tile_base = at(lay.tile_base); p.tile_seg = at(lay.tile_seg);
  p.tile_row0 = at(lay.tile_row0); p.tile_rows = at(lay.tile_rows);
  p.cross_ptr = at(lay.cross_ptr); p.cross_idx = at(lay.cross_idx);
  p.local_cnt = at(lay.local_cnt); p.local_ptr = at(lay.local_ptr); p.local_idx = at(lay.local_idx);
  p.mblock_tile0 = at(lay.mblock_tile0); p.sched = at(lay.sched); p.counters = at(lay.counters);
  p.n_q_heads = s->n_q_heads; p.n_tiles = lay.n_tiles; p.cross_cap = lay.cross_cap; p.local_cap = lay.local_cap;
  p.n_mblocks = lay.n_mblocks; p.n_items = lay.n_items;
  cudaGetLastError();
  sift_decode_lists_kernel<<<dim3(s->n_q_heads, s->n_layers), kDecodeThreads, 0, st>>>(dt, p);
  sift_schedule_kernel<<<s->n_layers, kSchedThreads, 0, st>>>(p, s->n_docs, s->n_layers);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return set_error(SIFT_ERR_CUDA, "decode launch: %s", cudaGetErrorString(e));
  count_launch(2);
  return SIFT_OK;
}

}  // namespace sift
