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
constexpr int kWPT = 4;    // CA words per thread and pass (a pass = 32768 key bits)
constexpr int kTPT = 2;    // tiles per thread and pass
constexpr int kMaxCrossParts = 4;   // CTAs that may share the cross list of one (layer, head) when the grid is small
constexpr int kStageEntries = 4096;   // shared-memory staging of one chunk: up to 50% of its 8192 bits set
constexpr int kSchedThreads = 1024;
constexpr int kCostBuckets = 4096;

struct DecodeParams {
  const uint8_t* la;
  const uint8_t* ca;
  int32_t *tile_base, *tile_seg, *tile_row0, *tile_rows;
  int32_t *cross_ptr, *cross_idx, *local_cnt, *local_ptr, *local_idx;
  int32_t *mblock_tile0, *sched, *counters;
  int32_t n_q_heads, n_kv_heads, n_tiles, cross_cap, local_cap, n_mblocks, n_items, gran;
  int32_t kv_per_group;   // kv heads whose work items are scheduled together (sched_kv_heads_per_group)
  int32_t cross_parts;    // CTAs per (layer, head) for the cross list: 4 when the grid would not fill the GPU, else 1
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

// K independent block-wide exclusive scans sharing one pair of barriers.  in[k] of thread t is element (k, t);
// out[k] = sum of in[k'][*] for k' < k  +  sum of in[k][t'] for t' < t  (i.e. the exclusive prefix in the order
// element index = k * THREADS + t).  Returns the total over all K * THREADS elements.  ws: [K][THREADS/32] ints;
// callers alternate between two buffers so that no trailing barrier is needed.
template <int K>
__device__ __forceinline__ int batched_exclusive_scan(const int (&in)[K], int (&out)[K], int* ws, int* chunk_start = nullptr,
                                                      int* chunk_total = nullptr) {
  constexpr int NW = kDecodeThreads / 32;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc[K];
#pragma unroll
  for (int k = 0; k < K; ++k) inc[k] = in[k];
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
    for (int k = 0; k < K; ++k) {
      const int n = __shfl_up_sync(0xffffffffu, inc[k], o);
      if (lane >= o) inc[k] += n;
    }
  }
  if (lane == 31) {
#pragma unroll
    for (int k = 0; k < K; ++k) ws[k * NW + wid] = inc[k];
  }
  __syncthreads();
  int carry = 0;
#pragma unroll
  for (int k = 0; k < K; ++k) {
    int before = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const int v = ws[k * NW + w];
      before += (w < wid) ? v : 0;
      tot += v;
    }
    out[k] = carry + before + inc[k] - in[k];
    if (chunk_start) { chunk_start[k] = carry; chunk_total[k] = tot; }
    carry += tot;
  }
  return carry;
}

// LA row i of a document: bits n0 .. n0+i of the MSB-first vector, n0 = i(i+1)/2, read a byte at a time
__device__ __forceinline__ int la_row_count(const uint8_t* __restrict__ v, int i) {
  int b = i * (i + 1) / 2;
  const int end = b + i + 1;
  int cnt = 0;
  while (b < end) {
    const int lo = b & 7, nb = min(8 - lo, end - b);
    const uint32_t x = ((uint32_t)__ldg(v + (b >> 3)) << lo) & 0xffu;   // first wanted bit at bit 7
    cnt += __popc(x >> (8 - nb));
    b += nb;
  }
  return cnt;
}
// writes base + j for every set bit (i, j), ascending j
__device__ __forceinline__ void la_row_fill(const uint8_t* __restrict__ v, int i, int base, int32_t* __restrict__ out) {
  const int n0 = i * (i + 1) / 2;
  int b = n0;
  const int end = b + i + 1;
  while (b < end) {
    const int lo = b & 7, nb = min(8 - lo, end - b);
    uint32_t x = (((uint32_t)__ldg(v + (b >> 3)) << lo) & 0xffu) >> (8 - nb);   // nb bits, first stream bit = bit nb-1
    while (x) {
      const int z = 31 - __clz(x);
      x &= ~(1u << z);
      *out++ = base + (b - n0) + (nb - 1 - z);
    }
    b += nb;
  }
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
  __shared__ int s_stage[kStageEntries];   // compacted entries of one 256-word chunk (denser chunks go straight to global)
  __shared__ int s_bscan[2][(kWPT > kTPT ? kWPT : kTPT) * (kDecodeThreads / 32)];

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
  // blockIdx.z splits a (layer, head): z < kCrossParts = one range of the cross list, z = kCrossParts = the local lists
  // (and, for the first head, the tile tables).  Shortens the latency chain of a CTA (a single layer is latency-bound).
  const int kCrossParts = p.cross_parts;
  const bool do_cross = ((int)blockIdx.z < kCrossParts);
  const bool writer = (h == 0 && l == 0 && !do_cross);
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
  // A pass covers kWPT * 256 words: every thread issues its kWPT word loads back to back (one DRAM round trip per
  // pass instead of one per 256 words), counts, and ONE batched block scan (kWPT independent prefix sums sharing the
  // same two barriers) turns the counts into offsets.
  int32_t* cross_ptr = p.cross_ptr + lh * (D + 1);
  int32_t* cross_idx = p.cross_idx + lh * p.cross_cap;
  // masked stream-order bits of word v of the head's virtual word sequence, the global coordinate of its bit 0 and
  // the document it closes (or -1)
  auto load_word = [&](int v, int& key0, int& closes) -> uint32_t {
    const int d = upper_seg(s_wstart, D, v);
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
    // global coordinate of stream bit 0 of this word: key row (G == 1) or tile id (G == tile; a page is a tile)
    key0 = (G == 1 ? dt.off[d] : s_tile_base[d]) + wi * 32 - lead;
    closes = (v + 1 == s_wstart[d + 1]) ? d : -1;
    return x & m;
  };
  // The word sequence of a head is cut into kCrossParts ranges, one CTA each (grid z): a CTA first popcounts the words
  // before its range (the bit vectors of a head are a few KB: re-reading them costs less than waiting for a prefix
  // from another CTA), which gives it the list offset of its first entry.
  const int all_words = s_wstart[D];
  const int per = (all_words + kCrossParts - 1) / kCrossParts;
  const int w_lo = do_cross ? min(all_words, (int)blockIdx.z * per) : 0;
  const int total_words = do_cross ? min(all_words, w_lo + per) : 0;      // end of this CTA's range
  int running = 0;
  if (do_cross) {
    int before = 0, k0, cl;
    for (int v = tid; v < w_lo; v += kDecodeThreads) before += __popc(load_word(v, k0, cl));
    int tot;
    block_exclusive_scan<kDecodeThreads>(before, s_scan, tot);
    running = tot;
    if (blockIdx.z == 0 && tid == 0) cross_ptr[0] = 0;
  }
  int scan_no = 0;   // the two scan buffers alternate over ALL scans of the kernel (no trailing barrier needed)
  for (int base = w_lo; base < total_words; base += kWPT * kDecodeThreads) {
    uint32_t bits[kWPT];
    int key0[kWPT], cnt[kWPT], dd[kWPT];
#pragma unroll
    for (int k = 0; k < kWPT; ++k) {
      const int v = base + k * kDecodeThreads + tid;
      bits[k] = 0; key0[k] = 0; dd[k] = -1;
      if (v < total_words) bits[k] = load_word(v, key0[k], dd[k]);
    }
#pragma unroll
    for (int k = 0; k < kWPT; ++k) cnt[k] = __popc(bits[k]);                     // pass 1: count
    int ex[kWPT], cs[kWPT], ct[kWPT];
    const int pass_total = batched_exclusive_scan<kWPT>(cnt, ex, s_bscan[scan_no++ & 1], cs, ct);   // offsets
    // pass 2: fill, global coordinates.  Each 256-word chunk is compacted into shared memory by a thread-per-word
    // ffs loop and then copied out with coalesced stores: scattering the ffs loop straight to global memory cost 32
    // sectors per store instruction, a warp-cooperative bit-per-lane fill cost ~1500 instructions per warp and made
    // the kernel issue-bound (65% issue-active, 56 us for the 32 layers of C5).
#pragma unroll
    for (int k = 0; k < kWPT; ++k) {
      if (dd[k] >= 0) cross_ptr[dd[k] + 1] = running + ex[k] + cnt[k];
      if (ct[k] == 0) continue;                        // block-uniform
      int32_t* dst = cross_idx + running + cs[k];
      int o = ex[k] - cs[k];
      uint32_t bk = bits[k];
      if (ct[k] <= kStageEntries) {                    // block-uniform
        while (bk) {
          const int sb = __ffs(bk) - 1;
          bk &= bk - 1;
          s_stage[o++] = key0[k] + sb;
        }
        __syncthreads();
        for (int i = tid; i < ct[k]; i += kDecodeThreads) dst[i] = s_stage[i];
        __syncthreads();
      } else {
        while (bk) {
          const int sb = __ffs(bk) - 1;
          bk &= bk - 1;
          dst[o++] = key0[k] + sb;
        }
      }
    }
    running += pass_total;
  }
  // entries in [total, roundup128(total)) must be valid rows: the attention kernel gathers whole groups
  if (do_cross) {
    if (blockIdx.z == kCrossParts - 1)
      for (int i = running + tid; i < ((running + 127) & ~127); i += kDecodeThreads) cross_idx[i] = 0;
    return;
  }

  // ---- local lists: LA row popcounts, offsets, fill -------------------------------------------------
  int32_t* local_cnt = p.local_cnt + lh * NT;
  int32_t* local_ptr = p.local_ptr + lh * (NT + 1);
  int32_t* local_idx = p.local_idx + lh * p.local_cap;
  running = 0;
  for (int base = 0; base < NT; base += kTPT * kDecodeThreads) {
    int cnt[kTPT], dd[kTPT], ii[kTPT];
    const uint8_t* lv[kTPT];
#pragma unroll
    for (int k = 0; k < kTPT; ++k) {
      const int t = base + k * kDecodeThreads + tid;
      cnt[k] = 0; dd[k] = 0; ii[k] = 0; lv[k] = nullptr;
      if (t < NT) {
        const int d = upper_seg(s_tile_base, D + 1, t);
        const int i = t - s_tile_base[d];
        dd[k] = d; ii[k] = i;
        const int seg_len = (d < D) ? dt.off[d + 1] - dt.off[d] : dt.query_len;
        if (writer) {
          p.tile_seg[t] = d;
          p.tile_row0[t] = dt.off[d] + i * T;
          p.tile_rows[t] = min(T, seg_len - i * T);
        }
        if (d == D) {
          cnt[k] = t + 1;                                             // query M-block: all causal N-blocks (L243)
        } else {
          const int pd = s_tile_base[d + 1] - s_tile_base[d];
          const int nbytes = (pd * (pd + 1) / 2 + 7) >> 3;
          lv[k] = p.la + dt.la_off[d] + lh * nbytes;
          cnt[k] = la_row_count(lv[k], i);
        }
      }
    }
    int ex[kTPT];
    const int pass_total = batched_exclusive_scan<kTPT>(cnt, ex, s_bscan[scan_no++ & 1]);
#pragma unroll
    for (int k = 0; k < kTPT; ++k) {
      const int t = base + k * kDecodeThreads + tid;
      if (t < NT) {
        int w0 = running + ex[k];
        local_cnt[t] = cnt[k];
        local_ptr[t] = w0;
        if (dd[k] == D) {
          for (int j = 0; j <= t; ++j) local_idx[w0 + j] = j;
        } else {
          la_row_fill(lv[k], ii[k], s_tile_base[dd[k]], local_idx + w0);
        }
      }
    }
    running += pass_total;
  }
  if (tid == 0) local_ptr[NT] = running;
}

// Work items (head, M-block) of one layer sorted by (kv-head group, descending cost) (counting sort): the persistent
// attention grid pulls them through an atomic counter.
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
      // steps of a document tile: groups of 128 gathered rows (G == 1) or one page per step (G == tile), plus local tiles
      if (seg < D) c += (p.gran == 1 ? (p.cross_ptr[lh * (D + 1) + seg] + 127) / 128 : p.cross_ptr[lh * (D + 1) + seg]) + p.local_cnt[lh * NT + t];
      else c += (p.tile_row0[t] + p.tile_rows[t] + 127) / 128;
    }
    // bucket = processing order: groups of kv heads one after the other (the q-heads of a kv head gather from the same
    // K/V, so the K/V working set of the grid stays L2-sized and K/V are read from HBM about once), longest items
    // first inside a group
    const int groups = (p.n_kv_heads + p.kv_per_group - 1) / p.kv_per_group, bpg = kCostBuckets / groups;
    const int g = h / (p.n_q_heads / p.n_kv_heads) / p.kv_per_group;
    return g * bpg + (bpg - 1 - min(c, bpg - 1));
  };
  // the cost of an item is a chain of dependent global loads: evaluate it once and keep it in registers for the
  // scatter pass (up to kCached items per thread; larger layers recompute)
  constexpr int kCached = 8;
  int ccost[kCached];
#pragma unroll
  for (int k = 0; k < kCached; ++k) {
    const int e = tid + k * kSchedThreads;
    ccost[k] = (e < p.n_items) ? cost_of(e) : 0;
  }
#pragma unroll
  for (int k = 0; k < kCached; ++k)
    if (tid + k * kSchedThreads < p.n_items) atomicAdd(&s_hist[ccost[k]], 1);
  for (int e = tid + kCached * kSchedThreads; e < p.n_items; e += kSchedThreads)
    atomicAdd(&s_hist[cost_of(e)], 1);
  __syncthreads();
  {  // exclusive scan over buckets (bucket 0 = first to be processed)
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
  auto place = [&](int e, int c) {
    const int h = e / NMB, mb = e - h * NMB;
    const int pos = atomicAdd(&s_hist[c], 1);
    sched[pos] = (h << 20) | mb;
  };
#pragma unroll
  for (int k = 0; k < kCached; ++k)
    if (tid + k * kSchedThreads < p.n_items) place(tid + k * kSchedThreads, ccost[k]);
  for (int e = tid + kCached * kSchedThreads; e < p.n_items; e += kSchedThreads) place(e, cost_of(e));
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
  p.n_q_heads = s->n_q_heads; p.n_kv_heads = s->n_kv_heads; p.n_tiles = lay.n_tiles; p.cross_cap = lay.cross_cap; p.local_cap = lay.local_cap;
  p.n_mblocks = lay.n_mblocks; p.n_items = lay.n_items; p.gran = s->cross_gran;
  // few (layer, head) pairs (one layer of an 8B-class model = 32): the call is latency-bound, cut each head's cross list
  // into ranges for separate CTAs; many (a whole stack = 1024): one CTA per list is more efficient (no re-counting)
  int num_sms = 0;
  if (int rc = device_sm_count(&num_sms)) return rc;
  p.cross_parts = ((int64_t)s->n_q_heads * s->n_layers <= num_sms) ? kMaxCrossParts : 1;
  p.kv_per_group = sched_kv_heads_per_group((int64_t)s->doc_offsets[s->n_docs] + s->query_len, s->head_dim, s->n_kv_heads);
  cudaGetLastError();
  sift_decode_lists_kernel<<<dim3(s->n_q_heads, s->n_layers, p.cross_parts + 1), kDecodeThreads, 0, st>>>(dt, p);
  sift_schedule_kernel<<<s->n_layers, kSchedThreads, 0, st>>>(p, s->n_docs, s->n_layers);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return set_error(SIFT_ERR_CUDA, "decode launch: %s", cudaGetErrorString(e));
  count_launch(2);
  return SIFT_OK;
}

}  // namespace sift
