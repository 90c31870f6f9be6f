// SIFT metadata decode for sm_100a (sec 5.1): bit vectors -> MD-v1 index lists, ONE launch.
//
// The paper launches one 128-thread CTA per (head, M-block) and replicates the CA entries into every
// M-block's list.  Here the CA entries of a head form ONE ascending list of which document d uses the prefix
// [0, cross_ptr[d]), so the CA bits are scanned once per head instead of once per M-block.
// Grid (q-head, layer, role): role < cross_parts = one range of the head's cross list, then the local lists, then
// (small grids only) the scheduler keys.  Pass 1 (count) = popc of masked 32-bit words, offsets = batched block scan
// (warp shuffles), pass 2 (fill) = ffs-compaction of the same registers into a warp-private slice of shared memory
// and a coalesced copy; the two passes of the paper are fused so the bit vectors are read from HBM once.
// The tile scheduler (a5) is fused as well: every (layer, head) publishes the sort key of its work items, and the
// CTA that finishes a layer last counting-sorts the layer's items (no second launch).
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
constexpr int kWarpStage = kStageEntries / (kDecodeThreads / 32);   // staging slice of a warp: its 32 words, <= 50% set
constexpr int kCostBuckets = 4096;    // buckets of the scheduler's counting sort (they reuse the staging buffer)
static_assert(kCostBuckets == kStageEntries, "the scheduler's (padded) histogram lives in the staging buffer");
static_assert(kCostBuckets / kDecodeThreads == 16, "histogram padding: one word per 16 buckets");

// "CTAs of this layer that have finished" counters of the fused scheduler: every decode call takes n_layers
// consecutive slots of this ring; the CTA that finishes a layer last sorts the layer's work items and puts the
// slot back to 0, so the ring is all-zero whenever no decode is in flight.
constexpr int kDoneRing = 1 << 16;
__device__ int32_t g_layer_done[kDoneRing];
static std::atomic<uint32_t> g_done_ticket{0};

struct DecodeParams {
  const uint8_t* la;
  const uint8_t* ca;
  int32_t *tile_base, *tile_seg, *tile_row0, *tile_rows;
  int32_t *cross_ptr, *cross_idx, *local_cnt, *local_ptr, *local_idx;
  int32_t *mblock_tile0, *sched, *counters, *sched_key, *seg_info;
  int32_t n_q_heads, n_kv_heads, n_tiles, cross_cap, local_cap, n_mblocks, n_items, gran;
  int32_t kv_per_group;   // kv heads whose work items are scheduled together (sched_kv_heads_per_group)
  int32_t cross_parts;    // CTAs per (layer, head) for the cross list: 4 when the grid would not fill the GPU, else 1
  int32_t tile_shift, gran_shift;   // tile and cross_gran are powers of two (64 | 128; 1 | tile): no integer divisions
  int32_t done_base;      // first slot of this call in g_layer_done
  int32_t fused;          // 1 (small grids): the scheduler runs inside this launch (a key CTA per (layer, head), the
                          // layer's last CTA sorts); 0 (whole stacks): sift_schedule_kernel follows
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
// Predicated probes (no data-dependent branch); top = largest power of two < n (upper_seg_top), so the depth follows the
// number of documents.
__device__ __forceinline__ int upper_seg_top(int n) { return n > 1 ? 1 << (31 - __clz(n - 1)) : 0; }
__device__ __forceinline__ int upper_seg(const int* tab, int n, int x, int top) {
  int lo = 0;
  for (int step = top; step > 0; step >>= 1) {
    const int mid = lo + step;
    const int v = tab[min(mid, n - 1)];
    lo = (mid < n && v <= x) ? mid : lo;
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
sift_decode_kernel(const __grid_constant__ DocTable dt, const DecodeParams p) {
  // tables per segment (documents and queries in token order; index S = totals)
  __shared__ int s_tile_base[kMaxSeg + 1];
  __shared__ int s_wstart[kMaxSeg + 1];
  __shared__ int s_mb_base[kMaxSeg + 1];
  // copies of the kernel-parameter table: a per-lane index into the constant bank is replayed once per distinct
  // address, shared memory is not
  __shared__ int s_off[kMaxSeg + 1];              // first row of the segment; s_off[S] = n_tokens
  __shared__ short s_sdoc[kMaxSeg], s_sfirst[kMaxSeg];   // document index (-1: query), first segment of the prompt
  __shared__ int s_ca_lead[kMaxSeg];              // bit offset of the head's CA vector inside its first covering word
  __shared__ int64_t s_doc64[2 * kMaxSeg];
  int64_t* s_ca_word = s_doc64;                   // index (in 32-bit words from the 4-byte aligned base of p.ca) of that word
  int64_t* s_la_off = s_doc64 + kMaxSeg;
  __shared__ int s_pad[kMaxSeg + 1];              // several prompts: list offset added to the raw bit rank (see below)
  __shared__ int s_scan[kDecodeThreads / 32 + 1];
  __shared__ __align__(16) int s_stage[kStageEntries + kStageEntries / 16];   // warp-private staging slices | per-segment counts | histogram
  __shared__ int s_bscan[2][(kWPT > kTPT ? kWPT : kTPT) * (kDecodeThreads / 32)];

  const int tid = threadIdx.x;
  const int h = blockIdx.x, l = blockIdx.y;
  const int S = dt.n_seg, D = dt.n_docs, T = dt.tile, G = dt.gran;
  const int64_t lh = (int64_t)l * p.n_q_heads + h;
  constexpr int NQ = SIFT_Q_TILES_PER_ITEM;

  // ---- step 0: per-segment tables (tiles, covering words of this head's CA vectors, M-blocks) ----------
  // One warp scans the segments 32 at a time (three running sums through shuffles); the other warps wait at a
  // single barrier.  (The first version ran three block-wide scans per 256 segments in every CTA.)
  const int tsh = p.tile_shift, gsh = p.gran_shift;
  if (tid < 32) {
    int carry_t = 0, carry_w = 0, carry_m = 0;
    for (int d0 = 0; d0 < S; d0 += 32) {
      const int d = d0 + tid;
      int pd = 0, nw = 0;
      if (d < S) {
        const int o0 = dt.off[d], len = dt.off[d + 1] - o0, dc = dt.doc[d];
        pd = (len + T - 1) >> tsh;
        s_off[d] = o0; s_sdoc[d] = (short)dc; s_sfirst[d] = dt.first[d];
        if (dc >= 0) {
          const int nbits = (len + G - 1) >> gsh;
          const uint64_t a = (reinterpret_cast<uintptr_t>(p.ca) & 3) + (uint64_t)(dt.ca_off[dc] + lh * ((nbits + 7) >> 3));
          const int lead = (int)(a & 3);
          nw = (lead * 8 + nbits + 31) >> 5;
          s_ca_lead[d] = lead * 8; s_ca_word[d] = (int64_t)(a >> 2); s_la_off[d] = dt.la_off[dc];
        }
      }
      int it = pd, iw = nw, im = (pd + NQ - 1) / NQ;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int a = __shfl_up_sync(0xffffffffu, it, o), b = __shfl_up_sync(0xffffffffu, iw, o),
                  c = __shfl_up_sync(0xffffffffu, im, o);
        if (tid >= o) { it += a; iw += b; im += c; }
      }
      if (d < S) {
        s_tile_base[d] = carry_t + it - pd;
        s_wstart[d] = carry_w + iw - nw;
        s_mb_base[d] = carry_m + im - (pd + NQ - 1) / NQ;
      }
      carry_t += __shfl_sync(0xffffffffu, it, 31);
      carry_w += __shfl_sync(0xffffffffu, iw, 31);
      carry_m += __shfl_sync(0xffffffffu, im, 31);
    }
    if (tid == 0) {
      s_tile_base[S] = carry_t;
      s_wstart[S] = carry_w;
      s_mb_base[S] = carry_m;
      s_off[S] = dt.off[S];
    }
  }
  __syncthreads();
  const int NT = s_tile_base[S];
  // blockIdx.z splits a (layer, head): z < kCrossParts = one range of the cross list, z = kCrossParts = the local lists
  // (and, for the first head, the tile tables).  Shortens the latency chain of a CTA (a single layer is latency-bound).
  const int kCrossParts = p.cross_parts;
  const bool do_cross = ((int)blockIdx.z < kCrossParts);
  // fused scheduler (small grids): the sort keys of the head's work items come from a CTA of their own (z = kCrossParts + 1)
  const bool do_local = ((int)blockIdx.z == kCrossParts);
  const bool do_keys = p.fused && ((int)blockIdx.z == kCrossParts + 1);
  const bool writer = (h == 0 && l == 0 && do_local);
  if (writer) {
    for (int d = tid; d <= S; d += kDecodeThreads) p.tile_base[d] = s_tile_base[d];
    for (int d = tid; d < S; d += kDecodeThreads) {
      const int pd = s_tile_base[d + 1] - s_tile_base[d];
      const int nb = (pd + NQ - 1) / NQ;
      for (int k = 0; k < nb; ++k) p.mblock_tile0[s_mb_base[d] + k] = s_tile_base[d] + k * NQ;
      const int f = s_sfirst[d];
      reinterpret_cast<int4*>(p.seg_info)[d] = make_int4(s_sdoc[d], s_sdoc[f], s_off[f], s_tile_base[f]);
    }
    if (tid == 0) p.mblock_tile0[s_mb_base[S]] = NT;
  }

  // ---- cross list: CA bits of all documents, one virtual word sequence ---------------------------------
  // A pass covers kWPT * 256 words: every thread issues its kWPT word loads back to back (one DRAM round trip per
  // pass instead of one per 256 words), counts, and ONE batched block scan (kWPT independent prefix sums sharing the
  // same two barriers) turns the counts into offsets.
  int32_t* cross_ptr = p.cross_ptr + lh * (D + 1);
  int32_t* cross_idx = p.cross_idx + lh * p.cross_cap;
  // masked stream-order bits of word v of the head's virtual word sequence, the global coordinate of its bit 0, the
  // segment it closes (or -1) and its segment
  const int top_s = upper_seg_top(S);
  const uint32_t* ca_words = reinterpret_cast<const uint32_t*>(reinterpret_cast<uintptr_t>(p.ca) & ~(uintptr_t)3);
  auto load_word = [&](int v, int& key0, int& closes, int* seg = nullptr) -> uint32_t {
    const int d = upper_seg(s_wstart, S, v, top_s);   // (segments without words share a start: the last one owns it)
    const int wi = v - s_wstart[d];
    const int len = s_off[d + 1] - s_off[d];
    const int nbits = (len + G - 1) >> gsh;
    const int lead = s_ca_lead[d];
    const uint32_t w = __ldg(ca_words + s_ca_word[d] + wi);
    // stream bit s (MSB-first within each byte, bytes ascending) -> bit s of x
    const uint32_t x = __brev(__byte_perm(w, 0, 0x0123));
    const int lo = max(0, lead - wi * 32);
    const int hi = min(32, lead + nbits - wi * 32);
    uint32_t m = (hi >= 32) ? 0xffffffffu : ((1u << hi) - 1u);
    m &= ~((lo >= 32) ? 0xffffffffu : ((1u << lo) - 1u));
    // global coordinate of stream bit 0 of this word: key row (G == 1) or tile id (G == tile; a page is a tile)
    key0 = (G == 1 ? s_off[d] : s_tile_base[d]) + wi * 32 - lead;
    closes = (v + 1 == s_wstart[d + 1]) ? d : -1;
    if (seg) *seg = d;
    return x & m;
  };
  const int all_words = s_wstart[S];
  // marked bits per segment, as an exclusive prefix in s_stage[0 .. S] (s_stage[s] = marked bits before segment s)
  auto count_segments = [&]() {
    int* s_ccnt = s_stage;
    for (int d = tid; d <= S; d += kDecodeThreads) s_ccnt[d] = 0;
    __syncthreads();
#pragma unroll 4
    for (int v = tid; v < all_words; v += kDecodeThreads) {
      int k0, cl, d;
      const int c = __popc(load_word(v, k0, cl, &d));
      if (c) atomicAdd(&s_ccnt[d + 1], c);
    }
    __syncthreads();
    if (tid < 32) {
      int carry = 0;
      for (int d0 = 0; d0 <= S; d0 += 32) {
        const int d = d0 + tid;
        int v = (d <= S) ? s_ccnt[d] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int n = __shfl_up_sync(0xffffffffu, v, o);
          if (tid >= o) v += n;
        }
        if (d <= S) s_ccnt[d] = carry + v;
        carry += __shfl_sync(0xffffffffu, v, 31);
      }
    }
    __syncthreads();
  };
  // Several prompts (MD-v1b): the list of every prompt starts at a multiple of 128 (the attention kernel reads whole
  // groups of 128 entries), so an entry's position is its rank among the head's marked bits plus s_pad[its segment].
  // s_pad[S] doubles as "several prompts".  One prompt: all zero, nothing to count.
  const bool multi = dt.n_prompts > 1;
  if (multi && do_cross) {
    count_segments();
    if (tid == 0) {
      int pad = 0;
      for (int sg = 0; sg < S; ++sg) {
        if (s_sfirst[sg] == sg) pad = ((s_stage[sg] + pad + 127) & ~127) - s_stage[sg];
        s_pad[sg] = pad;
      }
    }
    __syncthreads();
    // the tail of every prompt's list up to the next multiple of 128 must hold valid rows (gathered, then masked)
    if ((int)blockIdx.z == kCrossParts - 1) {
      for (int sg = 0; sg < S; ++sg) {
        if (s_sdoc[sg] >= 0) continue;                      // at a query segment: its prompt's documents are counted
        const int end = s_stage[sg] + s_pad[sg];
        for (int i = end + tid; i < ((end + 127) & ~127); i += kDecodeThreads) cross_idx[i] = 0;
      }
    }
    __syncthreads();                                        // (s_stage becomes the staging buffer)
  } else {
    for (int sg = tid; sg <= S; sg += kDecodeThreads) s_pad[sg] = 0;
    __syncthreads();
  }
  // list offset of the document that follows segment sg (= the end of sg's own entries; rounded up if a new prompt starts)
  auto next_doc_pad = [&](int sg) {
    int n = sg + 1;
    while (n < S && s_sdoc[n] < 0) ++n;
    return n < S ? s_pad[n] : s_pad[sg];
  };
  // The word sequence of a head is cut into kCrossParts ranges, one CTA each (grid z): a CTA first popcounts the words
  // before its range (the bit vectors of a head are a few KB: re-reading them costs less than waiting for a prefix
  // from another CTA), which gives it the list offset of its first entry.
  const int per = (all_words + kCrossParts - 1) / kCrossParts;
  const int w_lo = do_cross ? min(all_words, (int)blockIdx.z * per) : 0;
  const int total_words = do_cross ? min(all_words, w_lo + per) : 0;      // end of this CTA's range
  int running = 0;
  if (do_cross) {
    int before = 0, k0, cl;
#pragma unroll 4
    for (int v = tid; v < w_lo; v += kDecodeThreads) before += __popc(load_word(v, k0, cl));
    int tot;
    block_exclusive_scan<kDecodeThreads>(before, s_scan, tot);
    running = tot;
    if (blockIdx.z == 0 && tid == 0) cross_ptr[0] = 0;
  }
  int scan_no = 0;   // the two scan buffers alternate over ALL scans of the kernel (no trailing barrier needed)
  for (int base = w_lo; base < total_words; base += kWPT * kDecodeThreads) {
    uint32_t bits[kWPT];
    int key0[kWPT], cnt[kWPT], dd[kWPT], pad[kWPT];
#pragma unroll
    for (int k = 0; k < kWPT; ++k) {
      const int v = base + k * kDecodeThreads + tid;
      bits[k] = 0; key0[k] = 0; dd[k] = -1; pad[k] = 0;
      if (v < total_words) {
        int sg;
        bits[k] = load_word(v, key0[k], dd[k], &sg);
        pad[k] = s_pad[sg];
      }
    }
#pragma unroll
    for (int k = 0; k < kWPT; ++k) cnt[k] = __popc(bits[k]);                     // pass 1: count
    int ex[kWPT];
    const int pass_total = batched_exclusive_scan<kWPT>(cnt, ex, s_bscan[scan_no++ & 1]);   // offsets
    // pass 2: fill, global coordinates.  Every warp compacts its own 32 words with a thread-per-word ffs loop into a
    // private slice of shared memory and copies the slice out with coalesced stores: no block barrier in the fill (the
    // first version staged 256 words per block between two __syncthreads, eight barriers per pass), and no scattered
    // 4-byte stores (32 sectors per store instruction when the ffs loop wrote straight to global memory).
#pragma unroll
    for (int k = 0; k < kWPT; ++k) {
      if (dd[k] >= 0) cross_ptr[s_sdoc[dd[k]] + 1] = running + ex[k] + cnt[k] + next_doc_pad(dd[k]);
      const int lane = tid & 31, wid = tid >> 5;
      const int wbase = __shfl_sync(0xffffffffu, ex[k], 0);                      // list offset of the warp's first entry
      const int wtot = __shfl_sync(0xffffffffu, ex[k] + cnt[k], 31) - wbase;     // entries of the warp's 32 words
      if (wtot == 0) continue;                                                   // warp-uniform
      // (a warp whose words straddle two prompts has two different pads: it writes straight to global memory)
      const int pmin = __reduce_min_sync(0xffffffffu, cnt[k] ? pad[k] : 0x7fffffff);
      const int pmax = __reduce_max_sync(0xffffffffu, cnt[k] ? pad[k] : -1);
      int32_t* dst = cross_idx + running + wbase;
      int o = ex[k] - wbase;
      uint32_t bk = bits[k];
      if (wtot <= kWarpStage - 4 && pmin == pmax) {
        // the slice is filled at the destination's misalignment (mod 4 entries), so that both sides of the copy are
        // 16-byte aligned: whole int4 where all four entries belong to the warp, single entries at the two edges
        // (the scalar copy was 12% of the kernel's instructions)
        dst += pmin;
        const int mis = (int)((running + wbase + pmin) & 3);      // cross_idx rows start 128-byte aligned
        int* stage = s_stage + wid * kWarpStage + mis;
        while (bk) {
          const int sb = __ffs(bk) - 1;
          bk &= bk - 1;
          stage[o++] = key0[k] + sb;
        }
        __syncwarp();
        const int4* st4 = reinterpret_cast<const int4*>(stage - mis);
        int4* dst4 = reinterpret_cast<int4*>(dst - mis);
        const int pend = mis + wtot;
        for (int v = lane; v * 4 < pend; v += 32) {
          const int4 x = st4[v];
          const int p0 = v * 4;
          if (p0 >= mis && p0 + 4 <= pend) {
            dst4[v] = x;
          } else {
            int32_t* d = reinterpret_cast<int32_t*>(dst4 + v);
            if (p0 >= mis && p0 < pend) d[0] = x.x;
            if (p0 + 1 >= mis && p0 + 1 < pend) d[1] = x.y;
            if (p0 + 2 >= mis && p0 + 2 < pend) d[2] = x.z;
            if (p0 + 3 >= mis && p0 + 3 < pend) d[3] = x.w;
          }
        }
        __syncwarp();
      } else {                                            // more than half of the warp's 1024 bits set, or two prompts
        dst += pad[k];
        while (bk) {
          const int sb = __ffs(bk) - 1;
          bk &= bk - 1;
          dst[o++] = key0[k] + sb;
        }
      }
    }
    running += pass_total;
  }
  if (do_cross) {
    // entries in [total, roundup128(total)) must be valid rows: the attention kernel gathers whole groups
    if (!multi && (int)blockIdx.z == kCrossParts - 1)
      for (int i = running + tid; i < ((running + 127) & ~127); i += kDecodeThreads) cross_idx[i] = 0;
  } else if (do_local) {
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
          const int d = upper_seg(s_tile_base, S, t, top_s);
          const int i = t - s_tile_base[d];
          dd[k] = d; ii[k] = i;
          const int seg_len = s_off[d + 1] - s_off[d];
          if (writer) {
            p.tile_seg[t] = d;
            p.tile_row0[t] = s_off[d] + i * T;
            p.tile_rows[t] = min(T, seg_len - i * T);
          }
          if (s_sdoc[d] < 0) {
            cnt[k] = t - s_tile_base[s_sfirst[d]] + 1;                  // query M-block: all causal N-blocks of its prompt (L243)
          } else {
            const int pd = s_tile_base[d + 1] - s_tile_base[d];
            const int nbytes = (pd * (pd + 1) / 2 + 7) >> 3;
            lv[k] = p.la + s_la_off[d] + lh * nbytes;
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
          const int w0 = running + ex[k];
          local_cnt[t] = cnt[k];
          local_ptr[t] = w0;
          if (s_sdoc[dd[k]] >= 0) la_row_fill(lv[k], ii[k], s_tile_base[dd[k]], local_idx + w0);
        }
      }
      running += pass_total;
    }
    if (tid == 0) local_ptr[NT] = running;
    __syncthreads();
    // query tile t lists the tiles f .. t of its prompt: written by the whole block with coalesced stores (one thread
    // per tile wrote up to ~500 entries one after the other in the first version)
    for (int sg = 0; sg < S; ++sg) {
      if (s_sdoc[sg] >= 0) continue;
      const int f = s_tile_base[s_sfirst[sg]];
      for (int t = s_tile_base[sg]; t < s_tile_base[sg + 1]; ++t) {
        const int w0 = __ldcg(local_ptr + t);              // (written above by this block)
        for (int j = tid; j <= t - f; j += kDecodeThreads) local_idx[w0 + j] = f + j;
      }
    }
  }
  if (do_keys) {
    // ---- scheduler keys of this head's work items (a5).  key = processing order: groups of kv heads one after the
    // other (the q-heads of a kv head gather from the same K/V, so the K/V working set of the grid stays L2-sized and
    // K/V are read from HBM about once), longest items first inside a group.  cost = steps of the item's tiles: groups
    // of 128 gathered rows (G == 1) or one page per step (G == tile) + local tiles | dense steps of query tiles.
    // The counts are recounted here from the bits (a few KB, read by the list CTAs at the same time) instead of waiting
    // for the lists: every CTA of the layer only publishes, and the CTA that finishes last just sorts the keys.
    __syncthreads();                                         // (the local lists above are done with s_stage / s_scan)
    count_segments();
    const int* s_ccnt = s_stage;
    const int groups = (p.n_kv_heads + p.kv_per_group - 1) / p.kv_per_group, bpg = kCostBuckets / groups;
    const int g = h / ((p.n_q_heads / p.n_kv_heads) * p.kv_per_group);
    int32_t* key = p.sched_key + (int64_t)l * p.n_items + (int64_t)h * p.n_mblocks;
    static_assert(NQ == 2, "cost of an M-block: two tiles");
    for (int mb = tid; mb < p.n_mblocks; mb += kDecodeThreads) {
      const int seg = upper_seg(s_mb_base, S, mb, top_s);
      const int t0 = s_tile_base[seg] + (mb - s_mb_base[seg]) * NQ;
      const bool two = t0 + 1 < s_tile_base[seg + 1];
      const int f = s_sfirst[seg];
      int c;
      if (s_sdoc[seg] >= 0) {
        const int cp = s_ccnt[seg] - s_ccnt[f];              // marked keys of the prompt's earlier documents
        const int cross_steps = (G == 1) ? (cp + 127) >> 7 : cp;
        const int pd = s_tile_base[seg + 1] - s_tile_base[seg], i0 = t0 - s_tile_base[seg];
        const uint8_t* lv = p.la + s_la_off[seg] + lh * ((pd * (pd + 1) / 2 + 7) >> 3);
        c = (two ? 2 : 1) * cross_steps + la_row_count(lv, i0) + (two ? la_row_count(lv, i0 + 1) : 0);
      } else {
        // dense steps of the query tiles: keys from the prompt's first row to the tile's last row
        const int r0 = s_off[seg] - s_off[f] + (t0 - s_tile_base[seg]) * T, rend = s_off[seg + 1] - s_off[f];
        c = (min(r0 + T, rend) + 127) >> 7;
        if (two) c += (min(r0 + 2 * T, rend) + 127) >> 7;
      }
      key[mb] = g * bpg + (bpg - 1 - min(c, bpg - 1));
    }
  }

  // ---- scheduler (a5), fused: the CTA that finishes a layer last sorts the layer's work items (head, M-block) by
  // key = (kv-head group, descending cost) with a counting sort in shared memory; the persistent attention grid pulls
  // them through an atomic counter.  The keys of the other CTAs are published by the fence + counter below.
  if (!p.fused) return;
  __shared__ int s_last;
  __threadfence();
  __syncthreads();
  int32_t* done = &g_layer_done[(uint32_t)(p.done_base + l) % kDoneRing];
  if (tid == 0) s_last = (atomicAdd(done, 1) == (int)(gridDim.x * gridDim.z) - 1);
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  {
    int* s_hist = s_stage;
    const int NMB = p.n_mblocks;
    auto hx = [](int b) { return b + (b >> 4); };   // 16 consecutive buckets per thread in the scan: pad against bank conflicts
    for (int i = tid; i < kCostBuckets + kCostBuckets / 16; i += kDecodeThreads) s_hist[i] = 0;
    __syncthreads();
    // The sort runs once per layer, in a CTA that is alone on its SM, right after the L1 was invalidated: its code is
    // fetched cold.  So it is written as small loops (a 17x unrolled version spent 40K+ cycles on instruction fetch),
    // unrolled by 4 so that the loads of four items overlap.  Thread t owns items t*per .. t*per+per-1:
    // the items of a warp instruction are `per` apart (other documents, other costs), so its lanes seldom hit the same
    // histogram bucket (consecutive M-blocks of a head mostly do).
    const int32_t* key = p.sched_key + (int64_t)l * p.n_items;   // (plain loads: the fence above invalidated this SM's L1)
    const int n_items = p.n_items;
    const int per = (n_items + kDecodeThreads - 1) / kDecodeThreads, e0 = tid * per, e1 = min(n_items, e0 + per);
#pragma unroll 4
    for (int e = e0; e < e1; ++e) {
      atomicAdd(&s_hist[hx(key[e])], 1);
    }
    __syncthreads();
    {  // exclusive scan over buckets (bucket 0 = first to be processed)
      constexpr int PER = kCostBuckets / kDecodeThreads;
      int sum = 0;
#pragma unroll 4
      for (int k = 0; k < PER; ++k) sum += s_hist[hx(tid * PER + k)];
      int tot;
      int ex = block_exclusive_scan<kDecodeThreads>(sum, s_scan, tot);
#pragma unroll 4
      for (int k = 0; k < PER; ++k) { const int c = s_hist[hx(tid * PER + k)]; s_hist[hx(tid * PER + k)] = ex; ex += c; }
    }
    __syncthreads();
    int32_t* sched = p.sched + (int64_t)l * n_items;
#pragma unroll 4
    for (int e = e0; e < e1; ++e) {
      const int b = key[e];
      const int h2 = e / NMB;
      sched[atomicAdd(&s_hist[hx(b)], 1)] = (h2 << 20) | (e - h2 * NMB);
    }
    if (tid < 2) p.counters[l * 2 + tid] = 0;
    if (tid == 0) *done = 0;
  }
}

// Scheduler as a launch of its own (whole stacks, p.fused == 0): one 1024-thread CTA per layer computes the same sort
// keys from the decoded counts and counting-sorts the layer's work items.
constexpr int kSchedThreads = 1024;
__global__ void __launch_bounds__(kSchedThreads)
sift_schedule_kernel(const DecodeParams p, int n_docs) {
  __shared__ int s_hist[kCostBuckets];
  __shared__ int s_scan[kSchedThreads / 32 + 1];
  constexpr int NQ = SIFT_Q_TILES_PER_ITEM;
  const int l = blockIdx.x, tid = threadIdx.x;
  const int D = n_docs, NT = p.n_tiles, NMB = p.n_mblocks;
  for (int i = tid; i < kCostBuckets; i += kSchedThreads) s_hist[i] = 0;
  __syncthreads();
  const int groups = (p.n_kv_heads + p.kv_per_group - 1) / p.kv_per_group, bpg = kCostBuckets / groups;
  auto key_of = [&](int e) {
    const int h = e / NMB, mb = e - h * NMB;
    const int64_t lh = (int64_t)l * p.n_q_heads + h;
    const int t0 = p.mblock_tile0[mb], t1 = min(p.mblock_tile0[mb + 1], t0 + NQ);
    const int4 si = reinterpret_cast<const int4*>(p.seg_info)[p.tile_seg[t0]];
    int c = 0;
    if (si.x >= 0) {
      const int cp = p.cross_ptr[lh * (D + 1) + si.x] - p.cross_ptr[lh * (D + 1) + si.y];
      const int cross_steps = (p.gran == 1) ? (cp + 127) >> 7 : cp;
      for (int t = t0; t < t1; ++t) c += cross_steps + p.local_cnt[lh * NT + t];
    } else {
      for (int t = t0; t < t1; ++t) c += (p.tile_row0[t] - si.z + p.tile_rows[t] + 127) >> 7;
    }
    const int g = h / (p.n_q_heads / p.n_kv_heads) / p.kv_per_group;
    return g * bpg + (bpg - 1 - min(c, bpg - 1));
  };
  // the key of an item is a chain of dependent global loads: evaluate it once and keep it in registers for the
  // scatter pass (up to kCached items per thread; larger layers recompute)
  constexpr int kCached = 8;
  int ck[kCached];
#pragma unroll
  for (int k = 0; k < kCached; ++k) {
    const int e = tid + k * kSchedThreads;
    ck[k] = (e < p.n_items) ? key_of(e) : 0;
  }
#pragma unroll
  for (int k = 0; k < kCached; ++k)
    if (tid + k * kSchedThreads < p.n_items) atomicAdd(&s_hist[ck[k]], 1);
  for (int e = tid + kCached * kSchedThreads; e < p.n_items; e += kSchedThreads) atomicAdd(&s_hist[key_of(e)], 1);
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
  auto place = [&](int e, int b) {
    const int h = e / NMB;
    sched[atomicAdd(&s_hist[b], 1)] = (h << 20) | (e - h * NMB);
  };
#pragma unroll
  for (int k = 0; k < kCached; ++k)
    if (tid + k * kSchedThreads < p.n_items) place(tid + k * kSchedThreads, ck[k]);
  for (int e = tid + kCached * kSchedThreads; e < p.n_items; e += kSchedThreads) place(e, key_of(e));
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
  p.sched_key = at(sched_key_offset(lay, s->n_layers));
  p.seg_info = at(lay.seg_info);
  p.n_q_heads = s->n_q_heads; p.n_kv_heads = s->n_kv_heads; p.n_tiles = lay.n_tiles; p.cross_cap = lay.cross_cap; p.local_cap = lay.local_cap;
  p.n_mblocks = lay.n_mblocks; p.n_items = lay.n_items; p.gran = s->cross_gran;
  // few (layer, head) pairs (one layer of an 8B-class model = 32): the call is latency-bound, cut each head's cross list
  // into ranges for separate CTAs; many (a whole stack = 1024): one CTA per list is more efficient (no re-counting)
  int num_sms = 0;
  if (int rc = device_sm_count(&num_sms)) return rc;
  p.cross_parts = ((int64_t)s->n_q_heads * s->n_layers <= num_sms) ? kMaxCrossParts : 1;
  // one layer: a second launch would double the latency of the call, so the scheduler is fused (21 vs 26 us at 32K);
  // whole stacks: the recount behind the keys and the per-layer sort tails cost more than a second launch that sorts
  // all layers in parallel (32 layers of C3: 66 us fused, 50 us with the separate kernel)
  p.fused = (p.cross_parts > 1);
  p.kv_per_group = sched_kv_heads_per_group(lay.n_tokens, s->head_dim, s->n_kv_heads);
  p.tile_shift = (s->tile == 128) ? 7 : 6;
  p.gran_shift = (s->cross_gran == 1) ? 0 : p.tile_shift;
  if (s->n_layers > kDoneRing / 4) return set_error(SIFT_ERR_UNSUPPORTED, "too many layers in one decode call");
  p.done_base = (int32_t)(g_done_ticket.fetch_add((uint32_t)s->n_layers, std::memory_order_relaxed) % kDoneRing);
  cudaGetLastError();
  sift_decode_kernel<<<dim3(s->n_q_heads, s->n_layers, p.cross_parts + 1 + p.fused), kDecodeThreads, 0, st>>>(dt, p);
  if (!p.fused) sift_schedule_kernel<<<s->n_layers, kSchedThreads, 0, st>>>(p, s->n_docs);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return set_error(SIFT_ERR_CUDA, "decode launch: %s", cudaGetErrorString(e));
  count_launch(p.fused ? 1 : 2);
  return SIFT_OK;
}

}  // namespace sift
