// Internal declarations shared by the translation units of libsift_b200.so (not part of the ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <atomic>

#include "sift.h"

#ifndef SIFT_Q_TILES_PER_ITEM
#define SIFT_Q_TILES_PER_ITEM 2   // query tiles (of `tile` rows) one attention work item covers
#endif

namespace sift {

// Passed by value as a kernel parameter (CUDA >= 12.1 allows 32 KB of parameters): the decode grid and
// the tile tables depend on the document offsets, which the ABI hands over as HOST memory.
// Segments = documents and queries in token order (one prompt: its documents, then the query; several prompts: one
// after the other).
constexpr int kMaxSeg = SIFT_MAX_DOCS + 1;
struct DocTable {
  int32_t n_seg;
  int32_t n_docs;
  int32_t n_prompts;
  int32_t tile;
  int32_t gran;
  int32_t off[kMaxSeg + 1];        // first row of segment s; off[n_seg] = N
  int16_t doc[kMaxSeg];            // document index of segment s, -1 for a query segment
  int16_t first[kMaxSeg];          // first segment of s's prompt
  int64_t la_off[SIFT_MAX_DOCS];   // by document index
  int64_t ca_off[SIFT_MAX_DOCS];
};
// fills n_seg, n_docs, n_prompts, tile, gran, off, doc, first from a validated shape
void build_segments(const sift_shape* s, DocTable* dt);
int64_t shape_n_tokens(const sift_shape* s);

int set_error(int code, const char* fmt, ...);
int validate_shape(const sift_shape* s);
int compute_layout(const sift_shape* s, sift_md_layout* out);
void count_launch(int n = 1);

int launch_decode(const sift_shape* s, const sift_md_layout& lay, const DocTable& dt,
                  const uint8_t* la_base, const uint8_t* ca_base, void* md, cudaStream_t st);

// 2-D tensor [rows][cols] of bf16 (elem_bytes 2) or bytes (1: e4m3) with a row stride of `row_stride` elements; box = 128
// bytes of a row x box_rows, 128-byte swizzle (the image tcgen05's SWIZZLE_128B descriptors read).  Shared by the
// attention and the encoder launchers.
int make_tensor_map_2d(CUtensorMap* m, const void* base, int64_t rows, int64_t cols, int64_t row_stride, int box_rows,
                       int elem_bytes = 2);
// SM count of the current device, and the once-per-(device, kernel) opt-in to `bytes` of dynamic shared memory.
// `slot` numbers the kernels of the library (kSmemSlot*): cudaFuncSetAttribute is a per-device attribute.
int device_sm_count(int* num_sms);
enum { kSmemSlotAttn64 = 0, kSmemSlotAttn128, kSmemSlotEnc64, kSmemSlotEnc128, kSmemSlotAttnF8, kSmemSlots };
int ensure_dynamic_smem(const void* func, int bytes, int slot);

static inline int ceil_div_i(int a, int b) { return (a + b - 1) / b; }
// private array behind `counters`: the sort key of every work item, [L][n_items] int32 (compute_layout reserves it)
static inline size_t sched_key_offset(const sift_md_layout& lay, int n_layers) {
  return (lay.counters + (size_t)n_layers * 2 * 4 + 127) / 128 * 128;
}

// How many kv heads the scheduler lets the grid work on at a time: as many as keep their K and V (n_tokens x head_dim
// bf16 each) within ~72 MB of the 126 MB L2.  Measured on B200: C3 32K is fastest with >= 4 of its 8
// kv heads active (fewer concentrates the traffic on too few L2 slices: K/V rows of one kv head are 256 B out of every
// 2 KB), C4 64K with 2; DRAM traffic drops from 2.0x to 1.0-1.25x the algorithmic bytes.
static inline int sched_kv_heads_per_group(int64_t n_tokens, int head_dim, int n_kv_heads) {
  const int64_t per_head = n_tokens * head_dim * 2 * 2;
  int64_t k = (72ll << 20) / (per_head > 0 ? per_head : 1);
  if (k < 1) k = 1;
  if (k > n_kv_heads) k = n_kv_heads;
  return (int)k;
}

}  // namespace sift
