// Internal declarations shared by the translation units of libsift_b200.so (not part of the ABI).
#pragma once
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
struct DocTable {
  int32_t n_docs;
  int32_t query_len;
  int32_t tile;
  int32_t gran;
  int32_t off[SIFT_MAX_DOCS + 1];
  int64_t la_off[SIFT_MAX_DOCS];
  int64_t ca_off[SIFT_MAX_DOCS];
};

int set_error(int code, const char* fmt, ...);
int validate_shape(const sift_shape* s);
int compute_layout(const sift_shape* s, sift_md_layout* out);
void count_launch(int n = 1);

int launch_decode(const sift_shape* s, const sift_md_layout& lay, const DocTable& dt,
                  const uint8_t* la_base, const uint8_t* ca_base, void* md, cudaStream_t st);

static inline int ceil_div_i(int a, int b) { return (a + b - 1) / b; }

}  // namespace sift
