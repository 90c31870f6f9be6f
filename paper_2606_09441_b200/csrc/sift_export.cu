// The paper's own index layout, materialised from MD-v1 (sec 5.1).
//
// The paper's decode kernel emits `sparse_n_indices`: for every (head, M-block) ONE packed int32 list, the CA entries of
// all earlier documents first, then the M-block's LA entries, at a designated offset; a query M-block lists all causal
// N-blocks.  MD-v1 stores the CA entries of a head once (document d uses the prefix [cross_ptr[d0], cross_ptr[d]) of one
// list) and only the LA lists per M-block.  These two kernels rebuild the paper's replicated layout on the GPU so that
// its size and the time to write it can be measured beside MD-v1's (bench.py extra.paper_indices), and so that a
// consumer written against the paper's layout can be fed.  No new information: list(h, t) = cross prefix ++ local list.
#include "sift_common.h"

namespace sift {

constexpr int kExportThreads = 256;

struct ExportParams {
  const int32_t *tile_seg, *seg_info, *cross_ptr, *cross_idx, *local_cnt, *local_ptr, *local_idx;   // offset to the layer
  int32_t n_tiles, n_docs, cross_cap, local_cap;
};

__device__ __forceinline__ void tile_cross_range(const ExportParams& p, int h, int t, int& c0, int& c1) {
  const int4 si = reinterpret_cast<const int4*>(p.seg_info)[p.tile_seg[t]];   // {document, first document of the prompt, ..}
  c0 = c1 = 0;
  if (si.x >= 0) {
    const int32_t* cp = p.cross_ptr + (int64_t)h * (p.n_docs + 1);
    c0 = cp[si.y];
    c1 = cp[si.x];
  }
}

// ptr[h][t] = number of entries of the M-blocks 0 .. t-1 of head h; ptr[h][NT] = entries of the head.  One CTA per head.
__global__ void __launch_bounds__(kExportThreads)
sift_paper_offsets_kernel(const ExportParams p, int64_t* __restrict__ ptr) {
  __shared__ int64_t s_warp[kExportThreads / 32];
  __shared__ int64_t s_carry;
  const int h = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (tid == 0) s_carry = 0;
  __syncthreads();
  int64_t* out = ptr + (int64_t)h * (p.n_tiles + 1);
  for (int base = 0; base < p.n_tiles; base += kExportThreads) {
    const int t = base + tid;
    int64_t v = 0;
    if (t < p.n_tiles) {
      int c0, c1;
      tile_cross_range(p, h, t, c0, c1);
      v = (int64_t)(c1 - c0) + p.local_cnt[(int64_t)h * p.n_tiles + t];
    }
    int64_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int64_t n = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += n;
    }
    if (lane == 31) s_warp[wid] = inc;
    __syncthreads();
    int64_t before = s_carry;
    for (int w = 0; w < wid; ++w) before += s_warp[w];
    if (t < p.n_tiles) out[t] = before + inc - v;
    __syncthreads();
    if (tid == kExportThreads - 1) s_carry = before + inc;
    __syncthreads();
  }
  if (tid == 0) out[p.n_tiles] = s_carry;
}

// One CTA per (M-block, head): copies the cross prefix, then the local list, to idx[h * head_stride + ptr[h][t] ..).
__global__ void __launch_bounds__(kExportThreads)
sift_paper_export_kernel(const ExportParams p, const int64_t* __restrict__ ptr, int32_t* __restrict__ idx, int64_t head_stride) {
  const int t = blockIdx.x, h = blockIdx.y, tid = threadIdx.x;
  int c0, c1;
  tile_cross_range(p, h, t, c0, c1);
  const int64_t w0 = ptr[(int64_t)h * (p.n_tiles + 1) + t];
  int32_t* dst = idx + (int64_t)h * head_stride;
  const int32_t* cross = p.cross_idx + (int64_t)h * p.cross_cap + c0;
  const int nc = c1 - c0;
  for (int i = tid; i < nc; i += kExportThreads)
    if (w0 + i < head_stride) dst[w0 + i] = cross[i];
  const int nl = p.local_cnt[(int64_t)h * p.n_tiles + t];
  const int32_t* loc = p.local_idx + (int64_t)h * p.local_cap + p.local_ptr[(int64_t)h * (p.n_tiles + 1) + t];
  for (int i = tid; i < nl; i += kExportThreads)
    if (w0 + nc + i < head_stride) dst[w0 + nc + i] = loc[i];
}

static int fill_params(const sift_shape* shape, int32_t layer, const void* metadata, ExportParams* p, sift_md_layout* lay) {
  int rc = compute_layout(shape, lay);
  if (rc) return rc;
  if (layer < 0 || layer >= shape->n_layers) return set_error(SIFT_ERR_INVALID_ARG, "layer %d out of range", layer);
  if (!metadata) return set_error(SIFT_ERR_INVALID_ARG, "metadata is NULL");
  const char* b = static_cast<const char*>(metadata);
  auto at = [&](size_t off) { return reinterpret_cast<const int32_t*>(b + off); };
  const int64_t lh0 = (int64_t)layer * shape->n_q_heads;
  p->tile_seg = at(lay->tile_seg);
  p->seg_info = at(lay->seg_info);
  p->cross_ptr = at(lay->cross_ptr) + lh0 * (shape->n_docs + 1);
  p->cross_idx = at(lay->cross_idx) + lh0 * lay->cross_cap;
  p->local_cnt = at(lay->local_cnt) + lh0 * lay->n_tiles;
  p->local_ptr = at(lay->local_ptr) + lh0 * (lay->n_tiles + 1);
  p->local_idx = at(lay->local_idx) + lh0 * lay->local_cap;
  p->n_tiles = lay->n_tiles; p->n_docs = shape->n_docs; p->cross_cap = lay->cross_cap; p->local_cap = lay->local_cap;
  return SIFT_OK;
}

}  // namespace sift

using namespace sift;

extern "C" int sift_paper_index_offsets(const sift_shape* shape, int32_t layer, const void* metadata, int64_t* ptr,
                                        void* stream) {
  ExportParams p;
  sift_md_layout lay;
  int rc = fill_params(shape, layer, metadata, &p, &lay);
  if (rc) return rc;
  if (!ptr) return set_error(SIFT_ERR_INVALID_ARG, "ptr is NULL");
  cudaGetLastError();
  sift_paper_offsets_kernel<<<shape->n_q_heads, kExportThreads, 0, (cudaStream_t)stream>>>(p, ptr);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return set_error(SIFT_ERR_CUDA, "paper offsets launch: %s", cudaGetErrorString(e));
  count_launch(1);
  return SIFT_OK;
}

extern "C" int sift_export_paper_indices(const sift_shape* shape, int32_t layer, const void* metadata, const int64_t* ptr,
                                         int32_t* idx, int64_t head_stride, void* stream) {
  ExportParams p;
  sift_md_layout lay;
  int rc = fill_params(shape, layer, metadata, &p, &lay);
  if (rc) return rc;
  if (!ptr || !idx) return set_error(SIFT_ERR_INVALID_ARG, "ptr / idx is NULL");
  if (head_stride < 0) return set_error(SIFT_ERR_INVALID_ARG, "negative head_stride");
  if (lay.n_tiles == 0) return SIFT_OK;
  cudaGetLastError();
  sift_paper_export_kernel<<<dim3(lay.n_tiles, shape->n_q_heads), kExportThreads, 0, (cudaStream_t)stream>>>(p, ptr, idx, head_stride);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return set_error(SIFT_ERR_CUDA, "paper export launch: %s", cudaGetErrorString(e));
  count_launch(1);
  return SIFT_OK;
}
