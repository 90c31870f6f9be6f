// Host side of the C ABI: validation, MD-v1 layout arithmetic, error reporting, sift_decode_metadata entry.
#include <stdarg.h>
#include <string.h>

#include "sift_common.h"

namespace sift {

static thread_local char g_err[512] = "";
static std::atomic<int64_t> g_launches{0};

int set_error(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

static int shape_n_prompts(const sift_shape* s) {
  return (s->struct_size == sizeof(sift_shape) && s->n_prompts > 1) ? s->n_prompts : 1;
}
int64_t shape_n_tokens(const sift_shape* s) {
  int64_t n = s->doc_offsets[s->n_docs];
  const int np = shape_n_prompts(s);
  if (np > 1) { for (int p = 0; p < np; ++p) n += s->prompt_query_len[p]; } else n += s->query_len;
  return n;
}

int validate_shape(const sift_shape* s) {
  if (!s) return set_error(SIFT_ERR_INVALID_ARG, "shape is NULL");
  if (s->struct_size != sizeof(sift_shape) && s->struct_size != SIFT_SHAPE_SIZE_V1)
    return set_error(SIFT_ERR_INVALID_ARG, "shape.struct_size %u: expected %zu (or %u, the struct without the prompt fields)",
                     s->struct_size, sizeof(sift_shape), SIFT_SHAPE_SIZE_V1);
  if (!s->doc_offsets) return set_error(SIFT_ERR_INVALID_ARG, "shape.doc_offsets is NULL");
  if (s->n_layers < 1 || s->n_q_heads < 1 || s->n_kv_heads < 1 || s->n_docs < 0 || s->query_len < 0)
    return set_error(SIFT_ERR_INVALID_ARG, "negative or zero dimension");
  if (s->n_q_heads % s->n_kv_heads != 0)
    return set_error(SIFT_ERR_INVALID_ARG, "n_q_heads %d not a multiple of n_kv_heads %d", s->n_q_heads, s->n_kv_heads);
  if (s->n_q_heads > 255) return set_error(SIFT_ERR_UNSUPPORTED, "n_q_heads %d > 255", s->n_q_heads);
  if (s->head_dim != 64 && s->head_dim != 128)
    return set_error(SIFT_ERR_UNSUPPORTED, "head_dim %d not in {64,128}", s->head_dim);
  if (s->tile != 64 && s->tile != 128) return set_error(SIFT_ERR_UNSUPPORTED, "tile %d not in {64,128}", s->tile);
  if (s->cross_gran != 1 && s->cross_gran != s->tile)
    return set_error(SIFT_ERR_UNSUPPORTED, "cross_gran %d: 1 (per key token) or tile (per page, PAPER.md:L209)", s->cross_gran);
  if (s->n_docs > SIFT_MAX_DOCS) return set_error(SIFT_ERR_UNSUPPORTED, "n_docs %d > %d", s->n_docs, SIFT_MAX_DOCS);
  if (s->doc_offsets[0] != 0) return set_error(SIFT_ERR_INVALID_ARG, "doc_offsets[0] != 0");
  for (int d = 0; d < s->n_docs; ++d)
    if (s->doc_offsets[d + 1] <= s->doc_offsets[d])
      return set_error(SIFT_ERR_INVALID_ARG, "doc_offsets not strictly increasing at %d", d);
  const int np = shape_n_prompts(s);
  if (np > 1) {
    if (!s->prompt_doc_start || !s->prompt_query_len)
      return set_error(SIFT_ERR_INVALID_ARG, "n_prompts %d but prompt_doc_start / prompt_query_len is NULL", np);
    if (s->n_docs + np > SIFT_MAX_DOCS + 1)
      return set_error(SIFT_ERR_UNSUPPORTED, "n_docs + n_prompts = %d > %d", s->n_docs + np, SIFT_MAX_DOCS + 1);
    if (s->prompt_doc_start[0] != 0 || s->prompt_doc_start[np] != s->n_docs)
      return set_error(SIFT_ERR_INVALID_ARG, "prompt_doc_start must run from 0 to n_docs");
    for (int p = 0; p < np; ++p)
      if (s->prompt_doc_start[p + 1] < s->prompt_doc_start[p] || s->prompt_query_len[p] < 0)
        return set_error(SIFT_ERR_INVALID_ARG, "prompt %d: decreasing prompt_doc_start or negative query length", p);
  }
  int64_t n = shape_n_tokens(s);
  if (n < 1 || n > (1 << 20)) return set_error(SIFT_ERR_UNSUPPORTED, "prompt(s) of %lld rows (1 .. 2^20 supported)", (long long)n);
  return SIFT_OK;
}

void build_segments(const sift_shape* s, DocTable* dt) {
  const int np = shape_n_prompts(s);
  dt->n_docs = s->n_docs; dt->n_prompts = np; dt->tile = s->tile; dt->gran = s->cross_gran;
  int seg = 0, row = 0;
  for (int p = 0; p < np; ++p) {
    const int d0 = np > 1 ? s->prompt_doc_start[p] : 0, d1 = np > 1 ? s->prompt_doc_start[p + 1] : s->n_docs;
    const int qlen = np > 1 ? s->prompt_query_len[p] : s->query_len;
    const int first = seg;
    for (int d = d0; d < d1; ++d) {
      dt->off[seg] = row; dt->doc[seg] = (int16_t)d; dt->first[seg] = (int16_t)first;
      row += s->doc_offsets[d + 1] - s->doc_offsets[d];
      ++seg;
    }
    dt->off[seg] = row; dt->doc[seg] = -1; dt->first[seg] = (int16_t)first;
    row += qlen;
    ++seg;
  }
  dt->off[seg] = row;
  dt->n_seg = seg;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_tensor_map_2d(CUtensorMap* m, const void* base, int64_t rows, int64_t cols, int64_t row_stride, int box_rows,
                       int elem_bytes) {
  static std::atomic<EncodeTiledFn> cached{nullptr};
  EncodeTiledFn fn = cached.load(std::memory_order_acquire);
  if (!fn) {
    void* sym = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
      return set_error(SIFT_ERR_CUDA, "cuTensorMapEncodeTiled not available from the driver");
    fn = reinterpret_cast<EncodeTiledFn>(sym);
    cached.store(fn, std::memory_order_release);
  }
  cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t gstr[1] = {(cuuint64_t)row_stride * elem_bytes};
  cuuint32_t box[2] = {(cuuint32_t)(128 / elem_bytes), (cuuint32_t)box_rows};   // 128 bytes of a row: one swizzle row
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(m, elem_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(base), gdim, gstr, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return set_error(SIFT_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  return SIFT_OK;
}

// Per-device launch state: the SM count sizes the persistent grids, the shared-memory opt-in is a per-device
// attribute of each kernel (a process may call the library on several devices, from several threads).
constexpr int kMaxDevices = 64;
struct DeviceState {
  std::atomic<int> num_sms{0};
  std::atomic<int> smem_set[kSmemSlots];
};
static DeviceState g_dev[kMaxDevices];

static int current_device(int* dev) {
  if (cudaGetDevice(dev) != cudaSuccess || *dev < 0 || *dev >= kMaxDevices)
    return set_error(SIFT_ERR_CUDA, "no usable current CUDA device");
  return SIFT_OK;
}

int device_sm_count(int* num_sms) {
  int dev, rc;
  if ((rc = current_device(&dev))) return rc;
  int n = g_dev[dev].num_sms.load(std::memory_order_relaxed);
  if (n == 0) {
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0)
      return set_error(SIFT_ERR_CUDA, "cannot read the SM count of device %d", dev);
    g_dev[dev].num_sms.store(n, std::memory_order_relaxed);
  }
  *num_sms = n;
  return SIFT_OK;
}

int ensure_dynamic_smem(const void* func, int bytes, int slot) {
  int dev, rc;
  if ((rc = current_device(&dev))) return rc;
  if (g_dev[dev].smem_set[slot].load(std::memory_order_acquire)) return SIFT_OK;
  cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e != cudaSuccess) return set_error(SIFT_ERR_CUDA, "cudaFuncSetAttribute(smem=%d): %s", bytes, cudaGetErrorString(e));
  g_dev[dev].smem_set[slot].store(1, std::memory_order_release);
  return SIFT_OK;
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

int compute_layout(const sift_shape* s, sift_md_layout* out) {
  int rc = validate_shape(s);
  if (rc) return rc;
  const int T = s->tile, D = s->n_docs, NQ = SIFT_Q_TILES_PER_ITEM;
  static thread_local DocTable dt;
  build_segments(s, &dt);
  int64_t nt = 0, lcap = 0, nmb = 0, ccap = 0;
  int64_t ncross = 0, first_tile = 0;       // of the current prompt
  for (int sg = 0; sg < dt.n_seg; ++sg) {
    const int64_t len = dt.off[sg + 1] - dt.off[sg];
    const int64_t p = (len + T - 1) / T;
    if (dt.first[sg] == sg) { first_tile = nt; ncross = 0; }
    if (dt.doc[sg] >= 0) {
      ncross += (len + s->cross_gran - 1) / s->cross_gran;
      lcap += p * (p + 1) / 2;
    } else {
      for (int64_t t = nt; t < nt + p; ++t) lcap += t - first_tile + 1;   // a query tile lists its prompt's tiles up to itself
      ccap += (ncross + 127) / 128 * 128;   // one entry per CA bit at most; every prompt's list in whole gather groups
    }
    nt += p;
    nmb += (p + NQ - 1) / NQ;
  }
  if (lcap >= (1ll << 31) || ccap >= (1ll << 31)) return set_error(SIFT_ERR_UNSUPPORTED, "index capacity >= 2^31");
  if (lcap < 1) lcap = 1;
  const int64_t LH = (int64_t)s->n_layers * s->n_q_heads;
  memset(out, 0, sizeof(*out));
  out->struct_size = sizeof(sift_md_layout);
  out->n_tiles = (int32_t)nt;
  out->cross_cap = (int32_t)ccap;
  out->local_cap = (int32_t)lcap;
  out->n_mblocks = (int32_t)nmb;
  out->n_items = (int32_t)(nmb * s->n_q_heads);
  size_t o = 0;
  auto take = [&](int64_t n_int32) { size_t r = o; o = align_up(o + (size_t)n_int32 * 4, 128); return r; };
  out->tile_base = take(dt.n_seg + 1);
  out->tile_seg = take(nt);
  out->tile_row0 = take(nt);
  out->tile_rows = take(nt);
  out->cross_ptr = take(LH * (D + 1));
  out->cross_idx = take(LH * ccap);
  out->local_cnt = take(LH * nt);
  out->local_ptr = take(LH * (nt + 1));
  out->local_idx = take(LH * lcap);
  out->mblock_tile0 = take(nmb + 1);
  out->sched = take((int64_t)s->n_layers * out->n_items);
  out->counters = take((int64_t)s->n_layers * 2);
  take((int64_t)s->n_layers * out->n_items);   // scheduler keys (private, unnamed: sched_key_offset())
  out->seg_info = take((int64_t)dt.n_seg * 4);
  out->n_seg = dt.n_seg;
  out->n_tokens = dt.off[dt.n_seg];
  out->total_bytes = o;
  return SIFT_OK;
}

}  // namespace sift

using namespace sift;

extern "C" {

#define SIFT_STR2(x) #x
#define SIFT_STR(x) SIFT_STR2(x)
const char* sift_version(void) {
  return "sift-b200 0.1.0 (sm_100a; MD-v1; q_tiles_per_item=" SIFT_STR(SIFT_Q_TILES_PER_ITEM) ")";
}

const char* sift_last_error(void) { return g_err; }

int64_t sift_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int sift_metadata_layout(const sift_shape* shape, sift_md_layout* out) {
  if (!out) return set_error(SIFT_ERR_INVALID_ARG, "out is NULL");
  sift_md_layout lay;
  int rc = compute_layout(shape, &lay);
  if (rc) return rc;
  // a V1-sized shape comes from a caller whose sift_md_layout ends before n_seg: write no more than it owns
  const size_t n = shape->struct_size == SIFT_SHAPE_SIZE_V1 ? (size_t)SIFT_MD_LAYOUT_SIZE_V1 : sizeof(lay);
  lay.struct_size = (uint32_t)n;
  memcpy(out, &lay, n);
  return SIFT_OK;
}

int sift_metadata_size(const sift_shape* shape, size_t* bytes) {
  if (!bytes) return set_error(SIFT_ERR_INVALID_ARG, "bytes is NULL");
  sift_md_layout lay;
  int rc = compute_layout(shape, &lay);
  if (rc) return rc;
  *bytes = lay.total_bytes;
  return SIFT_OK;
}

int sift_decode_metadata(const sift_shape* shape, const uint8_t* la_base, const int64_t* la_doc_off,
                         const uint8_t* ca_base, const int64_t* ca_doc_off, void* metadata, size_t metadata_bytes,
                         void* stream) {
  sift_md_layout lay;
  int rc = compute_layout(shape, &lay);
  if (rc) return rc;
  if (!metadata) return set_error(SIFT_ERR_INVALID_ARG, "metadata is NULL");
  if (((uintptr_t)metadata & 15) != 0) return set_error(SIFT_ERR_INVALID_ARG, "metadata not 16-byte aligned");
  if (metadata_bytes < lay.total_bytes)
    return set_error(SIFT_ERR_WORKSPACE, "metadata buffer %zu < %zu bytes", metadata_bytes, lay.total_bytes);
  if (shape->n_docs > 0 && (!la_base || !ca_base || !la_doc_off || !ca_doc_off))
    return set_error(SIFT_ERR_INVALID_ARG, "bit-vector pointer is NULL");
  static thread_local DocTable dt;
  build_segments(shape, &dt);
  for (int d = 0; d < shape->n_docs; ++d) {
    if (la_doc_off[d] < 0 || ca_doc_off[d] < 0) return set_error(SIFT_ERR_INVALID_ARG, "negative blob offset at doc %d", d);
    dt.la_off[d] = la_doc_off[d];
    dt.ca_off[d] = ca_doc_off[d];
  }
  return launch_decode(shape, lay, dt, la_base, ca_base, metadata, (cudaStream_t)stream);
}

}  // extern "C"
