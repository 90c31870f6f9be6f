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

int validate_shape(const sift_shape* s) {
  if (!s) return set_error(SIFT_ERR_INVALID_ARG, "shape is NULL");
  if (s->struct_size != sizeof(sift_shape))
    return set_error(SIFT_ERR_INVALID_ARG, "shape.struct_size %u != %zu", s->struct_size, sizeof(sift_shape));
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
  int64_t n = (int64_t)s->doc_offsets[s->n_docs] + s->query_len;
  if (n < 1 || n > (1 << 20)) return set_error(SIFT_ERR_UNSUPPORTED, "prompt of %lld rows (1 .. 2^20 supported)", (long long)n);
  return SIFT_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_tensor_map_2d(CUtensorMap* m, const void* base, int64_t rows, int64_t cols, int64_t row_stride, int box_rows) {
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
  cuuint64_t gstr[1] = {(cuuint64_t)row_stride * 2};
  cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim, gstr, box, estr,
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
  int64_t nt = 0, lcap = 0, nmb = 0, ncross = 0;
  for (int d = 0; d < D; ++d) {
    int64_t p = ceil_div_i(s->doc_offsets[d + 1] - s->doc_offsets[d], T);
    ncross += ceil_div_i(s->doc_offsets[d + 1] - s->doc_offsets[d], s->cross_gran);
    nt += p;
    lcap += p * (p + 1) / 2;
    nmb += (p + NQ - 1) / NQ;
  }
  int64_t pq = ceil_div_i(s->query_len, T);
  for (int64_t t = nt; t < nt + pq; ++t) lcap += t + 1;
  nt += pq;
  nmb += (pq + NQ - 1) / NQ;
  int64_t ccap = (ncross + 127) / 128 * 128;   // one entry per CA bit at most, rounded up to whole gather groups
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
  out->tile_base = take(D + 2);
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
  return compute_layout(shape, out);
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
  dt.n_docs = shape->n_docs;
  dt.query_len = shape->query_len;
  dt.tile = shape->tile;
  dt.gran = shape->cross_gran;
  for (int d = 0; d <= shape->n_docs; ++d) dt.off[d] = shape->doc_offsets[d];
  for (int d = 0; d < shape->n_docs; ++d) {
    if (la_doc_off[d] < 0 || ca_doc_off[d] < 0) return set_error(SIFT_ERR_INVALID_ARG, "negative blob offset at doc %d", d);
    dt.la_off[d] = la_doc_off[d];
    dt.ca_off[d] = ca_doc_off[d];
  }
  return launch_decode(shape, lay, dt, la_base, ca_base, metadata, (cudaStream_t)stream);
}

}  // extern "C"
