// Host-buffer entry of one prefill layer (include/sift.h: sift_prefill_layer_host).
//
// PAPER.md:L225 (sec 4.4): the bit vectors arrive from CPU DRAM together with the retrieved documents; L331 (sec 7.4):
// they are copied to the GPU in one H2D transfer.  This call takes everything from HOST memory and returns O to HOST
// memory: the layer is cut into its kv-head groups (a kv head and its q-heads are an independent unit of the path,
// SURVEY.md 8(e)); per group the strided H2D copy of its Q columns, metadata decode + attention for its q-heads, and
// the D2H copy of its O columns run on three streams, so that PCIe traffic in both directions overlaps the kernels
// and each other.  Plumbing only: cudaMemcpy2DAsync + events around the same two kernels every other entry uses.
#include <string.h>

#include <mutex>

#include "sift_common.h"

namespace sift {

constexpr int kMaxGroups = 256;

struct HostCtx {
  int device = -1;
  cudaStream_t s_in = nullptr, s_cmp = nullptr, s_out = nullptr;
  cudaEvent_t ev_start = nullptr, ev_done = nullptr;
  cudaEvent_t ev_in[kMaxGroups], ev_cmp[kMaxGroups];
  int n_events = 0;
};

static size_t up256(size_t x) { return (x + 255) / 256 * 256; }

// A caller built against the older header passes a shape of SIFT_SHAPE_SIZE_V1 bytes: read no further than it says
// (validate_shape has accepted struct_size), the prompt fields it does not have read as "one prompt".
static void copy_shape(const sift_shape* s, sift_shape* out) {
  memset(out, 0, sizeof(*out));
  memcpy(out, s, s->struct_size < sizeof(*out) ? s->struct_size : sizeof(*out));
  out->struct_size = sizeof(*out);
}

// Device workspace: Q | K | V | O | LSE | LA blob | CA blob | one metadata buffer per kv-head group
struct HostLayout {
  size_t q, k, v, o, lse, la, ca, md, md_stride, total;
  sift_md_layout sub_lay;
};

static int host_layout(const sift_shape* s, size_t la_bytes, size_t ca_bytes, HostLayout* out) {
  int rc = validate_shape(s);
  if (rc) return rc;
  const int64_t n = shape_n_tokens(s);
  const int hpg = s->n_q_heads / s->n_kv_heads;
  sift_shape sub;
  copy_shape(s, &sub);
  sub.n_layers = 1; sub.n_q_heads = hpg; sub.n_kv_heads = 1;
  if ((rc = compute_layout(&sub, &out->sub_lay))) return rc;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o = up256(o + bytes); return r; };
  out->q = take((size_t)n * s->n_q_heads * s->head_dim * 2);
  out->k = take((size_t)n * s->n_kv_heads * s->head_dim * 2);
  out->v = take((size_t)n * s->n_kv_heads * s->head_dim * 2);
  out->o = take((size_t)n * s->n_q_heads * s->head_dim * 2);
  out->lse = take((size_t)n * s->n_q_heads * 4);
  out->la = take(la_bytes + 16);
  out->ca = take(ca_bytes + 16);
  out->md_stride = up256(out->sub_lay.total_bytes);
  out->md = take(out->md_stride * s->n_kv_heads);
  out->total = o;
  return SIFT_OK;
}

}  // namespace sift

using namespace sift;

#define SIFT_CUDA_TRY(expr, what)                                                                     \
  do {                                                                                                \
    cudaError_t e_ = (expr);                                                                          \
    if (e_ != cudaSuccess) return set_error(SIFT_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e_));  \
  } while (0)

extern "C" int sift_host_ctx_destroy(sift_host_ctx* ctx);

static int ctx_init(HostCtx* c) {
  SIFT_CUDA_TRY(cudaGetDevice(&c->device), "cudaGetDevice");
  SIFT_CUDA_TRY(cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking), "cudaStreamCreate");
  SIFT_CUDA_TRY(cudaStreamCreateWithFlags(&c->s_cmp, cudaStreamNonBlocking), "cudaStreamCreate");
  SIFT_CUDA_TRY(cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking), "cudaStreamCreate");
  SIFT_CUDA_TRY(cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming), "cudaEventCreate");
  SIFT_CUDA_TRY(cudaEventCreateWithFlags(&c->ev_done, cudaEventDisableTiming), "cudaEventCreate");
  return SIFT_OK;
}

extern "C" int sift_host_ctx_create(sift_host_ctx** out) {
  if (!out) return set_error(SIFT_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  HostCtx* c = new HostCtx();
  const int rc = ctx_init(c);
  if (rc) {   // whatever was created before the failure goes with the ctx
    sift_host_ctx_destroy(reinterpret_cast<sift_host_ctx*>(c));
    return rc;
  }
  *out = reinterpret_cast<sift_host_ctx*>(c);
  return SIFT_OK;
}

extern "C" int sift_host_ctx_destroy(sift_host_ctx* ctx) {
  if (!ctx) return SIFT_OK;
  HostCtx* c = reinterpret_cast<HostCtx*>(ctx);
  for (int i = 0; i < c->n_events; ++i) { cudaEventDestroy(c->ev_in[i]); cudaEventDestroy(c->ev_cmp[i]); }
  if (c->ev_start) cudaEventDestroy(c->ev_start);
  if (c->ev_done) cudaEventDestroy(c->ev_done);
  if (c->s_in) cudaStreamDestroy(c->s_in);
  if (c->s_cmp) cudaStreamDestroy(c->s_cmp);
  if (c->s_out) cudaStreamDestroy(c->s_out);
  delete c;
  return SIFT_OK;
}

extern "C" int sift_prefill_layer_host_workspace_size(const sift_shape* shape, size_t la_blob_bytes,
                                                      size_t ca_blob_bytes, size_t* bytes) {
  if (!bytes) return set_error(SIFT_ERR_INVALID_ARG, "bytes is NULL");
  HostLayout hl;
  int rc = host_layout(shape, la_blob_bytes, ca_blob_bytes, &hl);
  if (rc) return rc;
  *bytes = hl.total;
  return SIFT_OK;
}

extern "C" int sift_prefill_layer_host(sift_host_ctx* ctx, const sift_shape* shape, int32_t layer,
                                       const uint8_t* la_host, size_t la_blob_bytes, const int64_t* la_doc_off,
                                       const uint8_t* ca_host, size_t ca_blob_bytes, const int64_t* ca_doc_off,
                                       const void* Q_host, const void* K_host, const void* V_host, int64_t q_row_stride,
                                       int64_t k_row_stride, int64_t v_row_stride, void* O_host, int64_t o_row_stride,
                                       float* lse_host, float softmax_scale, void* workspace, size_t workspace_bytes,
                                       void* stream) {
  if (!ctx) return set_error(SIFT_ERR_INVALID_ARG, "ctx is NULL");
  HostCtx* c = reinterpret_cast<HostCtx*>(ctx);
  HostLayout hl;
  int rc = host_layout(shape, la_blob_bytes, ca_blob_bytes, &hl);
  if (rc) return rc;
  const int D = shape->n_docs, Hq = shape->n_q_heads, Hkv = shape->n_kv_heads, HD = shape->head_dim, hpg = Hq / Hkv;
  if (layer < 0 || layer >= shape->n_layers) return set_error(SIFT_ERR_INVALID_ARG, "layer %d out of range", layer);
  if (Hkv > kMaxGroups) return set_error(SIFT_ERR_UNSUPPORTED, "n_kv_heads %d > %d", Hkv, kMaxGroups);
  if (!Q_host || !K_host || !V_host || !O_host || !workspace) return set_error(SIFT_ERR_INVALID_ARG, "NULL pointer");
  if (D > 0 && (!la_host || !ca_host || !la_doc_off || !ca_doc_off)) return set_error(SIFT_ERR_INVALID_ARG, "bit-vector pointer is NULL");
  if (((uintptr_t)workspace & 255) != 0) return set_error(SIFT_ERR_INVALID_ARG, "workspace not 256-byte aligned");
  if (workspace_bytes < hl.total) return set_error(SIFT_ERR_WORKSPACE, "workspace %zu < %zu bytes", workspace_bytes, hl.total);
  if (q_row_stride < (int64_t)Hq * HD || o_row_stride < (int64_t)Hq * HD || k_row_stride < (int64_t)Hkv * HD ||
      v_row_stride < (int64_t)Hkv * HD)
    return set_error(SIFT_ERR_INVALID_ARG, "row stride smaller than heads*head_dim");
  int dev = -1;
  SIFT_CUDA_TRY(cudaGetDevice(&dev), "cudaGetDevice");
  if (dev != c->device) return set_error(SIFT_ERR_INVALID_ARG, "ctx was created on device %d, current device is %d", c->device, dev);
  while (c->n_events < Hkv) {
    SIFT_CUDA_TRY(cudaEventCreateWithFlags(&c->ev_in[c->n_events], cudaEventDisableTiming), "cudaEventCreate");
    SIFT_CUDA_TRY(cudaEventCreateWithFlags(&c->ev_cmp[c->n_events], cudaEventDisableTiming), "cudaEventCreate");
    ++c->n_events;
  }
  // byte sizes of one (layer, head) vector of each document, and the per-group blob offsets
  int64_t la_vec[SIFT_MAX_DOCS], ca_vec[SIFT_MAX_DOCS], lo[SIFT_MAX_DOCS], co[SIFT_MAX_DOCS];
  for (int d = 0; d < D; ++d) {
    const int64_t len = shape->doc_offsets[d + 1] - shape->doc_offsets[d];
    const int64_t p = (len + shape->tile - 1) / shape->tile, nb = (len + shape->cross_gran - 1) / shape->cross_gran;
    la_vec[d] = (p * (p + 1) / 2 + 7) / 8;
    ca_vec[d] = (nb + 7) / 8;
    if (la_doc_off[d] < 0 || ca_doc_off[d] < 0 ||
        (uint64_t)la_doc_off[d] + (uint64_t)shape->n_layers * Hq * la_vec[d] > la_blob_bytes ||
        (uint64_t)ca_doc_off[d] + (uint64_t)shape->n_layers * Hq * ca_vec[d] > ca_blob_bytes)
      return set_error(SIFT_ERR_INVALID_ARG, "blob of document %d lies outside the given la/ca bytes", d);
  }
  char* ws = static_cast<char*>(workspace);
  char *qd = ws + hl.q, *kd = ws + hl.k, *vd = ws + hl.v, *od = ws + hl.o;
  float* lsed = reinterpret_cast<float*>(ws + hl.lse);
  uint8_t *lad = reinterpret_cast<uint8_t*>(ws + hl.la), *cad = reinterpret_cast<uint8_t*>(ws + hl.ca);
  const int64_t n = shape_n_tokens(shape);
  const size_t d2 = (size_t)HD * 2, qp = (size_t)Hq * d2, kp = (size_t)Hkv * d2;   // device row pitches (dense)
  cudaStream_t user = (cudaStream_t)stream;

  // everything below is ordered after the caller's stream, and the caller's stream waits for all of it -- also when a
  // step fails half way: what was enqueued before the failure still reads the host buffers and writes the workspace,
  // so the caller's stream is made to wait for the three streams before the error is returned
  auto enqueue = [&]() -> int {
  SIFT_CUDA_TRY(cudaEventRecord(c->ev_start, user), "cudaEventRecord");
  SIFT_CUDA_TRY(cudaStreamWaitEvent(c->s_in, c->ev_start, 0), "cudaStreamWaitEvent");
  SIFT_CUDA_TRY(cudaStreamWaitEvent(c->s_cmp, c->ev_start, 0), "cudaStreamWaitEvent");
  SIFT_CUDA_TRY(cudaStreamWaitEvent(c->s_out, c->ev_start, 0), "cudaStreamWaitEvent");
  if (la_blob_bytes) SIFT_CUDA_TRY(cudaMemcpyAsync(lad, la_host, la_blob_bytes, cudaMemcpyHostToDevice, c->s_in), "H2D la");
  if (ca_blob_bytes) SIFT_CUDA_TRY(cudaMemcpyAsync(cad, ca_host, ca_blob_bytes, cudaMemcpyHostToDevice, c->s_in), "H2D ca");
  // K and V (1/4 of the input bytes under 4:1 GQA) go up front as whole-row copies: per-group column slices of
  // 256 B per row make poor DMA descriptors; Q and O are copied per group
  SIFT_CUDA_TRY(cudaMemcpy2DAsync(kd, kp, K_host, (size_t)k_row_stride * 2, kp, n, cudaMemcpyHostToDevice, c->s_in), "H2D K");
  SIFT_CUDA_TRY(cudaMemcpy2DAsync(vd, kp, V_host, (size_t)v_row_stride * 2, kp, n, cudaMemcpyHostToDevice, c->s_in), "H2D V");
  sift_shape sub;
  copy_shape(shape, &sub);
  sub.n_layers = 1; sub.n_q_heads = hpg; sub.n_kv_heads = 1;
  for (int g = 0; g < Hkv; ++g) {
    const int h0 = g * hpg;
    SIFT_CUDA_TRY(cudaMemcpy2DAsync(qd + h0 * d2, qp, static_cast<const char*>(Q_host) + h0 * d2, (size_t)q_row_stride * 2,
                                    hpg * d2, n, cudaMemcpyHostToDevice, c->s_in), "H2D Q");
    SIFT_CUDA_TRY(cudaEventRecord(c->ev_in[g], c->s_in), "cudaEventRecord");
    SIFT_CUDA_TRY(cudaStreamWaitEvent(c->s_cmp, c->ev_in[g], 0), "cudaStreamWaitEvent");
    // the q-heads of this group inside each document's [layer][q_head][bytes] blob
    for (int d = 0; d < D; ++d) {
      lo[d] = la_doc_off[d] + ((int64_t)layer * Hq + h0) * la_vec[d];
      co[d] = ca_doc_off[d] + ((int64_t)layer * Hq + h0) * ca_vec[d];
    }
    void* md = ws + hl.md + (size_t)g * hl.md_stride;
    if ((rc = sift_decode_metadata(&sub, lad, lo, cad, co, md, hl.md_stride, c->s_cmp))) return rc;
    if ((rc = sift_prefill_attention(&sub, 0, qd + h0 * d2, kd + g * d2, vd + g * d2, (int64_t)Hq * HD, (int64_t)Hkv * HD,
                                     (int64_t)Hkv * HD, md, od + h0 * d2, (int64_t)Hq * HD, lsed + (int64_t)h0 * n,
                                     softmax_scale, c->s_cmp)))
      return rc;
    SIFT_CUDA_TRY(cudaEventRecord(c->ev_cmp[g], c->s_cmp), "cudaEventRecord");
    SIFT_CUDA_TRY(cudaStreamWaitEvent(c->s_out, c->ev_cmp[g], 0), "cudaStreamWaitEvent");
    SIFT_CUDA_TRY(cudaMemcpy2DAsync(static_cast<char*>(O_host) + h0 * d2, (size_t)o_row_stride * 2, od + h0 * d2, qp, hpg * d2, n,
                                    cudaMemcpyDeviceToHost, c->s_out), "D2H O");
    if (lse_host)
      SIFT_CUDA_TRY(cudaMemcpyAsync(lse_host + (int64_t)h0 * n, lsed + (int64_t)h0 * n, (size_t)hpg * n * 4,
                                    cudaMemcpyDeviceToHost, c->s_out), "D2H lse");
  }
  SIFT_CUDA_TRY(cudaEventRecord(c->ev_done, c->s_out), "cudaEventRecord");
  SIFT_CUDA_TRY(cudaStreamWaitEvent(user, c->ev_done, 0), "cudaStreamWaitEvent");
  return SIFT_OK;
  };
  rc = enqueue();
  if (rc) {
    // best effort, return codes ignored: the error being reported is the first one (g_err keeps its text)
    cudaEventRecord(c->ev_in[0], c->s_in);
    cudaStreamWaitEvent(c->s_out, c->ev_in[0], 0);
    cudaEventRecord(c->ev_cmp[0], c->s_cmp);
    cudaStreamWaitEvent(c->s_out, c->ev_cmp[0], 0);
    cudaEventRecord(c->ev_done, c->s_out);
    cudaStreamWaitEvent(user, c->ev_done, 0);
  }
  return rc;
}
