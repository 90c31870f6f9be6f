/* sift.h -- C ABI of the B200-native SIFT hot path (arxiv/paper_2606_09441).
 *
 * Two operations, as the paper's implementation section states them:
 *   sift_decode_metadata    PAPER.md:L237-247 (sec 5.1)  bit vectors -> packed int32 index lists
 *   sift_prefill_attention  PAPER.md:L249-255 (sec 5.2)  block-sparse causal prefill attention driven by those lists
 * plus a dense causal comparator from the same build ("Full Recompute").
 *
 * Conventions
 *   - "dev" pointers are device memory owned by the caller; "HOST" pointers are host memory read during the
 *     call and not retained.  The library never allocates or frees device memory, never synchronises the
 *     stream and never reads device memory on the host.  All work is enqueued on `stream` (a cudaStream_t
 *     passed as void*; NULL = the legacy default stream).
 *   - Every call returns 0 (SIFT_OK) or a negative sift_status; on error nothing is enqueued.
 *     sift_last_error() returns a thread-local, NUL-terminated description of the last failure.
 *   - Prompt layout (Fig 6): n_docs documents concatenated, then the user query.
 *     doc_offsets[0] = 0 < doc_offsets[1] < ... < doc_offsets[n_docs]; N = doc_offsets[n_docs] + query_len rows.
 *   - Tiles are document-relative (reading A2): tile (d,i) covers rows doc_offsets[d] + i*tile ...;
 *     the user query is segment n_docs.  Global tile id = tile_base[d] + i.
 *   - Bit vectors: per (layer, q_head, document).  LA: lower triangle of the P x P tile
 *     grid, row-major (0,0),(1,0),(1,1),(2,0).., MSB-first, ceil(P(P+1)/16) bytes, P = ceil(len/tile).
 *     CA: one bit per group of `cross_gran` key tokens, MSB-first, ceil(ceil(len/cross_gran)/8) bytes.
 *     Bits after the last valid bit of a vector are ignored.  One blob per document laid out
 *     [layer][q_head][bytes]; la_doc_off[p] / ca_doc_off[p] = byte offset (from la_base / ca_base) of the blob
 *     of the document at prompt position p.  The allocations must extend at least 4 bytes past the last vector
 *     (the decoder reads aligned 32-bit words).
 *   - GQA: q-head h uses kv-head h / (n_q_heads / n_kv_heads).
 */
#ifndef SIFT_H_
#define SIFT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SIFT_MAX_DOCS 512

typedef enum {
  SIFT_OK = 0,
  SIFT_ERR_INVALID_ARG = -1, /* NULL pointer, non-increasing offsets, misaligned tensor, ... */
  SIFT_ERR_UNSUPPORTED = -2, /* head_dim not in {64,128}, tile not in {64,128}, cross_gran not in {1,tile}, n_docs > SIFT_MAX_DOCS */
  SIFT_ERR_WORKSPACE = -3,   /* metadata buffer too small */
  SIFT_ERR_CUDA = -4         /* launch / driver error */
} sift_status;

typedef struct {
  uint32_t struct_size; /* = sizeof(sift_shape) */
  int32_t n_layers, n_q_heads, n_kv_heads, head_dim;
  int32_t n_docs, query_len;
  int32_t tile;       /* T: 64 or 128 (M-block = N-block = T).  128 is the tuned size; 64 is
                         functional: a 64-row query tile still occupies a 128-lane accumulator and a 64-key local tile
                         a 128-key MMA step, so at most half of the tensor work is useful */
  int32_t cross_gran; /* G: 1 = one CA bit per key token (BASELINE.json configs); tile = one bit per page */
  const int32_t* doc_offsets; /* HOST, n_docs + 1 entries */
  /* ---- several prompts in one call (optional; struct_size = SIFT_SHAPE_SIZE_V1 or n_prompts <= 1: one prompt) ----
   * PAPER.md:L67 (TTFT gates decode batching), L267 (the paper itself measures one request at a time).
   * The prompts are packed back to back on the token axis: prompt p = documents [prompt_doc_start[p],
   * prompt_doc_start[p+1]) in order, then its query of prompt_query_len[p] rows; a row attends keys of its own prompt
   * only.  doc_offsets stays the running sum of the DOCUMENT lengths over all n_docs documents (queries not counted);
   * query_len is ignored; N = doc_offsets[n_docs] + sum of prompt_query_len.  A prompt may have no documents.
   * n_docs + n_prompts <= SIFT_MAX_DOCS + 1.  la_doc_off / ca_doc_off are indexed by the document's index. */
  int32_t n_prompts;
  const int32_t* prompt_doc_start; /* HOST, n_prompts + 1 entries, [0] = 0, [n_prompts] = n_docs, non-decreasing */
  const int32_t* prompt_query_len; /* HOST, n_prompts entries, >= 0 */
} sift_shape;
#define SIFT_SHAPE_SIZE_V1 ((uint32_t)offsetof(sift_shape, n_prompts)) /* the struct before the prompt fields */

/* Byte offsets (from the start of the metadata buffer) of the arrays of container "MD-v1".
 * All arrays are int32.  Canonical arrays (compared bit-exactly with the oracle):
 *   tile_base [n_docs+2]           first global tile id of each segment; tile_base[n_docs+1] = NT
 *   tile_seg/tile_row0/tile_rows [NT]
 *   cross_ptr [L][Hq][n_docs+1]    cross_ptr[d] = number of marked keys in documents 0..d-1
 *   cross_idx [L][Hq][cross_cap]   ascending global key rows (G = 1) or global tile ids (G = tile); rows of
 *                                  document d attend entries [0, cross_ptr[d])
 *   local_cnt [L][Hq][NT], local_ptr [L][Hq][NT+1], local_idx [L][Hq][local_cap]
 *                                  per M-block: ascending global tile ids of marked LA tiles; query M-block t: 0..t
 * Several prompts ("MD-v1b"): segments (documents and queries) and documents are numbered in token order,
 * tile_base has n_docs + n_prompts + 1 entries; the cross list of every prompt starts at a multiple of 128, so
 * cross_ptr[d] is a running count that is rounded up at each prompt's first document, and document d of a prompt
 * whose first document is d0 attends entries [cross_ptr[d0], cross_ptr[d]); query tile t of a prompt whose first tile
 * is f lists f..t.  One prompt: exactly the arrays above.
 * Private arrays: seg_info [n_seg][4], sched [L][n_items], counters [L][2], sort keys [L][n_items]. */
typedef struct {
  uint32_t struct_size;
  int32_t n_tiles;   /* NT */
  int32_t cross_cap; /* per (layer, head) stride of cross_idx: sum_d ceil(len_d / G) rounded up to 128 */
  int32_t local_cap; /* per (layer, head) stride of local_idx */
  int32_t n_mblocks; /* scheduler M-blocks per head */
  int32_t n_items;   /* work items per layer = n_q_heads * n_mblocks */
  size_t tile_base, tile_seg, tile_row0, tile_rows;
  size_t cross_ptr, cross_idx, local_cnt, local_ptr, local_idx;
  size_t mblock_tile0, sched, counters;
  size_t total_bytes;
  int32_t n_seg;     /* segments: n_docs + max(n_prompts, 1) */
  int32_t n_tokens;  /* N */
  size_t seg_info;   /* private: per segment {document index or -1, first document of its prompt, first row of its prompt, first tile of its prompt} */
} sift_md_layout;
/* The struct before n_seg / n_tokens / seg_info were added.  A caller that passes a shape of SIFT_SHAPE_SIZE_V1 bytes
 * was built against that older header and owns a sift_md_layout of this size: sift_metadata_layout then writes
 * exactly SIFT_MD_LAYOUT_SIZE_V1 bytes (struct_size says so) and nothing behind them.  The offsets and total_bytes
 * are the same either way; total_bytes already covers the private arrays. */
#define SIFT_MD_LAYOUT_SIZE_V1 ((uint32_t)offsetof(sift_md_layout, n_seg))

const char* sift_version(void);
const char* sift_last_error(void);

/* Size / layout of the metadata buffer for a shape.  Pure host arithmetic.  sift_metadata_layout writes
 * sizeof(sift_md_layout) bytes to `out`, or SIFT_MD_LAYOUT_SIZE_V1 bytes when shape->struct_size is SIFT_SHAPE_SIZE_V1
 * (see above); out->struct_size holds the number of bytes written. */
int sift_metadata_size(const sift_shape* shape, size_t* bytes);
int sift_metadata_layout(const sift_shape* shape, sift_md_layout* out);

/* PAPER.md:L237-247.  Pass 1 counts marked bits per (layer, head, M-block / document), an exclusive scan turns
 * counts into offsets, pass 2 compacts the set bits into index lists in global coordinates.  All layers and heads
 * in one call.  metadata: dev, 16-byte aligned, >= sift_metadata_size() bytes, fully overwritten. */
int sift_decode_metadata(const sift_shape* shape,
                         const uint8_t* la_base /*dev*/, const int64_t* la_doc_off /*HOST, n_docs*/,
                         const uint8_t* ca_base /*dev*/, const int64_t* ca_doc_off /*HOST, n_docs*/,
                         void* metadata /*dev, out*/, size_t metadata_bytes, void* stream);

/* PAPER.md:L249-255.  One layer per call.  Q [N][n_q_heads][head_dim], K,V [N][n_kv_heads][head_dim], bf16, dev;
 * row strides in elements (head stride = head_dim); bases and row strides 16-byte aligned.
 * O [N][n_q_heads][head_dim] bf16 dev (out); lse [n_q_heads][N] fp32 dev (out, may be NULL): natural-log
 * log-sum-exp of the scaled logits.  A row with no allowed key gets O = 0, lse = -inf.
 * softmax_scale <= 0 selects 1/sqrt(head_dim).  fp32 accumulation; P is rounded to bf16 before P*V.
 * Calls that use the same (metadata, layer) must be stream-ordered (they share a work counter). */
int sift_prefill_attention(const sift_shape* shape, int32_t layer,
                           const void* Q, const void* K, const void* V,
                           int64_t q_row_stride, int64_t k_row_stride, int64_t v_row_stride,
                           const void* metadata /*dev, from sift_decode_metadata*/,
                           void* O, int64_t o_row_stride, float* lse, float softmax_scale, void* stream);

/* Chunked prefill (sec 2: time to first token gates decode batching, so a serving engine runs a long
 * prompt in chunks between decode steps).  Rows [row_begin, row_end) of the packed token axis only:
 * the same metadata, the same kernel and the same schedule as sift_prefill_attention, with M-blocks that have no row
 * in the range skipped and tiles / rows outside it neither computed nor written.  O and lse are the full-size arrays
 * of sift_prefill_attention (same base pointers and strides); rows outside the range keep what they held.  Every row
 * in the range is bit-identical to what sift_prefill_attention writes for it (a row's steps and their order do not
 * depend on which other rows run).
 *   0 <= row_begin <= row_end <= N; an empty range launches nothing.  The range may cut tiles and documents anywhere;
 *   whole tiles (multiples of `tile` inside a segment) waste no work.
 *   K and V rows [0, E) must exist, E = min(N, e + 127), e = one past the last row of the last tile that intersects
 *   the range: the copy engine fetches 128-row boxes (a document tile's box starts at the tile, a query tile's boxes
 *   at multiples of 128 from its prompt's first row), so the last box reaches past a ragged tile end and past row_end.
 *   Keys at or after a row's own position are masked, but V rows of a fetched box enter the MMAs with weight 0, so V
 *   rows [row_end, E) must be finite (zeros will do; K and Q rows there may hold anything).  Rows >= E are never read.
 * Same ordering rule: calls on one (metadata, layer) are stream-ordered, whole-prompt and ranged ones alike. */
int sift_prefill_attention_rows(const sift_shape* shape, int32_t layer, int32_t row_begin, int32_t row_end,
                                const void* Q, const void* K, const void* V,
                                int64_t q_row_stride, int64_t k_row_stride, int64_t v_row_stride,
                                const void* metadata /*dev*/, void* O, int64_t o_row_stride, float* lse,
                                float softmax_scale, void* stream);

/* FP8 variant (sec 2.6 points at FP8 prefill; reading R7).  Q8 [N][n_q_heads][128], K8, V8
 * [N][n_kv_heads][128]: OCP e4m3 bytes, dev, row strides in elements (= bytes), bases and strides 16-byte aligned;
 * q_scale HOST [n_q_heads], k_scale / v_scale HOST [n_kv_heads], all > 0.  The result is sift_prefill_attention of the
 * dequantised values q_scale[h] * Q8, k_scale[g] * K8, v_scale[g] * V8 (O bf16, lse fp32 as there), computed with
 * kind::f8f6f4 tensor-core MMAs: the logits are exact products accumulated in fp32, P is rounded to e4m3 before P*V
 * (tolerance in DESIGN.md).  head_dim 128 only (SIFT_ERR_UNSUPPORTED otherwise).  Same metadata, same ordering rule. */
int sift_prefill_attention_fp8(const sift_shape* shape, int32_t layer,
                               const void* Q8, const void* K8, const void* V8,
                               int64_t q_row_stride, int64_t k_row_stride, int64_t v_row_stride,
                               const float* q_scale /*HOST*/, const float* k_scale /*HOST*/, const float* v_scale /*HOST*/,
                               const void* metadata /*dev*/, void* O, int64_t o_row_stride, float* lse,
                               float softmax_scale, void* stream);

/* Dense causal attention over n_tokens rows with the same kernel body (no metadata).  Calls may be in flight on
 * different streams at the same time: each call draws its own work counter (cleared on `stream` before the launch). */
int sift_dense_causal_attention(int32_t n_tokens, int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim,
                                const void* Q, const void* K, const void* V,
                                int64_t q_row_stride, int64_t k_row_stride, int64_t v_row_stride,
                                void* O, int64_t o_row_stride, float* lse, float softmax_scale, void* stream);

/* ---- one prefill layer from HOST buffers (sec 4.4: the bit vectors arrive from CPU DRAM with the
 * retrieved documents; L331 sec 7.4: one H2D copy of the vectors) ----
 * sift_prefill_layer_host takes the bit-vector blobs, Q, K, V from HOST memory and leaves O (and optionally the row
 * log-sum-exp) in HOST memory.  The layer is processed per kv-head group (a kv head with its q-heads is an independent
 * unit of the path): the H2D copy of a group's Q columns, its metadata decode + attention, and the D2H copy of its O
 * columns run on three internal streams, so both PCIe directions overlap the kernels and each other.  The results
 * are bit-identical to sift_decode_metadata + sift_prefill_attention over all heads at once.
 *   ctx        from sift_host_ctx_create on the current device: 3 non-blocking streams + events, NO device memory;
 *              one call at a time per ctx; destroy with sift_host_ctx_destroy (after the work has completed).
 *   la_host / ca_host  HOST blobs ([layer][q_head][bytes] per document, all n_layers present) of la_blob_bytes /
 *              ca_blob_bytes bytes; la_doc_off / ca_doc_off HOST, as in sift_decode_metadata.
 *   Q_host [N][n_q_heads][head_dim], K_host, V_host [N][n_kv_heads][head_dim], O_host [N][n_q_heads][head_dim] bf16
 *              HOST (pinned memory for the copies to be asynchronous), row strides in elements; lse_host
 *              [n_q_heads][N] fp32 HOST or NULL.
 *   workspace  dev, 256-byte aligned, >= sift_prefill_layer_host_workspace_size() bytes (device copies of the inputs,
 *              O, LSE and one metadata buffer per kv-head group); owned by the caller.
 * Ordering: all work is ordered after the work already enqueued on `stream`, and `stream` waits for all of it: after
 * cudaStreamSynchronize(stream) O_host is complete.  The call itself never synchronises.  Host buffers must stay
 * valid and unmodified until then.  Errors as everywhere (nothing useful is enqueued after a failure). */
typedef struct sift_host_ctx sift_host_ctx;
int sift_host_ctx_create(sift_host_ctx** out);
int sift_host_ctx_destroy(sift_host_ctx* ctx);
int sift_prefill_layer_host_workspace_size(const sift_shape* shape, size_t la_blob_bytes, size_t ca_blob_bytes,
                                           size_t* bytes);
int sift_prefill_layer_host(sift_host_ctx* ctx, const sift_shape* shape, int32_t layer,
                            const uint8_t* la_host, size_t la_blob_bytes, const int64_t* la_doc_off /*HOST*/,
                            const uint8_t* ca_host, size_t ca_blob_bytes, const int64_t* ca_doc_off /*HOST*/,
                            const void* Q_host, const void* K_host, const void* V_host,
                            int64_t q_row_stride, int64_t k_row_stride, int64_t v_row_stride,
                            void* O_host, int64_t o_row_stride, float* lse_host /*nullable*/, float softmax_scale,
                            void* workspace /*dev*/, size_t workspace_bytes, void* stream);

/* ---- offline metadata generation (sec 4.1, L209 sec 4.2, L223 sec 4.4) ----
 * Produces the LA / CA bit vectors of ONE document for the q-heads of one layer from the document's standalone dense
 * causal attention ("SIFT is created offline by performing dense prefill on each RAG document").
 *   LA bit (i, j) = 1 iff tile (i, j) of the document holds at least one probability >= alpha      (L201)
 *   CA bit g      = 1 iff (cells of key group g with probability >= beta) > gamma * (causal cells of key group g);
 *                   a key group is one key token (cross_gran = 1; "Key tokens with >10% concentration
 *                   of high scores") or a page of `tile` keys (cross_gran = tile; L209).  DESIGN.md reading R6.
 * Q [doc_len][n_q_heads][head_dim], K [doc_len][n_kv_heads][head_dim] bf16 dev (the document's rows only), row
 * strides in elements; lse [n_q_heads][doc_len] fp32 dev = the natural-log row log-sum-exp of the document's dense
 * causal attention with the same softmax_scale, e.g. from sift_dense_causal_attention on the same Q, K.
 * la_out [n_q_heads][ceil(P(P+1)/16)], ca_out [n_q_heads][ceil(ceil(doc_len/cross_gran)/8)] dev, MSB-first, padding
 * bits 0: the [q_head][bytes] slice of a document's blob for one layer.  workspace: dev, 16-byte aligned,
 * >= sift_encode_workspace_size() bytes (per-key counters and per-tile flags; cleared by the call). */
int sift_encode_workspace_size(int32_t doc_len, int32_t n_q_heads, int32_t tile, size_t* bytes);
/* bytes of ONE q-head's LA / CA vector of a document: ceil(P(P+1)/16), ceil(ceil(doc_len/cross_gran)/8) */
int sift_encode_output_sizes(int32_t doc_len, int32_t tile, int32_t cross_gran, size_t* la_bytes, size_t* ca_bytes);
int sift_encode_document(int32_t doc_len, int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, int32_t tile,
                         int32_t cross_gran, const void* Q, const void* K, int64_t q_row_stride, int64_t k_row_stride,
                         const float* lse, float alpha, float beta, float gamma, float softmax_scale,
                         uint8_t* la_out, uint8_t* ca_out, void* workspace, size_t workspace_bytes, void* stream);

/* ---- sift_encode_document for callers that cannot allocate device memory ----
 * sift_encode_document needs a scratch workspace, and a caller has to get that from somewhere.  Some cannot: a plug-in
 * or custom op that is handed its input and output buffers by a host framework and has no handle on that framework's
 * allocator; a serving process that gave all free HBM to its KV-cache pool at start-up, where a cudaMalloc may fail
 * and, if it succeeds, stalls every stream of the device while it runs.  sift_encode_document_static is the same
 * operation (same arguments minus the workspace, same kernels, bit-identical la_out / ca_out) with the scratch in a
 * fixed array that is part of the library's device image: SIFT_ENCODE_STATIC_SCRATCH_BYTES on every GPU the library
 * is used on, held from the moment the CUDA runtime loads the library's kernels on that GPU until the process exits.
 * The call itself makes no cudaMalloc / cudaFree and uses no routine that allocates.
 *   Limit     sift_encode_workspace_size(doc_len, n_q_heads, tile) <= SIFT_ENCODE_STATIC_SCRATCH_BYTES (4 MiB), i.e.
 *             n_q_heads * (doc_len rounded up to 128 + P(P+1)/2) * 4 bytes with P = ceil(doc_len / tile): 32 q-heads of a
 *             12,288-token document at tile 64, of a 16,384-token one at tile 128 (the paper's documents are <= 4096
 *             tokens).  Anything larger returns SIFT_ERR_WORKSPACE with the two sizes in sift_last_error() and enqueues
 *             nothing; encode fewer heads per call (Q, lse, la_out, ca_out are per-head slices) or use the workspace
 *             variant.
 *   Set-up    the first call on each device looks up the array's address on that device (cudaGetSymbolAddress, which
 *             may also make the runtime load the library's device code there) and keeps it; make that first call with
 *             the device current as for every other call, and make it before any stream capture is begun.  Later calls
 *             on that device do no set-up.  Thread-safe.
 *   Sharing   there is ONE array per GPU and every call on that GPU uses it.  A call first clears the part it needs,
 *             on `stream` (what the previous call left there is never read), so calls issued to one stream, or otherwise
 *             ordered one after the other, are independent.  Two calls that may run on the GPU at the same time (different
 *             streams without an event between them, two host threads, two libraries' worth of users in one process)
 *             race on the array and produce wrong bits without any error: order them, or give all but one of them a
 *             workspace through sift_encode_document.
 * Everything else (arguments, outputs, errors, stream semantics) is as in sift_encode_document. */
#define SIFT_ENCODE_STATIC_SCRATCH_BYTES (4u << 20)
size_t sift_encode_static_scratch_bytes(void); /* the value the library was built with */
int sift_encode_document_static(int32_t doc_len, int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, int32_t tile,
                                int32_t cross_gran, const void* Q, const void* K, int64_t q_row_stride, int64_t k_row_stride,
                                const float* lse, float alpha, float beta, float gamma, float softmax_scale,
                                uint8_t* la_out, uint8_t* ca_out, void* stream);

/* ---- the paper's own index layout (sec 5.1) ----
 * sparse_n_indices as the paper stores it: per (head, M-block t) ONE packed int32 list, the CA entries of all earlier
 * documents of the prompt first (key rows at G = 1, global tile ids at G = tile), then the M-block's LA entries (global
 * tile ids); a query M-block lists its causal N-blocks.  MD-v1 keeps the CA entries of a head once; these two calls
 * rebuild the replicated layout from a decoded metadata buffer, for one layer, on `stream`:
 *   sift_paper_index_offsets   ptr (dev, out) [n_q_heads][NT + 1] int64: ptr[h][t] = entries of the M-blocks before t,
 *                              ptr[h][NT] = entries of head h (read it back to size idx).
 *   sift_export_paper_indices  idx (dev, out) [n_q_heads][head_stride] int32: the list of (h, t) at
 *                              idx[h * head_stride + ptr[h][t] ..]; entries at or beyond head_stride are not written.
 * NT = sift_md_layout.n_tiles (an M-block here is one query tile of `tile` rows). */
int sift_paper_index_offsets(const sift_shape* shape, int32_t layer, const void* metadata /*dev*/, int64_t* ptr /*dev*/,
                             void* stream);
int sift_export_paper_indices(const sift_shape* shape, int32_t layer, const void* metadata /*dev*/,
                              const int64_t* ptr /*dev*/, int32_t* idx /*dev*/, int64_t head_stride, void* stream);

/* Number of kernels the library has launched in this process (bench.py's gpu_launches). */
int64_t sift_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* SIFT_H_ */
