/* Plain-C client of include/sift.h (no Python, no torch): proves the boundary is a C ABI.
 *   abi_smoke host   -> host-only calls: version, layout arithmetic, error codes        (runs without a GPU)
 *   abi_smoke gpu    -> decode + dense/sparse attention on a small prompt through cudaMalloc'd buffers, the same layer
 *                       from host buffers, two prompts in one call, the paper's index layout
 * Expected values are closed forms: all-ones bit vectors => counts are sizes; Q = 0 => uniform attention, so every
 * output row is the running mean of the V rows it may see, and LSE = ln(#keys). */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "sift.h"

#define CHECK(c) do { if (!(c)) { fprintf(stderr, "FAILED %s:%d: %s (last error: %s)\n", __FILE__, __LINE__, #c, sift_last_error()); return 1; } } while (0)

/* minimal CUDA runtime prototypes (the test links libcudart but needs no CUDA headers) */
extern int cudaMalloc(void** p, size_t n);
extern int cudaMemcpy(void* dst, const void* src, size_t n, int kind);
extern int cudaMemset(void* p, int v, size_t n);
extern int cudaDeviceSynchronize(void);
extern int cudaFree(void* p);
extern int cudaMallocHost(void** p, size_t n);
extern int cudaFreeHost(void* p);
extern int cudaStreamCreate(void** s);
extern int cudaStreamSynchronize(void* s);
extern int cudaStreamDestroy(void* s);

static uint16_t f2bf(float f) { uint32_t u; memcpy(&u, &f, 4); u += 0x7fffu + ((u >> 16) & 1u); return (uint16_t)(u >> 16); }
static float bf2f(uint16_t h) { uint32_t u = (uint32_t)h << 16; float f; memcpy(&f, &u, 4); return f; }

static int host_part(void) {
  int32_t off[3] = {0, 300, 500};
  sift_shape s = {sizeof(sift_shape), 2, 4, 2, 128, 2, 70, 128, 1, off};
  sift_md_layout lay;
  size_t nb = 0;
  CHECK(strstr(sift_version(), "sift-b200") != NULL);
  CHECK(sift_metadata_layout(&s, &lay) == SIFT_OK);
  CHECK(sift_metadata_size(&s, &nb) == SIFT_OK && nb == lay.total_bytes);
  CHECK(lay.n_tiles == 3 + 2 + 1);                       /* ceil(300/128) + ceil(200/128) + ceil(70/128) */
  CHECK(lay.cross_cap == 512);                           /* 500 key bits rounded up to 128 */
  CHECK(lay.local_cap == 6 + 3 + 6);                     /* 3*4/2 + 2*3/2 + (query tile with global id 5: 6 entries) */
  s.head_dim = 96;
  CHECK(sift_metadata_size(&s, &nb) == SIFT_ERR_UNSUPPORTED && strlen(sift_last_error()) > 0);
  s.head_dim = 128; off[2] = 300;
  CHECK(sift_metadata_size(&s, &nb) == SIFT_ERR_INVALID_ARG);
  CHECK(sift_metadata_size(NULL, &nb) == SIFT_ERR_INVALID_ARG);
  CHECK(sift_encode_workspace_size(300, 4, 128, &nb) == SIFT_OK && nb == 4u * (384u + 6u) * 4u);
  size_t lb = 0, cb = 0;
  CHECK(sift_encode_output_sizes(1024, 128, 128, &lb, &cb) == SIFT_OK && lb == 5 && cb == 1);   /* P = 8 -> 36 / 8 bits */
  CHECK(sift_encode_output_sizes(300, 128, 1, &lb, &cb) == SIFT_OK && lb == 1 && cb == 38);
  off[2] = 500;
  CHECK(sift_prefill_layer_host_workspace_size(&s, 100, 100, &nb) == SIFT_OK && nb > 2u * 570u * 4u * 128u * 2u);
  CHECK(sift_prefill_layer_host(NULL, &s, 0, NULL, 0, NULL, NULL, 0, NULL, NULL, NULL, NULL, 0, 0, 0, NULL, 0, NULL, 0.f, NULL, 0, NULL) == SIFT_ERR_INVALID_ARG);
  /* a caller built against the header before the prompt fields: a shape of SIFT_SHAPE_SIZE_V1 bytes (poison behind it)
   * and a sift_md_layout that ends before n_seg; the library reads / writes no further than that */
  {
    unsigned char sbuf[sizeof(sift_shape) + 32], obuf[sizeof(sift_md_layout) + 32];
    sift_md_layout full, v1;
    size_t nb1 = 0;
    CHECK(sift_metadata_layout(&s, &full) == SIFT_OK && full.struct_size == sizeof(sift_md_layout));
    memset(sbuf, 0xCD, sizeof(sbuf)); memset(obuf, 0xAB, sizeof(obuf));
    memcpy(sbuf, &s, SIFT_SHAPE_SIZE_V1);
    ((sift_shape*)sbuf)->struct_size = SIFT_SHAPE_SIZE_V1;
    CHECK(sift_metadata_layout((const sift_shape*)sbuf, (sift_md_layout*)obuf) == SIFT_OK);
    for (size_t i = SIFT_MD_LAYOUT_SIZE_V1; i < sizeof(obuf); ++i) CHECK(obuf[i] == 0xAB);
    memcpy(&v1, obuf, SIFT_MD_LAYOUT_SIZE_V1);
    CHECK(v1.struct_size == SIFT_MD_LAYOUT_SIZE_V1 && v1.total_bytes == full.total_bytes && v1.counters == full.counters &&
          v1.n_items == full.n_items);
    CHECK(sift_metadata_size((const sift_shape*)sbuf, &nb1) == SIFT_OK && nb1 == full.total_bytes);
  }
  printf("abi_smoke host ok\n");
  return 0;
}

static int gpu_part(void) {
  enum { L0 = 200, L1 = 150, LQ = 34, N = L0 + L1 + LQ, HQ = 2, HKV = 1, D = 64, T = 64 };
  int32_t off[3] = {0, L0, L0 + L1};
  sift_shape s = {sizeof(sift_shape), 1, HQ, HKV, D, 2, LQ, T, 1, off};
  sift_md_layout lay;
  CHECK(sift_metadata_layout(&s, &lay) == SIFT_OK);
  /* all-ones vectors: per document [layer][head][bytes]; P = 4 and 3 -> LA 10 / 6 bits -> 2 / 1 bytes; CA 25 / 19 bytes */
  const int la_b[2] = {2, 1}, ca_b[2] = {25, 19};
  uint8_t la[HQ * 3 + 16], ca[HQ * 44 + 16];
  memset(la, 0xff, sizeof(la)); memset(ca, 0xff, sizeof(ca));
  int64_t la_off[2] = {0, HQ * la_b[0]}, ca_off[2] = {0, HQ * ca_b[0]};
  void *d_la, *d_ca, *d_md, *d_q, *d_k, *d_v, *d_o, *d_lse;
  CHECK(cudaMalloc(&d_la, sizeof(la)) == 0 && cudaMalloc(&d_ca, sizeof(ca)) == 0 && cudaMalloc(&d_md, lay.total_bytes) == 0);
  CHECK(cudaMemcpy(d_la, la, sizeof(la), 1) == 0 && cudaMemcpy(d_ca, ca, sizeof(ca), 1) == 0);
  CHECK(sift_decode_metadata(&s, (const uint8_t*)d_la, la_off, (const uint8_t*)d_ca, ca_off, d_md, lay.total_bytes, NULL) == SIFT_OK);
  int32_t* md = (int32_t*)malloc(lay.total_bytes);
  CHECK(cudaDeviceSynchronize() == 0 && cudaMemcpy(md, d_md, lay.total_bytes, 2) == 0);
  const int32_t* cross_ptr = (const int32_t*)((const char*)md + lay.cross_ptr);
  const int32_t* local_ptr = (const int32_t*)((const char*)md + lay.local_ptr);
  const int32_t* cross_idx = (const int32_t*)((const char*)md + lay.cross_idx);
  for (int h = 0; h < HQ; ++h) {
    CHECK(cross_ptr[h * 3 + 0] == 0 && cross_ptr[h * 3 + 1] == L0 && cross_ptr[h * 3 + 2] == L0 + L1);   /* padding bits ignored */
    CHECK(local_ptr[h * (lay.n_tiles + 1) + lay.n_tiles] == 10 + 6 + 8);                                  /* + query tile id 7: 8 entries */
    for (int i = 0; i < L0 + L1; ++i) CHECK(cross_idx[(size_t)h * lay.cross_cap + i] == i);
  }
  /* Q = 0, K arbitrary, V[n][c] = n (exact in bf16 up to 256; use n mod 64): all bits set => dense causal attention */
  uint16_t* hq = (uint16_t*)calloc((size_t)N * HQ * D, 2);
  uint16_t* hk = (uint16_t*)malloc((size_t)N * HKV * D * 2);
  uint16_t* hv = (uint16_t*)malloc((size_t)N * HKV * D * 2);
  for (int n = 0; n < N; ++n) for (int c = 0; c < D; ++c) { hk[n * D + c] = f2bf((float)((n * 7 + c) % 5) - 2.f); hv[n * D + c] = f2bf((float)(n % 64)); }
  size_t qb = (size_t)N * HQ * D * 2, kb = (size_t)N * HKV * D * 2;
  CHECK(cudaMalloc(&d_q, qb) == 0 && cudaMalloc(&d_k, kb) == 0 && cudaMalloc(&d_v, kb) == 0 && cudaMalloc(&d_o, qb) == 0 && cudaMalloc(&d_lse, (size_t)HQ * N * 4) == 0);
  CHECK(cudaMemcpy(d_q, hq, qb, 1) == 0 && cudaMemcpy(d_k, hk, kb, 1) == 0 && cudaMemcpy(d_v, hv, kb, 1) == 0);
  uint16_t* ho = (uint16_t*)malloc(qb);
  uint16_t* ho_sparse = (uint16_t*)malloc(qb);
  float* hl = (float*)malloc((size_t)HQ * N * 4);
  float* hl_sparse = (float*)malloc((size_t)HQ * N * 4);
  for (int pass = 0; pass < 2; ++pass) {
    CHECK(cudaMemset(d_o, 0xff, qb) == 0);
    int rc = pass == 0 ? sift_prefill_attention(&s, 0, d_q, d_k, d_v, HQ * D, HKV * D, HKV * D, d_md, d_o, HQ * D, (float*)d_lse, 0.f, NULL)
                       : sift_dense_causal_attention(N, HQ, HKV, D, d_q, d_k, d_v, HQ * D, HKV * D, HKV * D, d_o, HQ * D, (float*)d_lse, 0.f, NULL);
    CHECK(rc == SIFT_OK);
    CHECK(cudaDeviceSynchronize() == 0 && cudaMemcpy(ho, d_o, qb, 2) == 0 && cudaMemcpy(hl, d_lse, (size_t)HQ * N * 4, 2) == 0);
    if (pass == 0) { memcpy(ho_sparse, ho, qb); memcpy(hl_sparse, hl, (size_t)HQ * N * 4); }
    double sum = 0;
    for (int n = 0; n < N; ++n) {
      sum += (double)(n % 64);
      const double mean = sum / (n + 1);
      for (int h = 0; h < HQ; ++h) {
        CHECK(fabs(bf2f(ho[((size_t)n * HQ + h) * D + 5]) - mean) <= 0.02 * (1.0 + mean));
        CHECK(fabs(hl[(size_t)h * N + n] - log((double)(n + 1))) <= 1e-3);
      }
    }
  }
  CHECK(sift_launch_count() >= 3); /* decode (1 launch when the scheduler is fused) + attention + dense */
  /* the same layer from HOST buffers through sift_prefill_layer_host: host -> host, bit-identical to the single call */
  {
    void *p_la, *p_ca, *p_q, *p_k, *p_v, *p_o, *p_lse, *d_ws, *st;
    size_t wsb = 0;
    sift_host_ctx* ctx = NULL;
    CHECK(cudaMallocHost(&p_la, sizeof(la)) == 0 && cudaMallocHost(&p_ca, sizeof(ca)) == 0 && cudaMallocHost(&p_q, qb) == 0 &&
          cudaMallocHost(&p_k, kb) == 0 && cudaMallocHost(&p_v, kb) == 0 && cudaMallocHost(&p_o, qb) == 0 &&
          cudaMallocHost(&p_lse, (size_t)HQ * N * 4) == 0);
    memcpy(p_la, la, sizeof(la)); memcpy(p_ca, ca, sizeof(ca)); memcpy(p_q, hq, qb); memcpy(p_k, hk, kb); memcpy(p_v, hv, kb);
    memset(p_o, 0xff, qb);
    CHECK(sift_prefill_layer_host_workspace_size(&s, sizeof(la), sizeof(ca), &wsb) == SIFT_OK);
    CHECK(cudaMalloc(&d_ws, wsb) == 0 && cudaStreamCreate(&st) == 0 && sift_host_ctx_create(&ctx) == SIFT_OK);
    CHECK(sift_prefill_layer_host(ctx, &s, 0, (const uint8_t*)p_la, sizeof(la), la_off, (const uint8_t*)p_ca, sizeof(ca), ca_off,
                                  p_q, p_k, p_v, HQ * D, HKV * D, HKV * D, p_o, HQ * D, (float*)p_lse, 0.f, d_ws, wsb - 1, st) == SIFT_ERR_WORKSPACE);
    for (int rep = 0; rep < 2; ++rep) {
      CHECK(sift_prefill_layer_host(ctx, &s, 0, (const uint8_t*)p_la, sizeof(la), la_off, (const uint8_t*)p_ca, sizeof(ca), ca_off,
                                    p_q, p_k, p_v, HQ * D, HKV * D, HKV * D, p_o, HQ * D, (float*)p_lse, 0.f, d_ws, wsb, st) == SIFT_OK);
      CHECK(cudaStreamSynchronize(st) == 0);
      CHECK(memcmp(p_o, ho_sparse, qb) == 0 && memcmp(p_lse, hl_sparse, (size_t)HQ * N * 4) == 0);
    }
    CHECK(sift_host_ctx_destroy(ctx) == SIFT_OK);
    cudaStreamDestroy(st); cudaFree(d_ws);
    cudaFreeHost(p_la); cudaFreeHost(p_ca); cudaFreeHost(p_q); cudaFreeHost(p_k); cudaFreeHost(p_v); cudaFreeHost(p_o); cudaFreeHost(p_lse);
  }
  /* chunked prefill: the prompt in three row ranges that cut a tile, a document and the query; O / LSE start poisoned
   * and must end bit-identical to the single call; a range that reaches past N is refused */
  {
    const int cut[4] = {0, 100, 333, N};
    CHECK(cudaMemset(d_o, 0xff, qb) == 0 && cudaMemset(d_lse, 0xff, (size_t)HQ * N * 4) == 0);
    for (int c = 0; c < 3; ++c)
      CHECK(sift_prefill_attention_rows(&s, 0, cut[c], cut[c + 1], d_q, d_k, d_v, HQ * D, HKV * D, HKV * D, d_md, d_o, HQ * D,
                                        (float*)d_lse, 0.f, NULL) == SIFT_OK);
    CHECK(cudaDeviceSynchronize() == 0 && cudaMemcpy(ho, d_o, qb, 2) == 0 && cudaMemcpy(hl, d_lse, (size_t)HQ * N * 4, 2) == 0);
    CHECK(memcmp(ho, ho_sparse, qb) == 0 && memcmp(hl, hl_sparse, (size_t)HQ * N * 4) == 0);
    CHECK(sift_prefill_attention_rows(&s, 0, 10, N + 1, d_q, d_k, d_v, HQ * D, HKV * D, HKV * D, d_md, d_o, HQ * D, NULL, 0.f, NULL) ==
          SIFT_ERR_INVALID_ARG);
  }
  /* two prompts in one call (sift_shape.n_prompts): the same prompt twice, packed back to back; every row must see its own
   * prompt only, i.e. both halves of O and LSE repeat the single-prompt result bit for bit.  Then the paper's index layout. */
  {
    int32_t off2[5] = {0, L0, L0 + L1, 2 * L0 + L1, 2 * (L0 + L1)}, pstart[3] = {0, 2, 4}, pq[2] = {LQ, LQ};
    sift_shape s2 = {sizeof(sift_shape), 1, HQ, HKV, D, 4, 0, T, 1, off2, 2, pstart, pq};
    sift_md_layout lay2;
    CHECK(sift_metadata_layout(&s2, &lay2) == SIFT_OK && lay2.n_tokens == 2 * N && lay2.n_seg == 6 && lay2.n_tiles == 2 * lay.n_tiles);
    int64_t la_off2[4] = {la_off[0], la_off[1], la_off[0], la_off[1]}, ca_off2[4] = {ca_off[0], ca_off[1], ca_off[0], ca_off[1]};
    void *d_md2, *d_q2, *d_k2, *d_v2, *d_o2, *d_lse2, *d_ptr, *d_idx;
    CHECK(cudaMalloc(&d_md2, lay2.total_bytes) == 0 && cudaMalloc(&d_q2, 2 * qb) == 0 && cudaMalloc(&d_k2, 2 * kb) == 0 &&
          cudaMalloc(&d_v2, 2 * kb) == 0 && cudaMalloc(&d_o2, 2 * qb) == 0 && cudaMalloc(&d_lse2, (size_t)HQ * 2 * N * 4) == 0);
    for (int rep = 0; rep < 2; ++rep)
      CHECK(cudaMemcpy((char*)d_q2 + rep * qb, hq, qb, 1) == 0 && cudaMemcpy((char*)d_k2 + rep * kb, hk, kb, 1) == 0 &&
            cudaMemcpy((char*)d_v2 + rep * kb, hv, kb, 1) == 0);
    CHECK(sift_decode_metadata(&s2, (const uint8_t*)d_la, la_off2, (const uint8_t*)d_ca, ca_off2, d_md2, lay2.total_bytes, NULL) == SIFT_OK);
    CHECK(sift_prefill_attention(&s2, 0, d_q2, d_k2, d_v2, HQ * D, HKV * D, HKV * D, d_md2, d_o2, HQ * D, (float*)d_lse2, 0.f, NULL) == SIFT_OK);
    uint16_t* ho2 = (uint16_t*)malloc(2 * qb);
    float* hl2 = (float*)malloc((size_t)HQ * 2 * N * 4);
    CHECK(cudaDeviceSynchronize() == 0 && cudaMemcpy(ho2, d_o2, 2 * qb, 2) == 0 && cudaMemcpy(hl2, d_lse2, (size_t)HQ * 2 * N * 4, 2) == 0);
    for (int rep = 0; rep < 2; ++rep) {
      CHECK(memcmp((char*)ho2 + rep * qb, ho_sparse, qb) == 0);
      for (int h = 0; h < HQ; ++h) CHECK(memcmp(hl2 + (size_t)h * 2 * N + rep * N, hl_sparse + (size_t)h * N, (size_t)N * 4) == 0);
    }
    /* sparse_n_indices as the paper lays it out from the single-prompt metadata: all bits are set,
     * so the list of document tile (d, i) is [all keys of the earlier documents] ++ [tiles 0..i of d] */
    int64_t hp[HQ * 16];
    CHECK(lay.n_tiles + 1 <= 16 && cudaMalloc(&d_ptr, sizeof(hp)) == 0);
    CHECK(sift_paper_index_offsets(&s, 0, d_md, (int64_t*)d_ptr, NULL) == SIFT_OK);
    CHECK(cudaDeviceSynchronize() == 0 && cudaMemcpy(hp, d_ptr, (size_t)HQ * (lay.n_tiles + 1) * 8, 2) == 0);
    /* doc 0: 4 tiles with 1,2,3,4 entries; doc 1: 3 tiles with L0 + 1,2,3; query tile (id 7): 8 */
    const int64_t want_total = 10 + 3 * (int64_t)L0 + 6 + 8;
    for (int h = 0; h < HQ; ++h) CHECK(hp[h * (lay.n_tiles + 1) + 0] == 0 && hp[h * (lay.n_tiles + 1) + 4] == 10 && hp[h * (lay.n_tiles + 1) + lay.n_tiles] == want_total);
    CHECK(cudaMalloc(&d_idx, (size_t)HQ * want_total * 4) == 0);
    CHECK(sift_export_paper_indices(&s, 0, d_md, (const int64_t*)d_ptr, (int32_t*)d_idx, want_total, NULL) == SIFT_OK);
    int32_t* hidx = (int32_t*)malloc((size_t)HQ * want_total * 4);
    CHECK(cudaDeviceSynchronize() == 0 && cudaMemcpy(hidx, d_idx, (size_t)HQ * want_total * 4, 2) == 0);
    for (int i = 0; i < L0; ++i) CHECK(hidx[10 + i] == i);              /* first tile of doc 1: the L0 keys of doc 0 ... */
    CHECK(hidx[10 + L0] == 4);                                          /* ... then its own tile (global id 4) */
    free(ho2); free(hl2); free(hidx);
    cudaFree(d_md2); cudaFree(d_q2); cudaFree(d_k2); cudaFree(d_v2); cudaFree(d_o2); cudaFree(d_lse2); cudaFree(d_ptr); cudaFree(d_idx);
  }
  cudaFree(d_la); cudaFree(d_ca); cudaFree(d_md); cudaFree(d_q); cudaFree(d_k); cudaFree(d_v); cudaFree(d_o); cudaFree(d_lse);
  printf("abi_smoke gpu ok\n");
  return 0;
}

int main(int argc, char** argv) {
  if (argc > 1 && strcmp(argv[1], "gpu") == 0) return gpu_part();
  return host_part();
}
