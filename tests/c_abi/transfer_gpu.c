/* The product path driven from plain C with the CUDA runtime only (no Python, no torch): two pools from cudaMalloc,
 * flowkv_plan + flowkv_transfer on a stream of its own, then the whole dst pool compared byte for byte with the CPU
 * oracle (oracle/flowkv_oracle.c, linked here as the checker).  Shape: 3 layers, 2 KV heads, head_dim 64, 2-byte
 * elements; src LKBTHD block 16 -> dst BLKHTD block 32 (layout + block-size conversion), 2 requests, ragged tails.
 * Prints "ok <launches>" and exits 0 on success. */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <cuda_runtime_api.h>
#include "flowkv.h"

typedef struct {                       /* mirrors okv_pool of oracle/flowkv_oracle.c */
  uint32_t num_layers, num_kv_heads, head_dim, elem_bytes, num_blocks, block_size;
  int64_t s_layer, s_kv, s_block, s_token, s_head;
  uint32_t layer0, _pad;
  const int64_t* plane_off;            /* NULL here: a stacked pool (reading A22 otherwise) */
} okv_pool;
int okv_transfer(const uint8_t* src, const okv_pool* sp, uint8_t* dst, const okv_pool* dp, const int32_t* src_tab,
                 const int32_t* dst_tab, uint32_t T, uint32_t l0, uint32_t l1);

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_)); return 10; } } while (0)
#define FK(x) do { flowkv_status s_ = (x); if (s_ != FLOWKV_OK) { fprintf(stderr, "%s: %s: %s\n", #x, flowkv_status_string(s_), flowkv_last_error()); return 11; } } while (0)

static okv_pool as_oracle(const flowkv_pool* p) {
  okv_pool o;
  memset(&o, 0, sizeof o);
  o.num_layers = p->num_layers; o.num_kv_heads = p->num_kv_heads; o.head_dim = p->head_dim; o.elem_bytes = p->elem_bytes;
  o.num_blocks = p->num_blocks; o.block_size = p->block_size;
  o.s_layer = p->stride_bytes[FLOWKV_S_LAYER]; o.s_kv = p->stride_bytes[FLOWKV_S_KV]; o.s_block = p->stride_bytes[FLOWKV_S_BLOCK];
  o.s_token = p->stride_bytes[FLOWKV_S_TOKEN]; o.s_head = p->stride_bytes[FLOWKV_S_HEAD];
  return o;
}

int main(void) {
  enum { L = 3, H = 2, D = 64, E = 2, NBS = 40, NBD = 24 };
  const int32_t s0[] = {7, 8, 9, 30, 31, 2, 39}, d0[] = {5, 6, 0, 23};       /* 103 tokens: 7 x 16, 4 x 32 */
  const int32_t s1[] = {12, 13, 20}, d1[] = {10, 11};                        /* 40 tokens                 */
  flowkv_pool src, dst;
  flowkv_request reqs[2];
  flowkv_plan_t* plan = NULL;
  cudaStream_t stream;
  size_t sbytes = (size_t)NBS * 16 * 2 * L * H * D * E, dbytes = (size_t)NBD * 32 * 2 * L * H * D * E, i;
  uint8_t *hs = malloc(sbytes), *hd = malloc(dbytes), *exp = malloc(dbytes);
  void *ds = NULL, *dd = NULL;
  okv_pool os, od;
  uint64_t n0;

  memset(&src, 0, sizeof src);
  src.num_layers = L; src.num_kv_heads = H; src.head_dim = D; src.elem_bytes = E;
  dst = src;
  src.num_blocks = NBS; src.block_size = 16; src.layout = FLOWKV_LAYOUT_LKBTHD;
  dst.num_blocks = NBD; dst.block_size = 32; dst.layout = FLOWKV_LAYOUT_BLKHTD;
  srand(2504);
  for (i = 0; i < sbytes; ++i) hs[i] = (uint8_t)rand();
  memset(exp, 0xA5, dbytes);
  CK(cudaMalloc(&ds, sbytes));
  CK(cudaMalloc(&dd, dbytes));
  CK(cudaMemcpy(ds, hs, sbytes, cudaMemcpyHostToDevice));
  CK(cudaMemset(dd, 0xA5, dbytes));
  CK(cudaStreamCreateWithFlags(&stream, cudaStreamNonBlocking));
  src.base = ds; dst.base = dd;
  FK(flowkv_pool_strides(&src));
  FK(flowkv_pool_strides(&dst));
  memset(reqs, 0, sizeof reqs);
  reqs[0].num_tokens = 103; reqs[0].src_blocks = s0; reqs[0].n_src_blocks = 7; reqs[0].dst_blocks = d0; reqs[0].n_dst_blocks = 4;
  reqs[1].num_tokens = 40;  reqs[1].src_blocks = s1; reqs[1].n_src_blocks = 3; reqs[1].dst_blocks = d1; reqs[1].n_dst_blocks = 2;
  n0 = flowkv_launch_count();
  FK(flowkv_plan(&src, &dst, reqs, 2, FLOWKV_CHECK_DST_ALIAS, NULL, stream, &plan));
  FK(flowkv_transfer(plan, stream));
  flowkv_plan_destroy(plan);                                   /* stream-ordered: the queued kernel stays valid */
  CK(cudaStreamSynchronize(stream));
  CK(cudaMemcpy(hd, dd, dbytes, cudaMemcpyDeviceToHost));
  os = as_oracle(&src); od = as_oracle(&dst);
  if (okv_transfer(hs, &os, exp, &od, s0, d0, 103, 0, L) || okv_transfer(hs, &os, exp, &od, s1, d1, 40, 0, L)) return 12;
  for (i = 0; i < dbytes; ++i)
    if (hd[i] != exp[i]) { fprintf(stderr, "byte %zu differs: got %u expected %u\n", i, hd[i], exp[i]); return 1; }
  printf("ok %llu\n", (unsigned long long)(flowkv_launch_count() - n0));
  return 0;
}
