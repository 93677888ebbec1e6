/* The boundary is a C ABI: this file is compiled as C99 against include/flowkv.h and linked with libflowkv.so.
 * It plans the hand-worked example of SURVEY §8c (src [5,6,7,20,21,9,3,4] -> dst [0..7], 120 tokens, block 16)
 * with the host-only planner and prints the segments: "first_token n_tokens src_block dst_block" per line. */
#include <stdio.h>
#include "flowkv.h"

int main(void) {
  flowkv_pool src, dst;
  flowkv_request req;
  flowkv_plan_t* plan = NULL;
  flowkv_plan_stats st;
  const flowkv_segment* segs = NULL;
  const int32_t s[8] = {5, 6, 7, 20, 21, 9, 3, 4}, d[8] = {0, 1, 2, 3, 4, 5, 6, 7};
  unsigned i;
  flowkv_status rc;

  src.base = (void*)0x1000; src.num_layers = 2; src.num_kv_heads = 2; src.head_dim = 64; src.elem_bytes = 2;
  src.num_blocks = 32; src.block_size = 16; src.layout = FLOWKV_LAYOUT_LKBTHD; src._reserved = 0; src.plane_offsets = NULL;
  dst = src;
  if (flowkv_pool_strides(&src) != FLOWKV_OK || flowkv_pool_strides(&dst) != FLOWKV_OK) return 2;
  req.num_tokens = 120; req.n_src_blocks = 8; req.src_blocks = s; req.dst_blocks = d; req.n_dst_blocks = 8; req._reserved = 0;
  rc = flowkv_plan_host(&src, &dst, &req, 1, FLOWKV_CHECK_DST_ALIAS, NULL, &plan);
  if (rc != FLOWKV_OK) { fprintf(stderr, "%s: %s\n", flowkv_status_string(rc), flowkv_last_error()); return 3; }
  if (flowkv_plan_info(plan, &st, &segs) != FLOWKV_OK) return 4;
  for (i = 0; i < st.n_segments; ++i)
    printf("%u %u %u %u\n", segs[i].first_token, segs[i].n_tokens, segs[i].src_block, segs[i].dst_block);
  /* a plan built without a device refuses to run, loudly */
  if (flowkv_transfer(plan, NULL) != FLOWKV_ERR_UNSUPPORTED) return 5;
  flowkv_plan_destroy(plan);
  /* error path: table too short */
  req.n_src_blocks = 7;
  if (flowkv_plan_host(&src, &dst, &req, 1, 0, NULL, &plan) != FLOWKV_ERR_TABLE_LEN) return 6;
  req.n_src_blocks = 8;
  /* a cache whose planes are separate allocations (plane_offsets): same segments, the layer and K|V strides
   * are ignored; an offset that is no multiple of 16 is refused */
  {
    int64_t off[4] = {3 * 65536, 0, 65536 + 4096, 7 * 65536};       /* planes (l0,K) (l0,V) (l1,K) (l1,V) */
    uint64_t nseg = 0;
    src.plane_offsets = off;
    src.stride_bytes[FLOWKV_S_LAYER] = 0;
    src.stride_bytes[FLOWKV_S_KV] = 0;
    if (flowkv_plan_host(&src, &dst, &req, 1, 0, NULL, &plan) != FLOWKV_OK) return 7;
    if (flowkv_plan_info(plan, &st, NULL) != FLOWKV_OK) return 8;
    nseg = st.n_segments;
    flowkv_plan_destroy(plan);
    if (nseg != 4 || st.mode_transfer != 1) return 9;               /* still span mode: strides inside a plane decide */
    off[2] += 8;
    if (flowkv_plan_host(&src, &dst, &req, 1, 0, NULL, &plan) != FLOWKV_ERR_ALIGN) return 10;
  }
  return 0;
}
