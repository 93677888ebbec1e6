/*
 * flowkv_oracle.c — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * A plain, slow, single-threaded CPU statement of what FlowKV's KV-cache transfer
 * computes (arXiv 2504.03775, /root/reference/PAPER.md, cited "P:Lnn").  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.  It shares no code, header, table or helper with the CUDA path
 * under paper_2504_03775_b200/csrc/ and neither includes the other.
 *
 * What the path is (§3.1): "transfers the KV Cache K and V from node P_p to
 * node D_d".  The KV cache is paged (§3.3: "logical-to-physical block
 * mapping"); each side holds a block-id list per request (§3.3
 * Fig. 5 caption).  The result therefore has a plain definition, which this file
 * writes out element by element (reading A4: token-granular):
 *
 *   for every request r, token t in [0,T_r), layer l, c in {K,V}, head h, dim d:
 *     dst[l, c, Dst_r[t div BS_d], t mod BS_d, h, d] := src[l, c, Src_r[t div BS_s], t mod BS_s, h, d]
 *
 * with each pool addressed by its own byte strides (Eq. 5, names two
 * orders of the same axes: (L,2,B,H) and (B,L,2,H); strides express both).
 * Elements move as raw bytes (never through a float type).  Every other byte of
 * dst is left alone; src is never written.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): numpy fancy-indexing
 * special cases, a self-describing pool decoded from the definition, identity
 * tables == memcmp, untouched-byte sentinels, all 65,536 16-bit patterns,
 * 1-, 4- and 8-byte elements against numpy item views (the generic branch of
 * okv_copy_elem), all 256 byte codes and fp32 NaN payloads,
 * pack∘unpack identity, layer windows and plane windows == planes cut out of the wire format,
 * pools whose planes are separate allocations (plane_off, A22 / A3) == numpy fancy indexing plane by plane,
 * brute-force minimal partition count on tiny tables,
 * the paper's "fully contiguous => 1 transfer" and
 * "calls per block = L x 2", hand-worked fixtures in tests/golden/.
 * Unpinned by the paper: its printed latencies and the 23,469-call average
 * — other hardware / unstated request mix; context only.
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>

/* Geometry of one paged pool.  Strides are in BYTES; dim stride is elem_bytes.
 * `layer0`: the buffer handed in starts at layer `layer0` of the logical pool
 * (lets a caller hand over one layer slab of a pool too big for host RAM). */
/* `plane_off` (readings A22 and A3): the pool the paper STARTS from keeps every layer in a tensor of its
 * own ("combines the separate tensor structures across all layer dimensions into a continuous tensor"), and K
 * and V may be separate tensors too (A3), so the planes — plane = 2*layer + (0 for K, 1 for V) — are separate
 * allocations with no common stride.  When plane_off != NULL, plane (l, c) begins plane_off[2*l + c] bytes after the
 * buffer's first byte and neither s_layer nor s_kv is used (layer0 must then be 0); inside a plane nothing changes. */
typedef struct {
  uint32_t num_layers, num_kv_heads, head_dim, elem_bytes;
  uint32_t num_blocks, block_size;
  int64_t  s_layer, s_kv, s_block, s_token, s_head;
  uint32_t layer0;
  uint32_t _pad;
  const int64_t* plane_off;
} okv_pool;

static inline int64_t okv_addr(const okv_pool* p, uint32_t l, uint32_t c, int64_t blk,
                               uint32_t tok, uint32_t h, uint32_t d) {
  const int64_t plane = p->plane_off ? p->plane_off[2 * l + c]
                                     : (int64_t)(l - p->layer0) * p->s_layer + (int64_t)c * p->s_kv;
  return plane + blk * p->s_block +
         (int64_t)tok * p->s_token + (int64_t)h * p->s_head + (int64_t)d * p->elem_bytes;
}

/* Copy one element of `e` raw bytes. */
static inline void okv_copy_elem(uint8_t* dst, const uint8_t* src, uint32_t e) {
  if (e == 2) { uint16_t w; memcpy(&w, src, 2); memcpy(dst, &w, 2); }
  else { for (uint32_t b = 0; b < e; ++b) dst[b] = src[b]; }
}

/* Transfer of ONE request, layers [l0,l1).  Definition above, loop order
 * request -> token -> layer -> K|V -> head -> dim (north_star
 * "copies token by token through both block tables").  Returns 0, or -1 on a
 * table entry out of range / shape mismatch (nothing is written before the check
 * of that token). */
int okv_transfer(const uint8_t* src, const okv_pool* sp, uint8_t* dst, const okv_pool* dp,
                 const int32_t* src_tab, const int32_t* dst_tab, uint32_t T,
                 uint32_t l0, uint32_t l1) {
  if (sp->num_layers != dp->num_layers || sp->num_kv_heads != dp->num_kv_heads ||
      sp->head_dim != dp->head_dim || sp->elem_bytes != dp->elem_bytes) return -1;
  const uint32_t e = sp->elem_bytes;
  for (uint32_t t = 0; t < T; ++t) {
    int64_t sb = src_tab[t / sp->block_size]; uint32_t so = t % sp->block_size;
    int64_t db = dst_tab[t / dp->block_size]; uint32_t dof = t % dp->block_size;
    if (sb < 0 || sb >= (int64_t)sp->num_blocks || db < 0 || db >= (int64_t)dp->num_blocks) return -1;
    for (uint32_t l = l0; l < l1; ++l)
      for (uint32_t c = 0; c < 2; ++c)
        for (uint32_t h = 0; h < sp->num_kv_heads; ++h)
          for (uint32_t d = 0; d < sp->head_dim; ++d)
            okv_copy_elem(dst + okv_addr(dp, l, c, db, dof, h, d),
                          src + okv_addr(sp, l, c, sb, so, h, d), e);
  }
  return 0;
}

/* Dense wire format (reading A12; P:L28 describes the competing
 * system's "continuous buffer" only in words):
 *   staging[request][layer][K|V][token][head][dim], requests concatenated,
 *   request r starting at byte req_tok_off * bytes_per_token,
 *   bytes_per_token = 2 * L * Hkv * Dh * e.
 * Pack = pool -> staging through the src table. */
static inline int64_t okv_staging_addr(const okv_pool* p, uint64_t req_tok_off, uint32_t T,
                                       uint32_t l, uint32_t c, uint32_t t, uint32_t h, uint32_t d) {
  int64_t bpt = (int64_t)2 * p->num_layers * p->num_kv_heads * p->head_dim * p->elem_bytes;
  int64_t idx = ((((int64_t)(l * 2 + c) * T + t) * p->num_kv_heads + h) * p->head_dim + d);
  return (int64_t)req_tok_off * bpt + idx * p->elem_bytes;
}

int okv_pack(const uint8_t* src, const okv_pool* sp, const int32_t* src_tab, uint32_t T,
             uint8_t* staging, uint64_t req_tok_off, uint32_t l0, uint32_t l1) {
  const uint32_t e = sp->elem_bytes;
  for (uint32_t t = 0; t < T; ++t) {
    int64_t sb = src_tab[t / sp->block_size]; uint32_t so = t % sp->block_size;
    if (sb < 0 || sb >= (int64_t)sp->num_blocks) return -1;
    for (uint32_t l = l0; l < l1; ++l)
      for (uint32_t c = 0; c < 2; ++c)
        for (uint32_t h = 0; h < sp->num_kv_heads; ++h)
          for (uint32_t d = 0; d < sp->head_dim; ++d)
            okv_copy_elem(staging + okv_staging_addr(sp, req_tok_off, T, l, c, t, h, d),
                          src + okv_addr(sp, l, c, sb, so, h, d), e);
  }
  return 0;
}

/* Unpack = staging -> pool through the dst table (inverse of okv_pack). */
int okv_unpack(const uint8_t* staging, uint64_t req_tok_off, uint8_t* dst, const okv_pool* dp,
               const int32_t* dst_tab, uint32_t T, uint32_t l0, uint32_t l1) {
  const uint32_t e = dp->elem_bytes;
  for (uint32_t t = 0; t < T; ++t) {
    int64_t db = dst_tab[t / dp->block_size]; uint32_t dof = t % dp->block_size;
    if (db < 0 || db >= (int64_t)dp->num_blocks) return -1;
    for (uint32_t l = l0; l < l1; ++l)
      for (uint32_t c = 0; c < 2; ++c)
        for (uint32_t h = 0; h < dp->num_kv_heads; ++h)
          for (uint32_t d = 0; d < dp->head_dim; ++d)
            okv_copy_elem(dst + okv_addr(dp, l, c, db, dof, h, d),
                          staging + okv_staging_addr(dp, req_tok_off, T, l, c, t, h, d), e);
  }
  return 0;
}

/* Layer-window wire format (reading A20): a message that carries only layers [w0,w1) — what a
 * layer-wise / pipelined sender puts on the wire ("layer by layer", P:L222-224 the layerwise ablation) —
 * is the wire format of a model that has just those w1-w0 layers:
 *   window[request][layer - w0][K|V][token][head][dim], requests concatenated,
 *   request r starting at byte req_tok_off * 2*(w1-w0)*Hkv*Dh*e.
 * The window [0,L) is the format of okv_pack. */
static inline int64_t okv_window_addr(const okv_pool* p, uint32_t w0, uint32_t w1, uint64_t req_tok_off, uint32_t T,
                                      uint32_t l, uint32_t c, uint32_t t, uint32_t h, uint32_t d) {
  int64_t bpt = (int64_t)2 * (w1 - w0) * p->num_kv_heads * p->head_dim * p->elem_bytes;
  int64_t idx = ((((int64_t)((l - w0) * 2 + c) * T + t) * p->num_kv_heads + h) * p->head_dim + d);
  return (int64_t)req_tok_off * bpt + idx * p->elem_bytes;
}

int okv_pack_window(const uint8_t* src, const okv_pool* sp, const int32_t* src_tab, uint32_t T,
                    uint8_t* window, uint64_t req_tok_off, uint32_t w0, uint32_t w1) {
  const uint32_t e = sp->elem_bytes;
  for (uint32_t t = 0; t < T; ++t) {
    int64_t sb = src_tab[t / sp->block_size]; uint32_t so = t % sp->block_size;
    if (sb < 0 || sb >= (int64_t)sp->num_blocks) return -1;
    for (uint32_t l = w0; l < w1; ++l)
      for (uint32_t c = 0; c < 2; ++c)
        for (uint32_t h = 0; h < sp->num_kv_heads; ++h)
          for (uint32_t d = 0; d < sp->head_dim; ++d)
            okv_copy_elem(window + okv_window_addr(sp, w0, w1, req_tok_off, T, l, c, t, h, d),
                          src + okv_addr(sp, l, c, sb, so, h, d), e);
  }
  return 0;
}

int okv_unpack_window(const uint8_t* window, uint64_t req_tok_off, uint8_t* dst, const okv_pool* dp,
                      const int32_t* dst_tab, uint32_t T, uint32_t w0, uint32_t w1) {
  const uint32_t e = dp->elem_bytes;
  for (uint32_t t = 0; t < T; ++t) {
    int64_t db = dst_tab[t / dp->block_size]; uint32_t dof = t % dp->block_size;
    if (db < 0 || db >= (int64_t)dp->num_blocks) return -1;
    for (uint32_t l = w0; l < w1; ++l)
      for (uint32_t c = 0; c < 2; ++c)
        for (uint32_t h = 0; h < dp->num_kv_heads; ++h)
          for (uint32_t d = 0; d < dp->head_dim; ++d)
            okv_copy_elem(dst + okv_addr(dp, l, c, db, dof, h, d),
                          window + okv_window_addr(dp, w0, w1, req_tok_off, T, l, c, t, h, d), e);
  }
  return 0;
}

/* Plane-window wire format (reading A21): the same idea one level finer — a message that carries only the
 * planes [p0,p1), plane = 2*layer + (0 for K, 1 for V), in wire order:
 *   window[request][plane - p0][token][head][dim], requests concatenated,
 *   request r starting at byte req_tok_off * (p1-p0)*Hkv*Dh*e.
 * The planes [2*w0, 2*w1) are the layer window [w0,w1) of okv_pack_window.  (The chunked pinned-host pipeline cuts a
 * transfer into such messages when it wants more chunks than the model has layers.) */
static inline int64_t okv_planes_addr(const okv_pool* p, uint32_t p0, uint32_t p1, uint64_t req_tok_off, uint32_t T,
                                      uint32_t plane, uint32_t t, uint32_t h, uint32_t d) {
  int64_t bpt = (int64_t)(p1 - p0) * p->num_kv_heads * p->head_dim * p->elem_bytes;
  int64_t idx = ((((int64_t)(plane - p0) * T + t) * p->num_kv_heads + h) * p->head_dim + d);
  return (int64_t)req_tok_off * bpt + idx * p->elem_bytes;
}

int okv_pack_planes(const uint8_t* src, const okv_pool* sp, const int32_t* src_tab, uint32_t T,
                    uint8_t* window, uint64_t req_tok_off, uint32_t p0, uint32_t p1) {
  const uint32_t e = sp->elem_bytes;
  for (uint32_t t = 0; t < T; ++t) {
    int64_t sb = src_tab[t / sp->block_size]; uint32_t so = t % sp->block_size;
    if (sb < 0 || sb >= (int64_t)sp->num_blocks) return -1;
    for (uint32_t plane = p0; plane < p1; ++plane)
      for (uint32_t h = 0; h < sp->num_kv_heads; ++h)
        for (uint32_t d = 0; d < sp->head_dim; ++d)
          okv_copy_elem(window + okv_planes_addr(sp, p0, p1, req_tok_off, T, plane, t, h, d),
                        src + okv_addr(sp, plane / 2, plane % 2, sb, so, h, d), e);
  }
  return 0;
}

int okv_unpack_planes(const uint8_t* window, uint64_t req_tok_off, uint8_t* dst, const okv_pool* dp,
                      const int32_t* dst_tab, uint32_t T, uint32_t p0, uint32_t p1) {
  const uint32_t e = dp->elem_bytes;
  for (uint32_t t = 0; t < T; ++t) {
    int64_t db = dst_tab[t / dp->block_size]; uint32_t dof = t % dp->block_size;
    if (db < 0 || db >= (int64_t)dp->num_blocks) return -1;
    for (uint32_t plane = p0; plane < p1; ++plane)
      for (uint32_t h = 0; h < dp->num_kv_heads; ++h)
        for (uint32_t d = 0; d < dp->head_dim; ++d)
          okv_copy_elem(dst + okv_addr(dp, plane / 2, plane % 2, db, dof, h, d),
                        window + okv_planes_addr(dp, p0, p1, req_tok_off, T, plane, t, h, d), e);
  }
  return 0;
}

/* ---- Plan oracle: bidirectional segment alignment (§3.3; Fig. 5) ----
 * "compare the block ID lists of both the sending and receiving instances,
 *  identifying N contiguous block IDs that are present on both sides.  Since these
 *  N block IDs are memory-contiguous, they can be transferred in a single operation."
 * Reading (A6-A8, A13): walk the request left to right in units of the
 * granule g = gcd(BS_s, BS_d) tokens; position q has pool-wide granule id
 *     a_x(q) = Table_x[(q*g) div BS_x] * (BS_x/g) + ((q*g) mod BS_x)/g
 * on side x; a new transfer starts at q=0 and wherever a_s or a_d does not step
 * by exactly +1.  A side given as NULL is a dense buffer (always contiguous). */
static uint32_t okv_gcd(uint32_t a, uint32_t b) { while (b) { uint32_t t = a % b; a = b; b = t; } return a; }

static int64_t okv_granule_id(const int32_t* tab, uint32_t bs, uint32_t g, uint64_t q) {
  uint64_t tok = q * g;
  return (int64_t)tab[tok / bs] * (int64_t)(bs / g) + (int64_t)((tok % bs) / g);
}

/* One output record per transfer: first token, number of tokens.  `out` may be
 * NULL to count only.  Returns the number of transfers (0 when T == 0). */
uint64_t okv_align(const int32_t* src_tab, uint32_t bs_s, const int32_t* dst_tab, uint32_t bs_d,
                   uint32_t T, uint32_t* out_first_tok, uint32_t* out_n_tok, uint64_t out_cap) {
  if (T == 0) return 0;
  uint32_t g;
  if (src_tab && dst_tab) g = okv_gcd(bs_s, bs_d); else g = src_tab ? bs_s : bs_d;
  uint64_t nq = ((uint64_t)T + g - 1) / g;
  uint64_t n = 0, start_q = 0;
  for (uint64_t q = 1; q <= nq; ++q) {
    int brk = (q == nq);
    if (!brk && src_tab && okv_granule_id(src_tab, bs_s, g, q) != okv_granule_id(src_tab, bs_s, g, q - 1) + 1) brk = 1;
    if (!brk && dst_tab && okv_granule_id(dst_tab, bs_d, g, q) != okv_granule_id(dst_tab, bs_d, g, q - 1) + 1) brk = 1;
    if (brk) {
      uint64_t first = start_q * g, end = q * g; if (end > T) end = T;
      if (out_first_tok && n < out_cap) { out_first_tok[n] = (uint32_t)first; out_n_tok[n] = (uint32_t)(end - first); }
      ++n; start_q = q;
    }
  }
  return n;
}

/* Call count of the pre-optimisation scheme (§3.3: the reshape "reduces the
 * number of NCCL API calls per KV block by a factor of L x 2", i.e. before it one
 * call per block per layer per K|V). */
uint64_t okv_blockwise_calls(uint32_t n_blocks, uint32_t num_layers) {
  return (uint64_t)n_blocks * num_layers * 2u;
}
