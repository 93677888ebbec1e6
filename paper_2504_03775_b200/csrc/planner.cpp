// planner.cpp — host side of the FlowKV transfer path: validation (a1), bidirectional segment
// alignment (a2; §3.3, Fig. 5) and the tile schedule (a3).  Pure integer code.
//
// Alignment rule (readings A6-A10): a request is walked left to right in pieces that
// never cross a block boundary on either side.  A piece extends the open segment iff its first
// token SLOT (block_id*block_size + offset_in_block) directly follows the segment's last slot on
// the src side AND on the dst side; otherwise it opens a new segment.  Segments never span two
// requests.  The partition is the unique coarsest one whose parts are memory-contiguous on both
// sides in token-slot space, i.e. "N contiguous block IDs present on both sides".
#include <algorithm>
#include <cstdio>

#include "flowkv_internal.h"

namespace flowkv {

static bool is_pow2(uint32_t x) { return x && !(x & (x - 1)); }

bool pool_is_span_capable(const flowkv_pool& p, const Geometry& g) {
  return p.stride_bytes[FLOWKV_S_HEAD] == (int64_t)g.row_bytes &&
         p.stride_bytes[FLOWKV_S_TOKEN] == (int64_t)g.tok_bytes &&
         p.stride_bytes[FLOWKV_S_BLOCK] == (int64_t)p.block_size * g.tok_bytes;
}

flowkv_status validate_pool(const flowkv_pool* p, const char* which, std::string& err) {
  char buf[256];
  auto fail = [&](flowkv_status s, const char* msg) {
    snprintf(buf, sizeof buf, "%s pool: %s", which, msg);
    err = buf;
    return s;
  };
  if (!p->base) return fail(FLOWKV_ERR_INVALID_ARG, "base is NULL");
  if (!p->num_layers || !p->num_kv_heads || !p->head_dim || !p->elem_bytes || !p->num_blocks)
    return fail(FLOWKV_ERR_INVALID_ARG, "a shape field is zero");
  if (!is_pow2(p->block_size)) return fail(FLOWKV_ERR_UNSUPPORTED, "block_size must be a power of two");
  if (p->layout > FLOWKV_LAYOUT_BLKTHD) return fail(FLOWKV_ERR_INVALID_ARG, "unknown layout");
  const uint64_t row = (uint64_t)p->head_dim * p->elem_bytes;
  if (row % 16) return fail(FLOWKV_ERR_ALIGN, "head_dim*elem_bytes is not a multiple of 16 bytes");
  if (row > (1u << 20)) return fail(FLOWKV_ERR_UNSUPPORTED, "row larger than 1 MiB");
  if ((uintptr_t)p->base % 16) return fail(FLOWKV_ERR_ALIGN, "base is not 16-byte aligned");
  // rows mode addresses a chunk (<= one block) with 32-bit offsets
  if ((uint64_t)p->stride_bytes[FLOWKV_S_TOKEN] * p->block_size + (uint64_t)p->stride_bytes[FLOWKV_S_HEAD] * p->num_kv_heads >=
      (1ull << 32))
    return fail(FLOWKV_ERR_UNSUPPORTED, "one block spans 4 GiB or more");
  for (int i = 0; i < 5; ++i) {
    if ((i == FLOWKV_S_LAYER || i == FLOWKV_S_KV) && p->plane_offsets) continue;   // replaced by the per-plane offsets (A22)
    if (p->stride_bytes[i] <= 0) return fail(FLOWKV_ERR_INVALID_ARG, "a stride is <= 0 (call flowkv_pool_strides)");
    if (p->stride_bytes[i] % 16) return fail(FLOWKV_ERR_ALIGN, "a stride is not a multiple of 16 bytes");
  }
  if (p->plane_offsets)
    for (uint32_t pl = 0; pl < 2 * p->num_layers; ++pl)
      if (p->plane_offsets[pl] % 16) return fail(FLOWKV_ERR_ALIGN, "a plane offset is not a multiple of 16 bytes");
  return FLOWKV_OK;
}

static uint32_t ceil_div(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a + b - 1) / b); }

flowkv_status validate_requests(const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs,
                                uint32_t n_reqs, uint32_t flags, std::string& err) {
  char buf[256];
  std::vector<uint8_t> seen;
  if (dst && (flags & FLOWKV_CHECK_DST_ALIAS)) seen.assign(dst->num_blocks, 0);
  for (uint32_t r = 0; r < n_reqs; ++r) {
    const flowkv_request& q = reqs[r];
    if (src) {
      const uint32_t need = ceil_div(q.num_tokens, src->block_size);
      if (q.n_src_blocks != need) {
        snprintf(buf, sizeof buf, "request %u: n_src_blocks=%u but ceil(%u/%u)=%u", r, q.n_src_blocks,
                 q.num_tokens, src->block_size, need);
        err = buf;
        return FLOWKV_ERR_TABLE_LEN;
      }
      if (need && !q.src_blocks) { err = "src_blocks is NULL"; return FLOWKV_ERR_INVALID_ARG; }
      for (uint32_t i = 0; i < need; ++i)
        if (q.src_blocks[i] < 0 || (uint32_t)q.src_blocks[i] >= src->num_blocks) {
          snprintf(buf, sizeof buf, "request %u: src block id %d at %u outside [0,%u)", r, q.src_blocks[i], i,
                   src->num_blocks);
          err = buf;
          return FLOWKV_ERR_BLOCK_OOB;
        }
    }
    if (dst) {
      const uint32_t need = ceil_div(q.num_tokens, dst->block_size);
      if (q.n_dst_blocks != need) {
        snprintf(buf, sizeof buf, "request %u: n_dst_blocks=%u but ceil(%u/%u)=%u", r, q.n_dst_blocks,
                 q.num_tokens, dst->block_size, need);
        err = buf;
        return FLOWKV_ERR_TABLE_LEN;
      }
      if (need && !q.dst_blocks) { err = "dst_blocks is NULL"; return FLOWKV_ERR_INVALID_ARG; }
      for (uint32_t i = 0; i < need; ++i) {
        const int32_t b = q.dst_blocks[i];
        if (b < 0 || (uint32_t)b >= dst->num_blocks) {
          snprintf(buf, sizeof buf, "request %u: dst block id %d at %u outside [0,%u)", r, b, i, dst->num_blocks);
          err = buf;
          return FLOWKV_ERR_BLOCK_OOB;
        }
        if (!seen.empty()) {
          if (seen[b]) {
            snprintf(buf, sizeof buf, "request %u: dst block id %d is named twice in the batch", r, b);
            err = buf;
            return FLOWKV_ERR_DST_ALIAS;
          }
          seen[b] = 1;
        }
      }
    }
  }
  return FLOWKV_OK;
}

void align_segments(const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs,
                    uint32_t n_reqs, std::vector<flowkv_segment>& out) {
  out.clear();
  const uint32_t bs_s = src ? src->block_size : 0, bs_d = dst ? dst->block_size : 0;
  uint64_t tok_base = 0;   // staging_tok_off of the current request
  for (uint32_t r = 0; r < n_reqs; ++r) {
    const uint32_t T = reqs[r].num_tokens;
    const int32_t* S = reqs[r].src_blocks;
    const int32_t* D = reqs[r].dst_blocks;
    if (src && dst && bs_s == bs_d && T) {
      // Equal block sizes (the common case): pieces are whole blocks, so walk the two id lists directly —
      // a segment continues while both ids step by +1 (same rule, ~10x fewer instructions per block).
      // Break detection is branch-free (a fragmented table breaks at every other block, which a predicted branch
      // mispredicts half the time: 11 ns per block became 2): cuts[] collects the block index of every segment start.
      const uint32_t nb = (uint32_t)(((uint64_t)T + bs_s - 1) / bs_s);
      static thread_local std::vector<uint32_t> cuts;
      if (cuts.size() < (size_t)nb + 1) cuts.resize((size_t)nb + 1);
      uint32_t* cp = cuts.data();
      uint32_t n_cuts = 1;
      cp[0] = 0;
      for (uint32_t b = 1; b < nb; ++b) {
        cp[n_cuts] = b;
        n_cuts += (uint32_t)((S[b] != S[b - 1] + 1) | (D[b] != D[b - 1] + 1));
      }
      cp[n_cuts] = nb;
      const size_t base = out.size();
      out.resize(base + n_cuts);
      flowkv_segment* sp = out.data() + base;
      for (uint32_t i = 0; i < n_cuts; ++i) {
        const uint32_t start = cp[i], end = cp[i + 1];
        flowkv_segment sg{};
        sg.request = r;
        sg.first_token = start * bs_s;
        sg.n_tokens = (end < nb ? end * bs_s : T) - sg.first_token;
        sg.src_block = (uint32_t)S[start];
        sg.dst_block = (uint32_t)D[start];
        sg.staging_tok_off = tok_base;
        sp[i] = sg;
      }
      tok_base += T;
      continue;
    }
    bool open = false;
    int64_t next_s = 0, next_d = 0;          // slot that would continue the open segment
    uint32_t t = 0;
    while (t < T) {
      uint32_t piece = T - t;
      int64_t slot_s = 0, slot_d = 0;
      uint32_t sb = 0, so = 0, db = 0, dof = 0;
      if (src) {
        so = t & (bs_s - 1);
        sb = (uint32_t)S[t / bs_s];
        slot_s = (int64_t)sb * bs_s + so;
        piece = std::min(piece, bs_s - so);
      }
      if (dst) {
        dof = t & (bs_d - 1);
        db = (uint32_t)D[t / bs_d];
        slot_d = (int64_t)db * bs_d + dof;
        piece = std::min(piece, bs_d - dof);
      }
      const bool cont = open && (!src || slot_s == next_s) && (!dst || slot_d == next_d);
      if (cont) {
        out.back().n_tokens += piece;
      } else {
        flowkv_segment sg{};
        sg.request = r;
        sg.first_token = t;
        sg.n_tokens = piece;
        sg.src_block = sb; sg.src_tok_off = so;
        sg.dst_block = db; sg.dst_tok_off = dof;
        sg.staging_tok_off = tok_base;
        out.push_back(sg);
        open = true;
      }
      next_s = slot_s + piece;
      next_d = slot_d + piece;
      t += piece;
    }
    tok_base += T;
  }
}

// Byte offset of token slot (block, off) of a pool, plane offset excluded.
static inline int64_t pool_off(const flowkv_pool* p, uint32_t block, uint32_t off) {
  return (int64_t)block * p->stride_bytes[FLOWKV_S_BLOCK] + (int64_t)off * p->stride_bytes[FLOWKV_S_TOKEN];
}

// One rows-mode chunk list for tokens [t, end) of a request: a chunk stays inside one block on each paged side.
static void rows_chunks(const flowkv_pool* src, const flowkv_pool* dst, const Geometry& g, const flowkv_request& rq,
                        uint32_t request, int64_t dense0, uint32_t t, uint32_t end, uint32_t tile_tokens,
                        std::vector<Chunk>& out) {
  const int32_t* S = rq.src_blocks;
  const int32_t* D = rq.dst_blocks;
  while (t < end) {
    uint32_t n = std::min(tile_tokens, end - t);
    Chunk c{};
    if (src) {
      const uint32_t so = t & (src->block_size - 1);
      n = std::min(n, src->block_size - so);
      c.src_off = pool_off(src, (uint32_t)S[t / src->block_size], so);
    } else {
      c.src_off = dense0 | (int64_t)t;
    }
    if (dst) {
      const uint32_t dof = t & (dst->block_size - 1);
      n = std::min(n, dst->block_size - dof);
      c.dst_off = pool_off(dst, (uint32_t)D[t / dst->block_size], dof);
    } else {
      c.dst_off = dense0 | (int64_t)t;
    }
    c.n = n;
    c.req_tokens = rq.num_tokens;
    c.request = request;
    out.push_back(c);
    t += n;
  }
}

bool pools_are_flat_congruent(const flowkv_pool& a, const flowkv_pool& b, const Geometry& g) {
  if (a.block_size != b.block_size) return false;
  if (a.plane_offsets || b.plane_offsets) return false;      // separate plane allocations: a block is not one range
  for (int i : {FLOWKV_S_LAYER, FLOWKV_S_KV, FLOWKV_S_BLOCK, FLOWKV_S_TOKEN, FLOWKV_S_HEAD})
    if (a.stride_bytes[i] != b.stride_bytes[i]) return false;
  // the interior of a block must be a dense bijection onto [0, s_block): sorted by stride, every axis
  // starts where the one below it ends, the smallest is one row, and the block stride closes the product
  struct Axis { int64_t stride; uint64_t extent; };
  Axis ax[4] = {{a.stride_bytes[FLOWKV_S_LAYER], g.L}, {a.stride_bytes[FLOWKV_S_KV], 2},
                {a.stride_bytes[FLOWKV_S_TOKEN], a.block_size}, {a.stride_bytes[FLOWKV_S_HEAD], g.Hkv}};
  std::sort(ax, ax + 4, [](const Axis& x, const Axis& y) { return x.stride < y.stride; });
  int64_t expect = g.row_bytes;
  for (const Axis& x : ax) {
    if (x.extent == 1) continue;            // a length-1 axis never contributes an offset
    if (x.stride != expect) return false;
    expect *= (int64_t)x.extent;
  }
  return a.stride_bytes[FLOWKV_S_BLOCK] == expect && (uint64_t)expect < (1ull << 32);
}

void build_schedule(const flowkv_pool* src, const flowkv_pool* dst, const Geometry& g,
                    const flowkv_request* reqs, const std::vector<flowkv_segment>& segs,
                    uint32_t tile_bytes, uint32_t /*vec_bytes*/, Schedule& out) {
  out.chunks.clear();
  out.n_flat = out.n_ragged = 0;
  const bool span = (!src || pool_is_span_capable(*src, g)) && (!dst || pool_is_span_capable(*dst, g));
  const bool flat = !span && src && dst && pools_are_flat_congruent(*src, *dst, g);
  out.mode = span ? MODE_SPAN : (flat ? MODE_FLAT : MODE_ROWS);
  const uint32_t tile_tokens = std::max<uint32_t>(1, tile_bytes / g.tok_bytes);
  if (flat) {
    // Equal block sizes: every segment starts on a block boundary on both sides (breaks only happen
    // between blocks), so it is  whole blocks  +  at most one partial block at the end of its request.
    const uint32_t bs = src->block_size;
    const int64_t blk = src->stride_bytes[FLOWKV_S_BLOCK];
    std::vector<Chunk> ragged;
    // One entry per piece of 2^shift tiles: the largest power of two <= 32 that divides the tiles of one
    // block, so whole-block ranges fill every slot of every piece (no idle tile slots).
    uint32_t shift = 0;
    if (blk % tile_bytes == 0)
      while (shift < 5 && (blk / tile_bytes) % (2u << shift) == 0) ++shift;
    out.flat_shift = shift;
    out.flat_tile = tile_bytes;
    const uint64_t piece = (uint64_t)tile_bytes << shift;
    for (const flowkv_segment& sg : segs) {
      const uint32_t T = reqs[sg.request].num_tokens;
      const uint64_t bytes = (uint64_t)(sg.n_tokens / bs) * (uint64_t)blk;
      const int64_t s0 = (int64_t)sg.src_block * blk, d0 = (int64_t)sg.dst_block * blk;
      for (uint64_t done = 0; done < bytes; done += piece) {
        Chunk c{};
        c.src_off = s0 + (int64_t)done;
        c.dst_off = d0 + (int64_t)done;
        c.n = (uint32_t)std::min<uint64_t>(piece, bytes - done);
        c.req_tokens = T;
        c.request = sg.request;
        out.chunks.push_back(c);
      }
      const uint32_t rem = sg.n_tokens % bs;
      if (rem) {
        const uint32_t end = sg.first_token + sg.n_tokens;
        rows_chunks(src, dst, g, reqs[sg.request], sg.request, 0, end - rem, end, tile_tokens, ragged);
      }
    }
    out.n_flat = (uint32_t)out.chunks.size();
    out.n_ragged = (uint32_t)ragged.size();
    out.chunks.insert(out.chunks.end(), ragged.begin(), ragged.end());
    for (const flowkv_segment& sg : segs)     // third part: everything in rows mode, for layer-range launches
      rows_chunks(src, dst, g, reqs[sg.request], sg.request, 0, sg.first_token, sg.first_token + sg.n_tokens,
                  tile_tokens, out.chunks);
    return;
  }
  // Schedule order.  The segment LIST is in request order, then token order (that is what flowkv_plan_info reports);
  // the SCHEDULE walks it in the order of the dst pool's addresses when the batch is scattered over the dst pool, so
  // that concurrently running tiles write one rising front through every dst plane (DRAM-page streaks on the write
  // side: +0.6 % on BASELINE configs[2], nothing to gain when dst is contiguous).  Results do not depend on the order:
  // dst tiles are disjoint.  A counting sort over dst block ids: O(#segments + #dst blocks), ~0.1 ms for 14.6k segments.
  std::vector<uint32_t> order;
  if (dst && segs.size() >= 64) {
    bool rising = true;
    for (size_t i = 1; i < segs.size() && rising; ++i)
      rising = segs[i].dst_block > segs[i - 1].dst_block || (segs[i].dst_block == segs[i - 1].dst_block && segs[i].dst_tok_off > segs[i - 1].dst_tok_off);
    if (!rising) {
      static thread_local std::vector<uint32_t> start;
      start.assign((size_t)dst->num_blocks + 1, 0);
      for (const flowkv_segment& sg : segs) ++start[sg.dst_block + 1];
      for (uint32_t b = 0; b < dst->num_blocks; ++b) start[b + 1] += start[b];
      order.resize(segs.size());
      for (uint32_t i = 0; i < (uint32_t)segs.size(); ++i) order[start[segs[i].dst_block]++] = i;   // stable within a block
    }
  }
  Chunk* span_out = nullptr;
  size_t n_span = 0;
  if (span) {
    uint64_t tokens = 0;
    for (const flowkv_segment& sg : segs) tokens += sg.n_tokens;
    out.chunks.resize(segs.size() + (size_t)(tokens / tile_tokens) + 1);      // >= sum of ceil(n_tokens / tile_tokens)
    span_out = out.chunks.data();
  }
  for (size_t oi = 0; oi < segs.size(); ++oi) {
    const flowkv_segment& sg = segs[order.empty() ? oi : order[oi]];
    const uint32_t T = reqs[sg.request].num_tokens;
    // dense side: (staging_tok_off << 32) | token_in_request; the kernel turns it into bytes for the layer
    // window the staging buffer holds (side_offset() in kernels.cu)
    const int64_t dense0 = (int64_t)(sg.staging_tok_off << 32);
    if (span) {
      // the whole segment is one contiguous byte range per plane on both sides; the chunk array was sized for the
      // worst case up front, so the inner loop is plain stores (no capacity checks, no reallocation)
      const int64_t s0 = src ? pool_off(src, sg.src_block, sg.src_tok_off) : dense0 | (int64_t)sg.first_token;
      const int64_t d0 = dst ? pool_off(dst, sg.dst_block, sg.dst_tok_off) : dense0 | (int64_t)sg.first_token;
      const int64_t s_step = src ? (int64_t)g.tok_bytes : 1, d_step = dst ? (int64_t)g.tok_bytes : 1;   // dense side counts tokens
      uint32_t done = 0;
      do {
        const uint32_t n = std::min(tile_tokens, sg.n_tokens - done);
        Chunk& c = span_out[n_span++];
        c.src_off = s0 + (int64_t)done * s_step;
        c.dst_off = d0 + (int64_t)done * d_step;
        c.n = n * g.tok_bytes;
        c.req_tokens = T;
        c.request = sg.request;
        c._pad = 0;
        done += n;
      } while (done < sg.n_tokens);
    } else {
      rows_chunks(src, dst, g, reqs[sg.request], sg.request, dense0, sg.first_token, sg.first_token + sg.n_tokens,
                  tile_tokens, out.chunks);
    }
  }
  if (span) out.chunks.resize(n_span);
}

}  // namespace flowkv
