// kernels.cu — the sm_100a copy kernels of the FlowKV transfer path (steps a5-a7).
//
// One launch moves a whole transfer batch ("from 23,469 [calls] to just 1").  Thread groups walk
// a linear tile space with a grid-stride loop
//     tile -> (plane, chunk)      plane = 2*layer + kv, chunk = entry of the plan's schedule
// and the grid is capped at 256 CTAs per SM: up to the cap every tile has its own CTA and the hardware CTA
// scheduler hands tiles to whichever SM frees up first (measured 3-6 % faster than an exactly-resident grid
// with a static stride); beyond the cap each CTA strides.  No per-block / per-layer launch, no
// atomics, no inter-CTA dependence.  The path is a pure byte move: no FP, no tensor cores; the bound is HBM
// bandwidth.
//
// Variants
//   ldst : registers.  256-bit (LDG.E.256 / STG.E.256, sm_100+) or 128-bit vector accesses,
//          UNROLL independent loads in flight per thread before the first store, streaming cache
//          hints (L1::no_allocate, L2::evict_first) because nothing is ever re-read.
//            span mode : a chunk is one byte range contiguous on both sides (per plane).
//            rows mode : a chunk is n tokens x Hkv rows of Dh*e bytes; each side has its own
//                        token / head stride (layout + block-size conversion, BASELINE configs[3]).
//            flat mode : both pools block-major with the same interior (Eq. 5's (B,L,2,H)): whole-block
//                        runs are plane-free byte ranges; partial last blocks ride along as rows tiles.
//   bulk : TMA bulk copies (cp.async.bulk -> UBLKCP) gmem -> smem -> gmem through an mbarrier
//          ring driven by ONE thread per CTA; span and flat modes (byte ranges).  Uses no registers or LSU slots
//          for payload, which is what a copy that co-runs with GEMMs wants.
//   tables : no schedule at all — the kernel reads device-resident block tables (flowkv_transfer_tables).
// Every scheduled kernel exists for a schedule in global memory and for one passed by value in the kernel parameters.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>
#include <utility>

#include "flowkv_internal.h"

namespace flowkv {

// ------------------------------------------------------------------------------------------------
// vector load / store with cache hints
// ------------------------------------------------------------------------------------------------
template <int VEC> struct Vec;
template <> struct alignas(16) Vec<16> { uint32_t x, y, z, w; };
template <> struct alignas(32) Vec<32> { uint64_t a, b, c, d; };

// HINT 0: default caching.  1: L1::no_allocate.  2: L1::no_allocate + L2::evict_first.
template <int VEC, int HINT> struct Mem;

template <int HINT> struct Mem<32, HINT> {
  static __device__ __forceinline__ Vec<32> ld(const char* p, uint64_t) {
    Vec<32> v;
    if (HINT == 0)
      asm volatile("ld.global.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(v.a), "=l"(v.b), "=l"(v.c), "=l"(v.d) : "l"(p));
    else if (HINT == 1)
      asm volatile("ld.global.L1::no_allocate.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(v.a), "=l"(v.b), "=l"(v.c), "=l"(v.d) : "l"(p));
    else
      asm volatile("ld.global.L1::no_allocate.L2::evict_first.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(v.a), "=l"(v.b), "=l"(v.c), "=l"(v.d) : "l"(p));
    return v;
  }
  static __device__ __forceinline__ void st(char* p, const Vec<32>& v, uint64_t) {
    if (HINT == 0)
      asm volatile("st.global.v4.b64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(v.a), "l"(v.b), "l"(v.c), "l"(v.d) : "memory");
    else if (HINT == 1)
      asm volatile("st.global.L1::no_allocate.v4.b64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(v.a), "l"(v.b), "l"(v.c), "l"(v.d) : "memory");
    else
      asm volatile("st.global.L1::no_allocate.L2::evict_first.v4.b64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(v.a), "l"(v.b), "l"(v.c), "l"(v.d) : "memory");
  }
};

template <int HINT> struct Mem<16, HINT> {
  static __device__ __forceinline__ Vec<16> ld(const char* p, uint64_t pol) {
    Vec<16> v;
    if (HINT == 0)
      asm volatile("ld.global.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    else if (HINT == 1)
      asm volatile("ld.global.L1::no_allocate.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    else   // 128-bit forms take the L2 priority through a policy operand
      asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v4.b32 {%0,%1,%2,%3}, [%4], %5;"
                   : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(pol));
    return v;
  }
  static __device__ __forceinline__ void st(char* p, const Vec<16>& v, uint64_t pol) {
    if (HINT == 0)
      asm volatile("st.global.v4.b32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
    else if (HINT == 1)
      asm volatile("st.global.L1::no_allocate.v4.b32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
    else
      asm volatile("st.global.L1::no_allocate.L2::cache_hint.v4.b32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "r"(v.x), "r"(v.y),
                   "r"(v.z), "r"(v.w), "l"(pol) : "memory");
  }
};

// Programmatic dependent launch (sm_90+): every copy kernel lets the NEXT kernel in the stream start its CTAs and
// prologue while this one drains (launch_dependents, issued at entry), and waits for the PREVIOUS kernel's memory
// to be complete and visible (wait) before it touches global memory.  Back-to-back small batches thereby overlap
// their launch ramps with each other's tails.  Without the launch attribute both instructions are no-ops.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait_prior_grid() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}

__device__ __forceinline__ Chunk load_chunk(const Chunk* p) {
  // 32-byte read-only load of one schedule entry (every thread of the group reads the same one)
  Chunk c;
  uint64_t a, b, d, e;
  asm volatile("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(d), "=l"(e) : "l"(p));
  c.src_off = (int64_t)a;
  c.dst_off = (int64_t)b;
  c.n = (uint32_t)d;
  c.req_tokens = (uint32_t)(d >> 32);
  c.request = (uint32_t)e;
  c._pad = 0;
  return c;
}

// Where a kernel finds its schedule: in global memory (uploaded by flowkv_plan), or — for small plans —
// inside the kernel parameters themselves, so that planning a small batch needs no allocation, no
// upload and no cross-stream dependency before the launch (step a4 "kernel params when tiny").
struct GlobalChunks {
  const Chunk* p;
  __device__ __forceinline__ Chunk get(uint32_t i) const { return load_chunk(p + i); }
};
template <uint32_t N> struct ParamChunks {
  Chunk c[N];
  __device__ __forceinline__ Chunk get(uint32_t i) const { return c[i]; }    // constant-bank load
};

// Byte offset of a chunk inside one plane of one side.
//   pool side  : layer*s_layer + kv*s_kv + off                                    (off in bytes);
//                plane_off[plane] in place of layer*s_layer + kv*s_kv when the planes are separate allocations (A22)
//   dense side : off = (staging_tok_off << 32) | token_in_request.  The buffer holds the layer window
//                [plane0/2, ...) in wire order [request][layer][K|V][token][head][dim] (A12), so the
//                chunk sits at  staging_tok_off * window_bytes_per_token            (request base)
//                             + (plane - plane0) * T_r * tok_bytes                  (plane slab)
//                             + token_in_request * tok_bytes.
// PO = true only in the *_po kernels, which serve pools whose planes are separate allocations (reading A22): `po` is
// then that side's DEVICE table of per-plane byte offsets (or NULL: that side is an ordinary pool).  Every other
// kernel passes PO = false and compiles to exactly the code it had before such pools existed.
template <bool PO>
__device__ __forceinline__ int64_t side_offset(const Side& s, const int64_t* po, int64_t off, uint32_t plane,
                                               uint32_t req_tokens, uint32_t tok_bytes) {
  if (s.dense) {
    const uint32_t tok0 = (uint32_t)((uint64_t)off >> 32), t = (uint32_t)off;
    return (int64_t)tok0 * s.s_layer + ((int64_t)(plane - s.plane0) * req_tokens + t) * (int64_t)tok_bytes;
  }
  if (PO && po) return __ldg(po + plane) + off;
  return (int64_t)(plane >> 1) * s.s_layer + (int64_t)(plane & 1) * s.s_kv + off;
}

__device__ __forceinline__ void decode_tile(const KernelParams& p, uint32_t tile, uint32_t& plane, uint32_t& ci) {
  if (p.tile_order == 0) { plane = tile / p.n_chunks; ci = tile - plane * p.n_chunks; }
  else                   { ci = tile / p.n_planes;    plane = tile - ci * p.n_planes; }
  plane += p.plane0;       // layer-range launches start at plane 2*layer_begin
}

// One contiguous byte range: UNROLL independent loads in flight per thread, then UNROLL stores; the
// last round is ragged.  `step` = bytes one round of the whole thread group covers.
template <int VEC, int UNROLL, int HINT>
__device__ __forceinline__ void copy_span(const char* __restrict__ s, char* __restrict__ d, uint32_t n, uint32_t lane,
                                          uint32_t step, uint64_t pol) {
  for (uint32_t off = lane * VEC; off < n; off += UNROLL * step) {
    Vec<VEC> v[UNROLL];
#pragma unroll
    for (int j = 0; j < UNROLL; ++j)
      if (off + j * step < n) v[j] = Mem<VEC, HINT>::ld(s + off + j * step, pol);
#pragma unroll
    for (int j = 0; j < UNROLL; ++j)
      if (off + j * step < n) Mem<VEC, HINT>::st(d + off + j * step, v[j], pol);
  }
}

// `ntok` tokens x Hkv rows of row_bytes, each side with its own token / head stride; vectors are
// indexed (token, head, vec) so consecutive lanes move consecutive bytes of a row.
template <int VEC, int UNROLL, int HINT>
__device__ __forceinline__ void copy_rows(const KernelParams& p, const char* __restrict__ s, char* __restrict__ d,
                                          uint32_t ntok, uint32_t lane, uint32_t G, uint32_t vpr, bool pow2,
                                          uint64_t pol) {
  const uint32_t pieces = ntok * p.heads * vpr;       // vectors in this chunk, (token, head, vec) order
  for (uint32_t i0 = lane; i0 < pieces; i0 += G * UNROLL) {
    Vec<VEC> v[UNROLL];
    uint32_t doff[UNROLL];          // offsets inside one block fit 32 bits (checked by the planner)
#pragma unroll
    for (int j = 0; j < UNROLL; ++j) {
      const uint32_t i = i0 + j * G;
      if (i < pieces) {
        uint32_t row, o, tok, h;
        if (pow2) {
          row = i >> p.vpr_log2;   o = i & (vpr - 1);
          tok = row >> p.heads_log2; h = row & (p.heads - 1);
        } else {
          row = i / vpr;       o = i - row * vpr;
          tok = row / p.heads; h = row - tok * p.heads;
        }
        const uint32_t soff = tok * (uint32_t)p.src.s_token + h * (uint32_t)p.src.s_head + o * VEC;
        doff[j] = tok * (uint32_t)p.dst.s_token + h * (uint32_t)p.dst.s_head + o * VEC;
        v[j] = Mem<VEC, HINT>::ld(s + soff, pol);
      }
    }
#pragma unroll
    for (int j = 0; j < UNROLL; ++j)
      if (i0 + j * G < pieces) Mem<VEC, HINT>::st(d + doff[j], v[j], pol);
  }
}

// ------------------------------------------------------------------------------------------------
// ldst / span
// ------------------------------------------------------------------------------------------------
template <int VEC, int UNROLL, int HINT, class CS, bool PO>
__device__ __forceinline__ void span_kernel(const KernelParams& p, const CS& cs, const int64_t* po_src, const int64_t* po_dst) {
  const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t G = 1u << p.group_log2;
  const uint32_t lane = gtid & (G - 1);
  const uint32_t n_groups = (gridDim.x * blockDim.x) >> p.group_log2;
  const uint32_t step = G * VEC;
  const uint64_t pol = (HINT == 2 && VEC == 16) ? policy_evict_first() : 0;

  pdl_launch_dependents();
  uint32_t tile = gtid >> p.group_log2;
  if (tile >= p.n_tiles) return;
  uint32_t plane, ci;
  decode_tile(p, tile, plane, ci);
  pdl_wait_prior_grid();
  Chunk c = cs.get(ci);
  for (; tile < p.n_tiles; tile += n_groups) {
    // fetch the NEXT tile's schedule entry now, so its latency hides behind this tile's copy
    const uint32_t next = tile + n_groups;
    uint32_t nplane = 0, nci = 0;
    Chunk cn = c;
    if (next < p.n_tiles) {
      decode_tile(p, next, nplane, nci);
      cn = cs.get(nci);
    }
    const char* __restrict__ s = p.src.base + side_offset<PO>(p.src, po_src, c.src_off, plane, c.req_tokens, p.tok_bytes);
    char* __restrict__ d = p.dst.base + side_offset<PO>(p.dst, po_dst, c.dst_off, plane, c.req_tokens, p.tok_bytes);
    copy_span<VEC, UNROLL, HINT>(s, d, c.n, lane, step, pol);
    c = cn;
    plane = nplane;
  }
}
template <int VEC, int UNROLL, int HINT, class CS>
__global__ void __launch_bounds__(512, 2) fk_span_ldst(const __grid_constant__ KernelParams p, const __grid_constant__ CS cs) {
  span_kernel<VEC, UNROLL, HINT, CS, false>(p, cs, nullptr, nullptr);
}
template <int VEC, int UNROLL, int HINT, class CS>     // planes of a side are separate allocations (A22)
__global__ void __launch_bounds__(512, 2) fk_span_ldst_po(const __grid_constant__ KernelParams p, const __grid_constant__ CS cs,
                                                          const __grid_constant__ PlaneOffs po) {
  span_kernel<VEC, UNROLL, HINT, CS, true>(p, cs, po.src, po.dst);
}

// ------------------------------------------------------------------------------------------------
// ldst / rows: token- and head-strided rows (layout and block-size conversion fused in the move)
// ------------------------------------------------------------------------------------------------
template <int VEC, int UNROLL, int HINT, class CS, bool PO>
__device__ __forceinline__ void rows_kernel(const KernelParams& p, const CS& cs, const int64_t* po_src, const int64_t* po_dst) {
  const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t G = 1u << p.group_log2;
  const uint32_t lane = gtid & (G - 1);
  const uint32_t n_groups = (gridDim.x * blockDim.x) >> p.group_log2;
  const uint64_t pol = (HINT == 2 && VEC == 16) ? policy_evict_first() : 0;
  const uint32_t vpr = p.row_bytes / VEC;            // vectors per row
  const bool pow2 = (p.vpr_log2 != 0xffffffffu) && (p.heads_log2 != 0xffffffffu);

  pdl_launch_dependents();
  uint32_t tile = gtid >> p.group_log2;
  if (tile >= p.n_tiles) return;
  uint32_t plane, ci;
  decode_tile(p, tile, plane, ci);
  pdl_wait_prior_grid();
  Chunk c = cs.get(ci);
  for (; tile < p.n_tiles; tile += n_groups) {
    const uint32_t next = tile + n_groups;           // prefetch the next schedule entry (see span_kernel)
    uint32_t nplane = 0, nci = 0;
    Chunk cn = c;
    if (next < p.n_tiles) {
      decode_tile(p, next, nplane, nci);
      cn = cs.get(nci);
    }
    const char* __restrict__ s = p.src.base + side_offset<PO>(p.src, po_src, c.src_off, plane, c.req_tokens, p.tok_bytes);
    char* __restrict__ d = p.dst.base + side_offset<PO>(p.dst, po_dst, c.dst_off, plane, c.req_tokens, p.tok_bytes);
    copy_rows<VEC, UNROLL, HINT>(p, s, d, c.n, lane, G, vpr, pow2, pol);
    c = cn;
    plane = nplane;
  }
}
template <int VEC, int UNROLL, int HINT, class CS>
__global__ void __launch_bounds__(512, 2) fk_rows_ldst(const __grid_constant__ KernelParams p, const __grid_constant__ CS cs) {
  rows_kernel<VEC, UNROLL, HINT, CS, false>(p, cs, nullptr, nullptr);
}
template <int VEC, int UNROLL, int HINT, class CS>     // planes of a side are separate allocations (A22)
__global__ void __launch_bounds__(512, 2) fk_rows_ldst_po(const __grid_constant__ KernelParams p, const __grid_constant__ CS cs,
                                                          const __grid_constant__ PlaneOffs po) {
  rows_kernel<VEC, UNROLL, HINT, CS, true>(p, cs, po.src, po.dst);
}

// ------------------------------------------------------------------------------------------------
// ldst / flat: both pools block-major with the same block interior, (B,L,2,H) on both sides — the
// paper's own scenario (Eq. 5, Fig. 5): a run of whole blocks whose ids are
// consecutive on both sides is ONE byte range covering every layer and K|V.  chunks[0, n_flat) are
// pieces of such ranges (no plane term), each owning 2^flat_shift tile slots of flat_tile bytes, so the
// schedule stays one entry per <= 2 MiB instead of one per tile; the tokens of a partial last block
// (reading A4: token-granular) follow as rows-mode tiles over (plane, chunk), chunks[n_flat ...].
// Still one launch.
// ------------------------------------------------------------------------------------------------
template <int VEC, int UNROLL, int HINT, class CS>
__global__ void __launch_bounds__(512, 2) fk_flat_ldst(const __grid_constant__ KernelParams p, const __grid_constant__ CS cs) {
  const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t G = 1u << p.group_log2;
  const uint32_t lane = gtid & (G - 1);
  const uint32_t group = gtid >> p.group_log2;
  const uint32_t n_groups = (gridDim.x * blockDim.x) >> p.group_log2;
  const uint32_t step = G * VEC;
  const uint64_t pol = (HINT == 2 && VEC == 16) ? policy_evict_first() : 0;

  pdl_launch_dependents();
  pdl_wait_prior_grid();
  const uint32_t n_flat_tiles = p.n_flat << p.flat_shift;
  for (uint32_t tile = group; tile < n_flat_tiles; tile += n_groups) {
    const Chunk c = cs.get(tile >> p.flat_shift);
    const uint32_t off = (tile & ((1u << p.flat_shift) - 1)) * p.flat_tile;
    if (off < c.n)      // the last piece of a range may leave slots empty
      copy_span<VEC, UNROLL, HINT>(p.src.base + c.src_off + off, p.dst.base + c.dst_off + off,
                                   min(p.flat_tile, c.n - off), lane, step, pol);
  }
  const uint32_t n_ragged = p.n_tiles - n_flat_tiles;  // = n_chunks * n_planes
  if (n_ragged == 0) return;
  const uint32_t vpr = p.row_bytes / VEC;
  const bool pow2 = (p.vpr_log2 != 0xffffffffu) && (p.heads_log2 != 0xffffffffu);
  // start the ragged tiles where the flat ones stopped so the last wave of groups shares them
  for (uint32_t tile = (group + n_groups - n_flat_tiles % n_groups) % n_groups; tile < n_ragged; tile += n_groups) {
    uint32_t plane, ci;
    decode_tile(p, tile, plane, ci);
    const Chunk c = cs.get(p.n_flat + ci);
    const char* s = p.src.base + side_offset<false>(p.src, nullptr, c.src_off, plane, c.req_tokens, p.tok_bytes);
    char* d = p.dst.base + side_offset<false>(p.dst, nullptr, c.dst_off, plane, c.req_tokens, p.tok_bytes);
    copy_rows<VEC, UNROLL, HINT>(p, s, d, c.n, lane, G, vpr, pow2, pol);
  }
}

// ------------------------------------------------------------------------------------------------
// bulk / span: TMA bulk copies through a shared-memory ring, one driving thread per CTA
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar, uint64_t pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(smem_dst)),
      "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* smem_src, uint32_t bytes, uint64_t pol) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(gdst),
               "r"(smem_u32(smem_src)), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() {
  asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

constexpr int kBulkMaxStages = 16;

// stage_bytes: size of one ring slot (>= every chunk's n).  n_stages in [2, kBulkMaxStages].
template <class CS, bool PO>
__device__ __forceinline__ void span_bulk_kernel(const KernelParams& p, const CS& cs, uint32_t stage_bytes, uint32_t n_stages,
                                                 const int64_t* po_src, const int64_t* po_dst) {
  extern __shared__ __align__(128) char ring[];
  __shared__ __align__(8) uint64_t full[kBulkMaxStages];
  pdl_launch_dependents();
  if (threadIdx.x != 0) return;                       // one thread drives the TMA unit
  for (uint32_t i = 0; i < n_stages; ++i) mbar_init(&full[i], 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  const uint64_t pol = policy_evict_first();
  pdl_wait_prior_grid();

  const uint32_t first = blockIdx.x, stride = gridDim.x;
  const uint32_t n_my = first < p.n_tiles ? (p.n_tiles - first + stride - 1) / stride : 0;
  const uint32_t ahead = n_stages - 1;                // loads kept in flight

  __shared__ char* dptr[kBulkMaxStages];              // where each slot's bytes go
  __shared__ uint32_t nbytes[kBulkMaxStages];

  auto issue_load = [&](uint32_t k) {
    uint32_t plane, ci;
    decode_tile(p, first + k * stride, plane, ci);
    const Chunk c = cs.get(ci);
    const char* s = p.src.base + side_offset<PO>(p.src, po_src, c.src_off, plane, c.req_tokens, p.tok_bytes);
    const uint32_t slot = k % n_stages;
    dptr[slot] = p.dst.base + side_offset<PO>(p.dst, po_dst, c.dst_off, plane, c.req_tokens, p.tok_bytes);
    nbytes[slot] = c.n;
    mbar_expect_tx(&full[slot], c.n);
    bulk_g2s(ring + (size_t)slot * stage_bytes, s, c.n, &full[slot], pol);
  };

  for (uint32_t k = 0; k < ahead && k < n_my; ++k) issue_load(k);
  for (uint32_t k = 0; k < n_my; ++k) {
    const uint32_t slot = k % n_stages;
    mbar_wait(&full[slot], (k / n_stages) & 1);       // tile k has landed in its slot
    bulk_s2g(dptr[slot], ring + (size_t)slot * stage_bytes, nbytes[slot], pol);
    bulk_commit();
    if (k + ahead < n_my) {
      // slot of tile k+ahead == slot of tile k-1: its store must have finished READING smem
      bulk_wait_read<1>();
      issue_load(k + ahead);
    }
  }
  bulk_wait_all();
}
template <class CS>
__global__ void __launch_bounds__(32, 1) fk_span_bulk(const __grid_constant__ KernelParams p, const __grid_constant__ CS cs,
                                                      uint32_t stage_bytes, uint32_t n_stages) {
  span_bulk_kernel<CS, false>(p, cs, stage_bytes, n_stages, nullptr, nullptr);
}
template <class CS>                                   // planes of a side are separate allocations (A22)
__global__ void __launch_bounds__(32, 1) fk_span_bulk_po(const __grid_constant__ KernelParams p, const __grid_constant__ CS cs,
                                                         uint32_t stage_bytes, uint32_t n_stages, const __grid_constant__ PlaneOffs po) {
  span_bulk_kernel<CS, true>(p, cs, stage_bytes, n_stages, po.src, po.dst);
}

// bulk / flat: the same TMA ring over the plane-free tiles of two congruent block-major pools (the paper's
// (B,L,2,H) layout next to the paper's SM-contention concern): thread 0 drives the ring; the few tiles
// of partial last blocks are then moved by the whole warp with 128-bit loads/stores.
template <class CS>
__global__ void __launch_bounds__(32, 1) fk_flat_bulk(const __grid_constant__ KernelParams p, const __grid_constant__ CS cs,
                                                      uint32_t stage_bytes, uint32_t n_stages) {
  extern __shared__ __align__(128) char ring[];
  __shared__ __align__(8) uint64_t full[kBulkMaxStages];
  __shared__ char* dptr[kBulkMaxStages];
  __shared__ uint32_t nbytes[kBulkMaxStages];
  const uint32_t n_flat_tiles = p.n_flat << p.flat_shift;
  pdl_launch_dependents();
  pdl_wait_prior_grid();
  if (threadIdx.x == 0) {
    for (uint32_t i = 0; i < n_stages; ++i) mbar_init(&full[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    const uint64_t pol = policy_evict_first();
    uint32_t cursor = blockIdx.x;                     // next tile of this CTA to look at
    uint32_t loaded = 0, stored = 0;                  // non-empty tiles whose load / store has been issued
    auto issue_next = [&]() -> bool {                 // skips the empty slots at the end of a range
      for (; cursor < n_flat_tiles; cursor += gridDim.x) {
        const Chunk c = cs.get(cursor >> p.flat_shift);
        const uint32_t off = (cursor & ((1u << p.flat_shift) - 1)) * p.flat_tile;
        if (off >= c.n) continue;
        const uint32_t n = min(p.flat_tile, c.n - off), slot = loaded % n_stages;
        dptr[slot] = p.dst.base + c.dst_off + off;
        nbytes[slot] = n;
        mbar_expect_tx(&full[slot], n);
        bulk_g2s(ring + (size_t)slot * stage_bytes, p.src.base + c.src_off + off, n, &full[slot], pol);
        ++loaded;
        cursor += gridDim.x;
        return true;
      }
      return false;
    };
    for (uint32_t k = 0; k + 1 < n_stages; ++k)
      if (!issue_next()) break;
    while (stored < loaded) {
      const uint32_t slot = stored % n_stages;
      mbar_wait(&full[slot], (stored / n_stages) & 1);
      bulk_s2g(dptr[slot], ring + (size_t)slot * stage_bytes, nbytes[slot], pol);
      bulk_commit();
      ++stored;
      // the next load reuses the slot of store `stored-2`: all but the latest store have finished reading smem
      bulk_wait_read<1>();
      issue_next();
    }
    bulk_wait_all();
  }
  __syncwarp();
  const uint32_t n_ragged = p.n_tiles - n_flat_tiles;   // partial last blocks: rows tiles, 128-bit vectors
  const uint32_t vpr = p.row_bytes / 16;
  for (uint32_t tile = blockIdx.x; tile < n_ragged; tile += gridDim.x) {
    uint32_t plane, ci;
    decode_tile(p, tile, plane, ci);
    const Chunk c = cs.get(p.n_flat + ci);
    const char* s = p.src.base + side_offset<false>(p.src, nullptr, c.src_off, plane, c.req_tokens, p.tok_bytes);
    char* d = p.dst.base + side_offset<false>(p.dst, nullptr, c.dst_off, plane, c.req_tokens, p.tok_bytes);
    copy_rows<16, 8, 0>(p, s, d, c.n, threadIdx.x, 32, vpr, false, 0);
  }
}

// ------------------------------------------------------------------------------------------------
// bulk / rows: the TMA TENSOR path (cp.async.bulk.tensor -> UTMALDG / UTMASTG).  Both pools are 5-D tensors over
// (row element, token in block, head, block, plane) — same dimension order, different strides (tma.cpp).  One
// thread per CTA loads a box of (row, box_tok tokens, Hkv heads) through the src map into a ring slot, where it
// sits as dense [head][token][row] bytes, and stores the slot through the dst map: the token-major -> head-major
// conversion and the block-size change (BASELINE configs[3]) happen in the TMA unit's address generation.  No payload
// registers, no LSU slots — the shape that co-runs with GEMMs.  Chunks shorter than a box (the
// ragged end of a request, reading A4) move token by token through 1-token boxes, so nothing past T_r is touched.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tma_load_5d(void* smem_dst, const CUtensorMap* map, uint32_t c1, uint32_t c3, uint32_t c4,
                                            uint64_t* bar, uint64_t pol) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3, %4, %5, %6}], [%7], %8;" ::"r"(smem_u32(smem_dst)),
      "l"(map), "r"(0), "r"(c1), "r"(0), "r"(c3), "r"(c4), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void tma_store_5d(const CUtensorMap* map, uint32_t c1, uint32_t c3, uint32_t c4, const void* smem_src,
                                             uint64_t pol) {
  asm volatile(
      "cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group.L2::cache_hint"
      " [%0, {%1, %2, %3, %4, %5}], [%6], %7;" ::"l"(map),
      "r"(0), "r"(c1), "r"(0), "r"(c3), "r"(c4), "r"(smem_u32(smem_src)), "l"(pol) : "memory");
}

struct RowsTmaParams {              // by value in the kernel parameters; the maps must be __grid_constant__
  CUtensorMap src_full, dst_full, src_one, dst_one;
  int64_t  src_s_block, dst_s_block, src_s_token, dst_s_token;
  uint32_t box_tok, tok_slot, stage_bytes, n_stages;
};

template <class CS>
__global__ void __launch_bounds__(32, 1) fk_rows_tma(const __grid_constant__ KernelParams p, const __grid_constant__ CS cs,
                                                     const __grid_constant__ RowsTmaParams tp) {
  extern __shared__ __align__(128) char ring[];
  __shared__ __align__(8) uint64_t full[kBulkMaxStages];
  __shared__ uint32_t s_db[kBulkMaxStages], s_dt[kBulkMaxStages], s_n[kBulkMaxStages], s_plane[kBulkMaxStages];
  pdl_launch_dependents();
  if (threadIdx.x != 0) return;                       // one thread drives the TMA unit
  for (uint32_t i = 0; i < tp.n_stages; ++i) mbar_init(&full[i], 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  const uint64_t pol = policy_evict_first();
  pdl_wait_prior_grid();

  const uint32_t first = blockIdx.x, stride = gridDim.x;
  const uint32_t n_my = first < p.n_tiles ? (p.n_tiles - first + stride - 1) / stride : 0;
  const uint32_t ahead = tp.n_stages - 1;

  auto issue_load = [&](uint32_t k) {
    uint32_t plane, ci;
    decode_tile(p, first + k * stride, plane, ci);
    const Chunk c = cs.get(ci);
    // chunk offsets are bytes inside one plane: block * s_block + token * s_token (planner.cpp pool_off)
    const uint32_t sb = (uint32_t)(c.src_off / tp.src_s_block), st = (uint32_t)((c.src_off - sb * tp.src_s_block) / tp.src_s_token);
    const uint32_t db = (uint32_t)(c.dst_off / tp.dst_s_block), dt = (uint32_t)((c.dst_off - db * tp.dst_s_block) / tp.dst_s_token);
    const uint32_t slot = k % tp.n_stages;
    s_db[slot] = db; s_dt[slot] = dt; s_n[slot] = c.n; s_plane[slot] = plane;
    char* buf = ring + (size_t)slot * tp.stage_bytes;
    if (c.n == tp.box_tok) {
      mbar_expect_tx(&full[slot], c.n * p.tok_bytes);
      tma_load_5d(buf, &tp.src_full, st, sb, plane, &full[slot], pol);
    } else {                                          // ragged chunk: token by token (A4: nothing past T_r moves)
      mbar_expect_tx(&full[slot], c.n * p.tok_bytes);
      for (uint32_t t = 0; t < c.n; ++t) tma_load_5d(buf + (size_t)t * tp.tok_slot, &tp.src_one, st + t, sb, plane, &full[slot], pol);
    }
  };

  for (uint32_t k = 0; k < ahead && k < n_my; ++k) issue_load(k);
  for (uint32_t k = 0; k < n_my; ++k) {
    const uint32_t slot = k % tp.n_stages;
    mbar_wait(&full[slot], (k / tp.n_stages) & 1);    // the box has landed in its slot
    const char* buf = ring + (size_t)slot * tp.stage_bytes;
    const uint32_t n = s_n[slot], db = s_db[slot], dt = s_dt[slot], plane = s_plane[slot];
    if (n == tp.box_tok) {
      tma_store_5d(&tp.dst_full, dt, db, plane, buf, pol);
    } else {
      for (uint32_t t = 0; t < n; ++t) tma_store_5d(&tp.dst_one, dt + t, db, plane, buf + (size_t)t * tp.tok_slot, pol);
    }
    bulk_commit();
    if (k + ahead < n_my) {
      bulk_wait_read<1>();                            // slot of tile k-1 has been read out by its store
      issue_load(k + ahead);
    }
  }
  bulk_wait_all();
}

// ------------------------------------------------------------------------------------------------
// launcher
// ------------------------------------------------------------------------------------------------
// One launch with the programmatic-stream-serialization attribute (see pdl_launch_dependents()).  FLOWKV_PDL=0 in
// the environment turns the attribute off (A/B measurements); results never depend on it.
static bool pdl_enabled() {
  static const bool on = [] { const char* e = getenv("FLOWKV_PDL"); return !(e && e[0] == '0'); }();
  return on;
}
template <class... KArgs, class... Args>
static cudaError_t launch_kernel(void (*kernel)(KArgs...), uint32_t grid, uint32_t block, size_t smem, cudaStream_t st,
                                 Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(block);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl_enabled() ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

template <int VEC, int UNROLL, class CS>
static cudaError_t launch_ldst(Mode mode, const KernelParams& kp, const CS& cs, const LaunchShape& ls, int hint,
                               cudaStream_t st) {
#define FK_LAUNCH(KERNEL)                                                                                  \
  switch (hint) {                                                                                          \
    case 0: return launch_kernel(KERNEL<VEC, UNROLL, 0, CS>, ls.grid, ls.threads, 0, st, kp, cs);          \
    case 1: return launch_kernel(KERNEL<VEC, UNROLL, 1, CS>, ls.grid, ls.threads, 0, st, kp, cs);          \
    default: return launch_kernel(KERNEL<VEC, UNROLL, 2, CS>, ls.grid, ls.threads, 0, st, kp, cs);         \
  }
  if (mode == MODE_SPAN) { FK_LAUNCH(fk_span_ldst) }
  else if (mode == MODE_FLAT) { FK_LAUNCH(fk_flat_ldst) }
  else { FK_LAUNCH(fk_rows_ldst) }
#undef FK_LAUNCH
}

uint32_t bulk_max_smem() {
  int dev = 0, v = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return 0;
  return (uint32_t)v;
}

template <class CS>
static int launch_with(Mode mode, const KernelParams& kp, const CS& cs, const LaunchShape& ls, cudaStream_t st,
                       const RowsTma* tma) {
  if (ls.variant == FLOWKV_VARIANT_BULK && mode == MODE_ROWS && tma && tma->ok) {
    RowsTmaParams tp;
    tp.src_full = tma->src_full; tp.dst_full = tma->dst_full; tp.src_one = tma->src_one; tp.dst_one = tma->dst_one;
    tp.src_s_block = tma->src_s_block; tp.dst_s_block = tma->dst_s_block;
    tp.src_s_token = tma->src_s_token; tp.dst_s_token = tma->dst_s_token;
    tp.box_tok = tma->box_tok; tp.tok_slot = tma->tok_slot; tp.stage_bytes = ls.stage_bytes; tp.n_stages = ls.n_stages;
    const uint32_t smem = ls.n_stages * ls.stage_bytes;
    cudaError_t e = cudaFuncSetAttribute(fk_rows_tma<CS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
    return (int)launch_kernel(fk_rows_tma<CS>, ls.grid, 32, smem, st, kp, cs, tp);
  }
  if (ls.variant == FLOWKV_VARIANT_BULK && mode == MODE_SPAN) {
    const uint32_t smem = ls.n_stages * ls.stage_bytes;
    cudaError_t e = cudaFuncSetAttribute(fk_span_bulk<CS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
    return (int)launch_kernel(fk_span_bulk<CS>, ls.grid, 32, smem, st, kp, cs, ls.stage_bytes, ls.n_stages);
  }
  if (ls.variant == FLOWKV_VARIANT_BULK && mode == MODE_FLAT) {
    const uint32_t smem = ls.n_stages * ls.stage_bytes;
    cudaError_t e = cudaFuncSetAttribute(fk_flat_bulk<CS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
    return (int)launch_kernel(fk_flat_bulk<CS>, ls.grid, 32, smem, st, kp, cs, ls.stage_bytes, ls.n_stages);
  }
  if (ls.vec_bytes == 32) return (int)launch_ldst<32, 4, CS>(mode, kp, cs, ls, (int)ls.hint, st);
  return (int)launch_ldst<16, 8, CS>(mode, kp, cs, ls, (int)ls.hint, st);
}

// Pools whose planes are separate allocations (reading A22): the *_po kernels take the per-plane offset tables as one
// more parameter.  They exist for the uploaded schedule and for three parameter forms (16, 96 and 512 entries), in span
// and rows mode — such pools are never flat and never on
// the TMA tensor path — so the kernels of every other pool stay exactly what they were.
template <class CS>
static int launch_with_po(Mode mode, const KernelParams& kp, const CS& cs, const LaunchShape& ls, cudaStream_t st,
                          const PlaneOffs& po) {
  if (mode != MODE_SPAN && mode != MODE_ROWS) return (int)cudaErrorInvalidValue;
  if (ls.variant == FLOWKV_VARIANT_BULK && mode == MODE_SPAN) {
    const uint32_t smem = ls.n_stages * ls.stage_bytes;
    cudaError_t e = cudaFuncSetAttribute(fk_span_bulk_po<CS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
    return (int)launch_kernel(fk_span_bulk_po<CS>, ls.grid, 32, smem, st, kp, cs, ls.stage_bytes, ls.n_stages, po);
  }
#define FK_LAUNCH_PO(KERNEL, VEC, UNROLL)                                                                       \
  switch ((int)ls.hint) {                                                                                      \
    case 0: return (int)launch_kernel(KERNEL<VEC, UNROLL, 0, CS>, ls.grid, ls.threads, 0, st, kp, cs, po);     \
    case 1: return (int)launch_kernel(KERNEL<VEC, UNROLL, 1, CS>, ls.grid, ls.threads, 0, st, kp, cs, po);     \
    default: return (int)launch_kernel(KERNEL<VEC, UNROLL, 2, CS>, ls.grid, ls.threads, 0, st, kp, cs, po);    \
  }
  if (mode == MODE_SPAN) {
    if (ls.vec_bytes == 32) { FK_LAUNCH_PO(fk_span_ldst_po, 32, 4) }
    FK_LAUNCH_PO(fk_span_ldst_po, 16, 8)
  }
  if (ls.vec_bytes == 32) { FK_LAUNCH_PO(fk_rows_ldst_po, 32, 4) }
  FK_LAUNCH_PO(fk_rows_ldst_po, 16, 8)
#undef FK_LAUNCH_PO
}

// The parameter block of the larger forms (8-16 KiB) is not built on the stack of every launch, nor allocated and freed
// per launch: each thread keeps one block per form for its lifetime (cudaLaunchKernelEx copies the arguments before it
// returns, so the block is free again at once).
template <uint32_t N>
static ParamChunks<N>& param_scratch() {
  static thread_local ParamChunks<N> pc;
  return pc;
}
template <uint32_t N>
static int launch_inline(Mode mode, const KernelParams& kp, const Chunk* host_chunks, uint32_t n, const LaunchShape& ls,
                         cudaStream_t st, const RowsTma* tma) {
  if (N <= 96) {
    ParamChunks<N> pc;
    memcpy(pc.c, host_chunks, (size_t)n * sizeof(Chunk));
    return launch_with(mode, kp, pc, ls, st, tma);
  }
  ParamChunks<N>& pc = param_scratch<N>();
  memcpy(pc.c, host_chunks, (size_t)n * sizeof(Chunk));
  return launch_with(mode, kp, pc, ls, st, tma);
}
template <uint32_t N>
static int launch_inline_po(Mode mode, const KernelParams& kp, const Chunk* host_chunks, uint32_t n, const LaunchShape& ls,
                            cudaStream_t st, const PlaneOffs& po) {
  if (N <= 96) {
    ParamChunks<N> pc;
    memcpy(pc.c, host_chunks, (size_t)n * sizeof(Chunk));
    return launch_with_po(mode, kp, pc, ls, st, po);
  }
  ParamChunks<N>& pc = param_scratch<N>();
  memcpy(pc.c, host_chunks, (size_t)n * sizeof(Chunk));
  return launch_with_po(mode, kp, pc, ls, st, po);
}

int launch_copy(Mode mode, const KernelParams& kp, const Chunk* device_chunks, const Chunk* host_chunks,
                uint32_t n_host_chunks, const LaunchShape& ls, void* stream, const RowsTma* tma, const PlaneOffs* po) {
  cudaStream_t st = (cudaStream_t)stream;
  if (host_chunks && n_host_chunks > kInlineChunks) return (int)cudaErrorInvalidValue;
  if (po && (po->src || po->dst)) {        // planes of a side are separate allocations (A22)
    if (!host_chunks) return launch_with_po(mode, kp, GlobalChunks{device_chunks}, ls, st, *po);
    // small schedules take the 512-byte / 3 KiB parameter forms like every other pool (parameter bytes cost launch
    // time); the larger ones share the 16 KiB form
    if (n_host_chunks <= kInlineTiers[0]) return launch_inline_po<kInlineTiers[0]>(mode, kp, host_chunks, n_host_chunks, ls, st, *po);
    if (n_host_chunks <= kInlineTiers[1]) return launch_inline_po<kInlineTiers[1]>(mode, kp, host_chunks, n_host_chunks, ls, st, *po);
    return launch_inline_po<kInlineTiers[3]>(mode, kp, host_chunks, n_host_chunks, ls, st, *po);
  }
  if (host_chunks) {                       // small plan: the schedule rides in the kernel parameters
    if (n_host_chunks <= kInlineTiers[0]) return launch_inline<kInlineTiers[0]>(mode, kp, host_chunks, n_host_chunks, ls, st, tma);
    if (n_host_chunks <= kInlineTiers[1]) return launch_inline<kInlineTiers[1]>(mode, kp, host_chunks, n_host_chunks, ls, st, tma);
    if (n_host_chunks <= kInlineTiers[2]) return launch_inline<kInlineTiers[2]>(mode, kp, host_chunks, n_host_chunks, ls, st, tma);
    return launch_inline<kInlineTiers[3]>(mode, kp, host_chunks, n_host_chunks, ls, st, tma);
  }
  GlobalChunks gc{device_chunks};
  return launch_with(mode, kp, gc, ls, st, tma);
}

// ------------------------------------------------------------------------------------------------
// ldst / tables: no host plan at all.  tile -> (plane, request, granule); the group reads its two block ids
// from device-resident tables and moves one granule (min(BS_s, BS_d) tokens) of one plane in rows form.
// Segments are irrelevant to this kernel (a granule of a plane is >= one block-plane of contiguous bytes on
// the token-major side), so nothing has to be coalesced, uploaded or even known on the host — the tables may
// change between replays of a captured graph.
// ------------------------------------------------------------------------------------------------
// Address of token t0 of request r in plane `plane` on one side; `ok` is cleared when a block id is out of range.
template <bool PO>
__device__ __forceinline__ int64_t tables_side(const Side& sd, const int64_t* po, const int32_t* tab, uint32_t max_blocks,
                                               uint32_t bs_log2, int64_t s_block, uint32_t num_blocks, uint32_t r, uint32_t t0,
                                               uint32_t plane, uint32_t T, uint64_t tok0, uint32_t tok_bytes, bool& ok) {
  if (sd.dense)       // layer window in wire order (A12/A20): request base + plane slab + token
    return (int64_t)tok0 * sd.s_layer + ((int64_t)(plane - sd.plane0) * T + t0) * (int64_t)tok_bytes;
  const int32_t b = __ldg(tab + (size_t)r * max_blocks + (t0 >> bs_log2));
  if ((uint32_t)b >= num_blocks) ok = false;
  const int64_t pl = (PO && po) ? __ldg(po + plane) : (int64_t)(plane >> 1) * sd.s_layer + (int64_t)(plane & 1) * sd.s_kv;
  return pl + (int64_t)b * s_block + (int64_t)(t0 & ((1u << bs_log2) - 1)) * sd.s_token;
}

template <int VEC, int UNROLL, int HINT, bool PO>
__device__ __forceinline__ void tables_kernel(const TablesParams& tp, const int64_t* po_src, const int64_t* po_dst) {
  const KernelParams& p = tp.kp;
  const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t G = 1u << p.group_log2;
  const uint32_t lane = gtid & (G - 1);
  const uint32_t n_groups = (gridDim.x * blockDim.x) >> p.group_log2;
  const uint64_t pol = (HINT == 2 && VEC == 16) ? policy_evict_first() : 0;
  const uint32_t vpr = p.row_bytes / VEC;
  const bool pow2 = (p.vpr_log2 != 0xffffffffu) && (p.heads_log2 != 0xffffffffu);
  const uint32_t g = 1u << tp.granule_log2;
  const uint32_t per_plane = tp.n_reqs * tp.q_per_req;
  pdl_launch_dependents();
  pdl_wait_prior_grid();               // the tables themselves may have been written by the previous kernel
  for (uint32_t tile = gtid >> p.group_log2; tile < tp.n_tiles; tile += n_groups) {
    const uint32_t pl = tile / per_plane, rq = tile - pl * per_plane;
    const uint32_t plane = pl + p.plane0;
    const uint32_t r = rq / tp.q_per_req, q = rq - r * tp.q_per_req;
    uint32_t T;
    uint64_t tok0 = 0;                                 // tokens of the requests before r (dense side only)
    if (tp.cu_tokens) { tok0 = __ldg(tp.cu_tokens + r); T = (uint32_t)(__ldg(tp.cu_tokens + r + 1) - tok0); }
    else              { T = __ldg(tp.num_tokens + r); }
    // A length above the host's max_tokens breaks the call's contract: the grid was sized from max_tokens, so the
    // tokens past it are never visited.  The host cannot see the lengths; the request's first tile reports it (bit 4).
    if (T > tp.max_tokens && q == 0 && pl == 0 && tp.error && lane == 0) atomicOr(tp.error, 4u);
    const uint32_t t0 = q << tp.granule_log2;
    if (t0 >= T) continue;
    const uint32_t n = min(g, T - t0);
    bool ok = true;
    const int64_t so = tables_side<PO>(p.src, po_src, tp.src_tables, tp.max_src_blocks, tp.src_bs_log2, tp.src_s_block, tp.src_num_blocks,
                                   r, t0, plane, T, tok0, p.tok_bytes, ok);
    const int64_t dof = tables_side<PO>(p.dst, po_dst, tp.dst_tables, tp.max_dst_blocks, tp.dst_bs_log2, tp.dst_s_block, tp.dst_num_blocks,
                                    r, t0, plane, T, tok0, p.tok_bytes, ok);
    uint32_t bad = ok ? 0u : 1u;
    if (tp.cu_tokens && (tok0 + T) * (uint64_t)(p.src.dense ? p.src.s_layer : p.dst.s_layer) > tp.dense_bytes) bad |= 2u;
    if (bad) {                                         // nothing out of bounds is touched; the caller reads the flag
      if (tp.error && lane == 0) atomicOr(tp.error, bad);
      continue;
    }
    copy_rows<VEC, UNROLL, HINT>(p, p.src.base + so, p.dst.base + dof, n, lane, G, vpr, pow2, pol);
  }
}
template <int VEC, int UNROLL, int HINT>
__global__ void __launch_bounds__(512, 2) fk_tables_ldst(const __grid_constant__ TablesParams tp) {
  tables_kernel<VEC, UNROLL, HINT, false>(tp, nullptr, nullptr);
}
template <int VEC, int UNROLL, int HINT>              // planes of a side are separate allocations (A22)
__global__ void __launch_bounds__(512, 2) fk_tables_ldst_po(const __grid_constant__ TablesParams tp,
                                                            const __grid_constant__ PlaneOffs po) {
  tables_kernel<VEC, UNROLL, HINT, true>(tp, po.src, po.dst);
}

int launch_tables(const TablesParams& tp, const LaunchShape& ls, void* stream, const PlaneOffs* po) {
  cudaStream_t st = (cudaStream_t)stream;
  if (po && (po->src || po->dst)) {
    if (ls.vec_bytes == 32) return (int)launch_kernel(fk_tables_ldst_po<32, 4, 2>, ls.grid, ls.threads, 0, st, tp, *po);
    return (int)launch_kernel(fk_tables_ldst_po<16, 8, 2>, ls.grid, ls.threads, 0, st, tp, *po);
  }
  if (ls.vec_bytes == 32) return (int)launch_kernel(fk_tables_ldst<32, 4, 2>, ls.grid, ls.threads, 0, st, tp);
  return (int)launch_kernel(fk_tables_ldst<16, 8, 2>, ls.grid, ls.threads, 0, st, tp);
}

// ------------------------------------------------------------------------------------------------
// flowkv_transfer_static: the schedule-in-global-memory kernels with the schedule in memory nobody allocates.
//
// A schedule of more than kInlineChunks entries does not fit the kernel parameters, so the ordinary path
// (flowkv_plan) puts it into a device buffer it allocates for the plan.  Some callers must not allocate on the
// device after start-up: a serving engine that has handed all of HBM to its own block pool (a later cudaMalloc
// can fail, or shrink what the engine believes it owns), a decode loop that cannot afford the device-wide
// synchronisation cudaMalloc / cudaFree imply, a process held to a fixed memory budget by its operator.  For them
// the schedule lives in the array below — part of the library's image, so every GPU that loads the library holds
// these kStaticChunks * 32 bytes (1 MiB) until the process exits, used or not.
//
// Host code cannot use the name `g_static_schedule` as a pointer: on the host it is only a handle for the
// runtime's symbol calls.  static_schedule_setup() asks the runtime for the array's address on the CURRENT device
// (once per device, remembered) and that address is what the kernel receives.
//
// The array is shared by every call on a device and keeps whatever the last call wrote.  Nothing in it has to
// start at zero: a launch reads entries [0, n) only, and the call has just written exactly those.  Two calls whose
// GPU work overlaps (different streams, no event between them) race on it; calls on one stream are ordered.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) Chunk g_static_schedule[kStaticChunks];

namespace {
struct StaticSetup { Chunk* addr = nullptr; uint32_t num_sms = 0; };
std::mutex g_static_mu;
StaticSetup g_static_setup[64];
}  // namespace

int static_schedule_setup(Chunk** addr, uint32_t* num_sms) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return (int)e;
  if (dev < 0 || dev >= 64) return (int)cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_static_mu);
  StaticSetup& su = g_static_setup[dev];
  if (!su.addr) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_schedule);       // the array's address on device `dev` (current)
    if (e != cudaSuccess) return (int)e;
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return (int)e;
    su.num_sms = (uint32_t)sms;
    su.addr = (Chunk*)p;
  }
  *addr = su.addr;
  *num_sms = su.num_sms;
  return 0;
}

int launch_copy_static(Mode mode, const KernelParams& kp, const Chunk* host_chunks, uint32_t n, Chunk* device_addr,
                       const LaunchShape& ls, void* stream) {
  if (!host_chunks || !device_addr || n == 0 || n > kStaticChunks || ls.variant != FLOWKV_VARIANT_LDST)
    return (int)cudaErrorInvalidValue;
  cudaStream_t st = (cudaStream_t)stream;
  // Pageable source: the runtime copies it into its own staging before it returns, so the caller may free the plan
  // right after this call; the copy itself is ordered on `st` like any other, behind the previous call's kernel.
  cudaError_t e = cudaMemcpyAsync(device_addr, host_chunks, (size_t)n * sizeof(Chunk), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return (int)e;
  return launch_with(mode, kp, GlobalChunks{device_addr}, ls, st, nullptr);
}

}  // namespace flowkv
