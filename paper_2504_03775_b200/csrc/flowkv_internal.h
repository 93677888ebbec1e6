// flowkv_internal.h — structures shared by the host planner, the C-ABI layer and the sm_100a
// kernels of the product path.  Nothing under oracle/ includes this file.
#pragma once

#include <cuda.h>          // CUtensorMap (types only; the driver is reached through cudaGetDriverEntryPoint)
#include <stdint.h>

#include <new>
#include <string>
#include <vector>

#include "../../include/flowkv.h"

namespace flowkv {

void set_last_error(const std::string& msg);     // api.cpp: thread-local text behind flowkv_last_error()

// Runs one C-ABI entry point's body; turns any C++ exception into a status code.
template <class F>
flowkv_status guarded(F&& f) noexcept {
  try {
    return f();
  } catch (const std::bad_alloc&) {
    try { set_last_error("out of host memory"); } catch (...) {}
    return FLOWKV_ERR_NOMEM;
  } catch (...) {
    try { set_last_error("unexpected C++ exception inside the library"); } catch (...) {}
    return FLOWKV_ERR_INVALID_ARG;
  }
}

// ---------------------------------------------------------------------------------------------
// Device-visible schedule entry ("chunk"): one unit of work of one plane.  The same chunk list
// serves every plane p = 2*layer + kv; the kernel adds the plane offset of each side:
//   pool side   : layer*s_layer + kv*s_kv
//   dense side  : (p - plane0) * req_tokens * tok_bytes (wire format A12: [req][l][c][t][h][d])
// span mode: `n` BYTES that are contiguous on both sides.
// rows mode: `n` TOKENS; token t, head h of the chunk sits at off + t*s_token + h*s_head per side.
// ---------------------------------------------------------------------------------------------
struct alignas(32) Chunk {
  int64_t  src_off;      // pool side: bytes from the base, plane offset excluded;
  int64_t  dst_off;      // dense side: (staging_tok_off << 32) | token_in_request (see side_offset())
  uint32_t n;            // span: bytes (multiple of the vector width); rows: tokens
  uint32_t req_tokens;   // T_r of the owning request (dense-side plane stride = T_r * tok_bytes)
  uint32_t request;      // owning request (reporting only)
  uint32_t _pad;
};
static_assert(sizeof(Chunk) == 32, "Chunk is loaded as one 32-byte vector");

// MODE_FLAT: chunks[0, n_flat) are plane-free byte ranges (whole-block runs of two congruent block-major
// pools); chunks[n_flat, n_flat + n_chunks) are rows-mode chunks (partial last blocks) served per plane.
enum Mode : uint32_t { MODE_ABSENT = 0, MODE_SPAN = 1, MODE_ROWS = 2, MODE_FLAT = 3 };

struct Side {            // one end of a copy as the kernel sees it
  char*    base;         // device (or mapped host) pointer
  int64_t  s_layer, s_kv, s_token, s_head;   // bytes; s_token/s_head used in rows mode only.  Dense side:
                         // s_layer = bytes per token of the layer window the buffer holds, s_kv unused
  uint32_t dense;        // 1: dense staging buffer, 0: paged pool
  uint32_t plane0;       // dense side: first plane of the layer window the buffer holds (0 = whole wire format)
};

// Pools whose planes are separate allocations (readings A22 / A3): per side a DEVICE array [2L] of byte offsets from the
// side's base (plane p starts at [p]; s_layer / s_kv are then unused), or NULL for an ordinary pool.  Handed to the
// *_po kernels as a parameter of their own, so that the kernels of ordinary pools are untouched by the feature.
struct PlaneOffs {
  const int64_t* src;
  const int64_t* dst;
};

// Plans whose every schedule has at most kInlineChunks entries pass them in the kernel parameters instead of
// uploading them (CUDA >= 12.1 allows 32 KiB of parameters): no allocation, no upload, no cross-stream event, no
// stream-ordered free — the whole step is ONE stream call.  Parameter bytes cost launch time (measured: ~1 us for
// 3 KiB), so four forms exist — 16 entries (512 B), 96 (3 KiB), 256 (8 KiB), 512 (16 KiB) — and a launch uses the
// smallest that holds its schedule.  Measured on configs[1] (478 entries, 16 KiB form): call-to-done latency
// 0.558 -> 0.540 ms, pipelined step 0.5243 -> 0.5232 ms, stream calls per step 6 -> 1.
constexpr uint32_t kInlineChunks = 512;
constexpr uint32_t kInlineTiers[4] = {16, 96, 256, 512};

struct KernelParams {
  Side         src, dst;
  uint32_t     n_chunks;     // per plane
  uint32_t     n_planes;     // planes this launch covers: 2*(layer_end - layer_begin)
  uint32_t     plane0;       // first plane: 2*layer_begin
  uint32_t     n_tiles;      // (n_flat << flat_shift) + n_chunks * n_planes
  uint32_t     n_flat;       // MODE_FLAT: plane-free entries at the front of chunks[] (0 otherwise)
  uint32_t     flat_shift;   // MODE_FLAT: each of them owns 2^flat_shift tile slots ...
  uint32_t     flat_tile;    //            ... of this many bytes
  uint32_t     row_bytes;    // Dh*e
  uint32_t     heads;        // Hkv
  uint32_t     tok_bytes;    // Hkv*Dh*e
  uint32_t     tile_order;   // 0 plane-major, 1 chunk-major (resolved by the plan)
  uint32_t     group_log2;   // log2(threads sharing a tile)
  uint32_t     vpr_log2;     // rows mode: log2(vectors per row) or 0xffffffff if not a power of two
  uint32_t     heads_log2;   // rows mode: log2(Hkv) or 0xffffffff
};

struct LaunchShape {
  uint32_t grid, threads, group_threads, vec_bytes;
  uint32_t variant;       // FLOWKV_VARIANT_LDST | FLOWKV_VARIANT_BULK
  uint32_t hint;          // ldst: 0 default caching, 1 L1::no_allocate, 2 + L2::evict_first
  uint32_t n_stages;      // bulk: ring depth
  uint32_t stage_bytes;   // bulk: bytes per ring slot (>= largest chunk)
};

// Rows mode through the TMA tensor path (cp.async.bulk.tensor): one 5-D tensor map per pool over
//   (row element, token in block, head, block, plane = 2*layer + kv)
// in that order on BOTH sides, whatever the pool's strides are.  A box of (row, box_tok tokens, Hkv heads, 1, 1)
// therefore lands in shared memory as dense [head][token][row] bytes and is stored through the other pool's map
// with the other pool's strides: the layout / block-size conversion is done by the TMA unit's address generation,
// one elected thread, no payload registers.  `one` = the same maps with a 1-token box for ragged chunks (A4).
struct RowsTma {
  CUtensorMap src_full, dst_full, src_one, dst_one;
  uint32_t box_tok = 0;        // tokens per full box (= largest chunk of the schedule)
  uint32_t tok_slot = 0;       // shared-memory bytes one token occupies in a ragged slot (tok_bytes rounded to 128)
  int64_t  src_s_block = 0, dst_s_block = 0, src_s_token = 0, dst_s_token = 0;
  bool     ok = false;
};
// tma.cpp — builds (and caches per pool pair) the maps; false + `why` when the shape cannot ride the tensor path
// (then the plan runs the register path and says so in flowkv_plan_stats.variant).
bool build_rows_tma(const flowkv_pool& src, const flowkv_pool& dst, const struct Geometry& g, uint32_t box_tok,
                    RowsTma& out, std::string& why);

// kernels.cu — launches exactly one kernel; returns cudaError_t as int.  The schedule entries come from
// `device_chunks`, or, when `host_chunks` is not NULL (n_host_chunks <= kInlineChunks), travel by value in
// the kernel parameters.
int launch_copy(Mode mode, const KernelParams& kp, const Chunk* device_chunks, const Chunk* host_chunks,
                uint32_t n_host_chunks, const LaunchShape& ls, void* stream, const RowsTma* tma = nullptr,
                const PlaneOffs* po = nullptr);
// Table-driven transfer (flowkv_transfer_tables): no host plan; the kernel walks device-resident block tables.
struct TablesParams {
  KernelParams    kp;          // src/dst sides, row_bytes, heads, tok_bytes, group_log2, vpr_log2, heads_log2, n_planes
  const int32_t*  src_tables;  // device [n_reqs][max_src_blocks]
  const int32_t*  dst_tables;  // device [n_reqs][max_dst_blocks]
  const uint32_t* num_tokens;  // device [n_reqs]               (pool -> pool)
  const uint64_t* cu_tokens;   // device [n_reqs + 1], exclusive prefix sums of the lengths (pack / unpack; else NULL)
  uint64_t        dense_bytes; // capacity of the dense side (pack / unpack)
  uint32_t*       error;       // device flag or NULL: set to 1 when a block id is out of range (that tile is skipped)
  int64_t         src_s_block, dst_s_block;
  uint32_t        n_reqs, max_src_blocks, max_dst_blocks;
  uint32_t        granule_log2;           // tokens per tile = min(BS_s, BS_d)
  uint32_t        src_bs_log2, dst_bs_log2;
  uint32_t        q_per_req;              // tiles per (request, plane) = ceil(max_tokens / granule)
  uint32_t        src_num_blocks, dst_num_blocks;
  uint32_t        n_tiles;                // n_planes * n_reqs * q_per_req
  uint32_t        max_tokens;             // the host's bound on the lengths; a longer request sets error bit 4
};
int launch_tables(const TablesParams& tp, const LaunchShape& ls, void* stream, const PlaneOffs* po = nullptr);

// flowkv_transfer_static (kernels.cu): the schedule sits in a file-scope __device__ array of kStaticChunks entries.
//   static_schedule_setup : address of that array on the CURRENT device + the device's SM count; the first call on a
//                           device asks the runtime (cudaGetSymbolAddress), later calls return the remembered values.
//   launch_copy_static    : copies `n` entries into the array on `stream`, then launches the one kernel (register path).
// Neither allocates anything.  cudaError_t as int.
constexpr uint32_t kStaticChunks = FLOWKV_STATIC_SCHEDULE_ENTRIES;
int static_schedule_setup(Chunk** addr, uint32_t* num_sms);
int launch_copy_static(Mode mode, const KernelParams& kp, const Chunk* host_chunks, uint32_t n, Chunk* device_addr,
                       const LaunchShape& ls, void* stream);

// Largest dynamic shared memory the bulk variant may use on the current device (0 on failure).
uint32_t bulk_max_smem();

// ---------------------------------------------------------------------------------------------
// Host planner (planner.cpp) — pure integer host code, no CUDA.
// ---------------------------------------------------------------------------------------------
struct Geometry {          // what both sides must agree on
  uint32_t L, Hkv, Dh, e;
  uint32_t row_bytes, tok_bytes;
  uint64_t bytes_per_token;
};

struct Schedule {
  Mode mode = MODE_ABSENT;
  std::vector<Chunk> chunks;     // MODE_FLAT: [flat spans][ragged rows chunks][rows chunks of everything]
  uint32_t n_flat = 0;           // MODE_FLAT: entries of the first part
  uint32_t flat_shift = 0;       // MODE_FLAT: log2(tile slots per entry); an entry covers <= tile_bytes << flat_shift
  uint32_t flat_tile = 0;        // MODE_FLAT: bytes per tile slot
  uint32_t n_ragged = 0;         // MODE_FLAT: entries of the second part
  // MODE_FLAT keeps a complete rows-mode schedule as its third part: layer-range launches use it,
  // because a layer range of a block-major pool is not one byte range per block run.
  uint32_t n_per_plane() const { return mode == MODE_FLAT ? n_ragged : (uint32_t)chunks.size(); }
};

// Is a pool's block interior token-major and dense, with consecutive blocks abutting per plane?
bool pool_is_span_capable(const flowkv_pool& p, const Geometry& g);
// Are both pools block-major (a block = one dense byte range holding all its planes, blocks abutting)
// with the same block size and the same interior strides?  Then whole-block runs are flat byte ranges.
bool pools_are_flat_congruent(const flowkv_pool& a, const flowkv_pool& b, const Geometry& g);

// Byte offset of plane (l, c) from the pool's base (uniform strides, or the caller's per-plane offsets: reading A22).
inline int64_t pool_plane_off(const flowkv_pool& p, uint32_t l, uint32_t c) {
  return p.plane_offsets ? p.plane_offsets[2 * l + c]
                         : (int64_t)l * p.stride_bytes[FLOWKV_S_LAYER] + (int64_t)c * p.stride_bytes[FLOWKV_S_KV];
}

flowkv_status validate_pool(const flowkv_pool* p, const char* which, std::string& err);
flowkv_status validate_requests(const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs,
                                uint32_t n_reqs, uint32_t flags, std::string& err);

// Bidirectional segment alignment.  `src`/`dst` may be NULL (dense side).
void align_segments(const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs,
                    uint32_t n_reqs, std::vector<flowkv_segment>& out);

// Cut aligned segments into chunks no larger than tile_bytes.
void build_schedule(const flowkv_pool* src, const flowkv_pool* dst, const Geometry& g,
                    const flowkv_request* reqs, const std::vector<flowkv_segment>& segs,
                    uint32_t tile_bytes, uint32_t vec_bytes, Schedule& out);

}  // namespace flowkv
