/*
 * flowkv.h — C-ABI boundary of the B200-native FlowKV KV-cache transfer path.
 *
 * What the path is (arXiv 2504.03775; "P:Lnn" = /root/reference/PAPER.md line nn):
 *   P:L69  §3.1   "transfers the KV Cache K and V from node P_p to node D_d"
 *   P:L92  §3.3   the KV cache is paged (logical -> physical block mapping), so a request's
 *                 cache is many small scattered chunks
 *   P:L98-103 Eq.5  two orders of the same pool axes, (L,2,B,H) and (B,L,2,H)
 *   P:L107 §3.3, Fig.5  "bidirectional segment alignment": compare the block-id lists
 *                 of sender and receiver, merge ids that are memory-contiguous on BOTH sides into
 *                 one transfer
 * Restated for one B200 (BASELINE.json north_star): the "transfer" is a block-table driven
 * gather / layout-convert / scatter between two pools in HBM (or a dense staging buffer in
 * device or mapped pinned host memory), executed by ONE persistent sm_100a kernel per batch.
 *
 * Result that every entry point below reaches exactly (pure byte movement):
 *   for every request r, token t in [0,T_r), layer l, c in {K,V}, head h, dim d
 *     dst[l, c, Dst_r[t div BS_d], t mod BS_d, h, d] := src[l, c, Src_r[t div BS_s], t mod BS_s, h, d]
 *   each side addressed as base + l*s_layer + c*s_kv + blk*s_block + tok*s_token + h*s_head + d*e
 *   (plane_offsets[2*l + c] in place of l*s_layer + c*s_kv for a pool whose planes are separate allocations).
 *   Every other byte of dst keeps its value; src is never written.
 *
 * Conventions
 *   - All functions return a flowkv_status, never throw, never abort, never call exit.
 *   - "host" / "device" is stated for every pointer.  Pools, staging buffers and streams are
 *     the caller's; the library never allocates, frees or reallocs them.  A plan owns only
 *     its own small descriptor buffers (host + device).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - All validation happens in flowkv_plan(); flowkv_transfer / pack / unpack and their layer
 *     forms enqueue EXACTLY ONE kernel on the caller's stream (zero for an empty plan or range)
 *     and return without synchronising.  flowkv_transfer_via_host is the one composite call
 *     (2 kernels per layer chunk); it does not synchronise either.
 *   - A built plan's flowkv_transfer is capturable into a CUDA graph (it is one launch).
 *   - Every kernel is launched with the programmatic-stream-serialization attribute: it lets the next kernel of the
 *     stream become resident while it drains, and waits for the previous kernel's memory before touching any
 *     (griddepcontrol), so stream order holds as usual.  FLOWKV_PDL=0 in the environment turns the attribute off.
 *   - There is no CPU fallback and no other backend: without a CUDA device every call that
 *     needs one returns FLOWKV_ERR_CUDA.
 *   - Thread safety: distinct plans may be used from distinct threads; one plan is run from one
 *     thread at a time (flowkv_transfer_via_host keeps its helper streams and events in the
 *     plan); flowkv_last_error() is thread-local.
 */
#ifndef FLOWKV_H_
#define FLOWKV_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FLOWKV_VERSION 4

#if defined(__GNUC__)
#define FLOWKV_API __attribute__((visibility("default")))
#else
#define FLOWKV_API
#endif

typedef enum {
  FLOWKV_OK = 0,
  FLOWKV_ERR_INVALID_ARG = 1,      /* NULL where a pointer is required, bad enum / flag           */
  FLOWKV_ERR_BLOCK_OOB = 2,        /* a block id is < 0 or >= num_blocks of its pool               */
  FLOWKV_ERR_TABLE_LEN = 3,        /* n_*_blocks != ceil(num_tokens / block_size)                  */
  FLOWKV_ERR_DST_ALIAS = 4,        /* same dst block named twice in the batch (write race)        */
  FLOWKV_ERR_ALIGN = 5,            /* a base, stride or the row size is not a multiple of 16 B     */
  FLOWKV_ERR_SHAPE_MISMATCH = 6,   /* src and dst pools differ in L, Hkv, Dh or elem_bytes         */
  FLOWKV_ERR_UNSUPPORTED = 7,      /* e.g. block_size not a power of two, plan lacks the operation */
  FLOWKV_ERR_STAGING_TOO_SMALL = 8,
  FLOWKV_ERR_NOMEM = 9,
  FLOWKV_ERR_CUDA = 10             /* a CUDA runtime call failed; flowkv_last_error() has its text */
} flowkv_status;

/* Pool layouts.  `dim` (head_dim elements of elem_bytes) is always innermost and contiguous.
 *   LKBTHD  [layer][K|V][block][token][head][dim]  — Eq. 5 left side  (L,2,B,H), H=[token][head][dim]
 *   BLKHTD  [block][layer][K|V][head][token][dim]  — Eq. 5 right side (B,L,2,H), H=[head][token][dim]
 *   STRIDED caller fills stride_bytes[] itself (separate K and V tensors, padded blocks, ...).
 *   BLKTHD  [block][layer][K|V][token][head][dim]  — Eq. 5 right side (B,L,2,H) with H exactly as on the
 *           left side: the paper's own re-order, which only moves the block axis outwards.          */
typedef enum {
  FLOWKV_LAYOUT_LKBTHD = 0,
  FLOWKV_LAYOUT_BLKHTD = 1,
  FLOWKV_LAYOUT_STRIDED = 2,
  FLOWKV_LAYOUT_BLKTHD = 3
} flowkv_layout;

enum { FLOWKV_S_LAYER = 0, FLOWKV_S_KV = 1, FLOWKV_S_BLOCK = 2, FLOWKV_S_TOKEN = 3, FLOWKV_S_HEAD = 4 };

/* A paged KV pool.  Caller-owned memory. */
typedef struct {
  void*    base;            /* DEVICE pointer to element [0,0,0,0,0,0]; 16-B aligned (32-B enables 256-bit accesses) */
  uint32_t num_layers;      /* L                                                                    */
  uint32_t num_kv_heads;    /* Hkv                                                                  */
  uint32_t head_dim;        /* Dh; head_dim*elem_bytes (one "row") must be a multiple of 16 bytes   */
  uint32_t elem_bytes;      /* e; the library is dtype-agnostic, bytes move verbatim                */
  uint32_t num_blocks;      /* NB                                                                   */
  uint32_t block_size;      /* BS, tokens per block; power of two                                   */
  uint32_t layout;          /* flowkv_layout                                                        */
  uint32_t _reserved;
  int64_t  stride_bytes[5]; /* layer, kv, block, token, head — see FLOWKV_S_*; multiples of 16      */
  const int64_t* plane_offsets; /* NULL, or HOST array [2*num_layers] (borrowed for the call; a plan keeps a copy): plane
                             * p = 2*layer + (0 for K, 1 for V) starts plane_offsets[p] bytes from `base`, and
                             * stride_bytes[FLOWKV_S_LAYER] and [FLOWKV_S_KV] are ignored.  For a cache whose layers — and
                             * possibly K and V inside a layer — are separate allocations: the state the paper starts
                             * from, "separate tensor structures across all layer dimensions" (DESIGN.md readings
                             * A22, A3).  Set base to any one of the tensors and the offsets to the signed distances;
                             * multiples of 16, any order, gaps allowed.  One tensor per layer with K and V stacked inside
                             * is plane_offsets[2l + c] = layer_offset[l] + c * s_kv.  The block, token and head strides
                             * describe one plane.  Such pools run the register / bulk-copy paths (no flat mode, no TMA
                             * tensor path) through kernels of their own; a schedule of <= 512 entries then always rides
                             * in the 512-byte, 3 KiB or 16 KiB parameter form (16 / 96 / 512 entries). */
} flowkv_pool;

/* One request: its length and both sides' block-id lists.
 * HOST pointers, borrowed only for the duration of flowkv_plan().
 * A request need not start at token 0 of a sequence: to move only tokens [t0, T) — the suffix a prefix-cache match on
 * the decode side leaves, or the chunk a chunked prefill has just produced — pass the tables from entry
 * t0 / block_size on and num_tokens = T - t0 (t0 a multiple of both block sizes). */
typedef struct {
  uint32_t       num_tokens;     /* T_r; 0 is legal (contributes nothing)                          */
  uint32_t       n_src_blocks;   /* must equal ceil(T_r / src.block_size) when src pool is given   */
  const int32_t* src_blocks;     /* HOST; may be NULL when the plan has no src pool                */
  const int32_t* dst_blocks;     /* HOST; may be NULL when the plan has no dst pool                */
  uint32_t       n_dst_blocks;   /* must equal ceil(T_r / dst.block_size) when dst pool is given   */
  uint32_t       _reserved;
} flowkv_request;

/* One aligned segment (read-only view for tests / reporting): a maximal stretch of a request whose
 * token slots are consecutive on BOTH sides (unique, in request order then token order). */
typedef struct {
  uint32_t request;         /* index into reqs[]                                                    */
  uint32_t first_token;     /* first token of the stretch within its request                        */
  uint32_t n_tokens;
  uint32_t src_block, src_tok_off;   /* where it starts on the src side (0,0 without a src pool)    */
  uint32_t dst_block, dst_tok_off;   /* where it starts on the dst side (0,0 without a dst pool)    */
  uint32_t _reserved;
  uint64_t staging_tok_off; /* exclusive prefix sum of T over the requests before `request`         */
} flowkv_segment;

/* Plan flags */
#define FLOWKV_CHECK_DST_ALIAS   (1u << 0)  /* reject a dst block id used twice (A9)                 */
#define FLOWKV_PLAN_NO_TRANSFER  (1u << 1)  /* do not build the pool->pool schedule                  */
#define FLOWKV_PLAN_NO_PACK      (1u << 2)  /* do not build the pool->staging schedule               */
#define FLOWKV_PLAN_NO_UNPACK    (1u << 3)  /* do not build the staging->pool schedule               */

/* Optional tuning; zero-initialise for defaults.  Never changes results, only the schedule. */
typedef struct {
  uint32_t tile_bytes;      /* max bytes one thread group copies per tile (0 = auto; pow2, 1 KiB..1 MiB) */
  uint32_t ctas_per_sm;     /* resident CTAs per SM of the persistent grid (0 = auto)               */
  uint32_t max_sms;         /* SM budget: grid = min(#SMs, max_sms) * ctas_per_sm (0 = all SMs; P:L92 co-run) */
  uint32_t threads;         /* threads per CTA (0 = auto; power of two in [32, 512])                */
  uint32_t group_threads;   /* threads that share one tile (0 = auto; 32..threads, power of two)    */
  uint32_t variant;         /* flowkv_variant (0 = auto)                                            */
  uint32_t tile_order;      /* 0 = auto, 1 = plane-major (all tiles of plane 0, then plane 1, ...), 2 = chunk-major */
  uint32_t cache_hint;      /* ldst: 0 = auto, 1 = default caching, 2 = L1::no_allocate, 3 = + L2::evict_first */
  uint32_t stages;          /* bulk: ring depth (0 = auto; 2..16)                                   */
  uint32_t plan_in_params;  /* 0 = auto: a plan whose schedules have <= 512 entries each is passed in the kernel
                             *     parameters (no device allocation, no upload, no event, no free: one stream call per
                             *     step; plan_device_bytes == 0).  Four parameter forms — 16 entries (512 B), 96
                             *     (3 KiB), 256 (8 KiB), 512 (16 KiB) — the smallest that fits is used per launch;
                             * 1 = always upload                                                    */
  uint32_t _reserved[2];
} flowkv_tuning;

typedef enum {
  FLOWKV_VARIANT_AUTO = 0,
  FLOWKV_VARIANT_LDST = 1,   /* register path: 128/256-bit ld.global / st.global, unrolled        */
  FLOWKV_VARIANT_BULK = 2    /* TMA path: cp.async.bulk gmem->smem->gmem ring driven by one thread  */
} flowkv_variant;

typedef struct flowkv_plan_s flowkv_plan_t;

typedef struct {
  uint64_t n_requests, n_segments;
  uint64_t total_tokens, payload_bytes;     /* payload = total_tokens * 2*L*Hkv*Dh*e                */
  uint64_t staging_bytes;                   /* dense wire size == payload_bytes                     */
  uint64_t n_chunks_transfer, n_chunks_pack, n_chunks_unpack;  /* schedule entries per plane         */
  uint64_t plan_device_bytes;               /* descriptor bytes resident on the device              */
  uint32_t n_planes;                        /* 2*L                                                  */
  uint32_t mode_transfer, mode_pack, mode_unpack;   /* 0 = absent, 1 = span (contiguous per plane), 2 = rows,
                                                     * 3 = flat (block-major both sides, same interior: a run of
                                                     *     whole blocks is one byte range over all layers, Eq. 5) */
  uint32_t grid, threads, group_threads, tile_bytes, variant, vec_bytes;   /* launch shape in use   */
  uint32_t tile_order, cache_hint, stages, smem_bytes;                     /* (resolved, not 0)     */
  uint32_t num_sms;
  uint32_t n_flat_chunks;                   /* mode 3: whole-block byte ranges (no plane term; <= 32 tiles each) among n_chunks_transfer */
} flowkv_plan_stats;

/* Fill stride_bytes[] of a LKBTHD / BLKHTD / BLKTHD pool from its shape.  STRIDED: validates only.
 * pool: HOST pointer, read-write. */
FLOWKV_API flowkv_status flowkv_pool_strides(flowkv_pool* pool);

/* Build a plan: validate (a1), bidirectional segment alignment (a2), tile schedule (a3),
 * upload (a4; one stream-ordered allocation from a library-owned memory pool + one cudaMemcpyAsync from cached pinned memory on a library-owned
 * upload stream; `stream` only waits on the upload's event.  The call does not synchronise with `stream` or with
 * any caller kernel, so planning and uploading batch k+1 overlap the move of batch k: pinned staging buffers
 * whose previous upload is still in flight are skipped (cudaEventQuery) and a fresh one is taken; only with 256
 * uploads in flight at once does the call wait for the oldest — a few-KiB DMA on the library's own stream.  Small
 * plans are not uploaded at all: their schedule travels in the kernel parameters, see
 * flowkv_tuning.plan_in_params).
 *   src, dst : HOST pointers to pool descriptors; either may be NULL (pack-only / unpack-only).
 *   reqs     : HOST array of n_reqs requests (n_reqs may be 0).
 *   tuning   : HOST pointer or NULL.
 *   out      : HOST pointer; receives the plan (caller destroys it).  Untouched on error.
 * The plan stays valid until destroyed; pools must stay alive while it is run.  The first plan (or table-driven call)
 * that names a new plane_offsets[] array copies it to the device once (16*L bytes on the library's own stream, waited
 * for; cached by content, at most 64 tables, see flowkv_trim) — the one exception to "does not synchronise".  Inside a
 * stream capture the table must already be cached: make one call (or build any plan) with the same offsets first.
 * Errors (nothing is allocated or enqueued when one is returned):
 *   INVALID_ARG  out NULL, both pools NULL, reqs NULL with n_reqs > 0, a table pointer NULL, unknown flag /
 *                layout / tuning value, a zero shape field or a stride <= 0
 *   ALIGN        a base, a stride, a plane offset or head_dim*elem_bytes is not a multiple of 16 bytes
 *   SHAPE_MISMATCH  src and dst differ in L, Hkv, Dh or elem_bytes
 *   TABLE_LEN    n_*_blocks != ceil(num_tokens / block_size);  BLOCK_OOB  an id outside [0, num_blocks)
 *   DST_ALIAS    (only with FLOWKV_CHECK_DST_ALIAS) a dst block id named twice in the batch
 *   UNSUPPORTED  block_size not a power of two, a block spanning >= 4 GiB, a row > 1 MiB, a token > 16 MiB per plane,
 *                >= 2^31 tiles in one batch (split it)
 *   NOMEM        host allocation failed;  CUDA  a runtime call failed (no device, allocation, upload) */
FLOWKV_API flowkv_status flowkv_plan(const flowkv_pool* src, const flowkv_pool* dst,
                          const flowkv_request* reqs, uint32_t n_reqs, uint32_t flags,
                          const flowkv_tuning* tuning, void* stream, flowkv_plan_t** out);

/* Host-only variant of the same planner: no CUDA call at all (segments + stats only; the plan
 * cannot be run).  Used by host-logic tests and multi-process sharding tests. */
FLOWKV_API flowkv_status flowkv_plan_host(const flowkv_pool* src, const flowkv_pool* dst,
                               const flowkv_request* reqs, uint32_t n_reqs, uint32_t flags,
                               const flowkv_tuning* tuning, flowkv_plan_t** out);

/* stats: HOST out.  segments: HOST out, receives a pointer owned by the plan (n_segments entries,
 * valid until flowkv_plan_destroy); may be NULL. */
FLOWKV_API flowkv_status flowkv_plan_info(const flowkv_plan_t* plan, flowkv_plan_stats* stats,
                               const flowkv_segment** segments);

/* Pool -> pool (a5; "transfers the KV Cache K and V from node P_p to node D_d", through both block tables
 * P:L107).  One kernel launch on `stream`; no host synchronisation.  dst may be device memory of this GPU or a
 * peer's pool mapped into this process (CUDA IPC / peer access).
 * Errors: INVALID_ARG plan NULL; UNSUPPORTED the plan has no pool->pool schedule (one pool NULL or
 * FLOWKV_PLAN_NO_TRANSFER) or was built by flowkv_plan_host; CUDA the launch failed. */
FLOWKV_API flowkv_status flowkv_transfer(const flowkv_plan_t* plan, void* stream);

/* Pool -> dense staging (a6) / dense staging -> pool (a7).  Wire format (A12):
 * [request][layer][K|V][token][head][dim], requests concatenated; request r starts at byte
 * staging_tok_off(r) * bytes_per_token.  `staging`: DEVICE pointer, or a mapped pinned HOST
 * pointer reachable from the device (UVA); 16-B aligned; `bytes` >= staging_bytes.
 * Errors: INVALID_ARG plan or staging NULL; ALIGN staging not 16-B aligned; STAGING_TOO_SMALL; UNSUPPORTED the plan
 * lacks that schedule (pool NULL / FLOWKV_PLAN_NO_PACK / _NO_UNPACK / host plan); CUDA the launch failed. */
FLOWKV_API flowkv_status flowkv_pack(const flowkv_plan_t* plan, void* staging, uint64_t bytes, void* stream);
FLOWKV_API flowkv_status flowkv_unpack(const flowkv_plan_t* plan, const void* staging, uint64_t bytes, void* stream);

/* Layer-range variants (S§8f NEXT-2; the paper's "layerwise" ablation P:L222-224 and the overlap of transfer
 * with prefill of later layers): only layers [layer_begin, layer_end) move; everything else —
 * including the wire-format slabs of other layers in `staging` — is untouched.  One launch each
 * (zero when the range is empty).  FLOWKV_ERR_INVALID_ARG if the range is not inside [0, num_layers]. */
FLOWKV_API flowkv_status flowkv_transfer_layers(const flowkv_plan_t* plan, uint32_t layer_begin, uint32_t layer_end, void* stream);
FLOWKV_API flowkv_status flowkv_pack_layers(const flowkv_plan_t* plan, void* staging, uint64_t bytes,
                                            uint32_t layer_begin, uint32_t layer_end, void* stream);
FLOWKV_API flowkv_status flowkv_unpack_layers(const flowkv_plan_t* plan, const void* staging, uint64_t bytes,
                                              uint32_t layer_begin, uint32_t layer_end, void* stream);

/* Layer-window variants: `window` is a dense buffer that holds ONLY layers [layer_begin, layer_end), in the wire
 * order of a model with that many layers: [request][layer - layer_begin][K|V][token][head][dim], requests
 * concatenated; request r starts at byte staging_tok_off(r) * 2*(layer_end-layer_begin)*Hkv*Dh*e.  Each window is a
 * self-contained contiguous message of flowkv_window_bytes() bytes — what a layer-wise / pipelined sender puts
 * on the wire — so a transfer can be cut into layer chunks that need no full-size staging
 * buffer.  The window [0, num_layers) is the wire format of flowkv_pack.  One launch each (zero if empty).
 * `window`: DEVICE or mapped pinned HOST pointer, 16-B aligned, `bytes` >= flowkv_window_bytes(). */
FLOWKV_API flowkv_status flowkv_window_bytes(const flowkv_plan_t* plan, uint32_t layer_begin, uint32_t layer_end, uint64_t* bytes);
FLOWKV_API flowkv_status flowkv_pack_window(const flowkv_plan_t* plan, void* window, uint64_t bytes,
                                            uint32_t layer_begin, uint32_t layer_end, void* stream);
FLOWKV_API flowkv_status flowkv_unpack_window(const flowkv_plan_t* plan, const void* window, uint64_t bytes,
                                              uint32_t layer_begin, uint32_t layer_end, void* stream);

/* Pool -> pinned host -> pool with both PCIe directions busy at once (S§8f NEXT-3: chunked pinned-host
 * pipeline; the host buffer stands in for the network endpoint, BASELINE.json north_star).  dst ends up exactly
 * as after flowkv_transfer.  The layers are cut into `n_chunks` groups (0 = default; clamped to [1, L]); a chunk
 * comes back as soon as it has landed on the host, so the outbound leg of chunk c+1 overlaps the inbound leg of
 * chunk c.  The helper streams and events are library-owned (cached between plans); `stream` is made to wait for
 * the last inbound chunk, so callers see ordinary stream order.  Two modes:
 *   device_scratch == NULL — direct: the pack / unpack kernels store to / load from host memory themselves (UVA);
 *     no extra device memory.  host_staging holds the wire format of flowkv_pack.  Default 16 chunks.
 *     `ctas_per_kernel` caps each kernel's grid (0 = 64: a PCIe-bound kernel needs few CTAs and both kernels must
 *     be co-resident).
 *   device_scratch != NULL — copy engines, four queues: chunk c is packed into a scratch slot in HBM
 *     (flowkv_pack_window, on `stream`), moved D2H and H2D by cudaMemcpyAsync on two copy queues of their own, and
 *     unpacked from a second slot (flowkv_unpack_window, on a fourth queue), so neither engine ever waits behind a
 *     kernel.  On B200 the copy engines sustain ~50 GB/s in both directions at once where SM loads over PCIe drop
 *     to ~38 GB/s.  n_chunks is clamped to [1, 2L]; default (0) = the divisor of 2L nearest sqrt(payload_bytes / 400 KB),
 *     within [4, 64] (equal chunks):
 *     the first outbound and the last inbound chunk cross the link alone, so many small chunks win until the
 *     hand-over between the queues (a few microseconds per chunk) outweighs the shorter head — 16 chunks for a
 *     500-token Llama-3-8B request, 64 from 12,000 tokens up.  host_staging then holds the chunks back to back: with n <= L
 *     chunk c = the layer window [L*c/n, L*(c+1)/n) at byte offset flowkv_window_bytes(0, L*c/n) (== the wire
 *     format when n_chunks == 1); with n > L chunk c = the PLANES [2L*c/n, 2L*(c+1)/n) (plane = 2*layer + K|V) in
 *     wire order [request][plane - first][token][head][dim] at byte offset total_tokens * first * Hkv*Dh*e — a layer
 *     window cut once more between K and V.  device_scratch: DEVICE
 *     pointer, 256-B aligned, scratch_bytes >= flowkv_via_host_scratch_bytes(plan, n_chunks) (4 slots of the
 *     largest chunk); caller-owned, reusable once `stream` has passed this call.  `ctas_per_kernel`: 0 = the
 *     plan's grid.
 * Launches: 2 * (non-empty chunks).  host_staging: pinned HOST pointer (mapped / UVA for the direct mode; a device
 * pointer also works in direct mode), 16-B aligned, bytes >= staging_bytes. */
FLOWKV_API flowkv_status flowkv_via_host_scratch_bytes(const flowkv_plan_t* plan, uint32_t n_chunks, uint64_t* bytes);
FLOWKV_API flowkv_status flowkv_transfer_via_host(const flowkv_plan_t* plan, void* host_staging, uint64_t bytes,
                                                  uint32_t n_chunks, uint32_t ctas_per_kernel,
                                                  void* device_scratch, uint64_t scratch_bytes, void* stream);

/* Table-driven transfer: no plan.  The block tables and lengths are DEVICE-resident (as in servers that keep
 * their block tables in HBM) and are read by the kernel itself; the host never sees them, so nothing is planned,
 * allocated or uploaded, and the call can be captured in a CUDA graph and replayed while the tables' CONTENTS change.
 * Same result as flowkv_plan + flowkv_transfer on the same tables (the definition at the top of this file); segments
 * play no role because one kernel moves everything (a tile = min(BS_s, BS_d) tokens of one plane).  One launch.
 *   src_tables  DEVICE int32 [n_reqs][max_src_blocks], row r = request r's src block ids (padding ignored)
 *   dst_tables  DEVICE int32 [n_reqs][max_dst_blocks]
 *   num_tokens  DEVICE uint32 [n_reqs]; request r moves tokens [0, num_tokens[r]); must be <= max_tokens
 *   max_tokens  upper bound of num_tokens[] known to the host (sizes the grid; tiles past a request's end exit)
 *   error_flag  DEVICE uint32 or NULL: OR-ed with 1 if a block id in use is outside its pool (that tile is
 *               skipped, nothing out of bounds is touched); the host cannot validate what it never sees.
 *               OR-ed with 4 if a request's length on the device is above max_tokens: the grid was sized from
 *               max_tokens, so that request's tokens from max_tokens (rounded up to a tile) on are NOT moved.
 *               The library only ever ORs bits into the flag and never clears or reads it: the CALLER zeroes it
 *               (cudaMemsetAsync on `stream` before the call, or once if it reads "any error since then") and
 *               reads it back after synchronising `stream`.
 *               A dst block named twice is NOT detected (undefined result, as without FLOWKV_CHECK_DST_ALIAS).
 *   tuning      threads, group_threads, max_sms, ctas_per_sm are honoured; may be NULL.
 * Errors: INVALID_ARG, ALIGN, SHAPE_MISMATCH, UNSUPPORTED as for flowkv_plan; TABLE_LEN if max_*_blocks cannot
 * hold max_tokens; CUDA.  n_reqs == 0 or max_tokens == 0: FLOWKV_OK, zero launches. */
FLOWKV_API flowkv_status flowkv_transfer_tables(const flowkv_pool* src, const flowkv_pool* dst,
                                                const int32_t* src_tables, const int32_t* dst_tables,
                                                const uint32_t* num_tokens, uint32_t n_reqs,
                                                uint32_t max_src_blocks, uint32_t max_dst_blocks, uint32_t max_tokens,
                                                uint32_t* error_flag, const flowkv_tuning* tuning, void* stream);

/* Layer-range form of flowkv_transfer_tables (S§8f NEXT-2): only layers [layer_begin, layer_end)
 * move, everything else in dst is untouched.  One launch per call (zero when the range is empty), so a layer-wise
 * sender that overlaps the transfer with the prefill of later layers needs no host plan and can live inside a
 * captured CUDA graph whose tables change between replays.  flowkv_transfer_tables == the range [0, num_layers).
 * Errors as flowkv_transfer_tables, plus INVALID_ARG for a range outside [0, num_layers]. */
FLOWKV_API flowkv_status flowkv_transfer_tables_layers(const flowkv_pool* src, const flowkv_pool* dst,
                                                       const int32_t* src_tables, const int32_t* dst_tables,
                                                       const uint32_t* num_tokens, uint32_t n_reqs,
                                                       uint32_t max_src_blocks, uint32_t max_dst_blocks, uint32_t max_tokens,
                                                       uint32_t layer_begin, uint32_t layer_end,
                                                       uint32_t* error_flag, const flowkv_tuning* tuning, void* stream);

/* Table-driven pack / unpack of the layer window [layer_begin, layer_end) (the window [0, num_layers) is the wire
 * format of flowkv_pack): the same kernel with one side dense.  Tables as for flowkv_transfer_tables; lengths come as
 *   cu_tokens   DEVICE uint64 [n_reqs + 1], exclusive prefix sums of the request lengths (cu_tokens[0] == 0): request r
 *               has cu_tokens[r+1] - cu_tokens[r] tokens (<= max_tokens) and starts at wire token offset cu_tokens[r]
 *               — the "cumulative sequence lengths" array servers already keep on the device.
 *   window      DEVICE or mapped pinned HOST pointer, 16-B aligned; `bytes` = its capacity.  The host cannot see the
 *               total length, so the bound is enforced on the device: a request that would reach past `bytes` is
 *               skipped whole and error_flag is OR-ed with 2 (1 = a block id out of range, 4 = a request longer
 *               than max_tokens, as above).
 * One launch (zero if n_reqs, max_tokens or the layer range is empty).  Errors as flowkv_transfer_tables, plus
 * INVALID_ARG for a layer range outside [0, num_layers] or a NULL window / cu_tokens, ALIGN for the window. */
FLOWKV_API flowkv_status flowkv_pack_tables(const flowkv_pool* src, const int32_t* src_tables, const uint64_t* cu_tokens,
                                            uint32_t n_reqs, uint32_t max_src_blocks, uint32_t max_tokens,
                                            void* window, uint64_t bytes, uint32_t layer_begin, uint32_t layer_end,
                                            uint32_t* error_flag, const flowkv_tuning* tuning, void* stream);
FLOWKV_API flowkv_status flowkv_unpack_tables(const flowkv_pool* dst, const int32_t* dst_tables, const uint64_t* cu_tokens,
                                              uint32_t n_reqs, uint32_t max_dst_blocks, uint32_t max_tokens,
                                              const void* window, uint64_t bytes, uint32_t layer_begin, uint32_t layer_end,
                                              uint32_t* error_flag, const flowkv_tuning* tuning, void* stream);

/* Pool -> pool for callers that must not allocate device memory: same result as flowkv_transfer, and the call itself
 * makes no cudaMalloc / cudaFree / pool allocation of any kind (no pinned host allocation either).
 *
 * Who needs it.  flowkv_plan() keeps a schedule of more than 512 entries in a device buffer it allocates per plan.
 * That is unwelcome where the process may not touch the device allocator once it is serving: an engine that gave all
 * of HBM to its own KV block pool at start-up (a later allocation can fail outright, or eat into memory the engine
 * has already promised to requests), a latency-bound loop that cannot take the device-wide stall a cudaMalloc or
 * cudaFree may bring, a tenant held to a fixed memory budget.  Such a caller plans on the host — flowkv_plan_host()
 * makes no CUDA call — and runs the plan here.
 *
 * How.  The schedule goes into a fixed array inside the library's own device image,
 * FLOWKV_STATIC_SCHEDULE_ENTRIES entries of 32 bytes = 1 MiB.  Every GPU that loads the library carries that 1 MiB
 * until the process ends, whether or not this function is ever called.  Per call: one cudaMemcpyAsync of the
 * schedule (from ordinary pageable host memory, which the runtime may hold back until earlier work on `stream` is
 * done) and one kernel launch, both on `stream`; no host synchronisation beyond that.  The plan may be destroyed as
 * soon as the call returns.
 *   plan    built by flowkv_plan_host (or flowkv_plan) with both pools; the pools are the caller's inputs / outputs
 *           as everywhere else.  Register path only: tuning.variant must be 0 or FLOWKV_VARIANT_LDST.
 *   stream  cudaStream_t as void*.
 * First call on a device: with that device current, the library looks up the array's device address once
 * (cudaGetSymbolAddress) and the SM count, and remembers both.  Make that first call outside any stream capture.
 * Sharing: all calls on a device use the one array, and it keeps the previous call's entries.  Nothing in it needs
 * clearing — a launch reads only the entries its own call has just written — but two calls whose GPU work can
 * overlap (different streams with no event between them, or two threads) race on the array and move garbage.
 * Calls on a single stream are safe back to back.
 * Errors (nothing is enqueued): INVALID_ARG plan NULL; UNSUPPORTED the plan has no pool->pool schedule, needs more
 * than FLOWKV_STATIC_SCHEDULE_ENTRIES entries (flowkv_plan_stats.n_chunks_transfer tells beforehand; split the
 * batch), asks for the bulk variant, or names a pool with plane_offsets (their device tables would have to be
 * allocated); CUDA a runtime call failed.  An empty plan is FLOWKV_OK with nothing enqueued. */
#define FLOWKV_STATIC_SCHEDULE_ENTRIES 32768u
FLOWKV_API flowkv_status flowkv_transfer_static(const flowkv_plan_t* plan, void* stream);

/* Frees the plan.  Its device buffer is released in stream order on the stream flowkv_plan() was
 * given, so kernels already queued on THAT stream stay valid; if the plan was run on another stream,
 * synchronise that stream first.  NULL is ignored. */
FLOWKV_API void flowkv_plan_destroy(flowkv_plan_t* plan);

/* Process-lifetime caches, for long-lived servers.  The library keeps, per process: the device copies of
 * plane_offsets[] tables (at most 64; beyond that the least recently used table that no plan holds is dropped, after a
 * device-wide synchronisation), pinned host buffers that stage plan uploads (64 KiB and up each, at most 256, only
 * as many as there were uploads in flight at once), and the helper streams / events of flowkv_transfer_via_host (at
 * most 8 sets).  flowkv_trim() gives back everything that is idle right now: tables no plan references (it
 * synchronises the device first — call it from a quiet moment, never inside a stream capture), staging buffers whose
 * upload has finished, unused helper streams.  Plans stay valid.  flowkv_cache_counts() reports what is held
 * (either pointer may be NULL). */
FLOWKV_API flowkv_status flowkv_trim(void);
FLOWKV_API flowkv_status flowkv_cache_counts(uint32_t* plane_offset_tables, uint32_t* pinned_buffers);

/* FLOWKV_VERSION the library was built with.  The layout of flowkv_pool changed in version 4 (plane_offsets): a caller
 * compiled against another header must not pass structs to this library — compare before the first call. */
FLOWKV_API uint32_t flowkv_version(void);

FLOWKV_API const char* flowkv_status_string(flowkv_status s);
FLOWKV_API const char* flowkv_last_error(void);          /* thread-local text of the last failure          */

/* Number of kernels this library has launched in this process (monotonic; for launch accounting). */
FLOWKV_API uint64_t flowkv_launch_count(void);
/* Number of CUDA runtime calls this library has made that put work on a stream or (de)allocate stream-ordered
 * memory — kernel launches, cudaMemcpyAsync, cudaMallocAsync / cudaFreeAsync, event records and waits
 * (monotonic).  A plan of <= 512 schedule entries makes 1 such call per step (plan + transfer + destroy: the
 * launch); an uploaded plan's step makes 6. */
FLOWKV_API uint64_t flowkv_api_call_count(void);

/* ---- comparison baselines (BASELINE.json north_star; they are NOT the product path) ----------
 * Each issues cudaMemcpyAsync D2D copies on `stream` and writes the number issued to *n_calls.
 * They require equal block sizes and either two token-major pools (LKBTHD or equivalent strides) or two
 * block-major pools with the same interior (BLKHTD/BLKTHD; FLOWKV_ERR_UNSUPPORTED otherwise).
 *   blockwise : the pre-optimisation scheme of P:L92/L103 — one copy per (block, layer, K|V) for token-major
 *               pools; for (B,L,2,H) pools one copy per whole block (Eq. 5 makes a block one range).  A partial
 *               last block copies only its valid tokens (per plane; per plane and head when head-major).
 *   segmentwise: the paper's coalescing with cudaMemcpyAsync in place of ncclSend/ncclRecv — one copy
 *               per (aligned segment, layer, K|V); for (B,L,2,H) pools ONE copy per segment (Fig. 5).    */
FLOWKV_API flowkv_status flowkv_baseline_blockwise(const flowkv_pool* src, const flowkv_pool* dst,
                                        const flowkv_request* reqs, uint32_t n_reqs,
                                        void* stream, uint64_t* n_calls);
FLOWKV_API flowkv_status flowkv_baseline_segmentwise(const flowkv_plan_t* plan, void* stream, uint64_t* n_calls);

/* ---- segment-based block allocator (S§8f NEXT-1; §3.3) ----------------------------------
 * "FlowKV manages free memory blocks with segment-based minimum heaps.  It chooses the right segments
 *  during allocation to minimize waste and merges adjacent free segments during deallocation."
 * Host-only (no CUDA).  A segment is a maximal run of consecutive free block ids.  Policy (A19):
 *   allocate(n): if some free segment holds >= n blocks, take the first n blocks of the SMALLEST such
 *   segment (ties: lowest start) — best fit, minimum waste, one segment.  Otherwise take whole free
 *   segments, largest first (ties: lowest start), until the rest fits one segment, then best-fit the
 *   rest — the fewest segments any choice can reach.  Ids are written in allocation order.
 *   free(ids): blocks return to the free set; adjacent free segments merge.
 * Errors: FLOWKV_ERR_NOMEM when fewer than n blocks are free (nothing is taken);
 *         FLOWKV_ERR_BLOCK_OOB / FLOWKV_ERR_INVALID_ARG for ids out of range / not currently allocated
 *         (nothing is freed).  All pointers are HOST pointers. */
typedef struct flowkv_allocator_s flowkv_allocator_t;
FLOWKV_API flowkv_status flowkv_alloc_create(uint32_t num_blocks, flowkv_allocator_t** out);
FLOWKV_API flowkv_status flowkv_alloc_allocate(flowkv_allocator_t* a, uint32_t n, int32_t* out_ids, uint32_t* n_segments);
FLOWKV_API flowkv_status flowkv_alloc_free(flowkv_allocator_t* a, const int32_t* ids, uint32_t n);
FLOWKV_API flowkv_status flowkv_alloc_stats(const flowkv_allocator_t* a, uint32_t* free_blocks, uint32_t* free_segments,
                                            uint32_t* largest_segment);
FLOWKV_API void flowkv_alloc_destroy(flowkv_allocator_t* a);

#ifdef __cplusplus
}
#endif
#endif /* FLOWKV_H_ */
