// api.cpp — the C-ABI of include/flowkv.h: plan objects, upload, launches, error text.
// Everything the hot path does on the device runs in kernels.cu; this file is host plumbing.
#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <unordered_map>

#include "flowkv_internal.h"

using namespace flowkv;

namespace {

thread_local std::string g_last_error;
std::atomic<uint64_t> g_launches{0};
// CUDA runtime calls that put work on a stream or (de)allocate stream-ordered memory, kernel launches
// included — the "total API calls per batch" of SURVEY §8d, next to the launch count.
std::atomic<uint64_t> g_api_calls{0};
struct EnqTag {};
inline cudaError_t operator<<(EnqTag, cudaError_t e) {
  g_api_calls.fetch_add(1, std::memory_order_relaxed);
  return e;
}
#define FK_ENQ EnqTag{} <<      /* prefix of a counted runtime call:  e = FK_ENQ cudaMemcpyAsync(...) */

flowkv_status fail(flowkv_status s, const std::string& msg) {
  g_last_error = msg;
  return s;
}
}  // namespace
namespace flowkv {
void set_last_error(const std::string& msg) { g_last_error = msg; }   // for the other translation units
}
namespace {
flowkv_status fail_cuda(cudaError_t e, const char* what) {
  g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
  return FLOWKV_ERR_CUDA;
}

bool is_pow2(uint32_t x) { return x && !(x & (x - 1)); }
uint32_t log2u(uint32_t x) { uint32_t l = 0; while ((1u << l) < x) ++l; return l; }
uint32_t log2_or_none(uint32_t x) { return is_pow2(x) ? log2u(x) : 0xffffffffu; }

// Pinned host staging for plan uploads.  A pageable cudaMemcpyAsync larger than the driver's inline
// limit waits for earlier work on the stream, which would serialise "plan batch k+1" behind "move
// batch k"; a pinned source keeps the upload a plain stream-ordered DMA.  Buffers are cached for the
// life of the process (grow-only); an event marks when the last upload that read a buffer is done.
struct PinnedBuf {
  void* p = nullptr;
  size_t cap = 0;
  cudaEvent_t ev = nullptr;
  bool pending = false;
};

class PinnedCache {
 public:
  // Never blocks on the common path: a cached buffer whose last upload is still in flight (cudaEventQuery) is
  // skipped and a fresh one is allocated instead.  Only when kMaxBuffers buffers exist and all of them are
  // pending does the call wait — outside the mutex — for the oldest upload (a few-KiB DMA on the library's own
  // upload stream, never a caller kernel: the plan pool does not reuse memory through cross-stream dependencies).
  cudaError_t acquire(size_t bytes, PinnedBuf& out) {
    PinnedBuf oldest{};
    {
      std::lock_guard<std::mutex> lk(mu_);
      for (size_t i = 0; i < free_.size(); ++i) {
        if (free_[i].cap < bytes) continue;
        if (free_[i].pending) {
          if (cudaEventQuery(free_[i].ev) != cudaSuccess) continue;     // upload still reading this buffer
          free_[i].pending = false;
        }
        out = free_[i];
        free_.erase(free_.begin() + i);
        return cudaSuccess;
      }
      if (n_alive_ >= kMaxBuffers)
        for (size_t i = 0; i < free_.size(); ++i)
          if (free_[i].cap >= bytes) { oldest = free_[i]; free_.erase(free_.begin() + i); break; }
      if (!oldest.p) ++n_alive_;
    }
    if (oldest.p) {
      cudaError_t e = cudaEventSynchronize(oldest.ev);
      if (e != cudaSuccess) { release(oldest); return e; }
      oldest.pending = false;
      out = oldest;
      return cudaSuccess;
    }
    size_t cap = 64 << 10;
    while (cap < bytes) cap <<= 1;
    PinnedBuf b;
    cudaError_t e = cudaHostAlloc(&b.p, cap, cudaHostAllocDefault);
    if (e == cudaSuccess) {
      e = cudaEventCreateWithFlags(&b.ev, cudaEventDisableTiming);
      if (e != cudaSuccess) cudaFreeHost(b.p);
    }
    if (e != cudaSuccess) {
      std::lock_guard<std::mutex> lk(mu_);
      --n_alive_;
      return e;
    }
    b.cap = cap;
    out = b;
    return cudaSuccess;
  }
  void release(const PinnedBuf& b) {
    if (!b.p) return;
    std::lock_guard<std::mutex> lk(mu_);
    free_.push_back(b);
  }
  // flowkv_trim(): give back every cached buffer whose last upload has finished (the others stay until a later trim).
  void trim() {
    std::vector<PinnedBuf> dead;
    {
      std::lock_guard<std::mutex> lk(mu_);
      for (size_t i = 0; i < free_.size();) {
        if (free_[i].pending && cudaEventQuery(free_[i].ev) != cudaSuccess) { ++i; continue; }
        dead.push_back(free_[i]);
        free_.erase(free_.begin() + i);
        --n_alive_;
      }
    }
    (void)cudaGetLastError();             // cudaErrorNotReady from the queries above is not an error
    for (PinnedBuf& b : dead) { cudaEventDestroy(b.ev); cudaFreeHost(b.p); }
  }
  size_t alive() {
    std::lock_guard<std::mutex> lk(mu_);
    return n_alive_;
  }

 private:
  static constexpr size_t kMaxBuffers = 256;
  std::mutex mu_;
  std::vector<PinnedBuf> free_;
  size_t n_alive_ = 0;
};
PinnedCache g_pinned;

// Plan uploads go through a library-owned non-blocking stream, so the upload for batch k+1 does not
// queue behind the kernel that is moving batch k on the caller's stream; the caller's stream only
// waits on the upload's event.  One stream per device, created on first use, never destroyed.
// Plan buffers come from a library-owned memory pool per device whose release threshold is "never": the default
// pool hands freed memory back to the OS at the next synchronisation, after which every cudaMallocAsync is a
// fresh driver allocation (slow, and ordered against running work).  A few hundred KiB per plan in flight stay
// cached for the life of the process.
std::mutex g_upload_mu;
cudaStream_t g_upload_stream[64] = {};
cudaMemPool_t g_plan_pool[64] = {};
cudaError_t upload_stream(int device, cudaStream_t* out, cudaMemPool_t* pool) {
  if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_upload_mu);
  if (!g_upload_stream[device]) {
    cudaStream_t st = nullptr;
    cudaError_t e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking);
    if (e != cudaSuccess) return e;
    cudaMemPoolProps props{};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = device;
    cudaMemPool_t mp = nullptr;
    e = cudaMemPoolCreate(&mp, &props);
    if (e == cudaSuccess) {
      uint64_t never = ~0ull;
      e = cudaMemPoolSetAttribute(mp, cudaMemPoolAttrReleaseThreshold, &never);
    }
    if (e == cudaSuccess) {
      // Plan buffers are freed on caller streams and allocated on the upload stream.  Reuse "through an internal
      // dependency" would make the upload of batch k+1 wait for the kernel of batch k to finish; only memory whose
      // free has already completed may be reused (otherwise the pool grows by one small buffer).
      int off = 0;
      e = cudaMemPoolSetAttribute(mp, cudaMemPoolReuseAllowInternalDependencies, &off);
    }
    if (e != cudaSuccess) {
      if (mp) cudaMemPoolDestroy(mp);
      cudaStreamDestroy(st);
      return e;
    }
    g_plan_pool[device] = mp;
    g_upload_stream[device] = st;
  }
  *out = g_upload_stream[device];
  *pool = g_plan_pool[device];
  return cudaSuccess;
}

// Per-plane offset tables (flowkv_pool.plane_offsets, reading A22) as the kernels read them: DEVICE arrays, uploaded
// once per distinct content and device and shared by every plan / call that names the same offsets.  The upload rides
// the library's own stream and is waited for — outside the cache's mutex, so a first-use upload on one thread does not
// stall planning on the others.  The cache is bounded: beyond kMaxEntries tables the least recently used one that no
// plan or running call holds is dropped, after a device-wide synchronisation (a kernel launched by a call that has
// already returned may still be reading it).  That costs a stall, but only a process that keeps re-allocating its
// per-layer cache tensors ever gets there; a server with a handful of pools never evicts.
class PlaneOffsetCache {
 public:
  static constexpr size_t kMaxEntries = 64;
  // Looks the table up (or uploads it) and takes a reference; the holder calls release() when it is done launching
  // (table-driven calls: right after the launch; plans: when the plan dies).
  cudaError_t get(int device, const int64_t* host, uint32_t n, const int64_t** out) {
    uint64_t h = 1469598103934665603ull ^ (uint64_t)device;           // FNV-1a over the offsets
    for (uint32_t i = 0; i < n; ++i) { h ^= (uint64_t)host[i]; h *= 1099511628211ull; }
    {
      std::lock_guard<std::mutex> lk(mu_);
      if (Entry* e = find(h, device, host, n)) { ++e->refs; e->last_use = ++tick_; *out = e->dev; return cudaSuccess; }
    }
    cudaStream_t up = nullptr;
    cudaMemPool_t mp = nullptr;
    cudaError_t e = upload_stream(device, &up, &mp);
    if (e != cudaSuccess) return e;
    Entry en;
    en.device = device;
    en.host.assign(host, host + n);
    e = cudaMalloc((void**)&en.dev, n * sizeof(int64_t));
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(en.dev, en.host.data(), n * sizeof(int64_t), cudaMemcpyHostToDevice, up);
    if (e == cudaSuccess) e = cudaStreamSynchronize(up);
    if (e != cudaSuccess) { cudaFree(en.dev); return e; }
    int64_t* spare = nullptr;             // ours, if another thread uploaded the same table meanwhile
    Entry victim;                         // the least recently used unreferenced table, if the cache is full
    {
      std::lock_guard<std::mutex> lk(mu_);
      if (Entry* hit = find(h, device, host, n)) {
        spare = en.dev;
        ++hit->refs; hit->last_use = ++tick_; *out = hit->dev;
      } else {
        en.refs = 1;
        en.last_use = ++tick_;
        *out = en.dev;
        entries_.emplace(h, std::move(en));
        if (entries_.size() > kMaxEntries) {
          auto lru = entries_.end();
          for (auto it = entries_.begin(); it != entries_.end(); ++it)
            if (it->second.refs == 0 && (lru == entries_.end() || it->second.last_use < lru->second.last_use)) lru = it;
          if (lru != entries_.end()) { victim = std::move(lru->second); entries_.erase(lru); }
        }
      }
    }
    if (spare) cudaFree(spare);           // never handed out
    if (victim.dev) retire(victim);
    return cudaSuccess;
  }
  void release(const int64_t* dev) {
    if (!dev) return;
    std::lock_guard<std::mutex> lk(mu_);
    for (auto& kv : entries_)
      if (kv.second.dev == dev) { if (kv.second.refs) --kv.second.refs; return; }
  }
  // flowkv_trim(): drop every table nobody holds.
  void trim() {
    std::vector<Entry> dead;
    {
      std::lock_guard<std::mutex> lk(mu_);
      for (auto it = entries_.begin(); it != entries_.end();)
        if (it->second.refs == 0) { dead.push_back(std::move(it->second)); it = entries_.erase(it); } else ++it;
    }
    for (Entry& e : dead) retire(e);
  }
  size_t size() {
    std::lock_guard<std::mutex> lk(mu_);
    return entries_.size();
  }

 private:
  struct Entry { int device = -1; std::vector<int64_t> host; int64_t* dev = nullptr; uint32_t refs = 0; uint64_t last_use = 0; };
  Entry* find(uint64_t h, int device, const int64_t* host, uint32_t n) {
    auto range = entries_.equal_range(h);
    for (auto it = range.first; it != range.second; ++it) {
      Entry& e = it->second;
      if (e.device == device && e.host.size() == n && memcmp(e.host.data(), host, n * sizeof(int64_t)) == 0) return &e;
    }
    return nullptr;
  }
  static void retire(Entry& e) {          // outside the mutex: wait for whatever may still read the table, then free it
    int cur = -1;
    cudaGetDevice(&cur);
    if (cur != e.device) cudaSetDevice(e.device);
    cudaDeviceSynchronize();
    cudaFree(e.dev);
    if (cur >= 0 && cur != e.device) cudaSetDevice(cur);
    e.dev = nullptr;
  }
  std::mutex mu_;
  std::unordered_multimap<uint64_t, Entry> entries_;
  uint64_t tick_ = 0;
};
PlaneOffsetCache g_plane_offsets;

// Helper streams and events of flowkv_transfer_via_host.  Created once and recycled between plans (a plan per
// batch would otherwise pay three cudaStreamCreate and ~100 cudaEventCreate per step).
struct ViaHostCtx {
  cudaStream_t q_d2h = nullptr, q_h2d = nullptr, q_unpack = nullptr;
  std::vector<cudaEvent_t> ev;
  int device = -1;
};
class ViaHostCache {
 public:
  ViaHostCtx* acquire(int device) {
    {
      std::lock_guard<std::mutex> lk(mu_);
      for (size_t i = 0; i < free_.size(); ++i)
        if (free_[i]->device == device) {
          ViaHostCtx* c = free_[i];
          free_.erase(free_.begin() + i);
          return c;
        }
    }
    ViaHostCtx* c = new (std::nothrow) ViaHostCtx();
    if (!c) return nullptr;
    c->device = device;
    if (cudaStreamCreateWithFlags(&c->q_d2h, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&c->q_h2d, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&c->q_unpack, cudaStreamNonBlocking) != cudaSuccess) {
      destroy(c);
      return nullptr;
    }
    return c;
  }
  void release(ViaHostCtx* c) {
    if (!c) return;
    std::lock_guard<std::mutex> lk(mu_);
    if (free_.size() < 8) { free_.push_back(c); return; }
    destroy(c);
  }
  void trim() {                           // flowkv_trim(): helper streams and events no plan is using
    std::vector<ViaHostCtx*> dead;
    {
      std::lock_guard<std::mutex> lk(mu_);
      dead.swap(free_);
    }
    for (ViaHostCtx* c : dead) destroy(c);
  }
  static void destroy(ViaHostCtx* c) {
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    if (c->q_d2h) cudaStreamDestroy(c->q_d2h);
    if (c->q_h2d) cudaStreamDestroy(c->q_h2d);
    if (c->q_unpack) cudaStreamDestroy(c->q_unpack);
    delete c;
  }

 private:
  std::mutex mu_;
  std::vector<ViaHostCtx*> free_;
};
ViaHostCache g_via_host;

struct Op {                  // one runnable operation of a plan
  Schedule sched;
  const Chunk* d_chunks = nullptr;
  LaunchShape shape{};
  uint32_t tile_order = 0;   // resolved: 0 plane-major, 1 chunk-major
  uint32_t max_chunk_bytes = 0;
  bool in_params = false;    // schedule small enough to ride in the kernel parameters (no upload)
  RowsTma tma;               // rows mode + bulk variant: the tensor maps of both pools (ok == false: register path)
};

}  // namespace

struct flowkv_plan_s {
  bool has_src = false, has_dst = false, on_device = false;
  flowkv_pool src{}, dst{};            // plane_offsets (if any) point into the copies below
  std::vector<int64_t> src_plane_off, dst_plane_off;
  const int64_t *d_src_plane_off = nullptr, *d_dst_plane_off = nullptr;   // their device copies (library cache)
  Geometry g{};
  flowkv_tuning tuning{};
  uint32_t tile_bytes = 0;
  std::vector<flowkv_segment> segments;      // the reported alignment
  std::vector<flowkv_segment> segs_pack, segs_unpack;
  Op transfer, pack, unpack;
  uint64_t n_requests = 0, total_tokens = 0;
  void* d_buf = nullptr;     // stream-ordered allocation on `stream`
  uint64_t d_bytes = 0;
  cudaStream_t stream = nullptr;   // the stream flowkv_plan() was given: it waits on the upload; the free is ordered on it
  PinnedBuf staging{};             // staging.ev = "upload done" event
  mutable std::atomic<bool> upload_seen_done{false};   // run(): the upload event has been observed complete
  // flowkv_transfer_via_host: helper streams + events, taken from a library cache on first use (plans are logically const)
  mutable ViaHostCtx* via = nullptr;
  int device = -1;
  uint32_t num_sms = 0, max_smem_optin = 0;
};

namespace {

// Planning a large batch builds vectors of a few hundred KiB (segments, schedules).  Fresh allocations of that
// size are mmap'd and page-faulted in on every plan (measured: 1.6 of 2.4 ms for configs[2]); recycling the
// vectors of destroyed plans keeps their pages.  At most kMaxCached sets, each vector capped at 64 MiB.
class VectorCache {
 public:
  void take(flowkv_plan_t* pl) {
    Set st;
    {
      std::lock_guard<std::mutex> lk(mu_);
      if (free_.empty()) return;
      st = std::move(free_.back());
      free_.pop_back();
    }
    pl->segments.swap(st.seg[0]); pl->segs_pack.swap(st.seg[1]); pl->segs_unpack.swap(st.seg[2]);
    pl->transfer.sched.chunks.swap(st.ch[0]); pl->pack.sched.chunks.swap(st.ch[1]); pl->unpack.sched.chunks.swap(st.ch[2]);
  }
  void give(flowkv_plan_t* pl) {
    Set st;
    st.seg[0].swap(pl->segments); st.seg[1].swap(pl->segs_pack); st.seg[2].swap(pl->segs_unpack);
    st.ch[0].swap(pl->transfer.sched.chunks); st.ch[1].swap(pl->pack.sched.chunks); st.ch[2].swap(pl->unpack.sched.chunks);
    size_t bytes = 0;
    for (auto& v : st.seg) { v.clear(); bytes = std::max(bytes, v.capacity() * sizeof(flowkv_segment)); }
    for (auto& v : st.ch) { v.clear(); bytes = std::max(bytes, v.capacity() * sizeof(Chunk)); }
    if (bytes < (16u << 10) || bytes > (64u << 20)) return;      // small ones are cheap to rebuild, huge ones are not kept
    std::lock_guard<std::mutex> lk(mu_);
    if (free_.size() < kMaxCached) free_.push_back(std::move(st));
  }

 private:
  static constexpr size_t kMaxCached = 8;
  struct Set { std::vector<flowkv_segment> seg[3]; std::vector<Chunk> ch[3]; };
  std::mutex mu_;
  std::vector<Set> free_;
};
VectorCache g_vectors;

void drop_plan(flowkv_plan_t* pl) {       // every way a plan object dies goes through here
  g_plane_offsets.release(pl->d_src_plane_off);
  g_plane_offsets.release(pl->d_dst_plane_off);
  g_vectors.give(pl);
  delete pl;
}

// vector width every address of an operation is aligned to
uint32_t pick_vec(const flowkv_pool* a, const flowkv_pool* b, const Geometry& g) {
  auto ok32 = [&](const flowkv_pool* p) {
    if (!p) return true;
    if ((uintptr_t)p->base % 32) return false;
    for (int i = 0; i < 5; ++i)
      if (!((i == FLOWKV_S_LAYER || i == FLOWKV_S_KV) && p->plane_offsets) && p->stride_bytes[i] % 32) return false;
    if (p->plane_offsets)
      for (uint32_t q = 0; q < 2 * p->num_layers; ++q) if (p->plane_offsets[q] % 32) return false;
    return true;
  };
  return (g.row_bytes % 32 == 0 && ok32(a) && ok32(b)) ? 32 : 16;
}

void resolve_shape(flowkv_plan_t* pl, Op& op, const flowkv_pool* a, const flowkv_pool* b) {
  const flowkv_tuning& t = pl->tuning;
  LaunchShape& ls = op.shape;
  const uint32_t sms = pl->num_sms ? pl->num_sms : 148;
  const uint32_t use_sms = t.max_sms ? std::min(t.max_sms, sms) : sms;
  ls.vec_bytes = pick_vec(a, b, pl->g);
  ls.variant = t.variant ? t.variant : FLOWKV_VARIANT_LDST;
  op.max_chunk_bytes = 0;
  for (size_t i = 0; i < op.sched.chunks.size(); ++i) {
    const Chunk& c = op.sched.chunks[i];
    if (op.sched.mode == MODE_FLAT && i < op.sched.n_flat) continue;     // cut into flat_tile pieces by the kernel
    op.max_chunk_bytes = std::max(op.max_chunk_bytes, op.sched.mode == MODE_SPAN ? c.n : c.n * pl->g.tok_bytes);
  }
  op.tma.ok = false;
  if (op.sched.mode == MODE_ROWS && ls.variant == FLOWKV_VARIANT_BULK) {
    // rows mode rides the TMA TENSOR path when both sides are pools a 5-D tensor map can describe (tma.cpp); a dense
    // side (pack / unpack: its plane stride is T_r, per request) and host-only plans run the register path
    std::string why;
    const uint32_t box_tok = op.max_chunk_bytes / pl->g.tok_bytes;
    if (!(a && b && pl->device >= 0 && box_tok && build_rows_tma(*a, *b, pl->g, box_tok, op.tma, why)))
      ls.variant = FLOWKV_VARIANT_LDST;
  }
  op.tile_order = t.tile_order == 2 ? 1 : 0;
  // Auto: plane-major, except for a rows-mode move into a block-major pool of the same block size (Eq. 5's re-layout as
  // a move, `bench.py --config cfg2mig`): a chunk is then one whole block-plane, and chunk-major order makes the CTAs
  // that run together fill ONE dst block's 2L planes — one contiguous range — instead of one plane of many blocks
  // 2 MiB apart.  Same box, two runs each: 0.5333 -> 0.5264 ms (81.8 -> 82.9 % of 8 TB/s).  With unequal block sizes
  // (configs[3]: 4 KiB pieces into 16 KiB head slabs) the order makes no difference (82.39 vs 82.44 %): unchanged.
  if (t.tile_order == 0 && op.sched.mode == MODE_ROWS && a && b && a->block_size == b->block_size && !b->plane_offsets &&
      b->stride_bytes[FLOWKV_S_BLOCK] >= b->stride_bytes[FLOWKV_S_LAYER] * (int64_t)pl->g.L)
    op.tile_order = 1;
  const uint64_t n_tiles = ((uint64_t)op.sched.n_flat << op.sched.flat_shift) + (uint64_t)op.sched.n_per_plane() * 2 * pl->g.L;
  if (ls.variant == FLOWKV_VARIANT_BULK) {
    // a ring slot holds the largest chunk (span mode: at least one token's plane bytes); two slots must fit in
    // shared memory, else the plan runs the register path (reported in flowkv_plan_stats.variant)
    uint32_t stage_need = op.sched.mode == MODE_FLAT ? op.sched.flat_tile : op.max_chunk_bytes;
    if (op.sched.mode == MODE_ROWS)          // a ragged chunk parks each token at a 128-byte aligned offset
      stage_need = std::max<uint32_t>(stage_need, (op.tma.box_tok ? op.tma.box_tok - 1 : 0) * op.tma.tok_slot);
    const uint32_t stage = ((std::max<uint32_t>(stage_need, 1024)) + 127) & ~127u;
    const uint32_t cap = (pl->max_smem_optin ? pl->max_smem_optin : 232448) - 1024;
    if (2ull * stage > cap) ls.variant = FLOWKV_VARIANT_LDST;
    ls.stage_bytes = stage;
  }
  if (ls.variant == FLOWKV_VARIANT_BULK) {
    ls.threads = 32;
    ls.group_threads = 32;
    // like the ldst path the grid is oversubscribed (<= 256 CTAs per SM) and each CTA's ring is short:
    // several small CTAs per SM, scheduled by hardware, beat one long-lived CTA with a deep ring
    const uint32_t ctas = t.ctas_per_sm ? t.ctas_per_sm : 256;
    const uint32_t smem_cap = (pl->max_smem_optin ? pl->max_smem_optin : 232448) - 1024;
    const uint32_t resident = std::min<uint32_t>(ctas, 3);
    const uint32_t budget = std::min<uint32_t>(smem_cap, (228u * 1024 - 2048) / resident - 1024);
    uint32_t stages = t.stages ? t.stages : 2;
    stages = std::min<uint32_t>(stages, 16);
    while (stages > 2 && (uint64_t)stages * ls.stage_bytes > budget) --stages;
    ls.n_stages = stages;
    ls.hint = 2;
    ls.grid = (uint32_t)std::min<uint64_t>((uint64_t)use_sms * ctas, std::max<uint64_t>(n_tiles, 1));
    return;
  }
  // Defaults from the tuning sweeps on B200 (round 1):
  //  * one CTA-wide round of 512 threads x 4 x 32 B covers a 64 KiB tile;
  //  * the grid is a grid-stride loop capped at 256 CTAs per SM.  Up to that cap every tile gets its
  //    own CTA and the hardware CTA scheduler hands tiles to whichever SM frees up first, which
  //    measured 3-6 % faster than an exactly-resident persistent grid with a static tile stride
  //    (SMs do not all drain HBM at the same rate); beyond the cap each CTA strides over tiles;
  //  * rows mode (strided rows) prefers 128-thread groups: four tiles in flight per CTA.
  ls.threads = t.threads ? t.threads : std::min<uint32_t>(512, std::max<uint32_t>(128, pl->tile_bytes / 128));
  //  * span / flat mode: the whole CTA shares one tile (round 2 re-checked 256- and 128-thread groups on configs[1]:
  //    0.5242 / 0.5285 ms against 0.5182 ms — fewer, fatter CTAs lose the fine-grained hardware scheduling).
  const uint32_t group_auto = op.sched.mode == MODE_ROWS ? std::min<uint32_t>(128, ls.threads) : ls.threads;
  ls.group_threads = t.group_threads ? std::min(t.group_threads, ls.threads) : group_auto;
  ls.hint = t.cache_hint ? t.cache_hint - 1 : 2;
  ls.n_stages = 0;
  ls.stage_bytes = 0;
  const uint32_t ctas = t.ctas_per_sm ? t.ctas_per_sm : 256;
  const uint32_t groups_per_cta = ls.threads / ls.group_threads;
  const uint64_t ctas_needed = (n_tiles + groups_per_cta - 1) / groups_per_cta;
  ls.grid = (uint32_t)std::min<uint64_t>((uint64_t)use_sms * ctas, std::max<uint64_t>(ctas_needed, 1));
}

flowkv_status check_tuning(const flowkv_tuning& t) {
  if (t.tile_bytes && (!is_pow2(t.tile_bytes) || t.tile_bytes < 1024 || t.tile_bytes > (1u << 20)))
    return fail(FLOWKV_ERR_INVALID_ARG, "tuning.tile_bytes must be a power of two in [1 KiB, 1 MiB]");
  if (t.threads && (t.threads % 32 || t.threads > 512 || !is_pow2(t.threads)))
    return fail(FLOWKV_ERR_INVALID_ARG, "tuning.threads must be a power of two in [32, 512]");
  const uint32_t thr = t.threads ? t.threads : 512;      // with threads on auto the group is clamped to it later
  if (t.group_threads && (!is_pow2(t.group_threads) || t.group_threads < 32 || t.group_threads > thr))
    return fail(FLOWKV_ERR_INVALID_ARG, "tuning.group_threads must be a power of two in [32, threads]");
  if (t.variant > FLOWKV_VARIANT_BULK) return fail(FLOWKV_ERR_INVALID_ARG, "tuning.variant unknown");
  if (t.tile_order > 2) return fail(FLOWKV_ERR_INVALID_ARG, "tuning.tile_order unknown");
  if (t.cache_hint > 3) return fail(FLOWKV_ERR_INVALID_ARG, "tuning.cache_hint unknown");
  if (t.stages && (t.stages < 2 || t.stages > 16)) return fail(FLOWKV_ERR_INVALID_ARG, "tuning.stages must be in [2,16]");
  if (t.ctas_per_sm > 1024) return fail(FLOWKV_ERR_INVALID_ARG, "tuning.ctas_per_sm must be <= 1024");
  if (t.plan_in_params > 1) return fail(FLOWKV_ERR_INVALID_ARG, "tuning.plan_in_params unknown");
  if (t.variant == FLOWKV_VARIANT_BULK && t.tile_bytes > (64u << 10))
    return fail(FLOWKV_ERR_INVALID_ARG, "bulk variant: tile_bytes must be <= 64 KiB (two ring slots must fit in shared memory)");
  return FLOWKV_OK;
}

flowkv_status make_plan(const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs, uint32_t n_reqs,
                        uint32_t flags, const flowkv_tuning* tuning, bool device, void* stream, flowkv_plan_t** out) {
  if (!out) return fail(FLOWKV_ERR_INVALID_ARG, "out is NULL");
  if (!src && !dst) return fail(FLOWKV_ERR_INVALID_ARG, "both pools are NULL");
  if (n_reqs && !reqs) return fail(FLOWKV_ERR_INVALID_ARG, "reqs is NULL");
  if (flags & ~(FLOWKV_CHECK_DST_ALIAS | FLOWKV_PLAN_NO_TRANSFER | FLOWKV_PLAN_NO_PACK | FLOWKV_PLAN_NO_UNPACK))
    return fail(FLOWKV_ERR_INVALID_ARG, "unknown flag bit");
  std::string err;
  flowkv_status st;
  if (src && (st = validate_pool(src, "src", err)) != FLOWKV_OK) return fail(st, err);
  if (dst && (st = validate_pool(dst, "dst", err)) != FLOWKV_OK) return fail(st, err);
  if (src && dst &&
      (src->num_layers != dst->num_layers || src->num_kv_heads != dst->num_kv_heads ||
       src->head_dim != dst->head_dim || src->elem_bytes != dst->elem_bytes))
    return fail(FLOWKV_ERR_SHAPE_MISMATCH, "src and dst pools differ in num_layers, num_kv_heads, head_dim or elem_bytes");
  flowkv_tuning tn{};
  if (tuning) tn = *tuning;
  if ((st = check_tuning(tn)) != FLOWKV_OK) return st;
  if ((st = validate_requests(src, dst, reqs, n_reqs, flags, err)) != FLOWKV_OK) return fail(st, err);   // (guarded by the C-ABI wrapper)

  flowkv_plan_t* pl = new (std::nothrow) flowkv_plan_s();
  if (!pl) return fail(FLOWKV_ERR_NOMEM, "out of host memory");
  g_vectors.take(pl);
  try {
    const flowkv_pool* any = src ? src : dst;
    pl->has_src = src != nullptr;
    pl->has_dst = dst != nullptr;
    if (src) pl->src = *src;
    if (dst) pl->dst = *dst;
    if (src && src->plane_offsets) {       // the caller's array is borrowed for this call only
      pl->src_plane_off.assign(src->plane_offsets, src->plane_offsets + 2 * (size_t)src->num_layers);
      pl->src.plane_offsets = pl->src_plane_off.data();
    }
    if (dst && dst->plane_offsets) {
      pl->dst_plane_off.assign(dst->plane_offsets, dst->plane_offsets + 2 * (size_t)dst->num_layers);
      pl->dst.plane_offsets = pl->dst_plane_off.data();
    }
    pl->tuning = tn;
    Geometry& g = pl->g;
    g.L = any->num_layers; g.Hkv = any->num_kv_heads; g.Dh = any->head_dim; g.e = any->elem_bytes;
    g.row_bytes = g.Dh * g.e;
    g.tok_bytes = g.Hkv * g.row_bytes;
    g.bytes_per_token = 2ull * g.L * g.tok_bytes;
    pl->n_requests = n_reqs;
    for (uint32_t r = 0; r < n_reqs; ++r) pl->total_tokens += reqs[r].num_tokens;
    if ((uint64_t)g.Hkv * g.row_bytes > (1u << 24)) {
      drop_plan(pl);
      return fail(FLOWKV_ERR_UNSUPPORTED, "token larger than 16 MiB per plane");
    }

    if (device) {
      cudaError_t e = cudaGetDevice(&pl->device);
      if (e != cudaSuccess) { drop_plan(pl); return fail_cuda(e, "cudaGetDevice"); }
      // device attributes never change: query once per device, not once per plan
      static std::atomic<uint32_t> sms_of[64], smem_of[64];
      const int di = pl->device & 63;
      if (!sms_of[di].load(std::memory_order_acquire)) {
        int v = 0;
        e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, pl->device);
        if (e != cudaSuccess) { drop_plan(pl); return fail_cuda(e, "cudaDeviceGetAttribute"); }
        smem_of[di].store(bulk_max_smem(), std::memory_order_relaxed);
        sms_of[di].store((uint32_t)v, std::memory_order_release);
      }
      pl->num_sms = sms_of[di].load(std::memory_order_relaxed);
      pl->max_smem_optin = smem_of[di].load(std::memory_order_relaxed);
      if (!pl->src_plane_off.empty())
        e = g_plane_offsets.get(pl->device, pl->src_plane_off.data(), 2 * g.L, &pl->d_src_plane_off);
      if (e == cudaSuccess && !pl->dst_plane_off.empty())
        e = g_plane_offsets.get(pl->device, pl->dst_plane_off.data(), 2 * g.L, &pl->d_dst_plane_off);
      if (e != cudaSuccess) { drop_plan(pl); return fail_cuda(e, "upload of plane_offsets"); }
    } else {
      pl->num_sms = 148;
    }

    // tile size: default 64 KiB; shrink for small batches so every SM gets several tiles
    uint32_t tile = tn.tile_bytes;
    if (!tile) {
      // ldst: one CTA-wide round of 512 threads; bulk: 2 ring slots x 32 KiB keep 3 CTAs resident per SM
      tile = tn.variant == FLOWKV_VARIANT_BULK ? (32u << 10) : (64u << 10);
      // small batches: at least two tiles per SM, but no smaller than 16 KiB — a launch-bound copy wants few, fat
      // CTAs and a schedule short enough for the 512-byte parameter form (profiles/r02_sweep.md, tuning grid:
      // 128 tokens 11.2 us with 8 KiB tiles, 10.3 us with >= 16 KiB; the same-size cudaMemcpyAsync takes 10.2 us)
      const uint64_t want_tiles = 2ull * pl->num_sms;
      const uint64_t payload = pl->total_tokens * g.bytes_per_token;
      while (tile > 16384 && payload / tile < want_tiles) tile >>= 1;
      // ... and between two and four tiles per SM (a 256-token Llama-3-8B request: 32 MiB) halve the 64 KiB tile once:
      // 1,024 CTAs of 256 threads ramp up and drain faster than 512 of 512 (round 3, 40 repetitions, three runs
      // each: contiguous request 15.2-15.3 us -> 14.3-14.5 us, single-block runs unchanged at 14.3-14.4 us; the
      // same-size cudaMemcpyAsync takes 13.2-13.7 us).  Larger requests keep 64 KiB (1,024 tokens: 46.6-47.3 us
      // against 50.5-50.8 us with the small shape).
      if (tn.variant != FLOWKV_VARIANT_BULK && tile == (64u << 10) && payload / tile < 2 * want_tiles) tile >>= 1;
    }
    pl->tile_bytes = tile;

    const bool do_transfer = src && dst && !(flags & FLOWKV_PLAN_NO_TRANSFER);
    const bool do_pack = src && !(flags & FLOWKV_PLAN_NO_PACK);
    const bool do_unpack = dst && !(flags & FLOWKV_PLAN_NO_UNPACK);
    // the reported alignment: both sides when both pools are given, else one-sided
    align_segments(src, dst, reqs, n_reqs, pl->segments);
    if (do_transfer) {
      build_schedule(src, dst, g, reqs, pl->segments, tile, 0, pl->transfer.sched);
      resolve_shape(pl, pl->transfer, src, dst);
    }
    if (do_pack) {
      if (dst) align_segments(src, nullptr, reqs, n_reqs, pl->segs_pack);
      build_schedule(src, nullptr, g, reqs, dst ? pl->segs_pack : pl->segments, tile, 0, pl->pack.sched);
      resolve_shape(pl, pl->pack, src, nullptr);
    }
    if (do_unpack) {
      if (src) align_segments(nullptr, dst, reqs, n_reqs, pl->segs_unpack);
      build_schedule(nullptr, dst, g, reqs, src ? pl->segs_unpack : pl->segments, tile, 0, pl->unpack.sched);
      resolve_shape(pl, pl->unpack, nullptr, dst);
    }
    for (Op* op : {&pl->transfer, &pl->pack, &pl->unpack})
      if ((uint64_t)op->sched.chunks.size() * 2 * g.L + ((uint64_t)op->sched.n_flat << op->sched.flat_shift) >= (1ull << 31)) {
        drop_plan(pl);
        return fail(FLOWKV_ERR_UNSUPPORTED, "more than 2^31 tiles in one batch; split the batch");
      }

    if (device) {
      // a4: one stream-ordered allocation and ONE upload (from cached pinned memory) for all schedules,
      // issued on the library's upload stream; the caller's stream waits on the upload event
      // Small plans (every schedule <= kInlineChunks entries) skip all of that: their entries are passed by
      // value in the kernel parameters at launch, so nothing stands between planning and the launch.
      uint64_t bytes = 0;
      bool small = tn.plan_in_params != 1;
      for (Op* op : {&pl->transfer, &pl->pack, &pl->unpack}) {
        bytes += op->sched.chunks.size() * sizeof(Chunk);
        small = small && op->sched.chunks.size() <= kInlineChunks;
      }
      pl->stream = (cudaStream_t)stream;
      if (small) {
        for (Op* op : {&pl->transfer, &pl->pack, &pl->unpack}) op->in_params = true;
      } else if (bytes) {
        cudaStream_t up = nullptr;
        cudaMemPool_t mp = nullptr;
        cudaError_t e = upload_stream(pl->device, &up, &mp);
        if (e != cudaSuccess) { drop_plan(pl); return fail_cuda(e, "cudaStreamCreate(upload)"); }
        e = g_pinned.acquire(bytes, pl->staging);
        if (e != cudaSuccess) { drop_plan(pl); return fail_cuda(e, "cudaHostAlloc(plan staging)"); }
        e = FK_ENQ cudaMallocFromPoolAsync(&pl->d_buf, bytes, mp, up);
        if (e != cudaSuccess) { g_pinned.release(pl->staging); drop_plan(pl); return fail_cuda(e, "cudaMallocAsync(plan)"); }
        pl->d_bytes = bytes;
        uint64_t off = 0;
        for (Op* op : {&pl->transfer, &pl->pack, &pl->unpack}) {
          const uint64_t n = op->sched.chunks.size() * sizeof(Chunk);
          if (!n) continue;
          memcpy((char*)pl->staging.p + off, op->sched.chunks.data(), n);
          op->d_chunks = (const Chunk*)((char*)pl->d_buf + off);
          off += n;
        }
        e = FK_ENQ cudaMemcpyAsync(pl->d_buf, pl->staging.p, bytes, cudaMemcpyHostToDevice, up);
        if (e == cudaSuccess) e = FK_ENQ cudaEventRecord(pl->staging.ev, up);
        if (e == cudaSuccess) e = FK_ENQ cudaStreamWaitEvent(pl->stream, pl->staging.ev, 0);
        if (e != cudaSuccess) {
          FK_ENQ cudaFreeAsync(pl->d_buf, up);
          g_pinned.release(pl->staging);
          drop_plan(pl);
          return fail_cuda(e, "cudaMemcpyAsync(plan)");
        }
        pl->staging.pending = true;
      }
      pl->on_device = true;
    }
  } catch (...) {
    // any exception (bad_alloc, length_error from a vector, ...) ends here once, with everything the plan took so far
    // given back: the device buffer (stream-ordered, on the upload stream it came from), the pinned staging buffer,
    // the plane-offset references (drop_plan); guarded() then turns the exception into a status code
    if (pl->d_buf) {
      cudaStream_t up = nullptr;
      cudaMemPool_t mp = nullptr;
      if (upload_stream(pl->device, &up, &mp) == cudaSuccess) FK_ENQ cudaFreeAsync(pl->d_buf, up);
    }
    g_pinned.release(pl->staging);
    drop_plan(pl);
    throw;
  }
  *out = pl;
  return FLOWKV_OK;
}

Side pool_side(const flowkv_pool& p) {
  Side s{};
  s.base = (char*)p.base;
  s.s_layer = p.stride_bytes[FLOWKV_S_LAYER];
  s.s_kv = p.stride_bytes[FLOWKV_S_KV];
  s.s_token = p.stride_bytes[FLOWKV_S_TOKEN];
  s.s_head = p.stride_bytes[FLOWKV_S_HEAD];
  s.dense = 0;
  return s;
}

// A dense staging buffer that holds the layer window [w0, w1) in wire order (A12).  The whole wire format
// is the window [0, L).
// A dense buffer that holds the PLANES [p0, p1) (plane = 2*layer + kv) in wire order (A21).
Side dense_planes(const void* staging, const Geometry& g, uint32_t p0, uint32_t p1) {
  Side s{};
  s.base = (char*)staging;
  s.s_layer = (int64_t)(p1 - p0) * g.tok_bytes;   // bytes per token of the window
  s.s_kv = 0;                                     // plane stride comes from the chunk's req_tokens
  s.s_token = g.tok_bytes;
  s.s_head = g.row_bytes;
  s.dense = 1;
  s.plane0 = p0;
  return s;
}
Side dense_side(const void* staging, const Geometry& g, uint32_t w0, uint32_t w1) { return dense_planes(staging, g, 2 * w0, 2 * w1); }
Side dense_side(const void* staging, const Geometry& g) { return dense_side(staging, g, 0, g.L); }

struct RunOpts {
  bool ranged = false;                       // false: all layers
  uint32_t layer_begin = 0, layer_end = 0;   // [begin, end) when ranged
  bool by_planes = false;                    // ranged by PLANES [plane_begin, plane_end) instead (via-host chunks, A21)
  uint32_t plane_begin = 0, plane_end = 0;
  uint32_t max_grid = 0;                     // 0 = the plan's launch shape
};

flowkv_status run(const flowkv_plan_t* pl, const Op& op, const Side& s, const Side& d, uint32_t vec_bytes, void* stream,
                  const RunOpts& ro = RunOpts()) {
  if (!pl->on_device) return fail(FLOWKV_ERR_UNSUPPORTED, "plan was built by flowkv_plan_host and cannot run");
  const uint32_t l0 = ro.ranged ? ro.layer_begin : 0, l1 = ro.ranged ? ro.layer_end : pl->g.L;
  if (l0 > l1 || l1 > pl->g.L) return fail(FLOWKV_ERR_INVALID_ARG, "layer range outside [0, num_layers]");
  const uint32_t p0 = ro.by_planes ? ro.plane_begin : 2 * l0, p1 = ro.by_planes ? ro.plane_end : 2 * l1;
  if (p0 > p1 || p1 > 2 * pl->g.L) return fail(FLOWKV_ERR_INVALID_ARG, "plane range outside [0, 2*num_layers]");
  if (op.sched.chunks.empty() || p0 == p1) return FLOWKV_OK;       // A11: nothing to move, zero launches
  if ((cudaStream_t)stream != pl->stream && pl->staging.ev && !pl->upload_seen_done.load(std::memory_order_acquire)) {
    // A stream other than the plan's own has not been ordered after the plan upload yet.  Once the upload is known
    // to have finished no edge is needed — which also lets a long-lived plan be captured into a CUDA graph on any
    // stream (an edge to an event recorded outside the capture would invalidate it).  The query is made in relaxed
    // capture mode: it is a host-side read of an event that belongs to no capture.
    cudaStreamCaptureMode mode = cudaStreamCaptureModeRelaxed;
    cudaThreadExchangeStreamCaptureMode(&mode);
    cudaError_t q = cudaEventQuery(pl->staging.ev);
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (q != cudaSuccess) {
      (void)cudaGetLastError();
      cudaStreamIsCapturing((cudaStream_t)stream, &cap);
      // capturing and the few-KiB upload is still in flight: the only correct order is to let it finish first
      if (cap == cudaStreamCaptureStatusActive) q = cudaEventSynchronize(pl->staging.ev);
    }
    cudaThreadExchangeStreamCaptureMode(&mode);
    if (q == cudaSuccess) {
      pl->upload_seen_done.store(true, std::memory_order_release);
    } else {
      (void)cudaGetLastError();
      cudaError_t e = FK_ENQ cudaStreamWaitEvent((cudaStream_t)stream, pl->staging.ev, 0);
      if (e != cudaSuccess) return fail_cuda(e, "cudaStreamWaitEvent(plan upload)");
    }
  }
  KernelParams kp{};
  kp.src = s; kp.dst = d;
  Mode mode = op.sched.mode;
  uint32_t first = 0;                      // first schedule entry this launch uses
  kp.n_chunks = op.sched.n_per_plane();
  kp.n_flat = op.sched.n_flat;
  kp.flat_shift = op.sched.flat_shift;
  kp.flat_tile = op.sched.flat_tile;
  if (mode == MODE_FLAT && (p0 != 0 || p1 != 2 * pl->g.L)) {
    // a layer range of a block-major pool is not one byte range per block run: use the plan's
    // complete rows-mode schedule (third part of the chunk list)
    mode = MODE_ROWS;
    first = op.sched.n_flat + op.sched.n_ragged;
    kp.n_chunks = (uint32_t)op.sched.chunks.size() - first;
    kp.n_flat = 0;
  }
  kp.n_planes = p1 - p0;
  kp.plane0 = p0;
  kp.n_tiles = (kp.n_flat << kp.flat_shift) + kp.n_chunks * kp.n_planes;
  kp.row_bytes = pl->g.row_bytes;
  kp.heads = pl->g.Hkv;
  kp.tok_bytes = pl->g.tok_bytes;
  kp.tile_order = op.tile_order;
  LaunchShape ls = op.shape;
  ls.vec_bytes = vec_bytes;
  if (ls.variant == FLOWKV_VARIANT_BULK && mode == MODE_ROWS && !op.tma.ok) {
    // a layer range of a flat (block-major) bulk plan runs its rows schedule: no tensor maps for it, register path
    ls.variant = FLOWKV_VARIANT_LDST;
    ls.threads = 512;
    ls.group_threads = 128;
    ls.hint = 2;
    ls.grid = (pl->tuning.max_sms ? std::min(pl->tuning.max_sms, pl->num_sms) : pl->num_sms) *
              (pl->tuning.ctas_per_sm ? pl->tuning.ctas_per_sm : 256);
  }
  const uint32_t groups_per_cta = ls.variant == FLOWKV_VARIANT_BULK ? 1 : ls.threads / ls.group_threads;
  ls.grid = std::min<uint32_t>(ls.grid, (kp.n_tiles + groups_per_cta - 1) / groups_per_cta);
  if (ro.max_grid) ls.grid = std::min(ls.grid, ro.max_grid);
  kp.group_log2 = log2u(ls.group_threads);
  kp.vpr_log2 = log2_or_none(kp.row_bytes / ls.vec_bytes);
  kp.heads_log2 = log2_or_none(kp.heads);
  // per-plane offset tables (A22) of whichever side is a pool of this launch (a dense side has none)
  const PlaneOffs po{s.dense ? nullptr : pl->d_src_plane_off, d.dense ? nullptr : pl->d_dst_plane_off};
  const int e = op.in_params
                    ? launch_copy(mode, kp, nullptr, op.sched.chunks.data() + first, (uint32_t)op.sched.chunks.size() - first, ls, stream, &op.tma, &po)
                    : launch_copy(mode, kp, op.d_chunks + first, nullptr, 0, ls, stream, &op.tma, &po);
  if (e != 0) return fail_cuda((cudaError_t)e, "kernel launch");
  g_launches.fetch_add(1, std::memory_order_relaxed);
  g_api_calls.fetch_add(1, std::memory_order_relaxed);
  return FLOWKV_OK;
}

flowkv_status check_staging(const flowkv_plan_t* pl, const Op& op, const void* staging, uint64_t bytes, const char* what,
                            uint64_t need = ~0ull) {
  if (op.sched.mode == MODE_ABSENT)
    return fail(FLOWKV_ERR_UNSUPPORTED, std::string("plan has no ") + what + " schedule");
  if (op.sched.chunks.empty()) return FLOWKV_OK;
  if (!staging) return fail(FLOWKV_ERR_INVALID_ARG, "staging is NULL");
  if ((uintptr_t)staging % 16) return fail(FLOWKV_ERR_ALIGN, "staging is not 16-byte aligned");
  if (need == ~0ull) need = pl->total_tokens * pl->g.bytes_per_token;
  if (bytes < need) return fail(FLOWKV_ERR_STAGING_TOO_SMALL, "staging buffer too small");
  return FLOWKV_OK;
}

uint64_t window_bytes(const flowkv_plan_t* pl, uint32_t l0, uint32_t l1) {
  return pl->total_tokens * 2ull * (l1 - l0) * pl->g.tok_bytes;
}

}  // namespace

namespace impl {

flowkv_status flowkv_pool_strides(flowkv_pool* p) {
  if (!p) return fail(FLOWKV_ERR_INVALID_ARG, "pool is NULL");
  const int64_t row = (int64_t)p->head_dim * p->elem_bytes;
  if (p->layout == FLOWKV_LAYOUT_LKBTHD) {
    p->stride_bytes[FLOWKV_S_HEAD] = row;
    p->stride_bytes[FLOWKV_S_TOKEN] = row * p->num_kv_heads;
    p->stride_bytes[FLOWKV_S_BLOCK] = p->stride_bytes[FLOWKV_S_TOKEN] * p->block_size;
    p->stride_bytes[FLOWKV_S_KV] = p->stride_bytes[FLOWKV_S_BLOCK] * p->num_blocks;
    p->stride_bytes[FLOWKV_S_LAYER] = 2 * p->stride_bytes[FLOWKV_S_KV];
  } else if (p->layout == FLOWKV_LAYOUT_BLKHTD) {
    p->stride_bytes[FLOWKV_S_TOKEN] = row;
    p->stride_bytes[FLOWKV_S_HEAD] = row * p->block_size;
    p->stride_bytes[FLOWKV_S_KV] = p->stride_bytes[FLOWKV_S_HEAD] * p->num_kv_heads;
    p->stride_bytes[FLOWKV_S_LAYER] = 2 * p->stride_bytes[FLOWKV_S_KV];
    p->stride_bytes[FLOWKV_S_BLOCK] = p->stride_bytes[FLOWKV_S_LAYER] * p->num_layers;
  } else if (p->layout == FLOWKV_LAYOUT_BLKTHD) {
    p->stride_bytes[FLOWKV_S_HEAD] = row;
    p->stride_bytes[FLOWKV_S_TOKEN] = row * p->num_kv_heads;
    p->stride_bytes[FLOWKV_S_KV] = p->stride_bytes[FLOWKV_S_TOKEN] * p->block_size;
    p->stride_bytes[FLOWKV_S_LAYER] = 2 * p->stride_bytes[FLOWKV_S_KV];
    p->stride_bytes[FLOWKV_S_BLOCK] = p->stride_bytes[FLOWKV_S_LAYER] * p->num_layers;
  } else if (p->layout != FLOWKV_LAYOUT_STRIDED) {
    return fail(FLOWKV_ERR_INVALID_ARG, "unknown layout");
  }
  for (int i = 0; i < 5; ++i)
    if (!((i == FLOWKV_S_LAYER || i == FLOWKV_S_KV) && p->plane_offsets) && p->stride_bytes[i] <= 0) return fail(FLOWKV_ERR_INVALID_ARG, "a stride is <= 0");
  return FLOWKV_OK;
}

flowkv_status flowkv_plan(const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs, uint32_t n_reqs,
                          uint32_t flags, const flowkv_tuning* tuning, void* stream, flowkv_plan_t** out) {
  return make_plan(src, dst, reqs, n_reqs, flags, tuning, true, stream, out);
}

flowkv_status flowkv_plan_host(const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs,
                               uint32_t n_reqs, uint32_t flags, const flowkv_tuning* tuning, flowkv_plan_t** out) {
  return make_plan(src, dst, reqs, n_reqs, flags, tuning, false, nullptr, out);
}

flowkv_status flowkv_plan_info(const flowkv_plan_t* pl, flowkv_plan_stats* st, const flowkv_segment** segments) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  if (st) {
    memset(st, 0, sizeof *st);
    st->n_requests = pl->n_requests;
    st->n_segments = pl->segments.size();
    st->total_tokens = pl->total_tokens;
    st->payload_bytes = pl->total_tokens * pl->g.bytes_per_token;
    st->staging_bytes = st->payload_bytes;
    st->n_chunks_transfer = pl->transfer.sched.mode == MODE_FLAT
                                ? pl->transfer.sched.n_flat + pl->transfer.sched.n_ragged
                                : pl->transfer.sched.chunks.size();
    st->n_flat_chunks = pl->transfer.sched.n_flat;
    st->n_chunks_pack = pl->pack.sched.chunks.size();
    st->n_chunks_unpack = pl->unpack.sched.chunks.size();
    st->plan_device_bytes = pl->d_bytes;
    st->n_planes = 2 * pl->g.L;
    st->mode_transfer = pl->transfer.sched.mode;
    st->mode_pack = pl->pack.sched.mode;
    st->mode_unpack = pl->unpack.sched.mode;
    const Op& op = pl->transfer.sched.mode != MODE_ABSENT ? pl->transfer
                   : (pl->pack.sched.mode != MODE_ABSENT ? pl->pack : pl->unpack);
    st->grid = op.shape.grid;
    st->threads = op.shape.threads;
    st->group_threads = op.shape.group_threads;
    st->tile_bytes = pl->tile_bytes;
    st->variant = op.shape.variant;
    st->vec_bytes = op.shape.vec_bytes;
    st->tile_order = op.tile_order + 1;
    st->cache_hint = op.shape.hint + 1;
    st->stages = op.shape.n_stages;
    st->smem_bytes = op.shape.n_stages * op.shape.stage_bytes;
    st->num_sms = pl->num_sms;
  }
  if (segments) *segments = pl->segments.data();
  return FLOWKV_OK;
}

flowkv_status flowkv_transfer_layers(const flowkv_plan_t* pl, uint32_t layer_begin, uint32_t layer_end, void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  if (pl->transfer.sched.mode == MODE_ABSENT)
    return fail(FLOWKV_ERR_UNSUPPORTED, "plan has no pool-to-pool schedule (needs both pools, no FLOWKV_PLAN_NO_TRANSFER)");
  RunOpts ro;
  ro.ranged = true; ro.layer_begin = layer_begin; ro.layer_end = layer_end;
  return run(pl, pl->transfer, pool_side(pl->src), pool_side(pl->dst), pl->transfer.shape.vec_bytes, stream, ro);
}

flowkv_status flowkv_transfer(const flowkv_plan_t* pl, void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  return impl::flowkv_transfer_layers(pl, 0, pl->g.L, stream);
}

flowkv_status flowkv_pack_layers(const flowkv_plan_t* pl, void* staging, uint64_t bytes, uint32_t layer_begin,
                                 uint32_t layer_end, void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  flowkv_status st = check_staging(pl, pl->pack, staging, bytes, "pack");
  if (st != FLOWKV_OK || pl->pack.sched.chunks.empty()) return st;
  const uint32_t vec = ((uintptr_t)staging % 32 == 0) ? pl->pack.shape.vec_bytes : 16;
  RunOpts ro;
  ro.ranged = true; ro.layer_begin = layer_begin; ro.layer_end = layer_end;
  return run(pl, pl->pack, pool_side(pl->src), dense_side(staging, pl->g), vec, stream, ro);
}

flowkv_status flowkv_pack(const flowkv_plan_t* pl, void* staging, uint64_t bytes, void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  return impl::flowkv_pack_layers(pl, staging, bytes, 0, pl->g.L, stream);
}

flowkv_status flowkv_unpack_layers(const flowkv_plan_t* pl, const void* staging, uint64_t bytes, uint32_t layer_begin,
                                   uint32_t layer_end, void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  flowkv_status st = check_staging(pl, pl->unpack, staging, bytes, "unpack");
  if (st != FLOWKV_OK || pl->unpack.sched.chunks.empty()) return st;
  const uint32_t vec = ((uintptr_t)staging % 32 == 0) ? pl->unpack.shape.vec_bytes : 16;
  RunOpts ro;
  ro.ranged = true; ro.layer_begin = layer_begin; ro.layer_end = layer_end;
  return run(pl, pl->unpack, dense_side(staging, pl->g), pool_side(pl->dst), vec, stream, ro);
}

flowkv_status flowkv_unpack(const flowkv_plan_t* pl, const void* staging, uint64_t bytes, void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  return impl::flowkv_unpack_layers(pl, staging, bytes, 0, pl->g.L, stream);
}

flowkv_status flowkv_window_bytes(const flowkv_plan_t* pl, uint32_t layer_begin, uint32_t layer_end, uint64_t* bytes) {
  if (!pl || !bytes) return fail(FLOWKV_ERR_INVALID_ARG, "NULL argument");
  if (layer_begin > layer_end || layer_end > pl->g.L) return fail(FLOWKV_ERR_INVALID_ARG, "layer range outside [0, num_layers]");
  *bytes = window_bytes(pl, layer_begin, layer_end);
  return FLOWKV_OK;
}

flowkv_status flowkv_pack_window(const flowkv_plan_t* pl, void* window, uint64_t bytes, uint32_t layer_begin,
                                 uint32_t layer_end, void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  if (layer_begin > layer_end || layer_end > pl->g.L) return fail(FLOWKV_ERR_INVALID_ARG, "layer range outside [0, num_layers]");
  flowkv_status st = check_staging(pl, pl->pack, window, bytes, "pack", window_bytes(pl, layer_begin, layer_end));
  if (st != FLOWKV_OK || pl->pack.sched.chunks.empty()) return st;
  const uint32_t vec = ((uintptr_t)window % 32 == 0) ? pl->pack.shape.vec_bytes : 16;
  RunOpts ro;
  ro.ranged = true; ro.layer_begin = layer_begin; ro.layer_end = layer_end;
  return run(pl, pl->pack, pool_side(pl->src), dense_side(window, pl->g, layer_begin, layer_end), vec, stream, ro);
}

flowkv_status flowkv_unpack_window(const flowkv_plan_t* pl, const void* window, uint64_t bytes, uint32_t layer_begin,
                                   uint32_t layer_end, void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  if (layer_begin > layer_end || layer_end > pl->g.L) return fail(FLOWKV_ERR_INVALID_ARG, "layer range outside [0, num_layers]");
  flowkv_status st = check_staging(pl, pl->unpack, window, bytes, "unpack", window_bytes(pl, layer_begin, layer_end));
  if (st != FLOWKV_OK || pl->unpack.sched.chunks.empty()) return st;
  const uint32_t vec = ((uintptr_t)window % 32 == 0) ? pl->unpack.shape.vec_bytes : 16;
  RunOpts ro;
  ro.ranged = true; ro.layer_begin = layer_begin; ro.layer_end = layer_end;
  return run(pl, pl->unpack, dense_side(window, pl->g, layer_begin, layer_end), pool_side(pl->dst), vec, stream, ro);
}

namespace {
uint32_t via_host_chunks(const flowkv_plan_t* pl, uint32_t n_chunks, bool engines) {
  // defaults measured on B200 (profiles/r02_host_route.md): the first outbound and the last inbound chunk cross the
  // link alone, so the copy-engine pipeline wants many small chunks (up to one per plane) — as long as a chunk stays
  // large against the hand-over between the queues; the direct mode pays a kernel pair per chunk and stays at layer
  // granularity
  if (n_chunks == 0) {
    n_chunks = 16;
    if (engines) {
      // time ~ payload/bw * (1 + 1/n) + n * gap: the lonely head and tail shrink with n, every chunk costs a few
      // microseconds of queue hand-over.  The minimum sits at n = sqrt(payload / (bw * gap)) = sqrt(payload / 400 KB)
      // at ~50 GB/s and ~8 us; measured optimum on the paper's request sizes (profiles/r02_table3.md): 16 chunks at
      // 500 tokens (62.5 MiB), 32 at 4,000, 64 from 12,000 tokens up.
      const double payload = (double)pl->total_tokens * (double)pl->g.bytes_per_token;
      const double target = std::min(64.0, std::max(4.0, std::sqrt(payload / 400e3)));
      // ... and chunks of EQUAL size: among the counts that divide the 2L planes evenly, the one nearest the target
      // on a log scale (26 chunks of 2-3 planes measured 6.6 ms where 16 or 32 equal chunks take 6.1-6.2 ms)
      const uint32_t planes = 2 * pl->g.L;
      uint32_t best = std::min<uint32_t>(planes, 4);
      double best_err = 1e30;
      for (uint32_t d = std::min<uint32_t>(planes, 4); d <= std::min<uint32_t>(planes, 64); ++d) {
        if (planes % d) continue;
        const double err = std::fabs(std::log((double)d / target));
        if (err < best_err) { best_err = err; best = d; }
      }
      n_chunks = best;
    }
  }
  return std::max<uint32_t>(1, std::min(n_chunks, engines ? 2 * pl->g.L : pl->g.L));
}
// Chunk c of n covers the planes [first, last): whole layers while n <= L (the layer windows of A20), single planes
// or small groups of planes beyond that (plane windows, A21).
void via_host_chunk_planes(const flowkv_plan_t* pl, uint32_t n_chunks, uint32_t c, uint32_t& first, uint32_t& last) {
  const uint64_t L = pl->g.L;
  if (n_chunks <= L) { first = 2 * (uint32_t)(L * c / n_chunks); last = 2 * (uint32_t)(L * (c + 1) / n_chunks); }
  else               { first = (uint32_t)(2 * L * c / n_chunks); last = (uint32_t)(2 * L * (c + 1) / n_chunks); }
}
uint64_t planes_bytes(const flowkv_plan_t* pl, uint32_t p0, uint32_t p1) { return pl->total_tokens * (uint64_t)(p1 - p0) * pl->g.tok_bytes; }
uint64_t via_host_slot_bytes(const flowkv_plan_t* pl, uint32_t n_chunks) {
  uint32_t most = 0;                     // planes of the largest chunk
  for (uint32_t c = 0; c < n_chunks; ++c) {
    uint32_t a, b;
    via_host_chunk_planes(pl, n_chunks, c, a, b);
    most = std::max(most, b - a);
  }
  return (planes_bytes(pl, 0, most) + 255) & ~255ull;
}
}  // namespace

flowkv_status flowkv_via_host_scratch_bytes(const flowkv_plan_t* pl, uint32_t n_chunks, uint64_t* bytes) {
  if (!pl || !bytes) return fail(FLOWKV_ERR_INVALID_ARG, "NULL argument");
  *bytes = 4 * via_host_slot_bytes(pl, via_host_chunks(pl, n_chunks, true));
  return FLOWKV_OK;
}

flowkv_status flowkv_transfer_via_host(const flowkv_plan_t* pl, void* host_staging, uint64_t bytes, uint32_t n_chunks,
                                       uint32_t ctas_per_kernel, void* device_scratch, uint64_t scratch_bytes,
                                       void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  flowkv_status st = check_staging(pl, pl->pack, host_staging, bytes, "pack");
  if (st != FLOWKV_OK) return st;
  st = check_staging(pl, pl->unpack, host_staging, bytes, "unpack");
  if (st != FLOWKV_OK) return st;
  if (pl->pack.sched.chunks.empty()) return FLOWKV_OK;
  if (!pl->on_device) return fail(FLOWKV_ERR_UNSUPPORTED, "plan was built by flowkv_plan_host and cannot run");
  const uint32_t L = pl->g.L;
  const bool engines = device_scratch != nullptr;          // copy engines drive the link, kernels stay in HBM
  n_chunks = via_host_chunks(pl, n_chunks, engines);
  const uint64_t slot = via_host_slot_bytes(pl, n_chunks);
  if (engines) {
    if ((uintptr_t)device_scratch % 256) return fail(FLOWKV_ERR_ALIGN, "device_scratch is not 256-byte aligned");
    if (scratch_bytes < 4 * slot) return fail(FLOWKV_ERR_STAGING_TOO_SMALL, "device_scratch smaller than flowkv_via_host_scratch_bytes()");
  }
  cudaStream_t s = (cudaStream_t)stream;
  cudaError_t e;
  if (!pl->via) {
    pl->via = g_via_host.acquire(pl->device);
    if (!pl->via) return fail(FLOWKV_ERR_CUDA, "cudaStreamCreate(via-host helper streams)");
  }
  ViaHostCtx& vc = *pl->via;
  const size_t n_events = 4 * (size_t)n_chunks + 2;
  while (vc.ev.size() < n_events) {
    cudaEvent_t ev;
    e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
    if (e != cudaSuccess) return fail_cuda(e, "cudaEventCreate");
    vc.ev.push_back(ev);
  }
#define FK_TRY(call, what) do { if ((e = FK_ENQ call) != cudaSuccess) return fail_cuda(e, what); } while (0)
  RunOpts ro;
  ro.ranged = true;
  if (!engines) {
    // direct mode: the kernels touch host memory themselves; pack on `stream`, unpack on a helper stream.
    // A PCIe-bound kernel needs few CTAs and both directions' kernels must be co-resident.
    cudaStream_t aux = vc.q_unpack;
    cudaEvent_t e_start = vc.ev[4 * (size_t)n_chunks], e_done = vc.ev[4 * (size_t)n_chunks + 1];
    FK_TRY(cudaEventRecord(e_start, s), "cudaEventRecord");
    FK_TRY(cudaStreamWaitEvent(aux, e_start, 0), "cudaStreamWaitEvent");
    const uint32_t vec = ((uintptr_t)host_staging % 32 == 0) ? pl->pack.shape.vec_bytes : 16;
    const uint32_t vecu = ((uintptr_t)host_staging % 32 == 0) ? pl->unpack.shape.vec_bytes : 16;
    ro.max_grid = ctas_per_kernel ? ctas_per_kernel : 64;
    for (uint32_t c = 0; c < n_chunks; ++c) {
      ro.layer_begin = (uint32_t)((uint64_t)L * c / n_chunks);
      ro.layer_end = (uint32_t)((uint64_t)L * (c + 1) / n_chunks);
      if (ro.layer_begin == ro.layer_end) continue;
      st = run(pl, pl->pack, pool_side(pl->src), dense_side(host_staging, pl->g), vec, s, ro);          // D2H on `stream`
      if (st != FLOWKV_OK) return st;
      FK_TRY(cudaEventRecord(vc.ev[c], s), "cudaEventRecord");
      FK_TRY(cudaStreamWaitEvent(aux, vc.ev[c], 0), "cudaStreamWaitEvent");
      st = run(pl, pl->unpack, dense_side(host_staging, pl->g), pool_side(pl->dst), vecu, aux, ro);     // H2D on the helper
      if (st != FLOWKV_OK) return st;
    }
    FK_TRY(cudaEventRecord(e_done, aux), "cudaEventRecord");
    FK_TRY(cudaStreamWaitEvent(s, e_done, 0), "cudaStreamWaitEvent");
    return FLOWKV_OK;
  }
  // Copy-engine mode, four queues so that neither engine ever waits behind a kernel:
  //   `stream`  pack kernels      pool -> out slot (k & 1)           waits: D2H of chunk k-2 has drained that slot
  //   q_d2h     cudaMemcpyAsync   out slot -> host chunk             waits: pack k
  //   q_h2d     cudaMemcpyAsync   host chunk -> in slot 2 + (k & 1)  waits: D2H k; unpack k-2 has drained that slot
  //   q_unpack  unpack kernels    in slot -> pool                    waits: H2D k
  // Chunk k is its own dense message (a layer window, A20, or — with more chunks than layers — a plane window, A21)
  // at the host offset of its first plane.  While chunk k
  // crosses the link outbound, chunk k-1 crosses it inbound and chunks k+1 / k-2 are packed / unpacked in HBM.
  ro.max_grid = ctas_per_kernel;
  char* scratch = (char*)device_scratch;
  cudaEvent_t* packed = vc.ev.data();                       // [n_chunks] each
  cudaEvent_t* landed = packed + n_chunks;
  cudaEvent_t* arrived = landed + n_chunks;
  cudaEvent_t* unpacked = arrived + n_chunks;
  uint32_t k = 0;                                           // non-empty chunks so far
  int64_t prev1 = -1, prev2 = -1;                           // chunk indices of the two previous non-empty chunks
  ro.by_planes = true;
  ro.layer_begin = 0;
  ro.layer_end = L;
  for (uint32_t c = 0; c < n_chunks; ++c) {
    uint32_t p0, p1;
    via_host_chunk_planes(pl, n_chunks, c, p0, p1);
    if (p0 == p1) continue;
    ro.plane_begin = p0;
    ro.plane_end = p1;
    const uint64_t wb = planes_bytes(pl, p0, p1);
    char* out_slot = scratch + (k & 1) * slot;
    char* in_slot = scratch + (2 + (k & 1)) * slot;
    char* host = (char*)host_staging + planes_bytes(pl, 0, p0);
    if (prev2 >= 0) FK_TRY(cudaStreamWaitEvent(s, landed[prev2], 0), "cudaStreamWaitEvent");          // out slot free again
    st = run(pl, pl->pack, pool_side(pl->src), dense_planes(out_slot, pl->g, p0, p1), pl->pack.shape.vec_bytes, s, ro);
    if (st != FLOWKV_OK) return st;
    FK_TRY(cudaEventRecord(packed[c], s), "cudaEventRecord");
    FK_TRY(cudaStreamWaitEvent(vc.q_d2h, packed[c], 0), "cudaStreamWaitEvent");
    FK_TRY(cudaMemcpyAsync(host, out_slot, wb, cudaMemcpyDeviceToHost, vc.q_d2h), "cudaMemcpyAsync(D2H)");
    FK_TRY(cudaEventRecord(landed[c], vc.q_d2h), "cudaEventRecord");
    FK_TRY(cudaStreamWaitEvent(vc.q_h2d, landed[c], 0), "cudaStreamWaitEvent");
    if (prev2 >= 0) FK_TRY(cudaStreamWaitEvent(vc.q_h2d, unpacked[prev2], 0), "cudaStreamWaitEvent"); // in slot free again
    FK_TRY(cudaMemcpyAsync(in_slot, host, wb, cudaMemcpyHostToDevice, vc.q_h2d), "cudaMemcpyAsync(H2D)");
    FK_TRY(cudaEventRecord(arrived[c], vc.q_h2d), "cudaEventRecord");
    FK_TRY(cudaStreamWaitEvent(vc.q_unpack, arrived[c], 0), "cudaStreamWaitEvent");
    st = run(pl, pl->unpack, dense_planes(in_slot, pl->g, p0, p1), pool_side(pl->dst), pl->unpack.shape.vec_bytes, vc.q_unpack, ro);
    if (st != FLOWKV_OK) return st;
    FK_TRY(cudaEventRecord(unpacked[c], vc.q_unpack), "cudaEventRecord");
    prev2 = prev1;
    prev1 = c;
    ++k;
  }
  // `stream` continues only after the last chunk has been unpacked (q_unpack is in order, so that covers all)
  if (prev1 >= 0) FK_TRY(cudaStreamWaitEvent(s, unpacked[prev1], 0), "cudaStreamWaitEvent");
#undef FK_TRY
  return FLOWKV_OK;
}

namespace {
// Common body of the table-driven calls.  Exactly one of src / dst may be NULL: that side is then the dense
// buffer `dense` holding the layer window [l0, l1) (wire format A12 / A20) and `cu_tokens` gives each request's base.
flowkv_status tables_common(const flowkv_pool* src, const flowkv_pool* dst, const int32_t* src_tables, const int32_t* dst_tables,
                            const uint32_t* num_tokens, const uint64_t* cu_tokens, uint32_t n_reqs, uint32_t max_src_blocks,
                            uint32_t max_dst_blocks, uint32_t max_tokens, const void* dense, uint64_t dense_bytes,
                            uint32_t l0, uint32_t l1, uint32_t* error_flag, const flowkv_tuning* tuning, void* stream) {
  const flowkv_pool* any = src ? src : dst;
  if (!any) return fail(FLOWKV_ERR_INVALID_ARG, "a pool is NULL");
  std::string err;
  flowkv_status st;
  if (src && (st = validate_pool(src, "src", err)) != FLOWKV_OK) return fail(st, err);
  if (dst && (st = validate_pool(dst, "dst", err)) != FLOWKV_OK) return fail(st, err);
  if (src && dst &&
      (src->num_layers != dst->num_layers || src->num_kv_heads != dst->num_kv_heads || src->head_dim != dst->head_dim ||
       src->elem_bytes != dst->elem_bytes))
    return fail(FLOWKV_ERR_SHAPE_MISMATCH, "src and dst pools differ in num_layers, num_kv_heads, head_dim or elem_bytes");
  if (l0 > l1 || l1 > any->num_layers) return fail(FLOWKV_ERR_INVALID_ARG, "layer range outside [0, num_layers]");
  flowkv_tuning tn{};
  if (tuning) tn = *tuning;
  if ((st = check_tuning(tn)) != FLOWKV_OK) return st;
  if (n_reqs == 0 || max_tokens == 0 || l0 == l1) return FLOWKV_OK;    // A11: nothing to move, zero launches
  if ((src && !src_tables) || (dst && !dst_tables) || (!num_tokens && !cu_tokens))
    return fail(FLOWKV_ERR_INVALID_ARG, "a table pointer is NULL");
  if ((src && (uint64_t)max_src_blocks * src->block_size < max_tokens) ||
      (dst && (uint64_t)max_dst_blocks * dst->block_size < max_tokens))
    return fail(FLOWKV_ERR_TABLE_LEN, "max_*_blocks * block_size < max_tokens");
  if (!(src && dst)) {
    if (!dense) return fail(FLOWKV_ERR_INVALID_ARG, "staging is NULL");
    if ((uintptr_t)dense % 16) return fail(FLOWKV_ERR_ALIGN, "staging is not 16-byte aligned");
    if (!cu_tokens) return fail(FLOWKV_ERR_INVALID_ARG, "cu_tokens is NULL");
  }
  Geometry g{};
  g.L = any->num_layers; g.Hkv = any->num_kv_heads; g.Dh = any->head_dim; g.e = any->elem_bytes;
  g.row_bytes = g.Dh * g.e; g.tok_bytes = g.Hkv * g.row_bytes; g.bytes_per_token = 2ull * g.L * g.tok_bytes;
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return fail_cuda(e, "cudaGetDevice");
  const int64_t *d_slo = nullptr, *d_dlo = nullptr;      // device copies of the per-plane offsets (A22), cached
  if (src && src->plane_offsets) e = g_plane_offsets.get(dev, src->plane_offsets, 2 * src->num_layers, &d_slo);
  if (e == cudaSuccess && dst && dst->plane_offsets) e = g_plane_offsets.get(dev, dst->plane_offsets, 2 * dst->num_layers, &d_dlo);
  if (e != cudaSuccess) { g_plane_offsets.release(d_slo); return fail_cuda(e, "upload of plane_offsets"); }
  TablesParams tp{};
  tp.kp.src = src ? pool_side(*src) : dense_side(dense, g, l0, l1);
  tp.kp.dst = dst ? pool_side(*dst) : dense_side(dense, g, l0, l1);
  const PlaneOffs po{d_slo, d_dlo};
  tp.kp.n_planes = 2 * (l1 - l0);
  tp.kp.plane0 = 2 * l0;
  tp.kp.row_bytes = g.row_bytes;
  tp.kp.heads = g.Hkv;
  tp.kp.tok_bytes = g.tok_bytes;
  tp.src_tables = src_tables; tp.dst_tables = dst_tables; tp.num_tokens = num_tokens; tp.cu_tokens = cu_tokens;
  tp.dense_bytes = dense_bytes;
  tp.error = error_flag;
  tp.n_reqs = n_reqs; tp.max_src_blocks = max_src_blocks; tp.max_dst_blocks = max_dst_blocks;
  if (src) { tp.src_s_block = src->stride_bytes[FLOWKV_S_BLOCK]; tp.src_bs_log2 = log2u(src->block_size); tp.src_num_blocks = src->num_blocks; }
  if (dst) { tp.dst_s_block = dst->stride_bytes[FLOWKV_S_BLOCK]; tp.dst_bs_log2 = log2u(dst->block_size); tp.dst_num_blocks = dst->num_blocks; }
  tp.granule_log2 = src && dst ? std::min(tp.src_bs_log2, tp.dst_bs_log2) : (src ? tp.src_bs_log2 : tp.dst_bs_log2);
  tp.q_per_req = (uint32_t)(((uint64_t)max_tokens + (1u << tp.granule_log2) - 1) >> tp.granule_log2);
  const uint64_t n_tiles = (uint64_t)tp.kp.n_planes * n_reqs * tp.q_per_req;
  if (n_tiles >= (1ull << 31)) {
    g_plane_offsets.release(d_slo);
    g_plane_offsets.release(d_dlo);
    return fail(FLOWKV_ERR_UNSUPPORTED, "more than 2^31 tiles in one batch; split the batch");
  }
  tp.n_tiles = (uint32_t)n_tiles;
  tp.max_tokens = max_tokens;
  LaunchShape ls{};
  ls.vec_bytes = pick_vec(src, dst, g);
  if (!(src && dst) && (uintptr_t)dense % 32) ls.vec_bytes = 16;
  const uint32_t tile_bytes = (1u << tp.granule_log2) * g.tok_bytes;
  ls.threads = tn.threads ? tn.threads : 512;
  uint32_t grp = tn.group_threads ? std::min(tn.group_threads, ls.threads) : std::min<uint32_t>(128u, ls.threads);
  while (grp > 32 && grp * ls.vec_bytes > tile_bytes) grp >>= 1;       // no more threads than vectors in a tile
  ls.group_threads = grp;
  const uint32_t use_sms = tn.max_sms ? std::min<uint32_t>(tn.max_sms, (uint32_t)sms) : (uint32_t)sms;
  const uint32_t per_cta = ls.threads / ls.group_threads;
  ls.grid = (uint32_t)std::min<uint64_t>((uint64_t)use_sms * (tn.ctas_per_sm ? tn.ctas_per_sm : 256),
                                         (n_tiles + per_cta - 1) / per_cta);
  tp.kp.group_log2 = log2u(ls.group_threads);
  tp.kp.vpr_log2 = log2_or_none(g.row_bytes / ls.vec_bytes);
  tp.kp.heads_log2 = log2_or_none(g.Hkv);
  const int rc = launch_tables(tp, ls, stream, &po);
  g_plane_offsets.release(d_slo);        // held only while launching; an eviction waits for the device before it frees
  g_plane_offsets.release(d_dlo);
  if (rc != 0) return fail_cuda((cudaError_t)rc, "kernel launch");
  g_launches.fetch_add(1, std::memory_order_relaxed);
  g_api_calls.fetch_add(1, std::memory_order_relaxed);
  return FLOWKV_OK;
}
}  // namespace

flowkv_status flowkv_transfer_tables(const flowkv_pool* src, const flowkv_pool* dst, const int32_t* src_tables,
                                     const int32_t* dst_tables, const uint32_t* num_tokens, uint32_t n_reqs,
                                     uint32_t max_src_blocks, uint32_t max_dst_blocks, uint32_t max_tokens,
                                     uint32_t* error_flag, const flowkv_tuning* tuning, void* stream) {
  if (!src || !dst) return fail(FLOWKV_ERR_INVALID_ARG, "a pool is NULL");
  return tables_common(src, dst, src_tables, dst_tables, num_tokens, nullptr, n_reqs, max_src_blocks, max_dst_blocks,
                       max_tokens, nullptr, 0, 0, src->num_layers, error_flag, tuning, stream);
}

flowkv_status flowkv_transfer_tables_layers(const flowkv_pool* src, const flowkv_pool* dst, const int32_t* src_tables,
                                            const int32_t* dst_tables, const uint32_t* num_tokens, uint32_t n_reqs,
                                            uint32_t max_src_blocks, uint32_t max_dst_blocks, uint32_t max_tokens,
                                            uint32_t layer_begin, uint32_t layer_end, uint32_t* error_flag,
                                            const flowkv_tuning* tuning, void* stream) {
  if (!src || !dst) return fail(FLOWKV_ERR_INVALID_ARG, "a pool is NULL");
  return tables_common(src, dst, src_tables, dst_tables, num_tokens, nullptr, n_reqs, max_src_blocks, max_dst_blocks,
                       max_tokens, nullptr, 0, layer_begin, layer_end, error_flag, tuning, stream);
}

flowkv_status flowkv_pack_tables(const flowkv_pool* src, const int32_t* src_tables, const uint64_t* cu_tokens, uint32_t n_reqs,
                                 uint32_t max_src_blocks, uint32_t max_tokens, void* window, uint64_t bytes,
                                 uint32_t layer_begin, uint32_t layer_end, uint32_t* error_flag,
                                 const flowkv_tuning* tuning, void* stream) {
  if (!src) return fail(FLOWKV_ERR_INVALID_ARG, "pool is NULL");
  return tables_common(src, nullptr, src_tables, nullptr, nullptr, cu_tokens, n_reqs, max_src_blocks, 0, max_tokens, window,
                       bytes, layer_begin, layer_end, error_flag, tuning, stream);
}

flowkv_status flowkv_unpack_tables(const flowkv_pool* dst, const int32_t* dst_tables, const uint64_t* cu_tokens, uint32_t n_reqs,
                                   uint32_t max_dst_blocks, uint32_t max_tokens, const void* window, uint64_t bytes,
                                   uint32_t layer_begin, uint32_t layer_end, uint32_t* error_flag,
                                   const flowkv_tuning* tuning, void* stream) {
  if (!dst) return fail(FLOWKV_ERR_INVALID_ARG, "pool is NULL");
  return tables_common(nullptr, dst, nullptr, dst_tables, nullptr, cu_tokens, n_reqs, 0, max_dst_blocks, max_tokens, window,
                       bytes, layer_begin, layer_end, error_flag, tuning, stream);
}

// Pool -> pool with the schedule in the library's static device array (kernels.cu): for callers that must not
// allocate device memory.  Works on host plans (flowkv_plan_host makes no CUDA call) as well as device plans; the
// launch parameters are built here from the plan's host-side schedule, the ordinary run() path is not involved.
flowkv_status flowkv_transfer_static(const flowkv_plan_t* pl, void* stream) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  const Op& op = pl->transfer;
  if (op.sched.mode == MODE_ABSENT)
    return fail(FLOWKV_ERR_UNSUPPORTED, "plan has no pool-to-pool schedule (needs both pools, no FLOWKV_PLAN_NO_TRANSFER)");
  if (!pl->src_plane_off.empty() || !pl->dst_plane_off.empty())
    return fail(FLOWKV_ERR_UNSUPPORTED, "flowkv_transfer_static: pools with plane_offsets need a device table of their own, "
                                        "which this entry point will not allocate");
  if (op.shape.variant != FLOWKV_VARIANT_LDST)
    return fail(FLOWKV_ERR_UNSUPPORTED, "flowkv_transfer_static runs the register path only: plan with tuning.variant 0 or FLOWKV_VARIANT_LDST");
  // entries a whole-pool launch reads (a flat plan's third part serves layer ranges only)
  const uint64_t n = op.sched.mode == MODE_FLAT ? (uint64_t)op.sched.n_flat + op.sched.n_ragged : op.sched.chunks.size();
  if (n > kStaticChunks)
    return fail(FLOWKV_ERR_UNSUPPORTED, "flowkv_transfer_static: the schedule has " + std::to_string(n) + " entries, the static "
                "array holds " + std::to_string(kStaticChunks) + " (FLOWKV_STATIC_SCHEDULE_ENTRIES); split the batch");
  if (n == 0) return FLOWKV_OK;            // A11: nothing to move, nothing enqueued
  Chunk* d_sched = nullptr;
  uint32_t sms = 0;
  int rc = static_schedule_setup(&d_sched, &sms);
  if (rc != 0) return fail_cuda((cudaError_t)rc, "cudaGetSymbolAddress(static schedule)");
  KernelParams kp{};
  kp.src = pool_side(pl->src);
  kp.dst = pool_side(pl->dst);
  kp.n_chunks = op.sched.n_per_plane();
  kp.n_flat = op.sched.n_flat;
  kp.flat_shift = op.sched.flat_shift;
  kp.flat_tile = op.sched.flat_tile;
  kp.n_planes = 2 * pl->g.L;
  kp.plane0 = 0;
  kp.n_tiles = (kp.n_flat << kp.flat_shift) + kp.n_chunks * kp.n_planes;
  kp.row_bytes = pl->g.row_bytes;
  kp.heads = pl->g.Hkv;
  kp.tok_bytes = pl->g.tok_bytes;
  kp.tile_order = op.tile_order;
  LaunchShape ls = op.shape;
  const uint32_t groups_per_cta = ls.threads / ls.group_threads;
  const uint32_t use_sms = pl->tuning.max_sms ? std::min(pl->tuning.max_sms, sms) : sms;   // a host plan assumed 148 SMs
  const uint64_t cap = (uint64_t)use_sms * (pl->tuning.ctas_per_sm ? pl->tuning.ctas_per_sm : 256);
  ls.grid = (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>(cap, (kp.n_tiles + groups_per_cta - 1) / groups_per_cta));
  kp.group_log2 = log2u(ls.group_threads);
  kp.vpr_log2 = log2_or_none(kp.row_bytes / ls.vec_bytes);
  kp.heads_log2 = log2_or_none(kp.heads);
  rc = launch_copy_static(op.sched.mode, kp, op.sched.chunks.data(), (uint32_t)n, d_sched, ls, stream);
  if (rc != 0) return fail_cuda((cudaError_t)rc, "flowkv_transfer_static: schedule copy / kernel launch");
  g_launches.fetch_add(1, std::memory_order_relaxed);
  g_api_calls.fetch_add(2, std::memory_order_relaxed);     // the schedule copy and the launch
  return FLOWKV_OK;
}

void flowkv_plan_destroy(flowkv_plan_t* pl) {
  if (!pl) return;
  // via-host work on the helper streams was joined back into the caller's stream by an event, so the
  // stream-ordered free below is already behind it; the helper streams and events go back to the cache
  g_via_host.release(pl->via);
  if (pl->d_buf) FK_ENQ cudaFreeAsync(pl->d_buf, pl->stream);   // ordered after everything queued on the plan's stream
  g_pinned.release(pl->staging);
  drop_plan(pl);
}

flowkv_status flowkv_trim(void) {
  g_plane_offsets.trim();
  g_pinned.trim();
  g_via_host.trim();
  return FLOWKV_OK;
}

flowkv_status flowkv_cache_counts(uint32_t* plane_offset_tables, uint32_t* pinned_buffers) {
  if (plane_offset_tables) *plane_offset_tables = (uint32_t)g_plane_offsets.size();
  if (pinned_buffers) *pinned_buffers = (uint32_t)g_pinned.alive();
  return FLOWKV_OK;
}

const char* flowkv_status_string(flowkv_status s) {
  switch (s) {
    case FLOWKV_OK: return "FLOWKV_OK";
    case FLOWKV_ERR_INVALID_ARG: return "FLOWKV_ERR_INVALID_ARG";
    case FLOWKV_ERR_BLOCK_OOB: return "FLOWKV_ERR_BLOCK_OOB";
    case FLOWKV_ERR_TABLE_LEN: return "FLOWKV_ERR_TABLE_LEN";
    case FLOWKV_ERR_DST_ALIAS: return "FLOWKV_ERR_DST_ALIAS";
    case FLOWKV_ERR_ALIGN: return "FLOWKV_ERR_ALIGN";
    case FLOWKV_ERR_SHAPE_MISMATCH: return "FLOWKV_ERR_SHAPE_MISMATCH";
    case FLOWKV_ERR_UNSUPPORTED: return "FLOWKV_ERR_UNSUPPORTED";
    case FLOWKV_ERR_STAGING_TOO_SMALL: return "FLOWKV_ERR_STAGING_TOO_SMALL";
    case FLOWKV_ERR_NOMEM: return "FLOWKV_ERR_NOMEM";
    case FLOWKV_ERR_CUDA: return "FLOWKV_ERR_CUDA";
  }
  return "FLOWKV_ERR_?";
}

const char* flowkv_last_error(void) { return g_last_error.c_str(); }

uint64_t flowkv_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

uint64_t flowkv_api_call_count(void) { return g_api_calls.load(std::memory_order_relaxed); }

// ---- comparison baselines: many cudaMemcpyAsync calls (NOT the product path) --------------------
namespace {
// n tokens starting at token slot (block, off) on each side, every plane: the fewest contiguous copies the
// interior order allows (token-major: one per plane; head-major: one per plane and head).
flowkv_status memcpy_tokens(const flowkv_pool& S, const flowkv_pool& D, const Geometry& g, uint32_t sb, uint32_t so,
                            uint32_t db, uint32_t dof, uint32_t n, cudaStream_t st, uint64_t& calls) {
  auto token_major = [&](const flowkv_pool& p) {
    return p.stride_bytes[FLOWKV_S_HEAD] == (int64_t)g.row_bytes && p.stride_bytes[FLOWKV_S_TOKEN] == (int64_t)g.tok_bytes;
  };
  auto head_major = [&](const flowkv_pool& p) { return p.stride_bytes[FLOWKV_S_TOKEN] == (int64_t)g.row_bytes; };
  const bool tm = token_major(S) && token_major(D), hm = head_major(S) && head_major(D);
  if (!tm && !hm) return fail(FLOWKV_ERR_UNSUPPORTED, "memcpy baseline: block interiors are neither both token-major nor both head-major");
  for (uint32_t l = 0; l < g.L; ++l)
    for (uint32_t c = 0; c < 2; ++c)
      for (uint32_t h = 0; h < (tm ? 1u : g.Hkv); ++h) {
        const char* s = (const char*)S.base + pool_plane_off(S, l, c) + (int64_t)sb * S.stride_bytes[2] +
                        (int64_t)so * S.stride_bytes[3] + (int64_t)h * S.stride_bytes[4];
        char* d = (char*)D.base + pool_plane_off(D, l, c) + (int64_t)db * D.stride_bytes[2] +
                  (int64_t)dof * D.stride_bytes[3] + (int64_t)h * D.stride_bytes[4];
        cudaError_t e = FK_ENQ cudaMemcpyAsync(d, s, (size_t)n * (tm ? g.tok_bytes : g.row_bytes), cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return fail_cuda(e, "cudaMemcpyAsync");
        ++calls;
      }
  return FLOWKV_OK;
}
}  // namespace

flowkv_status flowkv_baseline_blockwise(const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs,
                                        uint32_t n_reqs, void* stream, uint64_t* n_calls) {
  if (!src || !dst || (n_reqs && !reqs)) return fail(FLOWKV_ERR_INVALID_ARG, "NULL argument");
  std::string err;
  flowkv_status st;
  if ((st = validate_pool(src, "src", err)) != FLOWKV_OK) return fail(st, err);
  if ((st = validate_pool(dst, "dst", err)) != FLOWKV_OK) return fail(st, err);
  if ((st = validate_requests(src, dst, reqs, n_reqs, 0, err)) != FLOWKV_OK) return fail(st, err);
  Geometry g{};
  g.L = src->num_layers; g.Hkv = src->num_kv_heads; g.Dh = src->head_dim; g.e = src->elem_bytes;
  g.row_bytes = g.Dh * g.e; g.tok_bytes = g.Hkv * g.row_bytes; g.bytes_per_token = 2ull * g.L * g.tok_bytes;
  const bool span = pool_is_span_capable(*src, g) && pool_is_span_capable(*dst, g);
  const bool flat = !span && pools_are_flat_congruent(*src, *dst, g);
  if (src->block_size != dst->block_size || (!span && !flat))
    return fail(FLOWKV_ERR_UNSUPPORTED, "blockwise baseline needs equal block sizes and two token-major pools, or two "
                                        "block-major pools with the same interior");
  uint64_t calls = 0;
  const uint32_t bs = src->block_size;
  for (uint32_t r = 0; r < n_reqs; ++r)
    for (uint32_t b = 0; b < reqs[r].n_src_blocks; ++b) {
      const uint32_t ntok = std::min(bs, reqs[r].num_tokens - b * bs);
      const uint32_t sb = (uint32_t)reqs[r].src_blocks[b], db = (uint32_t)reqs[r].dst_blocks[b];
      if (flat && ntok == bs) {
        // (B,L,2,H): the whole block, every layer and K|V, is one range (Eq. 5)
        cudaError_t e = FK_ENQ cudaMemcpyAsync((char*)dst->base + (int64_t)db * dst->stride_bytes[2],
                                        (const char*)src->base + (int64_t)sb * src->stride_bytes[2],
                                        (size_t)src->stride_bytes[2], cudaMemcpyDeviceToDevice, (cudaStream_t)stream);
        if (e != cudaSuccess) return fail_cuda(e, "cudaMemcpyAsync");
        ++calls;
      } else if ((st = memcpy_tokens(*src, *dst, g, sb, 0, db, 0, ntok, (cudaStream_t)stream, calls)) != FLOWKV_OK) {
        return st;
      }
    }
  if (n_calls) *n_calls = calls;
  return FLOWKV_OK;
}

flowkv_status flowkv_baseline_segmentwise(const flowkv_plan_t* pl, void* stream, uint64_t* n_calls) {
  if (!pl) return fail(FLOWKV_ERR_INVALID_ARG, "plan is NULL");
  const bool span = pl->has_src && pl->has_dst && pool_is_span_capable(pl->src, pl->g) && pool_is_span_capable(pl->dst, pl->g);
  const bool flat = pl->has_src && pl->has_dst && !span && pools_are_flat_congruent(pl->src, pl->dst, pl->g);
  if (!span && !flat)
    return fail(FLOWKV_ERR_UNSUPPORTED, "segmentwise baseline needs two token-major pools, or two block-major pools "
                                        "with the same interior and block size");
  uint64_t calls = 0;
  const flowkv_pool &S = pl->src, &D = pl->dst;
  flowkv_status st;
  for (const flowkv_segment& sg : pl->segments) {
    if (flat) {
      // whole blocks of the segment: ONE copy over all layers (Fig. 5); then the partial last block
      const uint32_t bs = S.block_size, nfull = sg.n_tokens / bs, rem = sg.n_tokens % bs;
      if (nfull) {
        cudaError_t e = FK_ENQ cudaMemcpyAsync((char*)D.base + (int64_t)sg.dst_block * D.stride_bytes[2],
                                        (const char*)S.base + (int64_t)sg.src_block * S.stride_bytes[2],
                                        (size_t)nfull * S.stride_bytes[2], cudaMemcpyDeviceToDevice, (cudaStream_t)stream);
        if (e != cudaSuccess) return fail_cuda(e, "cudaMemcpyAsync");
        ++calls;
      }
      if (rem && (st = memcpy_tokens(S, D, pl->g, sg.src_block + nfull, 0, sg.dst_block + nfull, 0, rem,
                                     (cudaStream_t)stream, calls)) != FLOWKV_OK)
        return st;
    } else if ((st = memcpy_tokens(S, D, pl->g, sg.src_block, sg.src_tok_off, sg.dst_block, sg.dst_tok_off, sg.n_tokens,
                                   (cudaStream_t)stream, calls)) != FLOWKV_OK) {
      return st;
    }
  }
  if (n_calls) *n_calls = calls;
  return FLOWKV_OK;
}

}  // namespace impl

// ---- the exported C ABI: every entry point runs its implementation under flowkv::guarded(), so that no C++
// exception (std::bad_alloc from a vector, a set insert, a string) ever crosses into a C caller: the header
// promises a status code, never a throw or an abort.
extern "C" {
flowkv_status flowkv_pool_strides(flowkv_pool* pool) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_pool_strides(pool); });
}
flowkv_status flowkv_plan(
    const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs, uint32_t n_reqs,
    uint32_t flags, const flowkv_tuning* tuning, void* stream, flowkv_plan_t** out) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_plan(src, dst, reqs, n_reqs, flags, tuning, stream, out); });
}
flowkv_status flowkv_plan_host(
    const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs, uint32_t n_reqs,
    uint32_t flags, const flowkv_tuning* tuning, flowkv_plan_t** out) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_plan_host(src, dst, reqs, n_reqs, flags, tuning, out); });
}
flowkv_status flowkv_plan_info(const flowkv_plan_t* plan, flowkv_plan_stats* stats, const flowkv_segment** segments) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_plan_info(plan, stats, segments); });
}
flowkv_status flowkv_transfer(const flowkv_plan_t* plan, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_transfer(plan, stream); });
}
flowkv_status flowkv_pack(const flowkv_plan_t* plan, void* staging, uint64_t bytes, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_pack(plan, staging, bytes, stream); });
}
flowkv_status flowkv_unpack(const flowkv_plan_t* plan, const void* staging, uint64_t bytes, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_unpack(plan, staging, bytes, stream); });
}
flowkv_status flowkv_transfer_layers(
    const flowkv_plan_t* plan, uint32_t layer_begin, uint32_t layer_end, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_transfer_layers(plan, layer_begin, layer_end, stream); });
}
flowkv_status flowkv_pack_layers(
    const flowkv_plan_t* plan, void* staging, uint64_t bytes, uint32_t layer_begin, uint32_t layer_end,
    void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_pack_layers(plan, staging, bytes, layer_begin, layer_end, stream); });
}
flowkv_status flowkv_unpack_layers(
    const flowkv_plan_t* plan, const void* staging, uint64_t bytes, uint32_t layer_begin,
    uint32_t layer_end, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_unpack_layers(plan, staging, bytes, layer_begin, layer_end, stream); });
}
flowkv_status flowkv_window_bytes(
    const flowkv_plan_t* plan, uint32_t layer_begin, uint32_t layer_end, uint64_t* bytes) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_window_bytes(plan, layer_begin, layer_end, bytes); });
}
flowkv_status flowkv_pack_window(
    const flowkv_plan_t* plan, void* window, uint64_t bytes, uint32_t layer_begin, uint32_t layer_end,
    void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_pack_window(plan, window, bytes, layer_begin, layer_end, stream); });
}
flowkv_status flowkv_unpack_window(
    const flowkv_plan_t* plan, const void* window, uint64_t bytes, uint32_t layer_begin,
    uint32_t layer_end, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_unpack_window(plan, window, bytes, layer_begin, layer_end, stream); });
}
flowkv_status flowkv_via_host_scratch_bytes(const flowkv_plan_t* plan, uint32_t n_chunks, uint64_t* bytes) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_via_host_scratch_bytes(plan, n_chunks, bytes); });
}
flowkv_status flowkv_transfer_via_host(
    const flowkv_plan_t* plan, void* host_staging, uint64_t bytes, uint32_t n_chunks,
    uint32_t ctas_per_kernel, void* device_scratch, uint64_t scratch_bytes, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_transfer_via_host(plan, host_staging, bytes, n_chunks, ctas_per_kernel, device_scratch, scratch_bytes, stream); });
}
flowkv_status flowkv_transfer_tables(
    const flowkv_pool* src, const flowkv_pool* dst, const int32_t* src_tables,
    const int32_t* dst_tables, const uint32_t* num_tokens, uint32_t n_reqs, uint32_t max_src_blocks,
    uint32_t max_dst_blocks, uint32_t max_tokens, uint32_t* error_flag, const flowkv_tuning* tuning,
    void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_transfer_tables(src, dst, src_tables, dst_tables, num_tokens, n_reqs, max_src_blocks, max_dst_blocks, max_tokens, error_flag, tuning, stream); });
}
flowkv_status flowkv_transfer_tables_layers(
    const flowkv_pool* src, const flowkv_pool* dst, const int32_t* src_tables,
    const int32_t* dst_tables, const uint32_t* num_tokens, uint32_t n_reqs, uint32_t max_src_blocks,
    uint32_t max_dst_blocks, uint32_t max_tokens, uint32_t layer_begin, uint32_t layer_end,
    uint32_t* error_flag, const flowkv_tuning* tuning, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_transfer_tables_layers(src, dst, src_tables, dst_tables, num_tokens, n_reqs, max_src_blocks, max_dst_blocks, max_tokens, layer_begin, layer_end, error_flag, tuning, stream); });
}
flowkv_status flowkv_pack_tables(
    const flowkv_pool* src, const int32_t* src_tables, const uint64_t* cu_tokens, uint32_t n_reqs,
    uint32_t max_src_blocks, uint32_t max_tokens, void* window, uint64_t bytes, uint32_t layer_begin,
    uint32_t layer_end, uint32_t* error_flag, const flowkv_tuning* tuning, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_pack_tables(src, src_tables, cu_tokens, n_reqs, max_src_blocks, max_tokens, window, bytes, layer_begin, layer_end, error_flag, tuning, stream); });
}
flowkv_status flowkv_unpack_tables(
    const flowkv_pool* dst, const int32_t* dst_tables, const uint64_t* cu_tokens, uint32_t n_reqs,
    uint32_t max_dst_blocks, uint32_t max_tokens, const void* window, uint64_t bytes,
    uint32_t layer_begin, uint32_t layer_end, uint32_t* error_flag, const flowkv_tuning* tuning,
    void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_unpack_tables(dst, dst_tables, cu_tokens, n_reqs, max_dst_blocks, max_tokens, window, bytes, layer_begin, layer_end, error_flag, tuning, stream); });
}
flowkv_status flowkv_trim(void) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_trim(); });
}
flowkv_status flowkv_cache_counts(uint32_t* plane_offset_tables, uint32_t* pinned_buffers) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_cache_counts(plane_offset_tables, pinned_buffers); });
}
flowkv_status flowkv_transfer_static(const flowkv_plan_t* plan, void* stream) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_transfer_static(plan, stream); });
}
void flowkv_plan_destroy(flowkv_plan_t* plan) {
  try { impl::flowkv_plan_destroy(plan); } catch (...) {}
}
const char* flowkv_status_string(flowkv_status s) {
  return impl::flowkv_status_string(s);
}
const char* flowkv_last_error(void) {
  return impl::flowkv_last_error();
}
uint32_t flowkv_version(void) {
  return FLOWKV_VERSION;
}
uint64_t flowkv_launch_count(void) {
  return impl::flowkv_launch_count();
}
uint64_t flowkv_api_call_count(void) {
  return impl::flowkv_api_call_count();
}
flowkv_status flowkv_baseline_blockwise(
    const flowkv_pool* src, const flowkv_pool* dst, const flowkv_request* reqs, uint32_t n_reqs,
    void* stream, uint64_t* n_calls) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_baseline_blockwise(src, dst, reqs, n_reqs, stream, n_calls); });
}
flowkv_status flowkv_baseline_segmentwise(const flowkv_plan_t* plan, void* stream, uint64_t* n_calls) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_baseline_segmentwise(plan, stream, n_calls); });
}
}  // extern "C"
