// tma.cpp — TMA tensor maps for rows mode (layout / block-size converting moves; BASELINE configs[3]).
//
// A pool is described to the TMA unit as ONE 5-D tensor of 4-byte elements
//     dim 0  row element      extent Dh*e/4      contiguous
//     dim 1  token in block   extent BS          stride s_token
//     dim 2  head             extent Hkv         stride s_head
//     dim 3  block            extent NB          stride s_block
//     dim 4  plane            extent 2*L         stride s_kv      (needs s_layer == 2*s_kv: true for every named layout)
// The dimension ORDER is the same for every pool; only the strides differ (LKBTHD: token 2 KiB / head 256 B;
// BLKHTD: token 256 B / head BS*256 B).  That is what makes a box loaded through the src map storable through the
// dst map unchanged.  Tensor maps depend on the pool, not on the batch: they are cached per (pool pair, box).
#include <cuda_runtime.h>

#include <cstring>
#include <mutex>

#include "flowkv_internal.h"

namespace flowkv {
namespace {

using EncodeTiled = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiled encode_fn() {
  static EncodeTiled fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    (void)cudaGetLastError();
    return (EncodeTiled)p;
  }();
  return fn;
}

bool encode_pool(const flowkv_pool& p, const Geometry& g, uint32_t box_tok, CUtensorMap* out, std::string& why) {
  EncodeTiled enc = encode_fn();
  if (!enc) { why = "cuTensorMapEncodeTiled is not available"; return false; }
  const cuuint64_t dims[5] = {g.row_bytes / 4, p.block_size, g.Hkv, p.num_blocks, 2ull * g.L};
  const cuuint64_t strides[4] = {(cuuint64_t)p.stride_bytes[FLOWKV_S_TOKEN], (cuuint64_t)p.stride_bytes[FLOWKV_S_HEAD],
                                 (cuuint64_t)p.stride_bytes[FLOWKV_S_BLOCK], (cuuint64_t)p.stride_bytes[FLOWKV_S_KV]};
  const cuuint32_t box[5] = {g.row_bytes / 4, box_tok, g.Hkv, 1, 1};
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_UINT32, 5, p.base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { why = "cuTensorMapEncodeTiled rejected the pool (CUresult " + std::to_string((int)r) + ")"; return false; }
  return true;
}

struct Key {
  flowkv_pool src, dst;
  uint32_t box_tok;
  int device;
};
bool same_pool(const flowkv_pool& a, const flowkv_pool& b) {
  return a.base == b.base && a.num_layers == b.num_layers && a.num_kv_heads == b.num_kv_heads && a.head_dim == b.head_dim &&
         a.elem_bytes == b.elem_bytes && a.num_blocks == b.num_blocks && a.block_size == b.block_size &&
         memcmp(a.stride_bytes, b.stride_bytes, sizeof a.stride_bytes) == 0;
}
struct Entry { Key k; RowsTma v; };
std::mutex g_mu;
std::vector<Entry> g_cache;          // most recently used first; a handful of pool pairs per process
constexpr size_t kMaxEntries = 32;

}  // namespace

bool build_rows_tma(const flowkv_pool& src, const flowkv_pool& dst, const Geometry& g, uint32_t box_tok, RowsTma& out,
                    std::string& why) {
  out.ok = false;
  // what the tensor path needs (everything else runs the register path)
  for (const flowkv_pool* p : {&src, &dst}) {
    if (p->plane_offsets) { why = "planes are separate allocations (no uniform plane stride)"; return false; }
    if (p->stride_bytes[FLOWKV_S_LAYER] != 2 * p->stride_bytes[FLOWKV_S_KV]) { why = "s_layer != 2*s_kv (plane axis is not uniform)"; return false; }
    for (int i = 0; i < 5; ++i)
      if ((uint64_t)p->stride_bytes[i] >= (1ull << 40)) { why = "a stride of 2^40 bytes or more"; return false; }
  }
  if (g.row_bytes / 4 > 256) { why = "rows longer than 1 KiB"; return false; }
  if (g.Hkv > 256 || box_tok == 0 || box_tok > 256) { why = "more than 256 heads or tokens per box"; return false; }
  if ((uint64_t)box_tok * g.tok_bytes > (96u << 10)) { why = "a box larger than 96 KiB"; return false; }
  int device = 0;
  if (cudaGetDevice(&device) != cudaSuccess) { (void)cudaGetLastError(); why = "no CUDA device"; return false; }
  {
    std::lock_guard<std::mutex> lk(g_mu);
    for (size_t i = 0; i < g_cache.size(); ++i) {
      const Key& k = g_cache[i].k;
      if (k.box_tok == box_tok && k.device == device && same_pool(k.src, src) && same_pool(k.dst, dst)) {
        out = g_cache[i].v;
        if (i) std::swap(g_cache[i], g_cache[0]);
        return out.ok;
      }
    }
  }
  RowsTma t;
  t.box_tok = box_tok;
  t.tok_slot = (g.tok_bytes + 127) & ~127u;
  t.src_s_block = src.stride_bytes[FLOWKV_S_BLOCK];
  t.dst_s_block = dst.stride_bytes[FLOWKV_S_BLOCK];
  t.src_s_token = src.stride_bytes[FLOWKV_S_TOKEN];
  t.dst_s_token = dst.stride_bytes[FLOWKV_S_TOKEN];
  t.ok = encode_pool(src, g, box_tok, &t.src_full, why) && encode_pool(dst, g, box_tok, &t.dst_full, why) &&
         encode_pool(src, g, 1, &t.src_one, why) && encode_pool(dst, g, 1, &t.dst_one, why);
  {
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_cache.size() >= kMaxEntries) g_cache.pop_back();
    g_cache.insert(g_cache.begin(), Entry{Key{src, dst, box_tok, device}, t});
  }
  out = t;
  return t.ok;
}

}  // namespace flowkv
