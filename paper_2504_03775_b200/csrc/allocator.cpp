// allocator.cpp — segment-based KV block allocator (§3.3).  Host only.
//
// Free space is a set of SEGMENTS (maximal runs of consecutive free block ids) kept in two ordered
// indexes: by (length, start) — the "segment-based minimum heap", with deletion — and by start, for
// merging neighbours on release.  Policy: include/flowkv.h and DESIGN.md reading A19.
#include <map>
#include <new>
#include <set>
#include <string>
#include <utility>
#include <vector>

#include "flowkv_internal.h"

struct flowkv_allocator_s {
  uint32_t num_blocks = 0, free_blocks = 0;
  std::set<std::pair<uint32_t, uint32_t>> by_len;   // (length, start)
  std::map<uint32_t, uint32_t> by_start;            // start -> length
  std::vector<uint8_t> used;                        // 1 = allocated

  void insert(uint32_t start, uint32_t len) {
    by_len.insert({len, start});
    by_start[start] = len;
  }
  void erase(uint32_t start, uint32_t len) {
    by_len.erase({len, start});
    by_start.erase(start);
  }
  // release [start, start+len) and merge with free neighbours
  void release(uint32_t start, uint32_t len) {
    auto next = by_start.lower_bound(start);
    if (next != by_start.end() && next->first == start + len) {
      const uint32_t nl = next->second, ns = next->first;
      erase(ns, nl);
      len += nl;
    }
    auto it = by_start.lower_bound(start);
    if (it != by_start.begin()) {
      --it;
      if (it->first + it->second == start) {
        const uint32_t ps = it->first, pl = it->second;
        erase(ps, pl);
        start = ps;
        len += pl;
      }
    }
    insert(start, len);
  }
};

// set by api.cpp's error channel
extern "C" const char* flowkv_last_error(void);
static flowkv_status fail(flowkv_status s, const char* msg) {
  flowkv::set_last_error(msg);
  return s;
}

namespace impl {

flowkv_status flowkv_alloc_create(uint32_t num_blocks, flowkv_allocator_t** out) {
  if (!out || !num_blocks) return fail(FLOWKV_ERR_INVALID_ARG, "allocator: out is NULL or num_blocks is 0");
  flowkv_allocator_s* a = new (std::nothrow) flowkv_allocator_s();
  if (!a) return fail(FLOWKV_ERR_NOMEM, "out of host memory");
  try {
    a->num_blocks = a->free_blocks = num_blocks;
    a->used.assign(num_blocks, 0);
    a->insert(0, num_blocks);
  } catch (...) {                  // the guard of the C ABI turns it into a status; do not leak the object
    delete a;
    throw;
  }
  *out = a;
  return FLOWKV_OK;
}

flowkv_status flowkv_alloc_allocate(flowkv_allocator_t* a, uint32_t n, int32_t* out_ids, uint32_t* n_segments) {
  if (!a || (n && !out_ids)) return fail(FLOWKV_ERR_INVALID_ARG, "allocator: NULL argument");
  if (n > a->free_blocks) return fail(FLOWKV_ERR_NOMEM, "allocator: not enough free blocks");
  uint32_t left = n, segs = 0, w = 0;
  while (left) {
    // best fit: the smallest segment that holds everything that is left
    auto fit = a->by_len.lower_bound({left, 0});
    uint32_t start, len, take;
    if (fit != a->by_len.end()) {
      len = fit->first; start = fit->second; take = left;
    } else {
      // nothing holds the rest: take the largest segment whole (lowest start among equals)
      const uint32_t maxlen = a->by_len.rbegin()->first;
      auto big = a->by_len.lower_bound({maxlen, 0});
      len = big->first; start = big->second; take = len;
    }
    a->erase(start, len);
    if (take < len) a->insert(start + take, len - take);
    for (uint32_t i = 0; i < take; ++i) {
      a->used[start + i] = 1;
      out_ids[w++] = (int32_t)(start + i);
    }
    left -= take;
    ++segs;
  }
  a->free_blocks -= n;
  if (n_segments) *n_segments = segs;
  return FLOWKV_OK;
}

flowkv_status flowkv_alloc_free(flowkv_allocator_t* a, const int32_t* ids, uint32_t n) {
  if (!a || (n && !ids)) return fail(FLOWKV_ERR_INVALID_ARG, "allocator: NULL argument");
  // validate first so that a bad call frees nothing
  for (uint32_t i = 0; i < n; ++i) {
    const bool oob = ids[i] < 0 || (uint32_t)ids[i] >= a->num_blocks;
    if (oob || a->used[ids[i]] != 1) {
      for (uint32_t j = 0; j < i; ++j) a->used[ids[j]] = 1;        // undo the marks made below
      return oob ? fail(FLOWKV_ERR_BLOCK_OOB, "allocator: block id out of range")
                 : fail(FLOWKV_ERR_INVALID_ARG, "allocator: block is not allocated (double free or duplicate id)");
    }
    a->used[ids[i]] = 2;                                           // marked for release (catches duplicates)
  }
  uint32_t i = 0;
  while (i < n) {                                                  // release run by run
    uint32_t j = i + 1;
    while (j < n && ids[j] == ids[j - 1] + 1) ++j;
    for (uint32_t k = i; k < j; ++k) a->used[ids[k]] = 0;
    a->release((uint32_t)ids[i], j - i);
    i = j;
  }
  a->free_blocks += n;
  return FLOWKV_OK;
}

flowkv_status flowkv_alloc_stats(const flowkv_allocator_t* a, uint32_t* free_blocks, uint32_t* free_segments,
                                 uint32_t* largest_segment) {
  if (!a) return fail(FLOWKV_ERR_INVALID_ARG, "allocator is NULL");
  if (free_blocks) *free_blocks = a->free_blocks;
  if (free_segments) *free_segments = (uint32_t)a->by_len.size();
  if (largest_segment) *largest_segment = a->by_len.empty() ? 0 : a->by_len.rbegin()->first;
  return FLOWKV_OK;
}

void flowkv_alloc_destroy(flowkv_allocator_t* a) { delete a; }

}  // namespace impl

// exported C ABI (exceptions never cross it; see api.cpp).  A std::bad_alloc inside allocate / free returns
// FLOWKV_ERR_NOMEM; the allocator must then be destroyed (its indexes may be half-updated).
extern "C" {
flowkv_status flowkv_alloc_create(uint32_t num_blocks, flowkv_allocator_t** out) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_alloc_create(num_blocks, out); });
}
flowkv_status flowkv_alloc_allocate(flowkv_allocator_t* a, uint32_t n, int32_t* out_ids, uint32_t* n_segments) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_alloc_allocate(a, n, out_ids, n_segments); });
}
flowkv_status flowkv_alloc_free(flowkv_allocator_t* a, const int32_t* ids, uint32_t n) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_alloc_free(a, ids, n); });
}
flowkv_status flowkv_alloc_stats(
    const flowkv_allocator_t* a, uint32_t* free_blocks, uint32_t* free_segments,
    uint32_t* largest_segment) {
  return flowkv::guarded([&]() -> flowkv_status { return impl::flowkv_alloc_stats(a, free_blocks, free_segments, largest_segment); });
}
void flowkv_alloc_destroy(flowkv_allocator_t* a) {
  try { impl::flowkv_alloc_destroy(a); } catch (...) {}
}
}  // extern "C"
