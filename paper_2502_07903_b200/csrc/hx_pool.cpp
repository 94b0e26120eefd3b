// Host page allocator: a LIFO free list of page ids.
// Paging is by citation only in the paper; running out of pages is the OOM the
// paper avoids by capping the online rate -> HX_ERR_NO_PAGES, all-or-nothing.
#include <cstdint>
#include <vector>

#include "hx.h"

namespace hx { void set_error(const char* fmt, ...); }

struct hx_page_pool {
  int32_t num_pages;
  std::vector<int32_t> free_list;   // back() is handed out next
  std::vector<uint8_t> is_free;
};

extern "C" {

int hx_pool_create(hx_page_pool** out, int32_t num_pages) {
  if (!out || num_pages < 0) { hx::set_error("hx_pool_create: out=%p num_pages=%d", (void*)out, num_pages); return HX_ERR_INVALID_ARG; }
  // No C++ exception may cross the C ABI: the only allocations of the pool's lifetime happen here (free_list is
  // sized to num_pages once, so hx_pool_free's push_back never reallocates) and are caught.
  hx_page_pool* p = nullptr;
  try {
    p = new hx_page_pool();
    p->num_pages = num_pages;
    p->free_list.resize(num_pages);
    for (int32_t i = 0; i < num_pages; ++i) p->free_list[i] = num_pages - 1 - i;   // page 0 first
    p->is_free.assign(num_pages, 1);
  } catch (...) {
    delete p;
    hx::set_error("hx_pool_create: out of host memory for %d pages", num_pages);
    return HX_ERR_NO_PAGES;
  }
  *out = p;
  return HX_OK;
}

static inline uint64_t splitmix64(uint64_t& s) {
  uint64_t z = (s += 0x9E3779B97F4A7C15ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

int hx_pool_shuffle(hx_page_pool* p, uint64_t seed) {
  if (!p) { hx::set_error("hx_pool_shuffle: NULL pool"); return HX_ERR_INVALID_ARG; }
  uint64_t s = seed;
  for (size_t i = p->free_list.size(); i > 1; --i) {          // Fisher-Yates
    size_t j = (size_t)(splitmix64(s) % i);
    int32_t t = p->free_list[i - 1]; p->free_list[i - 1] = p->free_list[j]; p->free_list[j] = t;
  }
  return HX_OK;
}

int hx_pool_alloc(hx_page_pool* p, int32_t n, int32_t* out_ids) {
  if (!p || n < 0 || (n > 0 && !out_ids)) { hx::set_error("hx_pool_alloc: bad arguments"); return HX_ERR_INVALID_ARG; }
  if ((size_t)n > p->free_list.size()) {
    hx::set_error("hx_pool_alloc: need %d pages, %zu free", n, p->free_list.size());
    return HX_ERR_NO_PAGES;
  }
  for (int32_t i = 0; i < n; ++i) {
    int32_t id = p->free_list.back(); p->free_list.pop_back();
    p->is_free[id] = 0; out_ids[i] = id;
  }
  return HX_OK;
}

int hx_pool_free(hx_page_pool* p, const int32_t* ids, int32_t n) {
  if (!p || n < 0 || (n > 0 && !ids)) { hx::set_error("hx_pool_free: bad arguments"); return HX_ERR_INVALID_ARG; }
  // validate first (bad id, already free, or repeated inside this call) so that nothing is freed on error
  for (int32_t i = 0; i < n; ++i) {
    int32_t id = ids[i];
    if (id < 0 || id >= p->num_pages || p->is_free[id]) {
      for (int32_t j = 0; j < i; ++j) p->is_free[ids[j]] = 0;
      hx::set_error("hx_pool_free: page id %d at index %d is out of range or already free", id, i);
      return HX_ERR_INVALID_ARG;
    }
    p->is_free[id] = 1;    // provisional mark also catches duplicates within ids[]
  }
  for (int32_t i = 0; i < n; ++i) p->free_list.push_back(ids[i]);   // within the capacity reserved at create: no allocation
  return HX_OK;
}

int32_t hx_pool_num_free(const hx_page_pool* p) { return p ? (int32_t)p->free_list.size() : -1; }
int32_t hx_pool_num_pages(const hx_page_pool* p) { return p ? p->num_pages : -1; }

int hx_pool_alloc_table(hx_page_pool* p, const int32_t* seq_lens, int32_t batch, int32_t page_size,
                        int32_t* block_table, int32_t stride) {
  if (!p || batch < 0 || page_size <= 0 || stride < 0 || (batch > 0 && (!seq_lens || !block_table))) {
    hx::set_error("hx_pool_alloc_table: bad arguments"); return HX_ERR_INVALID_ARG;
  }
  int64_t need = 0;
  for (int32_t i = 0; i < batch; ++i) {
    if (seq_lens[i] < 0) { hx::set_error("hx_pool_alloc_table: seq_lens[%d] < 0", i); return HX_ERR_INVALID_ARG; }
    int64_t k = ((int64_t)seq_lens[i] + page_size - 1) / page_size;
    if (k > stride) { hx::set_error("hx_pool_alloc_table: request %d needs %lld pages > stride %d", i, (long long)k, stride); return HX_ERR_INVALID_ARG; }
    need += k;
  }
  if (need > (int64_t)p->free_list.size()) {
    hx::set_error("hx_pool_alloc_table: need %lld pages, %zu free", (long long)need, p->free_list.size());
    return HX_ERR_NO_PAGES;
  }
  for (int32_t i = 0; i < batch; ++i) {
    int32_t k = (int32_t)(((int64_t)seq_lens[i] + page_size - 1) / page_size);
    int32_t* row = block_table + (int64_t)i * stride;
    hx_pool_alloc(p, k, row);
    for (int32_t j = k; j < stride; ++j) row[j] = -1;
  }
  return HX_OK;
}

void hx_pool_destroy(hx_page_pool* p) { delete p; }

}  // extern "C"
