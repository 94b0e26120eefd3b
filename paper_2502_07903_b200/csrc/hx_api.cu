// libhx C ABI: argument validation and dispatch.  Every step of the path runs in the CUDA
// kernels of ingest.cu / attention.cu; nothing here touches payload data.
#include <cstdio>
#include <cstring>
#include <mutex>

#include "handoff_tiles.cuh"
#include "hx_internal.h"

namespace hx {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
void clear_error() { g_err[0] = 0; }

int device_info(DeviceInfo* out) {
  static std::mutex mu;
  static DeviceInfo cache[64];
  int dev = 0;
  HX_CUDA_OK(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lock(mu);
  if (dev < 0 || dev >= 64) HX_FAIL(HX_ERR_CUDA, "device id %d out of range", dev);
  if (cache[dev].device != dev) {
    DeviceInfo d;
    d.device = dev;
    HX_CUDA_OK(cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev));
    HX_CUDA_OK(cudaDeviceGetAttribute(&d.max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    cache[dev] = d;
  }
  *out = cache[dev];
  return HX_OK;
}

static int check_cache(const hx_paged_cache* c, const char* who) {
  if (!c) HX_FAIL(HX_ERR_INVALID_ARG, "%s: cache is NULL", who);
  if (!c->k || !c->v) HX_FAIL(HX_ERR_INVALID_ARG, "%s: cache k/v pointer is NULL", who);
  if (!aligned16(c->k) || !aligned16(c->v)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: cache pointers must be 16-byte aligned", who);
  if (c->layers <= 0 || c->num_pages <= 0 || c->kv_heads <= 0 || c->page_size <= 0 || c->head_dim <= 0)
    HX_FAIL(HX_ERR_INVALID_ARG, "%s: cache dims must be positive (layers=%d pages=%d kv_heads=%d ps=%d D=%d)", who,
            c->layers, c->num_pages, c->kv_heads, c->page_size, c->head_dim);
  if (c->head_dim != 64 && c->head_dim != 128) HX_FAIL(HX_ERR_UNSUPPORTED, "%s: head_dim %d not in {64,128}", who, c->head_dim);
  if (c->page_size != 16) HX_FAIL(HX_ERR_UNSUPPORTED, "%s: page_size %d != 16", who, c->page_size);
  return HX_OK;
}

static int ingest_common(const void* const* src_k, const void* const* src_v, int32_t layers, int32_t heads,
                         int32_t head_dim, int32_t src_tp, int32_t dst_tp, int32_t dst_rank,
                         const hx_paged_cache* dst, const int32_t* block_table, int32_t stride,
                         const int32_t* cu_seqlens, const int32_t* seq_lens, int32_t batch,
                         int32_t total_tokens, int32_t max_seq_len, void* stream, bool gather,
                         const char* who, int32_t src_layers, int32_t src_layer0, int32_t dst_layer0,
                         bool dry_run = false, IngestParams* params_out = nullptr) {
  clear_error();
  if (layers < 0 || batch < 0 || total_tokens < 0 || max_seq_len < 0)
    HX_FAIL(HX_ERR_INVALID_ARG, "%s: negative size (layers=%d batch=%d total_tokens=%d max_seq_len=%d)", who, layers, batch, total_tokens, max_seq_len);
  if (heads <= 0 || src_tp <= 0 || dst_tp <= 0) HX_FAIL(HX_ERR_INVALID_ARG, "%s: heads/src_tp/dst_tp must be positive", who);
  if (src_tp > heads || dst_tp > heads) HX_FAIL(HX_ERR_UNSUPPORTED, "%s: TP degree above kv heads (replicated KV) is not supported (heads=%d src_tp=%d dst_tp=%d)", who, heads, src_tp, dst_tp);
  if (heads % src_tp || heads % dst_tp) HX_FAIL(HX_ERR_INVALID_ARG, "%s: heads=%d not divisible by src_tp=%d / dst_tp=%d", who, heads, src_tp, dst_tp);
  if (src_tp > 16) HX_FAIL(HX_ERR_UNSUPPORTED, "%s: src_tp %d > 16", who, src_tp);
  if (dst_rank < 0 || dst_rank >= dst_tp) HX_FAIL(HX_ERR_INVALID_ARG, "%s: dst_rank %d not in [0,%d)", who, dst_rank, dst_tp);
  int rc = check_cache(dst, who);
  if (rc) return rc;
  if (dst->head_dim != head_dim) HX_FAIL(HX_ERR_INVALID_ARG, "%s: head_dim %d != cache head_dim %d", who, head_dim, dst->head_dim);
  if (dst->kv_heads != heads / dst_tp) HX_FAIL(HX_ERR_INVALID_ARG, "%s: cache kv_heads %d != heads/dst_tp = %d", who, dst->kv_heads, heads / dst_tp);
  if (src_layers < 0) src_layers = layers;                     // plain ingest: the buffers hold exactly `layers`
  if (src_layer0 < 0 || dst_layer0 < 0 || (int64_t)src_layer0 + layers > src_layers)
    HX_FAIL(HX_ERR_INVALID_ARG, "%s: source layers [%d,%d) not inside [0,%d)", who, src_layer0, src_layer0 + layers, src_layers);
  if ((int64_t)dst_layer0 + layers > dst->layers)
    HX_FAIL(HX_ERR_INVALID_ARG, "%s: cache layers [%d,%d) not inside [0,%d)", who, dst_layer0, dst_layer0 + layers, dst->layers);
  if (batch == 0 || total_tokens == 0 || layers == 0) return HX_OK;
  if (!src_k || !src_v) HX_FAIL(HX_ERR_INVALID_ARG, "%s: src_k/src_v array is NULL", who);
  if (!block_table || !cu_seqlens || !seq_lens) HX_FAIL(HX_ERR_INVALID_ARG, "%s: block_table/cu_seqlens/seq_lens is NULL", who);
  if (max_seq_len > total_tokens) HX_FAIL(HX_ERR_INVALID_ARG, "%s: max_seq_len %d > total_tokens %d", who, max_seq_len, total_tokens);
  const int32_t ps = dst->page_size;
  if ((int64_t)stride * ps < (int64_t)max_seq_len) HX_FAIL(HX_ERR_INVALID_ARG, "%s: block_table_stride %d < ceil(max_seq_len %d / %d)", who, stride, max_seq_len, ps);
  if ((int64_t)src_layers * total_tokens * (heads / src_tp) * head_dim >= (int64_t)1 << 40) HX_FAIL(HX_ERR_UNSUPPORTED, "%s: shard too large", who);

  IngestParams p;
  memset(&p, 0, sizeof(p));
  p.hs = heads / src_tp; p.hd = heads / dst_tp; p.head0 = dst_rank * p.hd;
  const int r_lo = p.head0 / p.hs, r_hi = (p.head0 + p.hd - 1) / p.hs;
  for (int r = r_lo; r <= r_hi; ++r) {
    if (!src_k[r] || !src_v[r]) HX_FAIL(HX_ERR_INVALID_ARG, "%s: shard %d is needed by dst_rank %d but its pointer is NULL", who, r, dst_rank);
    if (!aligned16(src_k[r]) || !aligned16(src_v[r])) HX_FAIL(HX_ERR_INVALID_ARG, "%s: shard %d pointer not 16-byte aligned", who, r);
    p.src_k[r] = src_k[r]; p.src_v[r] = src_v[r];
  }
  p.dst_k = dst->k; p.dst_v = dst->v;
  p.block_table = block_table; p.cu_seqlens = cu_seqlens; p.seq_lens = seq_lens;
  p.layers = layers; p.total_tokens = total_tokens; p.batch = batch;
  p.src_layer0 = src_layer0; p.dst_layer0 = dst_layer0; p.src_layers = src_layers;
  p.head_dim = head_dim; p.page_size = ps; p.num_pages = dst->num_pages; p.bt_stride = stride;
  if (params_out) *params_out = p;                             // hx_decode_step(overlap_ingest): moved inside the attention kernel
  if (dry_run) return HX_OK;                                   // checks only (hx_decode_step validates before it enqueues)
  return launch_ingest(p, gather, static_cast<cudaStream_t>(stream));
}

}  // namespace hx

extern "C" {

int hx_version(void) { return HX_VERSION; }

const char* hx_status_string(int s) {
  switch (s) {
    case HX_OK: return "HX_OK";
    case HX_ERR_INVALID_ARG: return "HX_ERR_INVALID_ARG";
    case HX_ERR_UNSUPPORTED: return "HX_ERR_UNSUPPORTED";
    case HX_ERR_WORKSPACE: return "HX_ERR_WORKSPACE";
    case HX_ERR_CUDA: return "HX_ERR_CUDA";
    case HX_ERR_NO_PAGES: return "HX_ERR_NO_PAGES";
    default: return "HX_ERR_UNKNOWN";
  }
}

const char* hx_last_error(void) { return hx::g_err; }

size_t hx_paged_cache_bytes(int32_t layers, int32_t num_pages, int32_t kv_heads, int32_t page_size, int32_t head_dim) {
  if (layers <= 0 || num_pages <= 0 || kv_heads <= 0 || page_size <= 0 || head_dim <= 0) return 0;
  unsigned __int128 b = (unsigned __int128)layers * num_pages;
  b = b * kv_heads * page_size * head_dim * 2;
  if (b >> 62) return 0;
  return (size_t)b;
}

int hx_kv_ingest(const void* const* src_k, const void* const* src_v, int32_t layers, int32_t heads, int32_t head_dim,
                 int32_t src_tp, int32_t dst_tp, int32_t dst_rank, const hx_paged_cache* dst,
                 const int32_t* block_table, int32_t block_table_stride, const int32_t* cu_seqlens,
                 const int32_t* seq_lens, int32_t batch, int32_t total_tokens, int32_t max_seq_len, void* stream) {
  return hx::ingest_common(src_k, src_v, layers, heads, head_dim, src_tp, dst_tp, dst_rank, dst, block_table,
                           block_table_stride, cu_seqlens, seq_lens, batch, total_tokens, max_seq_len, stream, false,
                           "hx_kv_ingest", -1, 0, 0);
}

int hx_kv_ingest_stage(const void* const* src_k, const void* const* src_v, int32_t src_layers, int32_t src_layer0,
                       int32_t dst_layer0, int32_t layers, int32_t heads, int32_t head_dim, int32_t src_tp,
                       int32_t dst_tp, int32_t dst_rank, const hx_paged_cache* dst, const int32_t* block_table,
                       int32_t block_table_stride, const int32_t* cu_seqlens, const int32_t* seq_lens,
                       int32_t batch, int32_t total_tokens, int32_t max_seq_len, void* stream) {
  if (src_layers < 0) {
    hx::set_error("hx_kv_ingest_stage: src_layers %d is negative", src_layers);
    return HX_ERR_INVALID_ARG;
  }
  return hx::ingest_common(src_k, src_v, layers, heads, head_dim, src_tp, dst_tp, dst_rank, dst, block_table,
                           block_table_stride, cu_seqlens, seq_lens, batch, total_tokens, max_seq_len, stream, false,
                           "hx_kv_ingest_stage", src_layers, src_layer0, dst_layer0);
}

int hx_stage_overlap(int32_t src_first, int32_t src_count, int32_t dst_first, int32_t dst_count,
                     int32_t* src_layer0, int32_t* dst_layer0, int32_t* layers) {
  using namespace hx;
  clear_error();
  if (!src_layer0 || !dst_layer0 || !layers) HX_FAIL(HX_ERR_INVALID_ARG, "hx_stage_overlap: NULL output");
  if (src_first < 0 || src_count < 0 || dst_first < 0 || dst_count < 0) HX_FAIL(HX_ERR_INVALID_ARG, "hx_stage_overlap: negative input");
  const int64_t lo = src_first > dst_first ? src_first : dst_first;
  const int64_t se = (int64_t)src_first + src_count, de = (int64_t)dst_first + dst_count;
  const int64_t hi = se < de ? se : de;
  if (hi <= lo) { *src_layer0 = 0; *dst_layer0 = 0; *layers = 0; return HX_OK; }
  *src_layer0 = (int32_t)(lo - src_first); *dst_layer0 = (int32_t)(lo - dst_first); *layers = (int32_t)(hi - lo);
  return HX_OK;
}

int hx_kv_gather(void* const* src_k, void* const* src_v, int32_t layers, int32_t heads, int32_t head_dim,
                 int32_t src_tp, int32_t dst_tp, int32_t dst_rank, const hx_paged_cache* dst,
                 const int32_t* block_table, int32_t block_table_stride, const int32_t* cu_seqlens,
                 const int32_t* seq_lens, int32_t batch, int32_t total_tokens, int32_t max_seq_len, void* stream) {
  return hx::ingest_common(const_cast<const void* const*>(src_k), const_cast<const void* const*>(src_v), layers, heads,
                           head_dim, src_tp, dst_tp, dst_rank, dst, block_table, block_table_stride, cu_seqlens,
                           seq_lens, batch, total_tokens, max_seq_len, stream, true, "hx_kv_gather", -1, 0, 0);
}

size_t hx_decode_attention_workspace_bytes(int32_t batch, int32_t q_heads, int32_t kv_heads, int32_t head_dim,
                                           int32_t max_seq_len, int32_t page_size) {
  if (batch < 0 || q_heads <= 0 || kv_heads <= 0 || head_dim <= 0 || max_seq_len < 0 || page_size <= 0) return 0;
  return hx::attn_workspace_bytes(batch, q_heads, kv_heads, head_dim, max_seq_len, page_size);
}

// mode: 0 = hx_decode_attention (and _append / _overlapped), 1 = hx_decode_plan (writes `plan`), 2 = hx_decode_attention_planned
// pdl: 0 = plain launch; 3 = hx_decode_attention_overlapped(behind_ingest != 0): programmatic dependent of the ingest kernel
//      the caller says is directly before it; 1 / 2 = hx_decode_attention_chained (inputs_ready = 0 / 1)
static int attention_common(const char* who, void* out, const void* q, const void* k_new, const void* v_new, bool append, int pdl,
                            const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                            const int32_t* block_table, int32_t block_table_stride, const int32_t* seq_lens,
                            int32_t batch, int32_t max_seq_len, float sm_scale, void* workspace,
                            size_t workspace_bytes, void* stream, bool dry_run = false, int mode = 0,
                            void* plan = nullptr, size_t plan_bytes = 0, const hx::IngestParams* handoff = nullptr,
                            int32_t handoff_max_seq_len = 0, const hx::TileMaps* handoff_maps = nullptr) {
  using namespace hx;
  clear_error();
  if (batch < 0 || max_seq_len < 0) HX_FAIL(HX_ERR_INVALID_ARG, "%s: negative size (batch=%d max_seq_len=%d)", who, batch, max_seq_len);
  int rc = check_cache(cache, who);
  if (rc) return rc;
  if (layer < 0 || layer >= cache->layers) HX_FAIL(HX_ERR_INVALID_ARG, "%s: layer %d not in [0,%d)", who, layer, cache->layers);
  if (q_heads <= 0 || q_heads % cache->kv_heads) HX_FAIL(HX_ERR_INVALID_ARG, "%s: q_heads %d not a positive multiple of kv_heads %d", who, q_heads, cache->kv_heads);
  const int G = q_heads / cache->kv_heads;
  if (G != 1 && G != 2 && G != 4 && G != 8 && G != 16) HX_FAIL(HX_ERR_UNSUPPORTED, "%s: group size %d not in {1,2,4,8,16}", who, G);
  if (!(sm_scale == sm_scale) || sm_scale > 1e30f) HX_FAIL(HX_ERR_INVALID_ARG, "%s: sm_scale is NaN or too large", who);
  if (batch == 0) return HX_OK;
  if (mode != 1) {
    if (!out || !q) HX_FAIL(HX_ERR_INVALID_ARG, "%s: out/q is NULL", who);
    if (!aligned16(out) || !aligned16(q)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: out/q must be 16-byte aligned", who);
  }
  if (mode != 2 && (!block_table || !seq_lens)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: block_table/seq_lens is NULL", who);
  if (mode != 0) {
    if (!plan || !aligned16(plan)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: plan is NULL or not 16-byte aligned", who);
    const size_t pneed = attn_plan_bytes(batch, cache->kv_heads, max_seq_len, cache->page_size);
    if (plan_bytes < pneed) HX_FAIL(HX_ERR_WORKSPACE, "%s: plan buffer %zu bytes < required %zu", who, plan_bytes, pneed);
  }
  if (append) {
    if (!k_new || !v_new) HX_FAIL(HX_ERR_INVALID_ARG, "%s: k_new/v_new is NULL", who);
    if (!aligned16(k_new) || !aligned16(v_new)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: k_new/v_new must be 16-byte aligned", who);
  }
  if ((int64_t)block_table_stride * cache->page_size < (int64_t)max_seq_len)
    HX_FAIL(HX_ERR_INVALID_ARG, "%s: block_table_stride %d < ceil(max_seq_len %d / %d)", who, block_table_stride, max_seq_len, cache->page_size);
  // size limits of the launch itself, checked here so that a dry run (hx_decode_step validates the whole step before it
  // enqueues anything) sees them too; launch_stream / launch_plan repeat them
  if (mode != 1 && (uint64_t)cache->num_pages * cache->kv_heads * 16 * cache->layers >= (1ull << 31))
    HX_FAIL(HX_ERR_UNSUPPORTED, "%s: cache too large for one tensor map (%llu rows)", who,
            (unsigned long long)((uint64_t)cache->num_pages * cache->kv_heads * 16 * cache->layers));
  if ((long long)kAttnBatchPerLaunch * block_table_stride * cache->kv_heads >= (1ll << 28))
    HX_FAIL(HX_ERR_UNSUPPORTED, "%s: block_table_stride * kv_heads too large", who);
  if (mode != 0 && batch > kAttnBatchPerLaunch)
    HX_FAIL(HX_ERR_UNSUPPORTED, "%s: a plan covers at most %d requests (batch %d)", who, kAttnBatchPerLaunch, batch);
  const size_t need = mode == 1 ? 0 : attn_workspace_bytes(batch, q_heads, cache->kv_heads, cache->head_dim, max_seq_len, cache->page_size);
  if (need > 0 && (!workspace || workspace_bytes < need)) HX_FAIL(HX_ERR_WORKSPACE, "%s: workspace %zu bytes < required %zu (or NULL)", who, workspace_bytes, need);
  if (need > 0 && !aligned16(workspace)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: workspace must be 16-byte aligned", who);
  if (sm_scale <= 0.f) sm_scale = 1.0f / sqrtf((float)cache->head_dim);

  AttnParams p;
  memset(&p, 0, sizeof(p));
  p.out = out; p.q = q;
  p.k_base = cache->k; p.v_base = cache->v; p.layer = layer; p.layers = cache->layers;
  p.block_table = block_table; p.seq_lens = seq_lens;
  p.workspace = workspace; p.workspace_bytes = workspace_bytes;
  p.batch = batch; p.q_heads = q_heads; p.kv_heads = cache->kv_heads; p.head_dim = cache->head_dim;
  p.page_size = cache->page_size; p.num_pages = cache->num_pages; p.bt_stride = block_table_stride;
  p.max_seq_len = max_seq_len; p.sm_scale = sm_scale;
  p.k_new = append ? k_new : nullptr; p.v_new = append ? v_new : nullptr;
  p.overlap_prev = pdl;            // what the launch may overlap is the caller's explicit statement, never inferred
  p.plan = mode != 0 ? plan : nullptr;
  p.handoff = handoff; p.handoff_max_seq_len = handoff_max_seq_len; p.handoff_maps = handoff_maps;
  if (dry_run) return HX_OK;
  return mode == 1 ? launch_plan(p, static_cast<cudaStream_t>(stream)) : launch_attention(p, static_cast<cudaStream_t>(stream));
}

int hx_decode_attention(void* out, const void* q, const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                        const int32_t* block_table, int32_t block_table_stride, const int32_t* seq_lens,
                        int32_t batch, int32_t max_seq_len, float sm_scale, void* workspace,
                        size_t workspace_bytes, void* stream) {
  return attention_common("hx_decode_attention", out, q, nullptr, nullptr, false, 0, cache, layer, q_heads, block_table,
                          block_table_stride, seq_lens, batch, max_seq_len, sm_scale, workspace, workspace_bytes, stream);
}

int hx_decode_attention_append(void* out, const void* q, const void* k_new, const void* v_new,
                               const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                               const int32_t* block_table, int32_t block_table_stride, const int32_t* seq_lens,
                               int32_t batch, int32_t max_seq_len, float sm_scale, void* workspace,
                               size_t workspace_bytes, void* stream) {
  return attention_common("hx_decode_attention_append", out, q, k_new, v_new, true, 0, cache, layer, q_heads, block_table,
                          block_table_stride, seq_lens, batch, max_seq_len, sm_scale, workspace, workspace_bytes, stream);
}

int hx_decode_attention_overlapped(void* out, const void* q, const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                                   const int32_t* block_table, int32_t block_table_stride, const int32_t* seq_lens,
                                   int32_t batch, int32_t max_seq_len, float sm_scale, void* workspace,
                                   size_t workspace_bytes, int32_t behind_ingest, void* stream) {
  return attention_common("hx_decode_attention_overlapped", out, q, nullptr, nullptr, false, behind_ingest ? 3 : 0, cache, layer, q_heads,
                          block_table, block_table_stride, seq_lens, batch, max_seq_len, sm_scale, workspace,
                          workspace_bytes, stream);
}

// ---- hx_decode_attention_noalloc: the attention workspace for callers that cannot allocate one (include/hx.h) ----
// The scratch is a file-scope device array: it is part of this translation unit's device image, so the driver places it
// on every GPU that loads the image and releases it when the process exits; nobody calls cudaMalloc for it.
// Its zero-initialisation at load time only helps the very first call; after that it holds the last call's partials and
// counters, which is why every call clears the counter span of ITS shape first (the span's offset depends on the shape).
//
// g_noalloc_scratch is usable by name in device code only.  On the host the name is a stand-in symbol whose address is
// NOT a device address (passing it to a kernel faults, or silently reads host memory where the GPU can reach it), so
// host code asks the runtime for the real address once per device, with that device current, and caches it.
static __device__ __align__(256) unsigned char g_noalloc_scratch[HX_NOALLOC_SCRATCH_BYTES];

namespace {
std::mutex g_noalloc_mu;
void* g_noalloc_ptr[64] = {nullptr};   // device address of g_noalloc_scratch on device d; filled by the first call there

// Device address of the built-in scratch on the CURRENT device.  The first call per device does the look-up (it may
// load this module onto the device, so it belongs outside any stream capture); later calls only read the table.
int noalloc_scratch(void** out) {
  using namespace hx;
  int dev = 0;
  HX_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) HX_FAIL(HX_ERR_CUDA, "device id %d out of range", dev);
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    void* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
    if (e != cudaSuccess || !ptr)
      HX_FAIL(HX_ERR_CUDA, "hx_decode_attention_noalloc: cudaGetSymbolAddress(built-in scratch) on device %d: %s", dev,
              e != cudaSuccess ? cudaGetErrorString(e) : "returned a NULL address");
    g_noalloc_ptr[dev] = ptr;
  }
  *out = g_noalloc_ptr[dev];
  return HX_OK;
}
}  // namespace

int hx_decode_attention_noalloc(void* out, const void* q, const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                                const int32_t* block_table, int32_t block_table_stride, const int32_t* seq_lens,
                                int32_t batch, int32_t max_seq_len, float sm_scale, void* stream) {
  using namespace hx;
  const char* who = "hx_decode_attention_noalloc";
  // 1. every argument check of hx_decode_attention, without touching CUDA (a placeholder stands in for the workspace:
  //    a dry run reads neither the pointer's target nor the device)
  void* const placeholder = reinterpret_cast<void*>(static_cast<uintptr_t>(256));
  int rc = attention_common(who, out, q, nullptr, nullptr, false, 0, cache, layer, q_heads, block_table, block_table_stride,
                            seq_lens, batch, max_seq_len, sm_scale, placeholder, ~(size_t)0, stream, /*dry_run=*/true);
  if (rc) return rc;
  if (batch == 0) return HX_OK;                                 // nothing to do, as in hx_decode_attention
  // 2. does this shape fit the built-in array?
  const size_t need = attn_workspace_bytes(batch, q_heads, cache->kv_heads, cache->head_dim, max_seq_len, cache->page_size);
  if (need > HX_NOALLOC_SCRATCH_BYTES)
    HX_FAIL(HX_ERR_WORKSPACE, "%s: q_heads=%d kv_heads=%d head_dim=%d needs %zu bytes of scratch, the built-in array holds "
            "%zu (HX_NOALLOC_SCRATCH_BYTES); call hx_decode_attention with a workspace of your own for this shape",
            who, q_heads, cache->kv_heads, cache->head_dim, need, (size_t)HX_NOALLOC_SCRATCH_BYTES);
  // 3. the array's address on this device (looked up once per device)
  void* scratch = nullptr;
  rc = noalloc_scratch(&scratch);
  if (rc) return rc;
  // 4. the array still holds the previous call's contents, and for another shape the counters lie where that call kept
  //    partial results: clear this shape's counters, on the caller's stream, directly ahead of the kernel
  size_t zoff = 0, zbytes = 0;
  attn_workspace_zero_span(q_heads, cache->kv_heads, cache->head_dim, &zoff, &zbytes);
  HX_CUDA_OK(cudaMemsetAsync(static_cast<char*>(scratch) + zoff, 0, zbytes, static_cast<cudaStream_t>(stream)));
  // 5. the unchanged hx_decode_attention path, with the built-in array as its workspace
  return attention_common(who, out, q, nullptr, nullptr, false, 0, cache, layer, q_heads, block_table, block_table_stride,
                          seq_lens, batch, max_seq_len, sm_scale, scratch, HX_NOALLOC_SCRATCH_BYTES, stream);
}

int hx_kv_append(const void* k_new, const void* v_new, const hx_paged_cache* cache, int32_t layer,
                 const int32_t* block_table, int32_t block_table_stride, const int32_t* seq_lens, int32_t batch,
                 int32_t max_seq_len, void* stream) {
  using namespace hx;
  const char* who = "hx_kv_append";
  clear_error();
  if (batch < 0 || max_seq_len < 0) HX_FAIL(HX_ERR_INVALID_ARG, "%s: negative size (batch=%d max_seq_len=%d)", who, batch, max_seq_len);
  int rc = check_cache(cache, who);
  if (rc) return rc;
  if (layer < 0 || layer >= cache->layers) HX_FAIL(HX_ERR_INVALID_ARG, "%s: layer %d not in [0,%d)", who, layer, cache->layers);
  if (batch == 0) return HX_OK;
  if (!k_new || !v_new) HX_FAIL(HX_ERR_INVALID_ARG, "%s: k_new/v_new is NULL", who);
  if (!aligned16(k_new) || !aligned16(v_new)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: k_new/v_new must be 16-byte aligned", who);
  if (!block_table || !seq_lens) HX_FAIL(HX_ERR_INVALID_ARG, "%s: block_table/seq_lens is NULL", who);
  if ((int64_t)block_table_stride * cache->page_size < (int64_t)max_seq_len)
    HX_FAIL(HX_ERR_INVALID_ARG, "%s: block_table_stride %d < ceil(max_seq_len %d / %d)", who, block_table_stride, max_seq_len, cache->page_size);
  if ((int64_t)batch * 2 * cache->kv_heads * (cache->head_dim / 8) >= (int64_t)1 << 31) HX_FAIL(HX_ERR_UNSUPPORTED, "%s: batch too large", who);
  AppendParams p;
  const size_t layer_elems = (size_t)cache->num_pages * cache->kv_heads * cache->page_size * cache->head_dim;
  p.k_new = k_new; p.v_new = v_new;
  p.k = static_cast<uint16_t*>(cache->k) + layer_elems * layer;
  p.v = static_cast<uint16_t*>(cache->v) + layer_elems * layer;
  p.block_table = block_table; p.seq_lens = seq_lens;
  p.batch = batch; p.kv_heads = cache->kv_heads; p.head_dim = cache->head_dim; p.page_size = cache->page_size;
  p.bt_stride = block_table_stride;
  return launch_append(p, static_cast<cudaStream_t>(stream));
}

int hx_prefill_attention(void* out, const void* q, const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                         const int32_t* block_table, int32_t block_table_stride, const int32_t* seq_lens,
                         const int32_t* q_lens, const int32_t* cu_q_lens, int32_t batch, int32_t total_q_tokens,
                         int32_t max_q_len, int32_t max_seq_len, float sm_scale, void* stream) {
  using namespace hx;
  const char* who = "hx_prefill_attention";
  clear_error();
  if (batch < 0 || total_q_tokens < 0 || max_q_len < 0 || max_seq_len < 0)
    HX_FAIL(HX_ERR_INVALID_ARG, "%s: negative size (batch=%d total_q_tokens=%d max_q_len=%d max_seq_len=%d)", who, batch, total_q_tokens, max_q_len, max_seq_len);
  int rc = check_cache(cache, who);
  if (rc) return rc;
  if (layer < 0 || layer >= cache->layers) HX_FAIL(HX_ERR_INVALID_ARG, "%s: layer %d not in [0,%d)", who, layer, cache->layers);
  if (q_heads <= 0 || q_heads % cache->kv_heads) HX_FAIL(HX_ERR_INVALID_ARG, "%s: q_heads %d not a positive multiple of kv_heads %d", who, q_heads, cache->kv_heads);
  const int G = q_heads / cache->kv_heads;
  if (G != 1 && G != 2 && G != 4 && G != 8 && G != 16) HX_FAIL(HX_ERR_UNSUPPORTED, "%s: group size %d not in {1,2,4,8,16}", who, G);
  if (!(sm_scale == sm_scale) || sm_scale > 1e30f) HX_FAIL(HX_ERR_INVALID_ARG, "%s: sm_scale is NaN or too large", who);
  if (max_q_len > max_seq_len || max_q_len > total_q_tokens) HX_FAIL(HX_ERR_INVALID_ARG, "%s: max_q_len %d > max_seq_len %d or total_q_tokens %d", who, max_q_len, max_seq_len, total_q_tokens);
  if (batch == 0 || total_q_tokens == 0 || max_q_len == 0) return HX_OK;
  if (!out || !q) HX_FAIL(HX_ERR_INVALID_ARG, "%s: out/q is NULL", who);
  if (!aligned16(out) || !aligned16(q)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: out/q must be 16-byte aligned", who);
  if (!block_table || !seq_lens || !q_lens || !cu_q_lens) HX_FAIL(HX_ERR_INVALID_ARG, "%s: block_table/seq_lens/q_lens/cu_q_lens is NULL", who);
  if ((int64_t)block_table_stride * cache->page_size < (int64_t)max_seq_len)
    HX_FAIL(HX_ERR_INVALID_ARG, "%s: block_table_stride %d < ceil(max_seq_len %d / %d)", who, block_table_stride, max_seq_len, cache->page_size);
  if (sm_scale <= 0.f) sm_scale = 1.0f / sqrtf((float)cache->head_dim);
  PrefillArgs a;
  memset(&a, 0, sizeof(a));
  a.out = out; a.q = q; a.k_base = cache->k; a.v_base = cache->v;
  a.block_table = block_table; a.seq_lens = seq_lens; a.q_lens = q_lens; a.cu_q_lens = cu_q_lens;
  a.batch = batch; a.q_heads = q_heads; a.kv_heads = cache->kv_heads; a.head_dim = cache->head_dim;
  a.num_pages = cache->num_pages; a.bt_stride = block_table_stride; a.layer = layer; a.layers = cache->layers;
  a.total_q = total_q_tokens; a.max_q_len = max_q_len; a.sm_scale = sm_scale;
  return launch_prefill(a, static_cast<cudaStream_t>(stream));
}

size_t hx_decode_plan_bytes(int32_t batch, int32_t kv_heads, int32_t max_seq_len, int32_t page_size) {
  if (batch < 0 || kv_heads <= 0 || max_seq_len < 0 || page_size <= 0) return 0;
  return hx::attn_plan_bytes(batch, kv_heads, max_seq_len, page_size);
}

int hx_decode_plan(void* plan, size_t plan_bytes, const hx_paged_cache* cache, int32_t q_heads, const int32_t* block_table,
                   int32_t block_table_stride, const int32_t* seq_lens, int32_t batch, int32_t max_seq_len, void* stream) {
  return attention_common("hx_decode_plan", nullptr, nullptr, nullptr, nullptr, false, 0, cache, 0, q_heads, block_table,
                          block_table_stride, seq_lens, batch, max_seq_len, 0.f, nullptr, 0, stream, false, 1, plan, plan_bytes);
}

int hx_decode_attention_planned(void* out, const void* q, const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                                const void* plan, size_t plan_bytes, int32_t batch, int32_t max_seq_len, float sm_scale,
                                void* workspace, size_t workspace_bytes, void* stream) {
  const int32_t ps = (cache && cache->page_size > 0) ? cache->page_size : 16;
  return attention_common("hx_decode_attention_planned", out, q, nullptr, nullptr, false, 0, cache, layer, q_heads, nullptr,
                          (max_seq_len + ps - 1) / ps, nullptr, batch, max_seq_len, sm_scale, workspace, workspace_bytes, stream,
                          false, 2, const_cast<void*>(plan), plan_bytes);
}

int hx_decode_attention_chained(void* out, const void* q, const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                                const void* plan, size_t plan_bytes, int32_t batch, int32_t max_seq_len, float sm_scale,
                                void* workspace, size_t workspace_bytes, int32_t inputs_ready, void* stream) {
  const int32_t ps = (cache && cache->page_size > 0) ? cache->page_size : 16;
  return attention_common("hx_decode_attention_chained", out, q, nullptr, nullptr, false, inputs_ready ? 2 : 1, cache, layer, q_heads,
                          nullptr, (max_seq_len + ps - 1) / ps, nullptr, batch, max_seq_len, sm_scale, workspace, workspace_bytes,
                          stream, false, 2, const_cast<void*>(plan), plan_bytes);
}

// ---- whole decode step (row A9): library-owned side stream per device for the overlapped handoff ----
namespace {
struct SideStream { cudaStream_t stream = nullptr; cudaEvent_t fork = nullptr, join = nullptr; };
std::mutex g_step_mu;                 // held from fork to join: one step is enqueued at a time per process
SideStream g_side[64];

int side_stream(int* dev_out, SideStream** out) {
  using namespace hx;
  int dev = 0;
  HX_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) HX_FAIL(HX_ERR_CUDA, "device id %d out of range", dev);
  SideStream& s = g_side[dev];
  if (!s.stream) {
    // all three or none: a half-made set would be skipped by every later call and fail in cudaEventRecord for good
    SideStream made;
    cudaError_t e = cudaStreamCreateWithFlags(&made.stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&made.fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&made.join, cudaEventDisableTiming);
    if (e != cudaSuccess) {
      if (made.join) cudaEventDestroy(made.join);
      if (made.fork) cudaEventDestroy(made.fork);
      if (made.stream) cudaStreamDestroy(made.stream);
      HX_FAIL(HX_ERR_CUDA, "side stream / events for the overlapped handoff on device %d: %s", dev, cudaGetErrorString(e));
    }
    s = made;
  }
  *dev_out = dev; *out = &s;
  return HX_OK;
}

// The step on device buffers.  `h` (optional) adds the host<->device copies of hx_decode_step_host.
// query_fused != NULL: validate, decide whether the step would run as one fused kernel, report it and enqueue nothing.
int step_impl(const char* who, const hx_step_args* a, const hx_step_host_args* h, void* stream_, int32_t* query_fused = nullptr) {
  using namespace hx;
  cudaStream_t main_stream = static_cast<cudaStream_t>(stream_);
  const bool do_ing = a->ing_batch > 0, do_att = a->batch > 0;
  // ---- every host-side check first: nothing is enqueued unless the whole step is valid
  if (a->batch < 0 || a->ing_batch < 0) HX_FAIL(HX_ERR_INVALID_ARG, "%s: negative batch", who);
  if (!a->cache) HX_FAIL(HX_ERR_INVALID_ARG, "%s: cache is NULL", who);
  int rc;
  if (do_ing) {
    if (!a->src_k || !a->src_v) HX_FAIL(HX_ERR_INVALID_ARG, "%s: src_k/src_v is NULL", who);
    rc = ingest_common(a->src_k, a->src_v, a->ing_layers, a->heads, a->cache->head_dim, a->src_tp, a->dst_tp, a->dst_rank,
                       a->cache, a->ing_block_table, a->ing_block_table_stride, a->ing_cu_seqlens, a->ing_seq_lens,
                       a->ing_batch, a->ing_total_tokens, a->ing_max_seq_len, stream_, false, who, -1, 0, 0, /*dry_run=*/true);
    if (rc) return rc;
  }
  if (do_att) {
    rc = attention_common(who, a->out, a->q, nullptr, nullptr, false, 0, a->cache, a->layer, a->q_heads, a->block_table,
                          a->block_table_stride, a->seq_lens, a->batch, a->max_seq_len, a->sm_scale, a->workspace,
                          a->workspace_bytes, stream_, /*dry_run=*/true);
    if (rc) return rc;
  }
  size_t qbytes = 0, shard = 0;
  if (h) {
    if (do_att && (!h->q_host || !h->out_host)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: q_host/out_host is NULL", who);
    qbytes = (size_t)a->batch * a->q_heads * a->cache->head_dim * 2;
    if (do_ing) {
      if (!h->src_k_host || !h->src_v_host || !h->ing_block_table_host || !h->ing_cu_seqlens_host || !h->ing_seq_lens_host)
        HX_FAIL(HX_ERR_INVALID_ARG, "%s: host ingest buffers missing", who);
      if (!h->pull_src && (!h->src_k_dev || !h->src_v_dev)) HX_FAIL(HX_ERR_INVALID_ARG, "%s: device staging for the shards missing", who);
      shard = (size_t)a->ing_layers * a->ing_total_tokens * (a->heads / a->src_tp) * a->cache->head_dim * 2;
    }
  }

  // ---- enqueue.
  // overlap_ingest, device buffers: ONE kernel.  The attention kernel carries the handoff: every warp that has finished
  // its attention range moves (page, head) tiles of the new prompts with the copy engines (handoff_tiles.cuh) until none
  // are left, so the handoff runs in the slack the attention's uneven finish leaves, at warp granularity.
  // overlap_ingest, host buffers (hx_decode_step_host): the shards must cross PCIe first; copies + ingest go to the
  // library's side stream, forked from and joined to the caller's stream; once forked, every exit path joins.
  std::lock_guard<std::mutex> lock(g_step_mu);
  const bool overlap = a->overlap_ingest != 0 && do_ing && do_att;
  // an EMPTY handoff (every new prompt of length 0, or no layers) is a valid no-op for hx_kv_ingest; ingest_common then
  // returns before it fills `ip`, so such a step takes the in-order path (whose ingest half launches nothing)
  const bool handoff_empty = a->ing_total_tokens == 0 || a->ing_layers == 0;
  bool fused = overlap && !h && !handoff_empty && a->batch <= 2048 &&
               (int64_t)a->ing_layers * a->ing_batch * ((a->ing_max_seq_len + 15) / 16) * a->heads < ((int64_t)1 << 28);
  IngestParams ip{};
  TileMaps ip_maps;
  if (fused) {                       // the handoff's parameters and the tensor maps of its source shards (no launch yet)
    rc = ingest_common(a->src_k, a->src_v, a->ing_layers, a->heads, a->cache->head_dim, a->src_tp, a->dst_tp, a->dst_rank,
                       a->cache, a->ing_block_table, a->ing_block_table_stride, a->ing_cu_seqlens, a->ing_seq_lens,
                       a->ing_batch, a->ing_total_tokens, a->ing_max_seq_len, stream_, false, who, -1, 0, 0, /*dry_run=*/true, &ip);
    if (rc) return rc;
    rc = tile_maps(ip, &ip_maps, &fused);   // shards the copy engines cannot take (managed memory, > 8 shards): in order instead
    if (rc) return rc;
  }
  if (query_fused) { *query_fused = fused ? 1 : 0; return HX_OK; }
  const bool fork = overlap && h;
  SideStream* ss = nullptr;
  cudaStream_t ing_stream = main_stream;
  int dev = 0;
  if (fork) {
    rc = side_stream(&dev, &ss);
    if (rc) return rc;
    HX_CUDA_OK(cudaEventRecord(ss->fork, main_stream));
    HX_CUDA_OK(cudaStreamWaitEvent(ss->stream, ss->fork, 0));
    ing_stream = ss->stream;
  }
  rc = HX_OK;
  cudaError_t ce = cudaSuccess;
  const char* what = "";
#define STEP_CUDA(expr) do { if (rc == HX_OK && ce == cudaSuccess) { ce = (expr); if (ce != cudaSuccess) what = #expr; } } while (0)
  // the attention's small q upload goes first on the caller's stream so that it is not queued behind the shards
  if (h && do_att) STEP_CUDA(cudaMemcpyAsync(const_cast<void*>(a->q), h->q_host, qbytes, cudaMemcpyHostToDevice, main_stream));
  auto enqueue_attention = [&]() {
    if (rc == HX_OK && ce == cudaSuccess)
      rc = attention_common(who, a->out, a->q, nullptr, nullptr, false, 0, a->cache, a->layer, a->q_heads, a->block_table,
                            a->block_table_stride, a->seq_lens, a->batch, a->max_seq_len, a->sm_scale, a->workspace,
                            a->workspace_bytes, stream_);
  };
  auto enqueue_ingest = [&]() {
    if (rc == HX_OK && ce == cudaSuccess)
      rc = ingest_common(a->src_k, a->src_v, a->ing_layers, a->heads, a->cache->head_dim, a->src_tp, a->dst_tp, a->dst_rank,
                         a->cache, a->ing_block_table, a->ing_block_table_stride, a->ing_cu_seqlens, a->ing_seq_lens,
                         a->ing_batch, a->ing_total_tokens, a->ing_max_seq_len, static_cast<void*>(ing_stream), false, who, -1, 0, 0);
  };
  if (fused) {
    // one launch: the timing events (optional) bracket it
    if (a->ev_ingest_begin) STEP_CUDA(cudaEventRecord(static_cast<cudaEvent_t>(a->ev_ingest_begin), main_stream));
    if (a->ev_attention_begin) STEP_CUDA(cudaEventRecord(static_cast<cudaEvent_t>(a->ev_attention_begin), main_stream));
    if (rc == HX_OK && ce == cudaSuccess)
      rc = attention_common(who, a->out, a->q, nullptr, nullptr, false, 0, a->cache, a->layer, a->q_heads, a->block_table,
                            a->block_table_stride, a->seq_lens, a->batch, a->max_seq_len, a->sm_scale, a->workspace,
                            a->workspace_bytes, stream_, false, 0, nullptr, 0, &ip, a->ing_max_seq_len, &ip_maps);
    if (a->ev_attention_end) STEP_CUDA(cudaEventRecord(static_cast<cudaEvent_t>(a->ev_attention_end), main_stream));
    if (a->ev_ingest_end) STEP_CUDA(cudaEventRecord(static_cast<cudaEvent_t>(a->ev_ingest_end), main_stream));
  } else {
    if (do_ing) {
      if (h) {
        for (int r = 0; r < a->src_tp && !h->pull_src; ++r) {
          if (!h->src_k_host[r] || !h->src_k_dev[r]) continue;   // shard not needed by this rank
          STEP_CUDA(cudaMemcpyAsync(h->src_k_dev[r], h->src_k_host[r], shard, cudaMemcpyHostToDevice, ing_stream));
          STEP_CUDA(cudaMemcpyAsync(h->src_v_dev[r], h->src_v_host[r], shard, cudaMemcpyHostToDevice, ing_stream));
        }
        STEP_CUDA(cudaMemcpyAsync(const_cast<int32_t*>(a->ing_block_table), h->ing_block_table_host,
                                  (size_t)a->ing_batch * a->ing_block_table_stride * 4, cudaMemcpyHostToDevice, ing_stream));
        STEP_CUDA(cudaMemcpyAsync(const_cast<int32_t*>(a->ing_cu_seqlens), h->ing_cu_seqlens_host, (size_t)(a->ing_batch + 1) * 4,
                                  cudaMemcpyHostToDevice, ing_stream));
        STEP_CUDA(cudaMemcpyAsync(const_cast<int32_t*>(a->ing_seq_lens), h->ing_seq_lens_host, (size_t)a->ing_batch * 4,
                                  cudaMemcpyHostToDevice, ing_stream));
      }
      if (a->ev_ingest_begin) STEP_CUDA(cudaEventRecord(static_cast<cudaEvent_t>(a->ev_ingest_begin), ing_stream));
      enqueue_ingest();
      if (a->ev_ingest_end) STEP_CUDA(cudaEventRecord(static_cast<cudaEvent_t>(a->ev_ingest_end), ing_stream));
    }
    if (do_att) {
      if (a->ev_attention_begin) STEP_CUDA(cudaEventRecord(static_cast<cudaEvent_t>(a->ev_attention_begin), main_stream));
      enqueue_attention();
      if (a->ev_attention_end) STEP_CUDA(cudaEventRecord(static_cast<cudaEvent_t>(a->ev_attention_end), main_stream));
      if (h) STEP_CUDA(cudaMemcpyAsync(h->out_host, a->out, qbytes, cudaMemcpyDeviceToHost, main_stream));
    }
  }
#undef STEP_CUDA
  if (fork) {                                                   // join on every path, error or not
    cudaError_t j = cudaEventRecord(ss->join, ss->stream);
    if (j == cudaSuccess) j = cudaStreamWaitEvent(main_stream, ss->join, 0);
    if (j != cudaSuccess && rc == HX_OK && ce == cudaSuccess) { ce = j; what = "join of the side stream"; }
  }
  if (rc != HX_OK) return rc;                                   // hx_last_error() already holds the detail
  if (ce != cudaSuccess) HX_FAIL(HX_ERR_CUDA, "%s: %s: %s", who, what, cudaGetErrorString(ce));
  return HX_OK;
}
}  // namespace

int hx_decode_step(const hx_step_args* a, void* stream) {
  using namespace hx;
  clear_error();
  if (!a) HX_FAIL(HX_ERR_INVALID_ARG, "hx_decode_step: args is NULL");
  return step_impl("hx_decode_step", a, nullptr, stream);
}

int hx_decode_step_is_fused(const hx_step_args* a, int32_t* fused) {
  using namespace hx;
  clear_error();
  if (!a || !fused) HX_FAIL(HX_ERR_INVALID_ARG, "hx_decode_step_is_fused: args / fused is NULL");
  *fused = 0;
  return step_impl("hx_decode_step_is_fused", a, nullptr, nullptr, fused);
}

int hx_decode_step_host(const hx_step_host_args* h, void* stream) {
  using namespace hx;
  clear_error();
  if (!h) HX_FAIL(HX_ERR_INVALID_ARG, "hx_decode_step_host: args is NULL");
  hx_step_args a;
  memset(&a, 0, sizeof(a));
  a.out = h->out_dev; a.q = h->q_dev; a.cache = h->cache; a.layer = h->layer; a.q_heads = h->q_heads;
  a.block_table = h->block_table_dev; a.block_table_stride = h->block_table_stride; a.seq_lens = h->seq_lens_dev;
  a.batch = h->batch; a.max_seq_len = h->max_seq_len; a.sm_scale = h->sm_scale;
  a.workspace = h->workspace; a.workspace_bytes = h->workspace_bytes;
  // pull mode (F2): the ingest kernel reads the host shards over the link itself
  a.src_k = h->pull_src ? h->src_k_host : const_cast<const void* const*>(h->src_k_dev);
  a.src_v = h->pull_src ? h->src_v_host : const_cast<const void* const*>(h->src_v_dev);
  a.ing_layers = h->ing_layers; a.heads = h->heads; a.src_tp = h->src_tp; a.dst_tp = h->dst_tp; a.dst_rank = h->dst_rank;
  a.ing_block_table = h->ing_block_table_dev; a.ing_block_table_stride = h->ing_block_table_stride;
  a.ing_cu_seqlens = h->ing_cu_seqlens_dev; a.ing_seq_lens = h->ing_seq_lens_dev;
  a.ing_batch = h->ing_batch; a.ing_total_tokens = h->ing_total_tokens; a.ing_max_seq_len = h->ing_max_seq_len;
  a.overlap_ingest = h->overlap_ingest;
  return step_impl("hx_decode_step_host", &a, h, stream);
}

int hx_shutdown(void) {
  using namespace hx;
  clear_error();
  std::lock_guard<std::mutex> lock(g_step_mu);
  int cur = 0;
  HX_CUDA_OK(cudaGetDevice(&cur));
  for (int d = 0; d < 64; ++d) {
    SideStream& s = g_side[d];
    if (!s.stream) continue;
    HX_CUDA_OK(cudaSetDevice(d));
    cudaStreamSynchronize(s.stream);
    cudaEventDestroy(s.fork); cudaEventDestroy(s.join); cudaStreamDestroy(s.stream);
    s = SideStream();
  }
  HX_CUDA_OK(cudaSetDevice(cur));
  return HX_OK;
}

}  // extern "C"
