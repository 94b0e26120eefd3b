// Internal helpers shared by the libhx translation units (not part of the ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "hx.h"

namespace hx {

// Thread-local error text behind hx_last_error().
void set_error(const char* fmt, ...);
void clear_error();

#define HX_FAIL(status, ...)        \
  do {                              \
    ::hx::set_error(__VA_ARGS__);   \
    return (status);                \
  } while (0)

#define HX_CUDA_OK(expr)                                                              \
  do {                                                                                \
    cudaError_t e_ = (expr);                                                          \
    if (e_ != cudaSuccess) HX_FAIL(HX_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

struct DeviceInfo {
  int device = -1;
  int sm_count = 0;
  int max_smem_optin = 0;
};
// Properties of the current device (cached per device id).
int device_info(DeviceInfo* out);

// ---- launchers implemented in ingest.cu / attention.cu (arguments already validated) ----
struct TileUnits;
struct TileMaps;
struct IngestParams {
  const void* src_k[16];
  const void* src_v[16];
  void* dst_k;
  void* dst_v;
  const int32_t* block_table;
  const int32_t* cu_seqlens;
  const int32_t* seq_lens;
  int32_t layers, total_tokens, batch;
  int32_t src_layer0, dst_layer0;  // first source / cache layer of the call (pipeline-stage ingest)
  int32_t src_layers;              // layers the source buffers hold
  int32_t hs, hd, head0;          // heads per source shard, per dest rank, first owned global head
  int32_t head_dim, page_size, num_pages, bt_stride;
};
int launch_ingest(const IngestParams& p, bool gather, cudaStream_t stream);
// The tile mover (handoff_tiles.cuh): how it cuts a handoff into units for `workers` warps, and the tensor maps of the
// source shards.  tile_maps sets *ok = false (and returns HX_OK) when the call must use the rows kernel instead: more
// than kMaxTileShards source shards, a shard in managed or unregistered memory, or a shard too large for a map.  Shards in
// pinned host memory or in a peer GPU's memory are fine: the copy engines pull them over the link (F2).
TileUnits tile_units(const IngestParams& p, int32_t max_seq_len, long long workers);
int tile_maps(const IngestParams& p, TileMaps* maps, bool* ok);

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
int get_encode_fn(EncodeTiledFn* out);      // cuTensorMapEncodeTiled through the runtime's driver entry point (attention.cu)

struct AttnParams {
  void* out;
  const void* q;
  const void* k_base;             // whole cache (all layers)
  const void* v_base;
  const int32_t* block_table;
  const int32_t* seq_lens;
  void* workspace;
  size_t workspace_bytes;
  int32_t batch, q_heads, kv_heads, head_dim, page_size, num_pages, bt_stride, max_seq_len;
  int32_t layer, layers;
  float sm_scale;
  const void* k_new;              // fused append (hx_decode_attention_append); NULL otherwise
  const void* v_new;
  int32_t overlap_prev;           // 0, or launch as a programmatic dependent of the preceding kernel: 1 = wait before any read,
                                  // 2 = wait before the first global write (hx_decode_attention_chained), 3 = wait at exit only
                                  // (hx_decode_attention_overlapped); attention.cu PdlMode
  void* plan;                     // hx_decode_plan's output (written by launch_plan, read by a planned launch); NULL otherwise
  const IngestParams* handoff;    // hx_decode_step(overlap_ingest): the step's handoff, moved inside the attention kernel; NULL otherwise
  int32_t handoff_max_seq_len;
  const struct TileMaps* handoff_maps;
};
constexpr int kAttnBatchPerLaunch = 2048;   // requests one attention launch covers (attention.cu kBMax; larger batches are cut)
size_t attn_workspace_bytes(int32_t batch, int32_t q_heads, int32_t kv_heads, int32_t head_dim,
                            int32_t max_seq_len, int32_t page_size);
size_t attn_plan_bytes(int32_t batch, int32_t kv_heads, int32_t max_seq_len, int32_t page_size);
int launch_attention(const AttnParams& p, cudaStream_t stream);
int launch_plan(const AttnParams& p, cudaStream_t stream);
// where the two counters of the fused step's handoff live in the attention workspace (hx_decode_step)
size_t attn_workspace_claim_offset(int32_t q_heads, int32_t kv_heads, int32_t head_dim);
// which bytes of a workspace must be zero when a launch starts (the counters behind the partials)
void attn_workspace_zero_span(int32_t q_heads, int32_t kv_heads, int32_t head_dim, size_t* offset, size_t* bytes);

struct PrefillArgs {
  void* out;
  const void* q;
  const void* k_base;             // whole cache (all layers)
  const void* v_base;
  const int32_t* block_table;
  const int32_t* seq_lens;
  const int32_t* q_lens;
  const int32_t* cu_q_lens;
  int32_t batch, q_heads, kv_heads, head_dim, num_pages, bt_stride, layer, layers;
  int32_t total_q, max_q_len;
  float sm_scale;
};
int launch_prefill(const PrefillArgs& a, cudaStream_t stream);

struct AppendParams {
  const void* k_new;
  const void* v_new;
  void* k;                        // cache tensors, already offset to the layer
  void* v;
  const int32_t* block_table;
  const int32_t* seq_lens;
  int32_t batch, kv_heads, head_dim, page_size, bt_stride;
};
int launch_append(const AppendParams& p, cudaStream_t stream);

}  // namespace hx
