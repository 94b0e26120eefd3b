// hx_kv_ingest / hx_kv_gather kernels (SURVEY.md §8(a) rows A2 + A3).
//
// A bit copy with index math: every 16-byte chunk of every valid (layer, token, owned head,
// K|V) row moves once from its source shard to its slot in the paged cache (or back, gather).
// HBM-bound: algorithmic traffic = 2 x payload (read once, write once), zero flops.
//
// Kernel "rows": one thread owns one 16-byte column of one packed token for the whole call.
// It resolves (request, page, slot) ONCE (binary search over cu_seqlens + one block-table
// load), then streams every (layer, tensor, head) item of that token: 4 independent
// 16-byte loads are issued before the 4 stores (64 B in flight per thread).  A half-warp
// (D=128) covers one 256-byte row: reads and writes are both full 32-byte-sector runs, and
// the 16 tokens of a CTA tile that share a page write one contiguous 4 KiB (page, head) run.
//
// The same copy as a warp-level TILE MOVER on the copy engines lives in handoff_tiles.cuh; the decode-attention kernel
// runs it in its slack (hx_decode_step, overlap_ingest).  As a kernel of its own it was measured at 0.94-0.95 of this
// kernel's rate on configs[3] and equal on a one-layer handoff, so hx_kv_ingest stays here; this file only builds the
// mover's units and tensor maps (tile_units, tile_maps).
#include <cuda_fp16.h>

#include <mutex>

#include "handoff_tiles.cuh"
#include "hx_internal.h"

namespace hx {
namespace {

constexpr int kThreads = 256;
// 4 loads in flight per thread and at most 51 registers (48 used): five or more CTAs per SM.  (Eight loads in flight
// and 78 registers moved less: cfg4 6 511 -> 6 592 GB/s.)  A decode-attention CTA takes 236 registers x 256 threads and
// 165 KiB of shared memory, so an ingest CTA does NOT fit beside one: an ingest on a side stream or under
// hx_decode_attention_overlapped shares the GPU with the attention SM by SM, as attention CTAs leave or before they arrive.
constexpr int kBatch = 4;     // independent 16-byte loads in flight per thread
constexpr int kMinCtas = 5;   // __launch_bounds__ occupancy target (register cap)

__device__ __forceinline__ int4 ld_stream(const int4* p) {
  int4 r;
  uint64_t pol;                                   // the source shards are read once: evict-first in L2
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.L2::128B.v4.s32 {%0,%1,%2,%3}, [%4], %5;"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p), "l"(pol));
  return r;
}
__device__ __forceinline__ void st_stream(int4* p, const int4& v) {
  asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};"
               :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// One CTA tile: TOK packed tokens starting at token tile `tile`, layers l0, l0 + lstep, ... of the call.
template <int D, bool GATHER>
__device__ __forceinline__ void move_token_tile(const IngestParams& p, int tile, int l0, int lstep) {
  constexpr int CH = D / 8;                 // 16-byte chunks per row
  constexpr int TOK = kThreads / CH;        // packed tokens per CTA tile
  const int dc = threadIdx.x % CH;
  const int tk = tile * TOK + threadIdx.x / CH;
  if (tk >= p.total_tokens) return;

  // request i with cu[i] <= tk < cu[i+1] (largest i whose start is <= tk; empty requests skipped)
  int lo = 0, hi = p.batch;                 // invariant: cu[lo] <= tk < cu[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(p.cu_seqlens + mid) <= tk) lo = mid; else hi = mid;
  }
  const int t = tk - __ldg(p.cu_seqlens + lo);
  if (t >= __ldg(p.seq_lens + lo)) return;  // inconsistent cu/seq_lens: move nothing for this row
  const int ps = p.page_size;
  const int page = __ldg(p.block_table + (size_t)lo * p.bt_stride + t / ps);
  const int slot = t % ps;

  const int nitems = 2 * p.hd;              // (K|V) x owned heads
  const size_t src_layer = (size_t)p.total_tokens * p.hs * D;          // elements
  const size_t dst_layer = (size_t)p.num_pages * p.hd * ps * D;
  const size_t src_tok = ((size_t)tk * p.hs) * D + dc * 8;
  const size_t dst_tok = ((size_t)page * p.hd * ps + slot) * D + dc * 8;

  for (int l = l0; l < p.layers; l += lstep) {
    for (int base = 0; base < nitems; base += kBatch) {
      int4 val[kBatch];
      int4* wr[kBatch];
#pragma unroll
      for (int u = 0; u < kBatch; ++u) {
        const int it = base + u;
        if (it < nitems) {
          const int x = it >= p.hd;
          const int j = it - x * p.hd;
          const int h = p.head0 + j;
          const int r = h / p.hs;
          const __half* sbase = static_cast<const __half*>(x ? p.src_v[r] : p.src_k[r]);
          const __half* dbase = static_cast<const __half*>(x ? p.dst_v : p.dst_k);
          const __half* s = sbase + (size_t)(l + p.src_layer0) * src_layer + src_tok + (size_t)(h - r * p.hs) * D;
          const __half* d = dbase + (size_t)(l + p.dst_layer0) * dst_layer + dst_tok + (size_t)j * ps * D;
          const __half* from = GATHER ? d : s;
          const __half* to = GATHER ? s : d;
          val[u] = ld_stream(reinterpret_cast<const int4*>(from));
          wr[u] = reinterpret_cast<int4*>(const_cast<__half*>(to));
        }
      }
#pragma unroll
      for (int u = 0; u < kBatch; ++u)
        if (base + u < nitems) st_stream(wr[u], val[u]);
    }
  }
}

template <int D, bool GATHER>
__global__ void __launch_bounds__(kThreads, kMinCtas) ingest_rows_kernel(const __grid_constant__ IngestParams p, int layer_splits) {
  // a kernel launched as a programmatic dependent of this one (hx_decode_attention_overlapped) may start now;
  // without such a launch this is a no-op
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  move_token_tile<D, GATHER>(p, blockIdx.x, blockIdx.y, layer_splits);
}

// hx_kv_append: one thread per 16-byte chunk of one
// (request, K|V, kv head) row of the step's new token; B * 2 * Hkv * D/8 threads in all.
template <int D>
__global__ void __launch_bounds__(kThreads) append_kernel(const AppendParams p) {
  constexpr int CH = D / 8;
  const int idx = blockIdx.x * kThreads + threadIdx.x;
  const int per_req = 2 * p.kv_heads * CH;
  const int i = idx / per_req;
  if (i >= p.batch) return;
  const int n = __ldg(p.seq_lens + i);
  if (n <= 0) return;
  const int rem = idx - i * per_req;
  const int x = rem / (p.kv_heads * CH);
  const int gc = rem - x * (p.kv_heads * CH);
  const int g = gc / CH, c = gc - g * CH;
  const int t = n - 1;
  const int page = __ldg(p.block_table + (size_t)i * p.bt_stride + t / p.page_size);
  const __half* src = static_cast<const __half*>(x ? p.v_new : p.k_new) + ((size_t)i * p.kv_heads + g) * D + c * 8;
  __half* dst = static_cast<__half*>(x ? p.v : p.k) + (((size_t)page * p.kv_heads + g) * p.page_size + t % p.page_size) * D + c * 8;
  st_stream(reinterpret_cast<int4*>(dst), ld_stream(reinterpret_cast<const int4*>(src)));
}

}  // namespace

int launch_append(const AppendParams& p, cudaStream_t stream) {
  const long long threads = (long long)p.batch * 2 * p.kv_heads * (p.head_dim / 8);
  const int grid = (int)((threads + kThreads - 1) / kThreads);
  if (p.head_dim == 128) append_kernel<128><<<grid, kThreads, 0, stream>>>(p);
  else                   append_kernel<64><<<grid, kThreads, 0, stream>>>(p);
  HX_CUDA_OK(cudaGetLastError());
  return HX_OK;
}

// Units of the tile mover (handoff_tiles.cuh) for this handoff: split the owned heads into groups until there are enough units to balance
// `workers` warps (a unit is what one warp takes at a time).
TileUnits tile_units(const IngestParams& p, int32_t max_seq_len, long long workers) {
  TileUnits u;
  u.pages_per_req = (max_seq_len + 15) / 16;
  u.hg = p.hd;
  const long long slots = (long long)p.layers * 2 * p.batch * u.pages_per_req;
  while (u.hg % 2 == 0 && slots * (p.hd / u.hg) < 16 * workers) u.hg /= 2;
  u.units = slots * (p.hd / u.hg);
  return u;
}

// Tensor maps over the source shards, viewed as [src_layers * total_tokens][hs][D]: box {D, 1, 16} = the 16 token rows of
// one head, landing contiguously (no swizzle) — the layout of a (page, head) tile.  Maps are cached by (pointer, shape).
int tile_maps(const IngestParams& p, TileMaps* maps, bool* ok) {
  struct Entry { const void* ptr; uint64_t rows; int hs, D; CUtensorMap tm; };
  static std::mutex mu;
  static Entry cache[64];
  static int n = 0, next = 0;
  *ok = false;
  const int r_lo = p.head0 / p.hs, r_hi = (p.head0 + p.hd - 1) / p.hs;
  const uint64_t rows = (uint64_t)p.src_layers * p.total_tokens;
  if (r_hi - r_lo + 1 > kMaxTileShards || rows >= (1ull << 31)) return HX_OK;
  int dev = 0;
  HX_CUDA_OK(cudaGetDevice(&dev));
  EncodeTiledFn enc;
  int rc = get_encode_fn(&enc);
  if (rc) return rc;
  std::lock_guard<std::mutex> lock(mu);
  for (int r = r_lo; r <= r_hi; ++r)
    for (int x = 0; x < 2; ++x) {
      const void* ptr = x ? p.src_v[r] : p.src_k[r];
      cudaPointerAttributes at;
      if (cudaPointerGetAttributes(&at, ptr) != cudaSuccess) { cudaGetLastError(); return HX_OK; }
      // What the copy engines can load from is any address the GPU can: this device's HBM, pinned host memory (UVA) and a
      // peer GPU's memory with peer access enabled - the last two make the fused step a PULL-mode handoff (F2): each tile
      // crosses the link once, straight into its page.  Managed or unregistered memory: rows kernel.
      (void)dev;
      if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeHost) return HX_OK;
      CUtensorMap* out = x ? &maps->v[r - r_lo] : &maps->k[r - r_lo];
      bool hit = false;
      for (int e = 0; e < n && !hit; ++e)
        if (cache[e].ptr == ptr && cache[e].rows == rows && cache[e].hs == p.hs && cache[e].D == p.head_dim) { *out = cache[e].tm; hit = true; }
      if (hit) continue;
      Entry ent;
      ent.ptr = ptr; ent.rows = rows; ent.hs = p.hs; ent.D = p.head_dim;
      cuuint64_t dims[3] = {(cuuint64_t)p.head_dim, (cuuint64_t)p.hs, rows};
      cuuint64_t strides[2] = {(cuuint64_t)p.head_dim * 2, (cuuint64_t)p.hs * p.head_dim * 2};
      cuuint32_t box[3] = {(cuuint32_t)p.head_dim, 1, 16};
      cuuint32_t es[3] = {1, 1, 1};
      CUresult cr = enc(&ent.tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, es,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (cr != CUDA_SUCCESS) HX_FAIL(HX_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d) for source shard %d (%p, %llu rows)", (int)cr, r, ptr,
                                      (unsigned long long)rows);
      cache[next] = ent;
      next = (next + 1) % 64;
      if (n < 64) ++n;
      *out = ent.tm;
    }
  *ok = true;
  return HX_OK;
}

int launch_ingest(const IngestParams& p, bool gather, cudaStream_t stream) {
  DeviceInfo di;
  int rc = device_info(&di);
  if (rc) return rc;
  const int ch = p.head_dim / 8;
  const int tok = kThreads / ch;
  const int tiles = (p.total_tokens + tok - 1) / tok;
  // one layer per CTA (grid.y = layers, capped by the grid limit): many short CTAs hide the dependent
  // set-up hops and leave almost no tail.  Measured on cfg4 (80 layers): 6 236 GB/s with ~9 layers per
  // CTA, 6 350 / 6 421 / 6 504 / 6 511 GB/s with 4.5 / 2.3 / 1.2 / 1 layers per CTA.
  (void)di;
  int splits = p.layers;
  if (splits > 65535) splits = 65535;
  if (splits < 1) splits = 1;
  dim3 grid(tiles, splits);
  if (p.head_dim == 128) {
    if (gather) ingest_rows_kernel<128, true><<<grid, kThreads, 0, stream>>>(p, splits);
    else        ingest_rows_kernel<128, false><<<grid, kThreads, 0, stream>>>(p, splits);
  } else {
    if (gather) ingest_rows_kernel<64, true><<<grid, kThreads, 0, stream>>>(p, splits);
    else        ingest_rows_kernel<64, false><<<grid, kThreads, 0, stream>>>(p, splits);
  }
  HX_CUDA_OK(cudaGetLastError());
  return HX_OK;
}

}  // namespace hx
