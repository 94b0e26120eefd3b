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
#include <cuda_fp16.h>

#include <mutex>

#include "hx_internal.h"

namespace hx {
namespace {

constexpr int kThreads = 256;
// 4 loads in flight per thread and at most 51 registers (46 used): five or more CTAs per SM by themselves, and one
// CTA still fits beside a decode-attention CTA (51 K of the SM's 64 K registers), so an ingest on a side stream
// or under hx_decode_attention_overlapped keeps moving while attention runs.  cfg4: 6 511 -> 6 592 GB/s.
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

// The handoff as a TAIL FILLER (hx_decode_step, overlap_ingest): launched as a programmatic dependent of the attention
// kernel, whose CTAs release their dependents as soon as they start.  Every CTA of this grid REQUESTS more shared
// memory than an attention CTA leaves free (it uses none), so it is placed on an SM only when that SM's attention CTA
// has left: the handoff runs in the attention kernel's tail, on the SMs that finished early, instead of taking
// bandwidth from its main phase (both kernels are HBM-bound).  CTAs start at different times, so (token tile, layer)
// units are claimed from a counter; a bit copy does not care who moves what.  Each CTA waits for the attention grid
// before it exits: completion of this grid implies completion of both.
template <int D>
__global__ void __launch_bounds__(kThreads, 3) ingest_rows_tail_kernel(const __grid_constant__ IngestParams p, int tiles, int* claim) {
  __shared__ int unit[2];
  const int units = tiles * p.layers;
  if (threadIdx.x == 0) unit[0] = atomicAdd(claim, 1);
  __syncthreads();
  for (int it = 0;; ++it) {
    const int u = unit[it & 1];
    if (u >= units) break;
    if (threadIdx.x == 0) unit[(it + 1) & 1] = atomicAdd(claim, 1);      // next claim rides under this unit's copies
    move_token_tile<D, false>(p, u % tiles, u / tiles, p.layers);         // unit = one token tile of one layer
    __syncthreads();
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");
  // the last CTA out leaves the two counters at zero for the next call (plain stores, flushed at kernel end)
  if (threadIdx.x == 0 && atomicAdd(claim + 1, 1) == (int)gridDim.x - 1) { claim[0] = 0; claim[1] = 0; }
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

int launch_ingest_tail(const IngestParams& p, int32_t smem_request, int32_t* claim, cudaStream_t stream) {
  DeviceInfo di;
  int rc = device_info(&di);
  if (rc) return rc;
  const int tok = kThreads / (p.head_dim / 8);
  const int tiles = (p.total_tokens + tok - 1) / tok;
  if ((long long)tiles * p.layers >= (1ll << 30)) HX_FAIL(HX_ERR_UNSUPPORTED, "handoff too large for the overlapped step");
  const int max_dyn = di.max_smem_optin - 1024;               // (the kernel has a few bytes of static shared memory)
  if (smem_request > max_dyn) smem_request = max_dyn;
  if (smem_request < 0) smem_request = 0;
  {
    static std::mutex mu;
    static bool attr_set[64] = {false};
    std::lock_guard<std::mutex> lock(mu);
    if (!attr_set[di.device]) {
      HX_CUDA_OK(cudaFuncSetAttribute(ingest_rows_tail_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn));
      HX_CUDA_OK(cudaFuncSetAttribute(ingest_rows_tail_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn));
      attr_set[di.device] = true;
    }
  }
  long long grid = (long long)di.sm_count * 3;                 // what fits once every SM is free
  if (grid > (long long)tiles * p.layers) grid = (long long)tiles * p.layers;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(kThreads); cfg.dynamicSmemBytes = (size_t)smem_request; cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  if (p.head_dim == 128) HX_CUDA_OK(cudaLaunchKernelEx(&cfg, ingest_rows_tail_kernel<128>, p, tiles, claim));
  else                   HX_CUDA_OK(cudaLaunchKernelEx(&cfg, ingest_rows_tail_kernel<64>, p, tiles, claim));
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
