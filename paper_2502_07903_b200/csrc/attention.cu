// hx_decode_attention kernels (PAPER.md:L110 cites PagedAttention /
// FlashAttention and gives no kernel: the design below is ours, for sm_100a).
//
// Roofline: HBM.  Algorithmic bytes = sum_i n_i * kv_heads * head_dim * 2 tensors * 2 B; G flops
// per byte (G = q heads per kv head), so the job is to keep HBM saturated from every SM and to
// spend as few issue slots as possible per 8 KiB (page, kv-head) K+V tile.
//
// attn_stream_kernel — "stream-K over page tiles":
//  * The work is the linear sequence of (request, kv head, page) tiles.  Every warp of a
//    persistent grid (one CTA per SM, 8 warps) owns an equal contiguous range of that sequence
//    (row A4: the cut depends only on seq_lens and the grid size, never on page placement or on
//    timing, so the result is bit-identical under page permutation and from run to run).
//  * A tile is described by a 16-byte descriptor (cache row, first query row, context length, page
//    index).  Lanes produce descriptors 32-64 tiles ahead: either by a binary search over the page
//    prefix sums plus one block-table load (hx_decode_attention), or by one coalesced load from a
//    per-step PLAN that hx_decode_plan wrote once for all the layer calls of a decode step
//    (hx_decode_attention_planned: no prefix sums, no search, first TMA issued after one L2 hop).
//  * Each warp runs its own 2-stage ring: lane 0 issues one TMA tensor-tile load per K tile and
//    per V tile (cp.async.bulk.tensor, 128-byte swizzle, mbarrier complete_tx).  No CTA-wide
//    barrier after setup.  Two stages x 8 warps = 128 KiB in flight per SM: enough to saturate HBM
//    (6.9-7.4 TB/s of reads while all SMs stream), and the SMs share it far more evenly than with
//    three.
//  * Scores (row A5) and PV (row A7) run on mma.sync.m16n8k16 with the page as M (16 tokens) and
//    the GQA group as N (8 heads): S^T = K Q^T and O^T += V^T P^T, so one K/V tile serves all G
//    query heads from shared memory and nothing is padded along tokens.  Online softmax (row A6)
//    in fp32 on the accumulator fragments; P^T is re-laid for the second MMA with movmatrix.
//  * A range that covers a whole (request, kv head) writes fp16 output directly; a range that
//    starts or ends inside one writes an (m, l, acc) partial and bumps the pair's arrival counter;
//    the last arriver merges the pair's partials in worker order (= token order, so the result
//    does not depend on who arrives last), normalises and writes (row A8).  No second launch.
//  * APPEND (hx_decode_attention_append): the warp that streams the
//    last page of a (request, kv head) overlays the step's new K/V row on the tile in shared memory
//    and stores it to the page, so the decode step needs no separate append launch.
//  * Chained launches (hx_decode_attention_chained, row A9): the kernel can be launched as a programmatic dependent of
//    the kernel before it and then waits for that kernel either before its first global read or only before its first
//    global write (StreamParams::pdl_mode), so a layer loop's calls run in one another's tails.
//  * HANDOFF (attn_handoff_kernel, hx_decode_step with overlap_ingest, rows A2 + A3 + A9): warps that have finished their
//    attention range move (page, head) tiles of the step's KV handoff with the copy engines (handoff_tiles.cuh), so one
//    kernel does the whole decode step and the handoff fills the slack the attention's uneven finish leaves.
#include <cuda.h>
#include <cuda_fp16.h>

#include <cstring>
#include <mutex>

#include "handoff_tiles.cuh"
#include "hx_internal.h"

namespace hx {
namespace {

constexpr int kWarps = 8;          // warps (= independent workers) per CTA
constexpr int kBMax = kAttnBatchPerLaunch;   // 2048 requests per launch (prefix sums live in shared memory)
constexpr int kMaxWorkers = 2048;  // workspace is sized for this many workers (>= SMs * kWarps)
constexpr int kMaxSm = 256;        // CTAs (= SMs) per launch
constexpr float kLog2e = 1.4426950408889634f;
constexpr int kPlanMagic = 0x68785032;
constexpr int kPlanHeaderInts = 16;
enum PdlMode { kPdlNone = 0, kPdlInputs = 1, kPdlWrites = 2, kPdlEnd = 3 };

template <int D, int NT>
struct Cfg {
  static constexpr int kStages = 2;                  // 16 tiles (128 KiB) in flight per SM: see DESIGN.md 6.3
  static constexpr int kTile = 16 * D * 2;           // bytes of one (page, head) K or V tile
  static constexpr int kStage = 2 * kTile;           // K + V
  static constexpr int kQBytes = NT * 8 * D * 2;     // Q slot: NT*8 heads
  static constexpr int kKS = D / 16;                 // k-steps of QK^T
  static constexpr int kMT = D / 16;                 // m-tiles of PV
  static constexpr int kSlotFloats = NT * (kMT * 128 + 16);   // partial: acc[NT][MT][32][4], m[NT][8], l[NT][8]
  static constexpr int kSmem = kWarps * kStages * kStage + kWarps * kQBytes + kWarps * (kStages + 1 + tiles::kBufs) * 8 +
                               (kBMax + 1) * 4 + kBMax * 4 + 16;
  static_assert(kStages * kStage == tiles::kBufs * kTile, "a warp's ring doubles as the tile mover's four buffers");
};

// A per-step plan (hx_decode_plan), int32 words:
//   [0, 16)                header: magic, B, Hkv, Hq, nC, N (tiles), n_empty
//   [16, 16 + B)           indices of the requests with an empty context (n_empty of them)
//   first[W][32] x int4    the first 32 descriptors of every worker's range (so that a warp needs ONE load)
//   tiles[N] x int4        descriptor of every tile
struct PlanView {
  const int32_t* header;
  const int32_t* empty;
  const int4* first;
  const int4* tiles;
};
__host__ __device__ inline size_t plan_first_offset_ints(int B) { return (size_t)((kPlanHeaderInts + B + 3) & ~3); }

struct StreamParams {
  const __half* q;
  __half* out;
  const int32_t* bt;
  const int32_t* lens;
  float* partials;        // [2 * W][kSlotFloats]
  int32_t* counters;      // [B * Hkv] arrival counters of split pairs; zero between calls
  int32_t B, Hq, Hkv, G, bt_stride;
  uint32_t layer_row0;    // first tensor-map row of the layer
  float scale_log2;
  // fused append (hx_decode_attention_append): the step's new K/V rows [B][Hkv][D] and the layer's
  // cache tensors; the owner of the last page of (request, kv head) overlays and stores the row
  const __half* k_new;
  const __half* v_new;
  __half* kc;
  __half* vc;
  // Programmatic dependent launch: this grid may start while the kernel enqueued before it on the stream still runs.
  // Every CTA executes griddepcontrol.wait before it exits in every mode, so completion of this grid implies completion
  // (and visibility) of its predecessor; the mode says what else must wait:
  //   kPdlInputs (hx_decode_attention_chained, inputs_ready = 0): nothing is read from global memory before the wait;
  //              only the launch latency, the barrier set-up and the descriptor prefetch run under the predecessor.
  //   kPdlWrites (hx_decode_attention_chained, inputs_ready = 1): the caller asserts that nothing this grid READS is
  //              written by the predecessor; every global WRITE (out, partials, counters) comes after the wait, so the
  //              grid streams its first ranges under the predecessor's tail and may share its workspace and `out`.
  //   kPdlEnd    (hx_decode_attention_overlapped behind hx_kv_ingest): reads nothing and writes nothing the ingest
  //              touches; only the exit waits.
  int32_t pdl_mode;
  const int32_t* plan;    // hx_decode_attention_planned
  // HANDOFF (hx_decode_step, overlap_ingest): the step's KV handoff, moved by the warps that have finished their attention
  // range (handoff_tiles.cuh); claim[0] hands out units, claim[1] counts the warps that are done (both left at zero)
  IngestParams ing;
  TileUnits ing_units;
  int32_t* claim;
};

// ---------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  } while (!done);
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// K/V tiles are read once per call: evict-first keeps them from pushing the block table, Q and the
// partials out of L2.
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void tma_tile_3d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, uint32_t bar, uint64_t pol) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;"
      ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t movmatrix_t(uint32_t a) {
  uint32_t d;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
  return d;
}
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}


// ---------------------------------------------------------------------------- work partition (row A4)
// Tiles are ordered request-major, then kv head, then page: request i owns [Hkv*cum[i], Hkv*cum[i+1]).
// CTA-level range s of nC is [N*s/nC, N*(s+1)/nC); worker (s, j) owns the j-th of its 8 equal parts.
__device__ __forceinline__ int cta_lo(int s, int N, int nC) { return (int)((long long)N * s / nC); }
__device__ __forceinline__ int worker_lo(int ww, int N, int nC) {
  const int s = ww >> 3, j = ww & 7;
  const int lo = cta_lo(s, N, nC), hi = cta_lo(s + 1, N, nC);
  return lo + (int)((long long)(hi - lo) * j >> 3);
}
__device__ __forceinline__ int owner_of(int k, int N, int nC) {          // worker whose range holds tile k
  const int s = (int)((((long long)k + 1) * nC - 1) / N);               // largest s with cta_lo(s) <= k
  const int lo = cta_lo(s, N, nC), len = cta_lo(s + 1, N, nC) - lo;
  return s * 8 + (int)((((unsigned)(k - lo) + 1u) * 8u - 1u) / (unsigned)len);   // len < 2^28 (host check)
}

// descriptor of tile k: x = cache row of the tile's first token within a layer (page*Hkv*16 + g*16),
// y = first query row (i*Hq + g*G), z = context length n_i, w = page index j within the request
__device__ __forceinline__ int4 make_desc(long long k, const int* cum, const int* slen, int B, int Hkv, int Hq, int G,
                                          const int32_t* bt, int bt_stride) {
  int lo = 0, hi = B;     // invariant: Hkv*cum[lo] <= k < Hkv*cum[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if ((long long)Hkv * cum[mid] <= k) lo = mid; else hi = mid;
  }
  const int np = cum[lo + 1] - cum[lo];
  const int rem = (int)(k - (long long)Hkv * cum[lo]);
  const int g = rem / np, j = rem - g * np;
  const int page = __ldg(bt + (size_t)lo * bt_stride + j);
  return make_int4(page * (Hkv * 16) + g * 16, lo * Hq + g * G, slen[lo], j);
}

// Page-count prefix sums of the batch in shared memory: slen[i] = max(n_i, 0), cum[i] = pages before request i.
// Called by every thread of a 256-thread CTA; ends with a __syncthreads().
__device__ __forceinline__ void prefix_pages(const int32_t* lens, int B, int* slen, int* cum) {
  constexpr int PER = kBMax / (kWarps * 32);
  constexpr uint32_t FULL = 0xffffffffu;
  __shared__ int warp_tot[kWarps];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  int np[PER], sum = 0;
#pragma unroll
  for (int e = 0; e < PER; ++e) {
    const int i = tid * PER + e;
    const int n = (i < B) ? max(__ldg(lens + i), 0) : 0;
    if (i < B) slen[i] = n;
    np[e] = (n + 15) >> 4;
    sum += np[e];
  }
  int incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(FULL, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) warp_tot[warp] = incl;
  __syncthreads();
  int off = incl - sum;
  for (int w = 0; w < warp; ++w) off += warp_tot[w];
  if (tid == 0) cum[0] = 0;
#pragma unroll
  for (int e = 0; e < PER; ++e) {
    const int i = tid * PER + e;
    off += np[e];
    if (i < B) cum[i + 1] = off;
  }
  __syncthreads();
}

// ------------------------------------------------------------------------------------------
// hx_decode_plan: everything of a decode step's attention that depends only on seq_lens and the block table,
// computed once for all the layer calls of the step.  Same grid as the attention kernel.
__global__ void __launch_bounds__(kWarps * 32, 1)
plan_kernel(int32_t* plan, const int32_t* lens, const int32_t* bt, int B, int Hkv, int Hq, int bt_stride) {
  __shared__ int cum[kBMax + 1];
  __shared__ int slen[kBMax];
  __shared__ int n_empty;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nC = gridDim.x, G = Hq / Hkv;
  if (tid == 0) n_empty = 0;
  prefix_pages(lens, B, slen, cum);
  const int N = Hkv * cum[B];
  int4* first = reinterpret_cast<int4*>(plan + plan_first_offset_ints(B));
  int4* tiles = first + (size_t)nC * kWarps * 32;
  if (blockIdx.x == 0) {
    for (int i = tid; i < B; i += kWarps * 32)
      if (slen[i] == 0) plan[kPlanHeaderInts + atomicAdd(&n_empty, 1)] = i;       // (order is irrelevant: rows get zeros)
    __syncthreads();
    if (tid == 0) {
      plan[0] = kPlanMagic; plan[1] = B; plan[2] = Hkv; plan[3] = Hq; plan[4] = nC; plan[5] = N; plan[6] = n_empty;
    }
  }
  if (N == 0) return;
  const int w = blockIdx.x * kWarps + warp;
  const int k0 = worker_lo(w, N, nC), k1 = worker_lo(w + 1, N, nC);
  first[(size_t)w * 32 + lane] = (k0 + lane < k1) ? make_desc(k0 + lane, cum, slen, B, Hkv, Hq, G, bt, bt_stride) : make_int4(0, 0, 0, 0);
  for (long long k = (long long)blockIdx.x * (kWarps * 32) + tid; k < N; k += (long long)nC * (kWarps * 32))
    tiles[k] = make_desc(k, cum, slen, B, Hkv, Hq, G, bt, bt_stride);
}

// ------------------------------------------------------------------------------------------
template <int D, int NT, bool APPEND, bool PLANNED, bool HANDOFF>
__device__ __forceinline__ void attn_stream_body(const CUtensorMap& tmK, const CUtensorMap& tmV, const StreamParams& p,
                                                 const TileMaps* hmaps) {
  using C = Cfg<D, NT>;
  constexpr int kStages = C::kStages, kTile = C::kTile, kKS = C::kKS, kMT = C::kMT;
  constexpr uint32_t FULL = 0xffffffffu;
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* q_base = smem + kWarps * kStages * C::kStage;
  uint64_t* bars = reinterpret_cast<uint64_t*>(q_base + kWarps * C::kQBytes);
  uint64_t* hbars = bars + kWarps * (kStages + 1);                      // (HANDOFF only)
  int* cum = reinterpret_cast<int*>(hbars + kWarps * tiles::kBufs);    // (unplanned only)
  int* slen = cum + (kBMax + 1);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int B = p.B, Hkv = p.Hkv, G = p.G;
  const int nC = gridDim.x;
  if ((smem_u32(smem) & 1023u) != 0) __trap();       // the 128-byte-swizzle address math assumes a 1 KiB-aligned base
  if (tid == 32) {                                   // descriptor fetch off the first TMA's critical path
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmK) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmV) : "memory");
  }
  // a kernel launched as a programmatic dependent of this one (hx_decode_step's handoff) may be scheduled from now
  // on: it gets an SM only where this grid has left one; without such a launch this is a no-op
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int w = blockIdx.x * kWarps + warp;          // worker id
  if (lane == 0) {
    const uint32_t b0 = smem_u32(bars + warp * (kStages + 1));
    for (int s = 0; s <= kStages; ++s) mbar_init(b0 + 8 * s, 1);
    if (HANDOFF) for (int s = 0; s < tiles::kBufs; ++s) mbar_init(smem_u32(hbars + warp * tiles::kBufs) + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (p.pdl_mode == kPdlInputs) asm volatile("griddepcontrol.wait;" ::: "memory");
  bool pdl_pending = (p.pdl_mode == kPdlWrites);         // this thread has not yet waited for the preceding grid
  auto pdl_before_write = [&]() {
    if (pdl_pending) { asm volatile("griddepcontrol.wait;" ::: "memory"); pdl_pending = false; }
  };

  // ---- setup (row A4).  Unplanned: page-count prefix sums in shared memory (the only CTA-wide syncs).
  // Planned: the header and this worker's first 32 descriptors arrive with one round of loads; no CTA-wide sync.
  int N;
  PlanView pv = {nullptr, nullptr, nullptr, nullptr};
  int4 d_cur = make_int4(0, 0, 0, 0), d_nxt = make_int4(0, 0, 0, 0);    // lane L of round r describes tile k0 + 32 r + L
  if (PLANNED) {
    pv.header = p.plan;
    pv.empty = p.plan + kPlanHeaderInts;
    pv.first = reinterpret_cast<const int4*>(p.plan + plan_first_offset_ints(B));
    pv.tiles = pv.first + (size_t)nC * kWarps * 32;
    d_cur = __ldg(pv.first + (size_t)w * 32 + lane);
    const int hv = (lane < 8) ? __ldg(pv.header + lane) : 0;
    N = __shfl_sync(FULL, hv, 5);
    // a plan made for another batch, head layout or grid would send the warps to wrong tiles: stop loudly
    if (__shfl_sync(FULL, hv, 0) != kPlanMagic || __shfl_sync(FULL, hv, 1) != B || __shfl_sync(FULL, hv, 2) != Hkv ||
        __shfl_sync(FULL, hv, 3) != p.Hq || __shfl_sync(FULL, hv, 4) != nC) __trap();
    const int n_empty = __shfl_sync(FULL, hv, 6);
    if (n_empty > 0) pdl_before_write();
    for (int e = w; e < n_empty; e += nC * kWarps) {                     // reading S11: empty context -> zero row
      int4* row = reinterpret_cast<int4*>(p.out + (size_t)__ldg(pv.empty + e) * p.Hq * D);
      for (int x = lane; x < p.Hq * D / 8; x += 32) row[x] = make_int4(0, 0, 0, 0);
    }
    __syncwarp();
  } else {
    prefix_pages(p.lens, B, slen, cum);
    N = Hkv * cum[B];
    // reading S11: an empty context gives a zero output row (no tile ever touches it)
    for (int i = blockIdx.x * (kWarps * 32) + tid; i < B; i += gridDim.x * (kWarps * 32))
      if (slen[i] == 0) {
        pdl_before_write();
        int4* row = reinterpret_cast<int4*>(p.out + (size_t)i * p.Hq * D);
        for (int e = 0; e < p.Hq * D / 8; ++e) row[e] = make_int4(0, 0, 0, 0);
      }
  }

  do {
  if (N == 0) break;
  const int k0 = worker_lo(w, N, nC), k1 = worker_lo(w + 1, N, nC);
  if (k0 >= k1) break;

  uint8_t* my_stage = smem + warp * kStages * C::kStage;
  const uint32_t stage_u32 = smem_u32(my_stage);
  uint8_t* my_q = q_base + warp * C::kQBytes;
  const uint32_t q_u32 = smem_u32(my_q);
  const uint32_t bar_u32 = smem_u32(bars + warp * (kStages + 1));
  const uint32_t qbar = bar_u32 + 8 * kStages;
  const uint64_t kv_policy = policy_evict_first();

  auto load_round = [&](int r) -> int4 {
    const long long k = k0 + 32ll * r + lane;
    if (k >= k1) return make_int4(0, 0, 0, 0);
    if (PLANNED) return __ldg(pv.tiles + k);
    return make_desc(k, cum, slen, B, Hkv, p.Hq, G, p.bt, p.bt_stride);
  };
  if (!PLANNED) d_cur = load_round(0);
  d_nxt = load_round(1);
  int cur_round = 0;

  // descriptor fields of the tile in each stage (warp-uniform), stashed when the tile is issued
  int st_qrow[kStages], st_n[kStages], st_j[kStages], st_row[kStages];
#pragma unroll
  for (int s = 0; s < kStages; ++s) st_qrow[s] = st_n[s] = st_j[s] = st_row[s] = 0;
  int seg_j0 = 0, segs_started = 0;
  bool q_busy = false;

  // fragment-address constants
  const int a_row = (lane & 7) + ((lane >> 3) & 1) * 8;   // K (A, non-trans): token row
  const int a_csel = lane >> 4;                           //   chunk select within the k-step
  const int v_row = (lane & 7) + (lane >> 4) * 8;         // V (A, trans): token row
  const int v_csel = (lane >> 3) & 1;
  const int tok0 = lane >> 2;
  const int gshift = 31 - __clz(G);

  uint32_t qb[NT][kKS][2];
  float o[NT][kMT][4];
  float m_run[NT][2], l_run[NT][2];

  int pk = k0, ck = k0;
  while (ck < k1) {
    // ------------------------------------------------ produce: keep kStages tiles in flight
    while (pk < k1 && pk - ck < kStages) {
      const int idx = pk - k0;
      if ((idx >> 5) != cur_round) {
        d_cur = d_nxt;
        ++cur_round;
        d_nxt = load_round(cur_round + 1);
      }
      const int src = idx & 31;
      const int dj = __shfl_sync(FULL, d_cur.w, src);
      const bool segstart = (idx == 0) || (dj == 0);
      if (segstart && q_busy) break;
      const int drow = __shfl_sync(FULL, d_cur.x, src);
      const int dq = __shfl_sync(FULL, d_cur.y, src);
      const int dn = __shfl_sync(FULL, d_cur.z, src);
      const int stage = idx % kStages;
#pragma unroll
      for (int s = 0; s < kStages; ++s)
        if (s == stage) { st_qrow[s] = dq; st_n[s] = dn; st_j[s] = dj; st_row[s] = drow; }
      if (lane == 0) {
        if (segstart) {
          mbar_expect_tx(qbar, (uint32_t)(G * D * 2));
          bulk_load(q_u32, p.q + (size_t)dq * D, (uint32_t)(G * D * 2), qbar);
        }
        const uint32_t full = bar_u32 + 8 * stage;
        const uint32_t dst = stage_u32 + stage * C::kStage;
        const int row = (int)(p.layer_row0 + (uint32_t)drow);
        mbar_expect_tx(full, 2 * kTile);
        tma_tile_3d(dst, &tmK, 0, row, 0, full, kv_policy);
        tma_tile_3d(dst + kTile, &tmV, 0, row, 0, full, kv_policy);
      }
      if (segstart) q_busy = true;
      ++pk;
    }

    // ------------------------------------------------ consume tile ck
    const int idx = ck - k0;
    const int stage = idx % kStages;
    int c_qrow = 0, c_n = 0, c_j = 0, c_row = 0;
#pragma unroll
    for (int s = 0; s < kStages; ++s)
      if (s == stage) { c_qrow = st_qrow[s]; c_n = st_n[s]; c_j = st_j[s]; c_row = st_row[s]; }
    const int c_np = (c_n + 15) >> 4;
    if (c_j == 0 || idx == 0) {                      // segment start: fetch Q fragments, reset state
      mbar_wait(qbar, segs_started & 1);
      ++segs_started;
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        const int head = nt * 8 + (lane >> 2);
        const uint8_t* qrow = my_q + head * (D * 2) + (lane & 3) * 4;
#pragma unroll
        for (int ks = 0; ks < kKS; ++ks) {
          uint32_t b0 = *reinterpret_cast<const uint32_t*>(qrow + ks * 32);
          uint32_t b1 = *reinterpret_cast<const uint32_t*>(qrow + ks * 32 + 16);
          qb[nt][ks][0] = head < G ? b0 : 0u;
          qb[nt][ks][1] = head < G ? b1 : 0u;
        }
#pragma unroll
        for (int mt = 0; mt < kMT; ++mt) o[nt][mt][0] = o[nt][mt][1] = o[nt][mt][2] = o[nt][mt][3] = 0.f;
        m_run[nt][0] = m_run[nt][1] = -INFINITY;
        l_run[nt][0] = l_run[nt][1] = 0.f;
      }
      __syncwarp();
      q_busy = false;
      seg_j0 = c_j;
    }
    const bool last_page = (c_j == c_np - 1);
    const int valid = last_page ? c_n - 16 * (c_np - 1) : 16;
    const int pair = c_qrow >> gshift;               // request * Hkv + kv head (G is a power of two)
    // fused append (F1): token n-1 is the step's new token; its K/V row comes from k_new/v_new, not
    // from the page.  Fetch it (lanes [0,CH): K chunks, [CH,2CH): V chunks) while the tile lands.
    int4 new_row = make_int4(0, 0, 0, 0);
    if (APPEND && last_page) {
      constexpr int CH = D / 8;
      if (lane < 2 * CH) {
        const __half* src = (lane < CH ? p.k_new : p.v_new) + (size_t)pair * D + (lane % CH) * 8;
        new_row = __ldg(reinterpret_cast<const int4*>(src));
      }
    }
    mbar_wait(bar_u32 + 8 * stage, (idx / kStages) & 1);

    const uint32_t kb = stage_u32 + stage * C::kStage, vb = kb + kTile;
    if (APPEND && last_page) {
      // overlay the row on the tile in shared memory (same swizzle as the TMA box) and store it to
      // the page: cache and output both equal hx_kv_append followed by hx_decode_attention
      constexpr int CH = D / 8;
      const int r = valid - 1;
      pdl_before_write();
      if (lane < 2 * CH) {
        const int x = lane >= CH ? 1 : 0, ch = lane - x * CH;
        *reinterpret_cast<int4*>(my_stage + stage * C::kStage + x * kTile + (ch >> 3) * 2048 + r * 128 +
                                 (((ch & 7) ^ (r & 7)) << 4)) = new_row;
        __half* dstg = (x ? p.vc : p.kc) + ((size_t)c_row + r) * D + ch * 8;     // cache row of the tile's token r
        *reinterpret_cast<int4*>(dstg) = new_row;
      }
      __syncwarp();
    }
    if (valid < 16) {
      // tail slots may hold anything (NaN/Inf): P is 0 there, but 0 * Inf = NaN in the PV MMA,
      // so the V rows past the context end are zeroed in shared memory (reading S10).
      for (int e = lane; e < (16 - valid) * (D / 8); e += 32) {
        const int r = valid + e / (D / 8), ch = e % (D / 8);
        *reinterpret_cast<int4*>(my_stage + stage * C::kStage + kTile + (ch >> 3) * 2048 + r * 128 + (ch & 7) * 16) =
            make_int4(0, 0, 0, 0);
      }
      __syncwarp();
    }

    // ---- S^T[16 tok x 8 heads] = K[16 x D] Q^T   (row A5)
    float sacc[NT][2][4];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
      for (int h = 0; h < 2; ++h) sacc[nt][h][0] = sacc[nt][h][1] = sacc[nt][h][2] = sacc[nt][h][3] = 0.f;
#pragma unroll
    for (int ks = 0; ks < kKS; ++ks) {
      const int cidx = 2 * ks + a_csel;
      uint32_t a[4];
      ldsm_x4(kb + (cidx >> 3) * 2048 + a_row * 128 + (((cidx & 7) ^ (a_row & 7)) << 4), a);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) mma16816(sacc[nt][ks & 1], a, qb[nt][ks][0], qb[nt][ks][1]);
    }

    // ---- online softmax on the accumulator fragments (row A6)
    uint32_t pb[NT][2];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
      float s[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) s[r] = (sacc[nt][0][r] + sacc[nt][1][r]) * p.scale_log2;
      if (tok0 >= valid) s[0] = s[1] = -INFINITY;
      if (tok0 + 8 >= valid) s[2] = s[3] = -INFINITY;
      float pr[4], corr[2];
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        float mx = fmaxf(s[e], s[e + 2]);
        mx = fmaxf(mx, __shfl_xor_sync(FULL, mx, 4));
        mx = fmaxf(mx, __shfl_xor_sync(FULL, mx, 8));
        mx = fmaxf(mx, __shfl_xor_sync(FULL, mx, 16));
        const float m_new = fmaxf(m_run[nt][e], mx);        // finite: every tile has >= 1 valid token
        corr[e] = ex2(m_run[nt][e] - m_new);                // -inf -> 0 on the first tile
        m_run[nt][e] = m_new;
        pr[e] = ex2(s[e] - m_new);
        pr[e + 2] = ex2(s[e + 2] - m_new);
      }
      const __half2 p01 = __floats2half2_rn(pr[0], pr[1]);
      const __half2 p23 = __floats2half2_rn(pr[2], pr[3]);
      // l sums the ROUNDED weights so that numerator and denominator use the same weights
      l_run[nt][0] = l_run[nt][0] * corr[0] + __low2float(p01) + __low2float(p23);
      l_run[nt][1] = l_run[nt][1] * corr[1] + __high2float(p01) + __high2float(p23);
      pb[nt][0] = movmatrix_t(*reinterpret_cast<const uint32_t*>(&p01));   // P^T B-fragment, tokens 0-7
      pb[nt][1] = movmatrix_t(*reinterpret_cast<const uint32_t*>(&p23));   //                tokens 8-15
      if (__any_sync(FULL, corr[0] != 1.f || corr[1] != 1.f)) {
#pragma unroll
        for (int mt = 0; mt < kMT; ++mt) {
          o[nt][mt][0] *= corr[0]; o[nt][mt][1] *= corr[1];
          o[nt][mt][2] *= corr[0]; o[nt][mt][3] *= corr[1];
        }
      }
    }

    // ---- O^T[D x 8 heads] += V^T[D x 16 tok] P^T   (row A7)
#pragma unroll
    for (int mt = 0; mt < kMT; ++mt) {
      const int cidx = 2 * mt + v_csel;
      uint32_t a[4];
      ldsm_x4_t(vb + (cidx >> 3) * 2048 + v_row * 128 + (((cidx & 7) ^ (v_row & 7)) << 4), a);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) mma16816(o[nt][mt], a, pb[nt][0], pb[nt][1]);
    }
    __syncwarp();                                    // every lane is done reading this stage

    // ------------------------------------------------ segment end: output or partial (row A8)
    const bool seg_end = last_page || (ck == k1 - 1);
    bool wrote_smem = valid < 16 || (APPEND && last_page);
    if (seg_end) {
      pdl_before_write();
#pragma unroll
      for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          float l = l_run[nt][e];
          l += __shfl_xor_sync(FULL, l, 4);
          l += __shfl_xor_sync(FULL, l, 8);
          l += __shfl_xor_sync(FULL, l, 16);
          l_run[nt][e] = l;
        }
      bool emit = (seg_j0 == 0 && last_page);         // whole (request, kv head) inside this range
      if (!emit) {
        // ---- partial: first segment of this worker -> slot 2w, any later partial is its last -> 2w+1
        const bool first_seg = (segs_started == 1);
        float* dstp = p.partials + (size_t)(2 * w + (first_seg ? 0 : 1)) * C::kSlotFloats;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
          for (int mt = 0; mt < kMT; ++mt)
            __stcg(reinterpret_cast<float4*>(dstp) + (nt * kMT + mt) * 32 + lane,
                   make_float4(o[nt][mt][0], o[nt][mt][1], o[nt][mt][2], o[nt][mt][3]));
          if (lane < 4) {
            float* ml = dstp + NT * kMT * 128 + nt * 8 + 2 * lane;
            __stcg(reinterpret_cast<float2*>(ml), make_float2(m_run[nt][0], m_run[nt][1]));
            __stcg(reinterpret_cast<float2*>(ml + NT * 8), make_float2(l_run[nt][0], l_run[nt][1]));
          }
        }
        // ---- last arriver merges (row A8).  Owners of this pair's tiles [a, b): workers wa..wb.
        const int a = ck - c_j, b = a + c_np;
        const int wa = owner_of(a, N, nC), wb = owner_of(b - 1, N, nC);
        const bool dense = N >= 16 * nC;                       // then every worker's range is non-empty
        auto next_owner = [&](int ww) -> int {                 // next worker with a tile of the pair
          if (dense) return ww + 1;
          const int kn = worker_lo(ww + 1, N, nC);             // (workers with an empty range own none)
          return kn >= b ? wb + 1 : owner_of(kn, N, nC);
        };
        int nseg = wb - wa + 1;
        if (!dense) { nseg = 0; for (int ww = wa; ww <= wb; ww = next_owner(ww)) ++nseg; }
        int* counter = p.counters + pair;
        __threadfence();                                       // release: this warp's partial before its count-up
        __syncwarp();
        int old = 0;
        if (lane == 0) old = atomicAdd(counter, 1);
        old = __shfl_sync(FULL, old, 0);
        if (old == nseg - 1) {
          // Last arriver: every other owner's partial is in L2 (its fence precedes its count-up, and this warp saw
          // all the count-ups).  The loads below bypass L1 (ld.global.cg) and are issued after the atomic returned,
          // so no second fence is needed.  The counter goes back to zero with a plain store (flushed at kernel end).
          if (lane == 0) *counter = 0;
          const bool wa_first = (worker_lo(wa, N, nC) == a);
          auto slot_of = [&](int ww) -> const float* {
            return p.partials + (size_t)((ww == wa && !wa_first) ? 2 * ww + 1 : 2 * ww) * C::kSlotFloats;
          };
          const int hb = 2 * (lane & 3);
          // Online merge in worker (= token) order, deterministic; two partials are fetched per round trip.
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            float mr0 = -INFINITY, mr1 = -INFINITY, l0 = 0.f, l1 = 0.f;
#pragma unroll
            for (int mt = 0; mt < kMT; ++mt) o[nt][mt][0] = o[nt][mt][1] = o[nt][mt][2] = o[nt][mt][3] = 0.f;
            auto fetch = [&](const float* sl, float4 (&v)[kMT], float2& mv, float2& lv) {
              mv = __ldcg(reinterpret_cast<const float2*>(sl + NT * kMT * 128 + nt * 8 + hb));
              lv = __ldcg(reinterpret_cast<const float2*>(sl + NT * kMT * 128 + NT * 8 + nt * 8 + hb));
#pragma unroll
              for (int mt = 0; mt < kMT; ++mt) v[mt] = __ldcg(reinterpret_cast<const float4*>(sl) + (nt * kMT + mt) * 32 + lane);
            };
            auto fold = [&](const float4 (&v)[kMT], const float2 mv, const float2 lv) {
              const float n0 = fmaxf(mr0, mv.x), n1 = fmaxf(mr1, mv.y);
              const float r0 = ex2(mr0 - n0), r1 = ex2(mr1 - n1);       // 0 for the first partial (-inf)
              const float c0 = ex2(mv.x - n0), c1 = ex2(mv.y - n1);
              mr0 = n0; mr1 = n1;
              l0 = l0 * r0 + lv.x * c0; l1 = l1 * r1 + lv.y * c1;
#pragma unroll
              for (int mt = 0; mt < kMT; ++mt) {
                o[nt][mt][0] = o[nt][mt][0] * r0 + v[mt].x * c0; o[nt][mt][1] = o[nt][mt][1] * r1 + v[mt].y * c1;
                o[nt][mt][2] = o[nt][mt][2] * r0 + v[mt].z * c0; o[nt][mt][3] = o[nt][mt][3] * r1 + v[mt].w * c1;
              }
            };
            for (int ww = wa; ww <= wb;) {
              const int ww2 = next_owner(ww);
              const bool two = ww2 <= wb;
              float4 va[kMT], vb2[kMT];
              float2 ma, la, mb = make_float2(0.f, 0.f), lb = make_float2(0.f, 0.f);
              fetch(slot_of(ww), va, ma, la);
              if (two) fetch(slot_of(ww2), vb2, mb, lb);
              fold(va, ma, la);
              if (two) fold(vb2, mb, lb);
              ww = two ? next_owner(ww2) : wb + 1;
            }
            l_run[nt][0] = l0; l_run[nt][1] = l1;
          }
          emit = true;
        }
      }
      if (emit) {
        // normalise, transpose through the just-consumed K tile, 16-byte coalesced stores
        __half* scratch = reinterpret_cast<__half*>(my_stage + stage * C::kStage);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
          const float inv0 = 1.f / l_run[nt][0], inv1 = 1.f / l_run[nt][1];
          const int h0 = nt * 8 + 2 * (lane & 3);
#pragma unroll
          for (int mt = 0; mt < kMT; ++mt) {
            const int d0 = 16 * mt + tok0;
            scratch[h0 * D + d0] = __float2half_rn(o[nt][mt][0] * inv0);
            scratch[(h0 + 1) * D + d0] = __float2half_rn(o[nt][mt][1] * inv1);
            scratch[h0 * D + d0 + 8] = __float2half_rn(o[nt][mt][2] * inv0);
            scratch[(h0 + 1) * D + d0 + 8] = __float2half_rn(o[nt][mt][3] * inv1);
          }
        }
        __syncwarp();
        int4* dst = reinterpret_cast<int4*>(p.out + (size_t)c_qrow * D);
        const int4* srcv = reinterpret_cast<const int4*>(scratch);
        for (int e = lane; e < G * D / 8; e += 32) dst[e] = srcv[e];
        __syncwarp();
        wrote_smem = true;
      }
    }
    if (wrote_smem) { fence_proxy_async(); __syncwarp(); }   // generic writes before the TMA refill
    ++ck;
  }
  } while (false);
  if (HANDOFF) {
    // This warp's attention range is done (its partials stored, its merges written): it now moves tiles of the step's
    // KV handoff through its ring, claiming units from a global counter, until none are left.  The handoff writes pages
    // that this grid's attention does not read (the caller's assertion, include/hx.h), so no ordering between the two
    // is needed inside the kernel.
    __syncwarp();
    fence_proxy_async();                               // this warp's generic accesses to its ring precede the copy engines'
    __syncwarp();
    int32_t* claim = p.claim;
    tiles::move_tiles<D, tiles::kBufs, tiles::kAhead>(p.ing, p.ing_units, *hmaps, smem_u32(smem + warp * kStages * C::kStage), smem_u32(hbars + warp * tiles::kBufs),
                         [&]() -> long long { return lane == 0 ? (long long)atomicAdd(claim, 1) : 0ll; });
    // the last warp out leaves both counters at zero for the next call (plain stores, flushed at kernel end)
    if (lane == 0 && atomicAdd(claim + 1, 1) == (int)(gridDim.x * kWarps) - 1) { claim[0] = 0; claim[1] = 0; }
  }
  if (p.pdl_mode != kPdlNone) asm volatile("griddepcontrol.wait;" ::: "memory");
}

template <int D, int NT, bool APPEND, bool PLANNED>
__global__ void __launch_bounds__(kWarps * 32, 1)
attn_stream_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                   const __grid_constant__ StreamParams p) {
  attn_stream_body<D, NT, APPEND, PLANNED, false>(tmK, tmV, p, nullptr);
}

// hx_decode_step(overlap_ingest): the attention kernel that also carries the step's KV handoff
template <int D, int NT>
__global__ void __launch_bounds__(kWarps * 32, 1)
attn_handoff_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                    const __grid_constant__ StreamParams p, const __grid_constant__ TileMaps hmaps) {
  attn_stream_body<D, NT, false, false, true>(tmK, tmV, p, &hmaps);
}

// ---------------------------------------------------------------------------- host side
// Tensor map over a whole K or V cache viewed as [D/64 halves][rows][64] with rows = layers*P*Hkv*16:
// box {64, 16, D/64} = one (page, head) tile, landing in shared memory as [half][16 tok][128 B] with
// the 128-byte swizzle (conflict-free ldmatrix).
int make_tile_map(CUtensorMap* tm, const void* base, uint64_t rows, int D) {
  EncodeTiledFn enc;
  int rc = get_encode_fn(&enc);
  if (rc) return rc;
  cuuint64_t dims[3] = {64, rows, (cuuint64_t)(D / 64)};
  cuuint64_t strides[2] = {(cuuint64_t)D * 2, 128};
  cuuint32_t box[3] = {64, 16, (cuuint32_t)(D / 64)};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) HX_FAIL(HX_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d) for base=%p rows=%llu D=%d", (int)r, base,
                                 (unsigned long long)rows, D);
  return HX_OK;
}

struct MapCacheEntry { const void* k; const void* v; uint64_t rows; int D; CUtensorMap tk, tv; };

int get_tile_maps(const void* k, const void* v, uint64_t rows, int D, CUtensorMap* tk, CUtensorMap* tv) {
  static std::mutex mu;
  static MapCacheEntry cache[16];
  static int n = 0, next = 0;
  std::lock_guard<std::mutex> lock(mu);
  for (int e = 0; e < n; ++e)
    if (cache[e].k == k && cache[e].v == v && cache[e].rows == rows && cache[e].D == D) {
      *tk = cache[e].tk; *tv = cache[e].tv;
      return HX_OK;
    }
  MapCacheEntry ent;
  ent.k = k; ent.v = v; ent.rows = rows; ent.D = D;
  int rc = make_tile_map(&ent.tk, k, rows, D);
  if (rc) return rc;
  rc = make_tile_map(&ent.tv, v, rows, D);
  if (rc) return rc;
  cache[next] = ent;
  next = (next + 1) % 16;
  if (n < 16) ++n;
  *tk = ent.tk; *tv = ent.tv;
  return HX_OK;
}


template <int D, int NT, bool APPEND, bool PLANNED, bool HANDOFF = false>
int launch_stream(const AttnParams& a, const DeviceInfo& di, cudaStream_t stream) {
  using C = Cfg<D, NT>;
  {
    static std::mutex mu;
    static bool attr_set[64] = {false};
    std::lock_guard<std::mutex> lock(mu);
    if (!attr_set[di.device]) {
      if (C::kSmem > di.max_smem_optin) HX_FAIL(HX_ERR_UNSUPPORTED, "device offers %d B shared memory per CTA, kernel needs %d", di.max_smem_optin, C::kSmem);
      if constexpr (HANDOFF) HX_CUDA_OK(cudaFuncSetAttribute(attn_handoff_kernel<D, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmem));
      else HX_CUDA_OK(cudaFuncSetAttribute(attn_stream_kernel<D, NT, APPEND, PLANNED>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmem));
      attr_set[di.device] = true;
    }
  }
  const uint64_t rows_per_layer = (uint64_t)a.num_pages * a.kv_heads * 16;
  const uint64_t rows = rows_per_layer * a.layers;
  if (rows >= (1ull << 31)) HX_FAIL(HX_ERR_UNSUPPORTED, "cache too large for one tensor map (%llu rows)", (unsigned long long)rows);
  CUtensorMap tk, tv;
  int rc = get_tile_maps(a.k_base, a.v_base, rows, D, &tk, &tv);
  if (rc) return rc;

  int grid = di.sm_count;
  if (grid > kMaxSm) grid = kMaxSm;
  char* ws = static_cast<char*>(a.workspace);
  const size_t partial_bytes = (size_t)2 * kMaxWorkers * C::kSlotFloats * sizeof(float);
  if ((long long)kBMax * a.bt_stride * a.kv_heads >= (1ll << 28)) HX_FAIL(HX_ERR_UNSUPPORTED, "block_table_stride * kv_heads too large");
  if (PLANNED && a.batch > kBMax) HX_FAIL(HX_ERR_UNSUPPORTED, "a plan covers at most %d requests (batch %d)", kBMax, a.batch);
  for (int b0 = 0; b0 < a.batch; b0 += kBMax) {
    StreamParams p;
    memset(&p, 0, sizeof(p));
    p.B = (a.batch - b0 < kBMax) ? a.batch - b0 : kBMax;
    p.q = static_cast<const __half*>(a.q) + (size_t)b0 * a.q_heads * D;
    p.out = static_cast<__half*>(a.out) + (size_t)b0 * a.q_heads * D;
    p.bt = a.block_table ? a.block_table + (size_t)b0 * a.bt_stride : nullptr;
    p.lens = a.seq_lens ? a.seq_lens + b0 : nullptr;
    p.partials = reinterpret_cast<float*>(ws);
    p.counters = reinterpret_cast<int32_t*>(ws + partial_bytes);
    p.Hq = a.q_heads; p.Hkv = a.kv_heads; p.G = a.q_heads / a.kv_heads; p.bt_stride = a.bt_stride;
    p.layer_row0 = (uint32_t)(rows_per_layer * a.layer);
    p.scale_log2 = a.sm_scale * kLog2e;
    const size_t layer_elems = (size_t)rows_per_layer * D;
    p.k_new = APPEND ? static_cast<const __half*>(a.k_new) + (size_t)b0 * a.kv_heads * D : nullptr;
    p.v_new = APPEND ? static_cast<const __half*>(a.v_new) + (size_t)b0 * a.kv_heads * D : nullptr;
    p.kc = static_cast<__half*>(const_cast<void*>(a.k_base)) + layer_elems * a.layer;
    p.vc = static_cast<__half*>(const_cast<void*>(a.v_base)) + layer_elems * a.layer;
    p.plan = PLANNED ? static_cast<const int32_t*>(a.plan) : nullptr;
    if (HANDOFF) {
      if (a.batch > kBMax) HX_FAIL(HX_ERR_UNSUPPORTED, "the fused step covers at most %d requests (batch %d)", kBMax, a.batch);
      p.ing = *a.handoff;
      p.ing_units = tile_units(p.ing, a.handoff_max_seq_len, (long long)grid * kWarps);
      if (p.ing_units.units >= (1ll << 30)) HX_FAIL(HX_ERR_UNSUPPORTED, "handoff too large for the fused step");
      p.claim = reinterpret_cast<int32_t*>(ws + attn_workspace_claim_offset(a.q_heads, a.kv_heads, a.head_dim));
    }
    p.pdl_mode = (b0 == 0) ? a.overlap_prev : kPdlNone;
    if constexpr (HANDOFF) {
      attn_handoff_kernel<D, NT><<<grid, kWarps * 32, C::kSmem, stream>>>(tk, tv, p, *a.handoff_maps);
    } else if (p.pdl_mode != kPdlNone) {
      // programmatic dependent launch: this grid may start while the kernel enqueued just before it is still running
      // (at once if that kernel executes griddepcontrol.launch_dependents early, as the ingest and attention kernels
      // do; when it exits otherwise).  StreamParams::pdl_mode says what waits for that kernel's completion.
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(grid); cfg.blockDim = dim3(kWarps * 32); cfg.dynamicSmemBytes = C::kSmem; cfg.stream = stream;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      at[0].val.programmaticStreamSerializationAllowed = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      HX_CUDA_OK(cudaLaunchKernelEx(&cfg, attn_stream_kernel<D, NT, APPEND, PLANNED>, tk, tv, p));
    } else {
      attn_stream_kernel<D, NT, APPEND, PLANNED><<<grid, kWarps * 32, C::kSmem, stream>>>(tk, tv, p);
    }
    HX_CUDA_OK(cudaGetLastError());
  }
  return HX_OK;
}

}  // namespace

int get_encode_fn(EncodeTiledFn* out) {
  static EncodeTiledFn fn = nullptr;
  static std::mutex mu;
  std::lock_guard<std::mutex> lock(mu);
  if (!fn) {
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    HX_CUDA_OK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres));
    if (qres != cudaDriverEntryPointSuccess || !ptr) HX_FAIL(HX_ERR_CUDA, "cuTensorMapEncodeTiled not available from the driver");
    fn = reinterpret_cast<EncodeTiledFn>(ptr);
  }
  *out = fn;
  return HX_OK;
}

size_t attn_workspace_bytes(int32_t batch, int32_t q_heads, int32_t kv_heads, int32_t head_dim,
                            int32_t max_seq_len, int32_t page_size) {
  (void)batch; (void)max_seq_len; (void)page_size;
  const int G = q_heads / kv_heads;
  const int nt = G > 8 ? 2 : 1;
  const size_t slot = (size_t)nt * ((head_dim / 16) * 128 + 16) * sizeof(float);
  const size_t counter_bytes = ((size_t)kBMax * kv_heads * sizeof(int32_t) + 15) & ~(size_t)15;
  return 2 * (size_t)kMaxWorkers * slot + counter_bytes + 16;     // + the overlapped step's two claim counters
}

size_t attn_workspace_claim_offset(int32_t q_heads, int32_t kv_heads, int32_t head_dim) {
  return attn_workspace_bytes(0, q_heads, kv_heads, head_dim, 0, 16) - 16;
}

// The bytes of a workspace a launch expects to find at zero: the split pairs' arrival counters and, behind them, the two
// claim counters.  They sit BEHIND the partials, so their offset moves with (group size, head_dim); the partials
// themselves are written before they are read and need no clearing.  (hx_decode_attention_noalloc clears this span.)
void attn_workspace_zero_span(int32_t q_heads, int32_t kv_heads, int32_t head_dim, size_t* offset, size_t* bytes) {
  const size_t total = attn_workspace_bytes(0, q_heads, kv_heads, head_dim, 0, 16);
  const size_t counter_bytes = ((size_t)kBMax * kv_heads * sizeof(int32_t) + 15) & ~(size_t)15;
  *offset = total - counter_bytes - 16;
  *bytes = counter_bytes + 16;
}

// Upper bound of a plan's size: header + empty list + first[W][32] + one descriptor per possible tile.
size_t attn_plan_bytes(int32_t batch, int32_t kv_heads, int32_t max_seq_len, int32_t page_size) {
  const size_t tiles = (size_t)batch * kv_heads * ((max_seq_len + page_size - 1) / page_size);
  return plan_first_offset_ints(batch) * 4 + (size_t)kMaxSm * kWarps * 32 * 16 + tiles * 16;
}

int launch_plan(const AttnParams& a, cudaStream_t stream) {
  DeviceInfo di;
  int rc = device_info(&di);
  if (rc) return rc;
  if (a.batch > kBMax) HX_FAIL(HX_ERR_UNSUPPORTED, "a plan covers at most %d requests (batch %d)", kBMax, a.batch);
  if ((long long)kBMax * a.bt_stride * a.kv_heads >= (1ll << 28)) HX_FAIL(HX_ERR_UNSUPPORTED, "block_table_stride * kv_heads too large");
  const int grid = di.sm_count < kMaxSm ? di.sm_count : kMaxSm;
  plan_kernel<<<grid, kWarps * 32, 0, stream>>>(static_cast<int32_t*>(a.plan), a.seq_lens, a.block_table, a.batch, a.kv_heads,
                                               a.q_heads, a.bt_stride);
  HX_CUDA_OK(cudaGetLastError());
  return HX_OK;
}

int launch_attention(const AttnParams& a, cudaStream_t stream) {
  DeviceInfo di;
  int rc = device_info(&di);
  if (rc) return rc;
  const int G = a.q_heads / a.kv_heads;
  if (a.k_new) {
    if (a.head_dim == 128) return G > 8 ? launch_stream<128, 2, true, false>(a, di, stream) : launch_stream<128, 1, true, false>(a, di, stream);
    return G > 8 ? launch_stream<64, 2, true, false>(a, di, stream) : launch_stream<64, 1, true, false>(a, di, stream);
  }
  if (a.handoff) {
    if (a.head_dim == 128) return G > 8 ? launch_stream<128, 2, false, false, true>(a, di, stream) : launch_stream<128, 1, false, false, true>(a, di, stream);
    return G > 8 ? launch_stream<64, 2, false, false, true>(a, di, stream) : launch_stream<64, 1, false, false, true>(a, di, stream);
  }
  if (a.plan) {
    if (a.head_dim == 128) return G > 8 ? launch_stream<128, 2, false, true>(a, di, stream) : launch_stream<128, 1, false, true>(a, di, stream);
    return G > 8 ? launch_stream<64, 2, false, true>(a, di, stream) : launch_stream<64, 1, false, true>(a, di, stream);
  }
  if (a.head_dim == 128) return G > 8 ? launch_stream<128, 2, false, false>(a, di, stream) : launch_stream<128, 1, false, false>(a, di, stream);
  return G > 8 ? launch_stream<64, 2, false, false>(a, di, stream) : launch_stream<64, 1, false, false>(a, di, stream);
}

}  // namespace hx
