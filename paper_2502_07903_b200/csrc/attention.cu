// hx_decode_attention kernels (PAPER.md:L110 cites PagedAttention /
// FlashAttention and gives no kernel: the design below is ours, for sm_100a).
//
// Roofline: HBM.  Algorithmic bytes = sum_i n_i * kv_heads * head_dim * 2 tensors * 2 B; G flops
// per byte (G = q heads per kv head), so the job is to keep ~50 KB of loads in flight per SM and
// to spend as few issue slots as possible per 8 KiB (page, kv-head) K+V tile.
//
// attn_stream_kernel — "stream-K over page tiles":
//  * The work is the linear sequence of (request, kv head, page) tiles.  Every warp of a
//    persistent grid (one CTA per SM, 8 warps) owns an equal contiguous range of that sequence
//    (row A4: the cut depends only on seq_lens and the grid size, never on page placement, so the
//    result is bit-identical under page permutation and from run to run).
//  * Each warp runs its own 3-stage ring: lane 0 issues one TMA tensor-tile load per K tile and
//    per V tile (cp.async.bulk.tensor, 128-byte swizzle, mbarrier complete_tx); block-table
//    entries are fetched 32-64 tiles ahead, one per lane.  No CTA-wide barrier after setup.
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
#include <cuda.h>
#include <cuda_fp16.h>

#include <mutex>

#include "hx_internal.h"

namespace hx {
namespace {

constexpr int kWarps = 8;          // warps (= independent workers) per CTA
constexpr int kBMax = 2048;        // requests per launch (prefix sums live in shared memory)
constexpr int kMaxWorkers = 2048;  // workspace is sized for this many workers (>= SMs * kWarps)
constexpr int kMaxSm = 256;        // CTAs (= SMs) per launch
constexpr float kLog2e = 1.4426950408889634f;

template <int D, int NT>
struct Cfg {
  static constexpr int kStages = (NT == 1) ? 3 : 2;
  static constexpr int kTile = 16 * D * 2;           // bytes of one (page, head) K or V tile
  static constexpr int kStage = 2 * kTile;           // K + V
  static constexpr int kQBytes = NT * 8 * D * 2;     // Q slot: NT*8 heads
  static constexpr int kKS = D / 16;                 // k-steps of QK^T
  static constexpr int kMT = D / 16;                 // m-tiles of PV
  static constexpr int kSlotFloats = NT * (kMT * 128 + 16);   // partial: acc[NT][MT][32][4], m[NT][8], l[NT][8]
  static constexpr int kSmem = kWarps * kStages * kStage + kWarps * kQBytes + kWarps * (kStages + 1) * 8 +
                               (kBMax + 1) * 4 + kBMax * 4 + (kMaxSm + 1) * 4 + 16;
};

struct StreamParams {
  const __half* q;
  __half* out;
  const int32_t* bt;
  const int32_t* lens;
  float* partials;        // [2 * W][kSlotFloats]
  int32_t* counters;      // [B * Hkv] arrival counters of split pairs; zero between calls
  int32_t* claim;         // [kMaxSm] range-claim flags + [kMaxSm] finished-CTA counter; zero between calls
  int32_t B, Hq, Hkv, G, bt_stride;
  uint32_t layer_row0;    // first tensor-map row of the layer
  float scale_log2;
  // fused append (hx_decode_attention_append): the step's new K/V rows [B][Hkv][D] and the layer's
  // cache tensors; the owner of the last page of (request, kv head) overlays and stores the row
  const __half* k_new;
  const __half* v_new;
  __half* kc;
  __half* vc;
  // hx_decode_attention_overlapped: this grid was launched as a programmatic dependent of the ingest kernel and
  // reads nothing that kernel writes; every CTA executes griddepcontrol.wait before it exits, so completion of this
  // grid implies completion (and visibility) of the ingest
  int32_t pdl_wait_at_end;
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

struct Loc { int i, g, j, np; };

// tile index k -> (request, kv head, page-in-request).  Tiles are ordered request-major, then kv
// head, then page: request i owns [Hkv*cum[i], Hkv*cum[i+1]).
__device__ __forceinline__ Loc locate(long long k, const int* cum, int B, int Hkv) {
  int lo = 0, hi = B;     // invariant: Hkv*cum[lo] <= k < Hkv*cum[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if ((long long)Hkv * cum[mid] <= k) lo = mid; else hi = mid;
  }
  Loc r;
  r.i = lo;
  r.np = cum[lo + 1] - cum[lo];
  const int rem = (int)(k - (long long)Hkv * cum[lo]);
  r.g = rem / r.np;
  r.j = rem - r.g * r.np;
  return r;
}

// ------------------------------------------------------------------------------------------
// SM streaming-rate table (hx_tune_sm_rates).  On B200 the SMs do not stream from HBM at the same
// rate when all of them load at once: they fall into stable classes (about 1.19 / 1.00 / 0.88 of
// the mean; TPC pairs alike), a property of the chip's fabric.  With equal ranges the kernel waits
// for the slow class.  The table holds a per-SM weight in 1/256 of the median rate; range sizes
// follow it.  g_sm_w_n == 0 means "not tuned": equal ranges.
__device__ int g_sm_w[kMaxSm];
__device__ int g_sm_w_n;
__device__ unsigned int g_sm_cnt[kMaxSm];

// Every SM streams 8 KiB bulk copies from `scratch` through the same per-warp rings as the
// attention kernel for a fixed time window and counts what it got.
__global__ void __launch_bounds__(kWarps * 32, 1)
sm_rate_probe_kernel(const uint8_t* scratch, unsigned long long chunks, unsigned int window_ns) {
  extern __shared__ __align__(1024) uint8_t smem[];
  constexpr int kStages = 3, kStage = 8192;
  __shared__ uint64_t bars[kWarps * kStages];
  __shared__ unsigned int warp_cnt[kWarps];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(smem_u32(&bars[warp * kStages + s]), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  unsigned int smid;
  asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
  unsigned long long t0, t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
  unsigned long long h = (unsigned long long)(smid * kWarps + warp) * 0x9E3779B97F4A7C15ull + 12345;
  const uint32_t stage0 = smem_u32(smem + warp * kStages * kStage);
  auto issue = [&](int n) {
    h = h * 6364136223846793005ull + 1442695040888963407ull;
    const unsigned long long c = (h >> 20) % chunks;
    const uint32_t bar = smem_u32(&bars[warp * kStages + n % kStages]);
    mbar_expect_tx(bar, kStage);
    bulk_load(stage0 + (n % kStages) * kStage, scratch + c * kStage, kStage, bar);
  };
  unsigned int n = 0;
  if (lane == 0) for (int s = 0; s < kStages; ++s) issue(s);
  while (true) {
    mbar_wait(smem_u32(&bars[warp * kStages + n % kStages]), (n / kStages) & 1);
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    if (t - t0 >= window_ns) break;
    if (lane == 0) issue(n + kStages);
    ++n;
  }
  // drain what is still in flight so that no bulk copy outlives the CTA
  for (unsigned int e = n + 1; e < n + kStages; ++e) mbar_wait(smem_u32(&bars[warp * kStages + e % kStages]), (e / kStages) & 1);
  if (lane == 0) warp_cnt[warp] = n;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned int tot = 0;
    for (int w2 = 0; w2 < kWarps; ++w2) tot += warp_cnt[w2];
    if (smid < kMaxSm) atomicMax(&g_sm_cnt[smid], tot);
  }
}

// One CTA: raw[s] = count[s] / median count; weight[s] = 256 * (1 + damp * (raw - 1)) rounded to a
// multiple of 8 (3 %: keeps the table stable from run to run) and clamped to [192, 352].  damp < 1
// because HBM is a shared, saturated pie: an SM that is given more work also runs longer against
// fewer competitors, so the probe's rate spread overstates the spread that balances the kernel.
// SMs that saw no probe CTA get the nominal 256.
__global__ void sm_rate_finalize_kernel(int n_sm, int reset, int damp_256) {
  __shared__ unsigned int cnt[kMaxSm];
  __shared__ unsigned int median;
  const int t = threadIdx.x;
  if (reset) {
    if (t < kMaxSm) { g_sm_w[t] = 256; g_sm_cnt[t] = 0; }
    if (t == 0) g_sm_w_n = 0;
    return;
  }
  if (t < kMaxSm) cnt[t] = t < n_sm ? g_sm_cnt[t] : 0;
  if (t == 0) median = 0;
  __syncthreads();
  if (t < n_sm && cnt[t] > 0) {
    int below = 0, valid = 0;
    for (int u = 0; u < n_sm; ++u)
      if (cnt[u] > 0) { ++valid; below += (cnt[u] < cnt[t]) || (cnt[u] == cnt[t] && u < t); }
    if (below == valid / 2) median = cnt[t];
  }
  __syncthreads();
  if (t < kMaxSm) {
    int w = 256;
    if (t < n_sm && cnt[t] > 0 && median > 0) {
      const long long raw = (256ll * cnt[t]) / median;               // 1/256 units
      long long d = 256 + ((raw - 256) * damp_256) / 256;
      d = (d + 4) & ~7ll;
      w = (int)(d < 192 ? 192 : (d > 352 ? 352 : d));
    }
    g_sm_w[t] = w;
    g_sm_cnt[t] = 0;
  }
  if (t == 0) { __threadfence(); g_sm_w_n = n_sm; }
}

// ------------------------------------------------------------------------------------------
template <int D, int NT, bool APPEND>
__global__ void __launch_bounds__(kWarps * 32, 1)
attn_stream_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                   const StreamParams p) {
  using C = Cfg<D, NT>;
  constexpr int kStages = C::kStages, kTile = C::kTile, kKS = C::kKS, kMT = C::kMT;
  constexpr uint32_t FULL = 0xffffffffu;
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* q_base = smem + kWarps * kStages * C::kStage;
  uint64_t* bars = reinterpret_cast<uint64_t*>(q_base + kWarps * C::kQBytes);
  int* cum = reinterpret_cast<int*>(bars + kWarps * (kStages + 1));
  int* slen = cum + (kBMax + 1);
  int* smlo = slen + kBMax;            // [nC + 1] first tile of each CTA-level range; then [nC+1] = my slot
  int* my_slot = smlo + kMaxSm + 1;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int B = p.B, Hkv = p.Hkv, G = p.G;
  const int nC = gridDim.x;
  if ((smem_u32(smem) & 1023u) != 0) __trap();       // the 128-byte-swizzle address math assumes a 1 KiB-aligned base
  if (tid == 32) {                                   // descriptor fetch off the first TMA's critical path
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmK) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmV) : "memory");
  }

  // ---- which CTA-level range is mine.  Not tuned: range blockIdx.x.  Tuned (hx_tune_sm_rates):
  // range sizes follow the per-SM rate table, so the range of SM s belongs to the CTA running on
  // SM s; it is claimed with a flag, and a CTA that finds its SM's range taken (two CTAs landed on
  // one SM) takes any free one, so every range is processed exactly once whatever the placement.
  const bool tuned = (g_sm_w_n == nC);
  const int my_w = (tid < nC) ? (tuned ? g_sm_w[tid] : 256) : 0;   // weight of CTA-level range `tid`
  if (tid == 0) {
    int slot = blockIdx.x;
    if (tuned) {
      unsigned int smid;
      asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
      slot = (int)(smid % (unsigned)nC);
      while (atomicCAS(p.claim + slot, 0, 1) != 0) slot = (slot + 1 == nC) ? 0 : slot + 1;
    }
    *my_slot = slot;
  }

  // ---- setup: page-count prefix sums (row A4) and barrier init; the only CTA-wide syncs
  {
    constexpr int PER = kBMax / (kWarps * 32);
    __shared__ int warp_tot[kWarps], warp_tot_w[kWarps];
    int np[PER], sum = 0;
#pragma unroll
    for (int e = 0; e < PER; ++e) {
      const int i = tid * PER + e;
      const int n = (i < B) ? max(__ldg(p.lens + i), 0) : 0;
      if (i < B) slen[i] = n;
      np[e] = (n + 15) >> 4;
      sum += np[e];
    }
    int incl = sum, incl_w = my_w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(FULL, incl, o);
      const int tw = __shfl_up_sync(FULL, incl_w, o);
      if (lane >= o) { incl += t; incl_w += tw; }
    }
    if (lane == 31) { warp_tot[warp] = incl; warp_tot_w[warp] = incl_w; }
    if (lane == 0) {
      const uint32_t b0 = smem_u32(bars + warp * (kStages + 1));
      for (int s = 0; s <= kStages; ++s) mbar_init(b0 + 8 * s, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
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
    {
      // CTA-level range starts: smlo[s] = N * (weights before s) / (all weights)
      int before = incl_w - my_w, all = 0;
#pragma unroll
      for (int w2 = 0; w2 < kWarps; ++w2) { if (w2 < warp) before += warp_tot_w[w2]; all += warp_tot_w[w2]; }
      const long long Nt = (long long)Hkv * cum[B];
      if (tid < nC) smlo[tid] = (int)(Nt * before / all);
      if (tid == nC || (nC == kWarps * 32 && tid == 0)) smlo[nC] = (int)Nt;
    }
    __syncthreads();
    // reading S11: an empty context gives a zero output row (no tile ever touches it)
    for (int i = blockIdx.x * (kWarps * 32) + tid; i < B; i += gridDim.x * (kWarps * 32))
      if (slen[i] == 0) {
        int4* row = reinterpret_cast<int4*>(p.out + (size_t)i * p.Hq * D);
        for (int e = 0; e < p.Hq * D / 8; ++e) row[e] = make_int4(0, 0, 0, 0);
      }
  }

  // worker (slot s, warp j) owns [lo(s, j), lo(s, j + 1)): the CTA range cut in 8 equal parts
  auto w_lo = [&](int ww) -> int {
    const int s = ww >> 3, j = ww & 7;
    return smlo[s] + (int)((long long)(smlo[s + 1] - smlo[s]) * j >> 3);
  };
  auto owner_of = [&](int k) -> int {                       // worker whose range holds tile k
    int lo = 0, hi = nC;                                    // smlo[lo] <= k < smlo[hi]
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (smlo[mid] <= k) lo = mid; else hi = mid;
    }
    const int len = smlo[lo + 1] - smlo[lo];
    return lo * 8 + (int)((((unsigned)(k - smlo[lo]) + 1u) * 8u - 1u) / (unsigned)len);   // len < 2^28 (host check)
  };
  const int w = *my_slot * kWarps + warp;
  const int k0 = w_lo(w), k1 = w_lo(w + 1);
  do {
  if (k0 >= k1) break;

  uint8_t* my_stage = smem + warp * kStages * C::kStage;
  const uint32_t stage_u32 = smem_u32(my_stage);
  uint8_t* my_q = q_base + warp * C::kQBytes;
  const uint32_t q_u32 = smem_u32(my_q);
  const uint32_t bar_u32 = smem_u32(bars + warp * (kStages + 1));
  const uint32_t qbar = bar_u32 + 8 * kStages;
  const uint64_t kv_policy = policy_evict_first();

  // ---- per-lane lookahead: lane L of round r describes tile k0 + 32 r + L
  int page_cur = 0, gpart_cur = 0, meta_cur = 0, page_nxt = 0, gpart_nxt = 0, meta_nxt = 0;
  auto load_round = [&](int r, int& page, int& gpart, int& meta) {
    const long long k = k0 + 32ll * r + lane;
    page = 0; gpart = 0; meta = 0;
    if (k < k1) {
      const Loc t = locate(k, cum, B, Hkv);
      page = __ldg(p.bt + (size_t)t.i * p.bt_stride + t.j);
      gpart = t.g * 16;
      meta = ((t.i * p.Hq + t.g * G) << 1) | (t.j == 0 ? 1 : 0);
    }
  };
  load_round(0, page_cur, gpart_cur, meta_cur);
  load_round(1, page_nxt, gpart_nxt, meta_nxt);
  int cur_round = 0;

  // ---- consumer cursor (warp-uniform)
  Loc c = locate(k0, cum, B, Hkv);
  int cn = slen[c.i];
  int seg_j0 = 0, segs_started = 0;
  bool q_busy = false;

  // fragment-address constants
  const int a_row = (lane & 7) + ((lane >> 3) & 1) * 8;   // K (A, non-trans): token row
  const int a_csel = lane >> 4;                           //   chunk select within the k-step
  const int v_row = (lane & 7) + (lane >> 4) * 8;         // V (A, trans): token row
  const int v_csel = (lane >> 3) & 1;
  const int tok0 = lane >> 2;

  uint32_t qb[NT][kKS][2];
  float o[NT][kMT][4];
  float m_run[NT][2], l_run[NT][2];

  long long pk = k0, ck = k0;
  while (ck < k1) {
    // ------------------------------------------------ produce: keep kStages tiles in flight
    while (pk < k1 && pk - ck < kStages) {
      const int idx = (int)(pk - k0);
      if ((idx >> 5) != cur_round) {
        page_cur = page_nxt; gpart_cur = gpart_nxt; meta_cur = meta_nxt;
        ++cur_round;
        load_round(cur_round + 1, page_nxt, gpart_nxt, meta_nxt);
      }
      const int src = idx & 31;
      const int meta = __shfl_sync(FULL, meta_cur, src);
      const bool segstart = (idx == 0) || (meta & 1);
      if (segstart && q_busy) break;
      const int page = __shfl_sync(FULL, page_cur, src);
      const int gpart = __shfl_sync(FULL, gpart_cur, src);
      const int stage = idx % kStages;
      if (lane == 0) {
        if (segstart) {
          mbar_expect_tx(qbar, (uint32_t)(G * D * 2));
          bulk_load(q_u32, p.q + (size_t)(meta >> 1) * D, (uint32_t)(G * D * 2), qbar);
        }
        const uint32_t full = bar_u32 + 8 * stage;
        const uint32_t dst = stage_u32 + stage * C::kStage;
        const int row = (int)(p.layer_row0 + (uint32_t)page * (uint32_t)(Hkv * 16) + (uint32_t)gpart);
        mbar_expect_tx(full, 2 * kTile);
        tma_tile_3d(dst, &tmK, 0, row, 0, full, kv_policy);
        tma_tile_3d(dst + kTile, &tmV, 0, row, 0, full, kv_policy);
      }
      if (segstart) q_busy = true;
      ++pk;
    }

    // ------------------------------------------------ consume tile ck
    const int idx = (int)(ck - k0);
    const int stage = idx % kStages;
    if (c.j == 0 || idx == 0) {                      // segment start: fetch Q fragments, reset state
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
      seg_j0 = c.j;
    }
    const bool last_page = (c.j == c.np - 1);
    const int valid = last_page ? cn - 16 * (c.np - 1) : 16;
    // fused append (F1): token n-1 is the step's new token; its K/V row comes from k_new/v_new, not
    // from the page.  Fetch it (lanes [0,CH): K chunks, [CH,2CH): V chunks) while the tile lands.
    int4 new_row = make_int4(0, 0, 0, 0);
    int new_page = 0;
    if (APPEND && last_page) {
      constexpr int CH = D / 8;
      if (lane < 2 * CH) {
        const __half* src = (lane < CH ? p.k_new : p.v_new) + ((size_t)c.i * Hkv + c.g) * D + (lane % CH) * 8;
        new_row = __ldg(reinterpret_cast<const int4*>(src));
      }
      new_page = __ldg(p.bt + (size_t)c.i * p.bt_stride + c.j);
    }
    mbar_wait(bar_u32 + 8 * stage, (idx / kStages) & 1);

    const uint32_t kb = stage_u32 + stage * C::kStage, vb = kb + kTile;
    if (APPEND && last_page) {
      // overlay the row on the tile in shared memory (same swizzle as the TMA box) and store it to
      // the page: cache and output both equal hx_kv_append followed by hx_decode_attention
      constexpr int CH = D / 8;
      const int r = valid - 1;
      if (lane < 2 * CH) {
        const int x = lane >= CH ? 1 : 0, ch = lane - x * CH;
        *reinterpret_cast<int4*>(my_stage + stage * C::kStage + x * kTile + (ch >> 3) * 2048 + r * 128 +
                                 (((ch & 7) ^ (r & 7)) << 4)) = new_row;
        __half* dstg = (x ? p.vc : p.kc) + (((size_t)new_page * Hkv + c.g) * 16 + r) * D + ch * 8;
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
        const int a = Hkv * cum[c.i] + c.g * c.np, b = a + c.np;
        const int wa = owner_of(a), wb = owner_of(b - 1);
        const bool dense = smlo[nC] >= 16 * nC;                // then every worker's range is non-empty
        auto next_owner = [&](int ww) -> int {                 // next worker with a tile of the pair
          if (dense) return ww + 1;
          const int kn = w_lo(ww + 1);                         // (workers with an empty range own none)
          return kn >= b ? wb + 1 : owner_of(kn);
        };
        int nseg = wb - wa + 1;
        if (!dense) { nseg = 0; for (int ww = wa; ww <= wb; ww = next_owner(ww)) ++nseg; }
        int* counter = p.counters + c.i * Hkv + c.g;
        __threadfence();
        __syncwarp();
        int old = 0;
        if (lane == 0) old = atomicAdd(counter, 1);
        old = __shfl_sync(FULL, old, 0);
        if (old == nseg - 1) {
          if (lane == 0) *counter = 0;                           // leave the workspace clean for the next call
          __threadfence();
          const bool wa_first = (w_lo(wa) == a);
          auto slot_of = [&](int ww) -> const float* {
            return p.partials + (size_t)((ww == wa && !wa_first) ? 2 * ww + 1 : 2 * ww) * C::kSlotFloats;
          };
          const int hb = 2 * (lane & 3);
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            float mm0 = -INFINITY, mm1 = -INFINITY;
            for (int ww = wa; ww <= wb; ww = next_owner(ww)) {
              const float2 mv = __ldcg(reinterpret_cast<const float2*>(slot_of(ww) + NT * kMT * 128 + nt * 8 + hb));
              mm0 = fmaxf(mm0, mv.x); mm1 = fmaxf(mm1, mv.y);
            }
            float l0 = 0.f, l1 = 0.f;
#pragma unroll
            for (int mt = 0; mt < kMT; ++mt) o[nt][mt][0] = o[nt][mt][1] = o[nt][mt][2] = o[nt][mt][3] = 0.f;
            for (int ww = wa; ww <= wb; ww = next_owner(ww)) {     // fixed (token) order: deterministic
              const float* sl = slot_of(ww);
              const float2 mv = __ldcg(reinterpret_cast<const float2*>(sl + NT * kMT * 128 + nt * 8 + hb));
              const float2 lv = __ldcg(reinterpret_cast<const float2*>(sl + NT * kMT * 128 + NT * 8 + nt * 8 + hb));
              const float c0 = ex2(mv.x - mm0), c1 = ex2(mv.y - mm1);
              l0 += lv.x * c0; l1 += lv.y * c1;
#pragma unroll
              for (int mt = 0; mt < kMT; ++mt) {
                const float4 v = __ldcg(reinterpret_cast<const float4*>(sl) + (nt * kMT + mt) * 32 + lane);
                o[nt][mt][0] += v.x * c0; o[nt][mt][1] += v.y * c1;
                o[nt][mt][2] += v.z * c0; o[nt][mt][3] += v.w * c1;
              }
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
        int4* dst = reinterpret_cast<int4*>(p.out + ((size_t)c.i * p.Hq + (size_t)c.g * G) * D);
        const int4* srcv = reinterpret_cast<const int4*>(scratch);
        for (int e = lane; e < G * D / 8; e += 32) dst[e] = srcv[e];
        __syncwarp();
        wrote_smem = true;
      }
    }
    if (wrote_smem) { fence_proxy_async(); __syncwarp(); }   // generic writes before the TMA refill

    // ------------------------------------------------ advance the cursor
    ++ck;
    if (++c.j == c.np) {
      c.j = 0;
      if (++c.g == Hkv) {
        c.g = 0;
        do { ++c.i; } while (c.i < B && cum[c.i + 1] == cum[c.i]);
        if (c.i < B) { c.np = cum[c.i + 1] - cum[c.i]; cn = slen[c.i]; }
      }
    }
  }
  } while (false);
  if (p.pdl_wait_at_end) asm volatile("griddepcontrol.wait;" ::: "memory");

  // ---- tuned mode: the last CTA of the grid to finish clears the claim flags for the next call.
  // No fences: every CTA's claim (an atomic whose result it consumed) precedes its own count-up, and
  // the plain stores below are flushed by kernel completion.
  if (tuned) {
    __syncthreads();
    if (tid == 0 && atomicAdd(p.claim + kMaxSm, 1) == nC - 1)
      for (int s = 0; s <= kMaxSm; ++s) p.claim[s] = 0;
  }
}

// ---------------------------------------------------------------------------- host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

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

template <int D, int NT, bool APPEND>
int launch_stream(const AttnParams& a, const DeviceInfo& di, cudaStream_t stream) {
  using C = Cfg<D, NT>;
  {
    static std::mutex mu;
    static bool attr_set[64] = {false};
    std::lock_guard<std::mutex> lock(mu);
    if (!attr_set[di.device]) {
      if (C::kSmem > di.max_smem_optin) HX_FAIL(HX_ERR_UNSUPPORTED, "device offers %d B shared memory per CTA, kernel needs %d", di.max_smem_optin, C::kSmem);
      HX_CUDA_OK(cudaFuncSetAttribute(attn_stream_kernel<D, NT, APPEND>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmem));
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
  const size_t counter_bytes = ((size_t)kBMax * a.kv_heads * sizeof(int32_t) + 15) & ~(size_t)15;
  if ((long long)kBMax * a.bt_stride * a.kv_heads >= (1ll << 28)) HX_FAIL(HX_ERR_UNSUPPORTED, "block_table_stride * kv_heads too large");
  for (int b0 = 0; b0 < a.batch; b0 += kBMax) {
    StreamParams p;
    p.B = (a.batch - b0 < kBMax) ? a.batch - b0 : kBMax;
    p.q = static_cast<const __half*>(a.q) + (size_t)b0 * a.q_heads * D;
    p.out = static_cast<__half*>(a.out) + (size_t)b0 * a.q_heads * D;
    p.bt = a.block_table + (size_t)b0 * a.bt_stride;
    p.lens = a.seq_lens + b0;
    p.partials = reinterpret_cast<float*>(ws);
    p.counters = reinterpret_cast<int32_t*>(ws + partial_bytes);
    p.claim = reinterpret_cast<int32_t*>(ws + partial_bytes + counter_bytes);
    p.Hq = a.q_heads; p.Hkv = a.kv_heads; p.G = a.q_heads / a.kv_heads; p.bt_stride = a.bt_stride;
    p.layer_row0 = (uint32_t)(rows_per_layer * a.layer);
    p.scale_log2 = a.sm_scale * kLog2e;
    const size_t layer_elems = (size_t)rows_per_layer * D;
    p.k_new = APPEND ? static_cast<const __half*>(a.k_new) + (size_t)b0 * a.kv_heads * D : nullptr;
    p.v_new = APPEND ? static_cast<const __half*>(a.v_new) + (size_t)b0 * a.kv_heads * D : nullptr;
    p.kc = static_cast<__half*>(const_cast<void*>(a.k_base)) + layer_elems * a.layer;
    p.vc = static_cast<__half*>(const_cast<void*>(a.v_base)) + layer_elems * a.layer;
    p.pdl_wait_at_end = (a.overlap_prev && b0 == 0) ? 1 : 0;
    if (p.pdl_wait_at_end) {
      // programmatic dependent launch: this grid may start while the ingest kernel enqueued just before it (which
      // executes griddepcontrol.launch_dependents at once) is still running.  The caller asserted that it reads
      // nothing that kernel writes; each CTA waits for the ingest's completion before it exits, so that whatever is
      // ordered after this grid is ordered after the ingest too.
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(grid); cfg.blockDim = dim3(kWarps * 32); cfg.dynamicSmemBytes = C::kSmem; cfg.stream = stream;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      at[0].val.programmaticStreamSerializationAllowed = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      HX_CUDA_OK(cudaLaunchKernelEx(&cfg, attn_stream_kernel<D, NT, APPEND>, tk, tv, p));
    } else {
      attn_stream_kernel<D, NT, APPEND><<<grid, kWarps * 32, C::kSmem, stream>>>(tk, tv, p);
    }
    HX_CUDA_OK(cudaGetLastError());
  }
  return HX_OK;
}

}  // namespace

size_t attn_workspace_bytes(int32_t batch, int32_t q_heads, int32_t kv_heads, int32_t head_dim,
                            int32_t max_seq_len, int32_t page_size) {
  (void)batch; (void)max_seq_len; (void)page_size;
  const int G = q_heads / kv_heads;
  const int nt = G > 8 ? 2 : 1;
  const size_t slot = (size_t)nt * ((head_dim / 16) * 128 + 16) * sizeof(float);
  const size_t counter_bytes = ((size_t)kBMax * kv_heads * sizeof(int32_t) + 15) & ~(size_t)15;
  return 2 * (size_t)kMaxWorkers * slot + counter_bytes + (size_t)(2 * kMaxSm) * sizeof(int32_t);
}

int tune_sm_rates(const void* scratch, size_t bytes, cudaStream_t stream) {
  DeviceInfo di;
  int rc = device_info(&di);
  if (rc) return rc;
  const int grid = di.sm_count < kMaxSm ? di.sm_count : kMaxSm;
  if (!scratch || bytes == 0) {                              // back to equal ranges
    sm_rate_finalize_kernel<<<1, kMaxSm, 0, stream>>>(grid, 1, 0);
    HX_CUDA_OK(cudaGetLastError());
    return HX_OK;
  }
  constexpr int kProbeSmem = kWarps * 3 * 8192;
  {
    static std::mutex mu;
    static bool attr_set[64] = {false};
    std::lock_guard<std::mutex> lock(mu);
    if (!attr_set[di.device]) {
      HX_CUDA_OK(cudaFuncSetAttribute(sm_rate_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kProbeSmem));
      attr_set[di.device] = true;
    }
  }
  // three windows of 80 us: the counts of a window are max-merged per SM, which drops start-up noise
  for (int rep = 0; rep < 3; ++rep) {
    sm_rate_probe_kernel<<<grid, kWarps * 32, kProbeSmem, stream>>>(static_cast<const uint8_t*>(scratch), bytes / 8192, 80000u);
    HX_CUDA_OK(cudaGetLastError());
  }
  const int damp = 176;                                     // 0.69 (B200 sweep: 160-192 best), see sm_rate_finalize_kernel
  sm_rate_finalize_kernel<<<1, kMaxSm, 0, stream>>>(grid, 0, damp);
  HX_CUDA_OK(cudaGetLastError());
  return HX_OK;
}

int launch_attention(const AttnParams& a, cudaStream_t stream) {
  DeviceInfo di;
  int rc = device_info(&di);
  if (rc) return rc;
  const int G = a.q_heads / a.kv_heads;
  if (a.k_new) {
    if (a.head_dim == 128) return G > 8 ? launch_stream<128, 2, true>(a, di, stream) : launch_stream<128, 1, true>(a, di, stream);
    return G > 8 ? launch_stream<64, 2, true>(a, di, stream) : launch_stream<64, 1, true>(a, di, stream);
  }
  if (a.head_dim == 128) return G > 8 ? launch_stream<128, 2, false>(a, di, stream) : launch_stream<128, 1, false>(a, di, stream);
  return G > 8 ? launch_stream<64, 2, false>(a, di, stream) : launch_stream<64, 1, false>(a, di, stream);
}

}  // namespace hx
