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
//
// attn_simple_kernel — one CTA per (request, q head) on CUDA cores; bring-up/debug only
// (HX_ATTN_IMPL=simple).
#include <cuda.h>
#include <cuda_fp16.h>

#include <cstdlib>
#include <cstring>
#include <mutex>

#include "hx_internal.h"

namespace hx {
namespace {

constexpr int kWarps = 8;          // consumer warps per CTA; tile t of a chunk belongs to warp t % 8
constexpr int kBMax = 1024;        // requests per launch (prefix sums live in shared memory)
constexpr int kMaxChunks = 4608;   // bound on chunk ids: nCTA * (levels + 2), nCTA <= 256, levels <= 16
constexpr int kChunkRing = 32;     // per-CTA ring of claimed chunks
constexpr int kRS = 4;             // own tiles described per lookahead round (lanes 0..kRS-1)
constexpr float kLog2e = 1.4426950408889634f;

template <int D, int NT>
struct Cfg {
  static constexpr int kStages = (NT == 1) ? 3 : 2;
  static constexpr int kTile = 16 * D * 2;           // bytes of one (page, head) K or V tile
  static constexpr int kStage = 2 * kTile;           // K + V
  static constexpr int kQBytes = NT * 8 * D * 2;     // per-warp Q slot: NT*8 heads
  static constexpr int kKS = D / 16;                 // k-steps of QK^T
  static constexpr int kMT = D / 16;                 // m-tiles of PV
  static constexpr int kSlices = NT * kMT;           // 16-row slices of O^T, one float4 per lane each
  static constexpr int kSlotFloats = kSlices * 128 + NT * 16;   // partial: acc[slices][32][4], m[NT][8], l[NT][8]
  static constexpr int kCtl = 4 * kChunkRing * 4 + 64 + kWarps * (NT * 16 + 1) * 4 + (6 + 3 * 40) * 4 + 16;
  static constexpr int kSmem = kWarps * kStages * kStage + kWarps * kQBytes + kWarps * (kStages + 1) * 8 +
                               (kBMax + 1) * 4 + kBMax * 4 + kCtl;
  static_assert(kStage >= kSlices * 512, "a consumed stage must hold one warp's O^T as merge scratch");
};

struct StreamParams {
  const __half* q;
  __half* out;
  const int32_t* bt;
  const int32_t* lens;
  int32_t* ctrl;          // [0] next chunk id, [1] finished CTAs; zero between calls
  int32_t* counters;      // [B * Hkv] arrival counters of pairs split across chunks; zero between calls
  float* partials;        // [2 * kMaxChunks][kSlotFloats]
  int32_t B, Hq, Hkv, G, bt_stride;
  uint32_t layer_row0;    // first tensor-map row of the layer
  float scale_log2;
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

__device__ __forceinline__ void tma_tile_3d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
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
// Guided chunk schedule over the tile sequence [0, N): a deterministic function of (N, nC, M).
// Level l holds nC chunks of s_l = roundup8(R_l / (2 nC)) tiles (R_l = tiles left at the level's
// start), until s_l <= M; the rest goes out in chunks of M.  Chunk sizes are multiples of 8 (only
// the very last may be short), so tile t of a chunk always belongs to warp t % 8.
constexpr int kMaxLv = 40;
struct ChunkSched {        // level table, built once per CTA in shared memory
  int N, nC, M, n_lv;
  int tail_first, tail_base;
  int lv_first[kMaxLv], lv_base[kMaxLv], lv_size[kMaxLv];
};

__device__ void build_sched(ChunkSched* cs, int N, int nC) {
  int m = (N / (nC * 4)) & ~7;                               // ~4 minimum-size chunks per CTA
  cs->N = N; cs->nC = nC; cs->M = m < 8 ? 8 : (m > 32 ? 32 : m);
  int base = 0, R = N, first = 0, l = 0;
  while (l < kMaxLv) {
    const int s = (R / (2 * nC) + 7) & ~7;
    if (s <= cs->M) break;
    cs->lv_first[l] = first; cs->lv_base[l] = base; cs->lv_size[l] = s;
    base += nC * s; R -= nC * s; first += nC; ++l;
  }
  cs->n_lv = l; cs->tail_first = first; cs->tail_base = base;
}
__device__ __forceinline__ void chunk_range(const ChunkSched* cs, int id, int& start, int& size) {
  for (int l = 0; l < cs->n_lv; ++l)
    if (id < cs->lv_first[l] + cs->nC) {
      start = cs->lv_base[l] + (id - cs->lv_first[l]) * cs->lv_size[l];
      size = cs->lv_size[l];
      return;
    }
  const long long st = (long long)cs->tail_base + (long long)(id - cs->tail_first) * cs->M;
  start = st >= cs->N ? cs->N : (int)st;
  size = st >= cs->N ? 0 : min(cs->M, cs->N - (int)st);
}
__device__ __forceinline__ int chunk_of_tile(const ChunkSched* cs, int k) {
  for (int l = 0; l < cs->n_lv; ++l)
    if (k < cs->lv_base[l] + cs->nC * cs->lv_size[l]) return cs->lv_first[l] + (k - cs->lv_base[l]) / cs->lv_size[l];
  return cs->tail_first + (k - cs->tail_base) / cs->M;
}

constexpr int kEvRing = 16;        // split-pair events queued for the service warp
struct Ctl {
  int ch_start[kChunkRing], ch_size[kChunkRing], ch_id[kChunkRing], ev[2 * kEvRing];
  int n_chunks, exhausted, lock, ev_head, ev_tail, cons_done, pad2[10];
};

template <int D, int NT>
__global__ void __launch_bounds__(kWarps * 32 + 32, 1)
attn_stream_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                   const StreamParams p) {
  using C = Cfg<D, NT>;
  constexpr int kStages = C::kStages, kTile = C::kTile, kKS = C::kKS, kMT = C::kMT, kSlices = C::kSlices;
  constexpr uint32_t FULL = 0xffffffffu;
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* q_base = smem + kWarps * kStages * C::kStage;
  uint64_t* bars = reinterpret_cast<uint64_t*>(q_base + kWarps * C::kQBytes);
  int* cum = reinterpret_cast<int*>(bars + kWarps * (kStages + 1));
  int* slen = cum + (kBMax + 1);
  Ctl* ctl = reinterpret_cast<Ctl*>(slen + kBMax);
  float* ml = reinterpret_cast<float*>(ctl + 1);            // [kWarps][NT*16]: m[8], l[8] per nt
  int* sc_off = reinterpret_cast<int*>(ml + kWarps * NT * 16);
  ChunkSched* sched = reinterpret_cast<ChunkSched*>(sc_off + kWarps);
  static_assert(sizeof(Ctl) == 4 * kChunkRing * 4 + 64 && 2 * kEvRing == kChunkRing, "Ctl size");

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int B = p.B, Hkv = p.Hkv, G = p.G;
#ifdef HX_TRACE
  unsigned long long tr[5] = {0, 0, 0, 0, 0};
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tr[0]));
#define HX_STAMP(x) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tr[x]))
#else
#define HX_STAMP(x)
#endif

  // ---- setup: page-count prefix sums (row A4), control block, barrier init
  {
    constexpr int PER = kBMax / (kWarps * 32);
    __shared__ int warp_tot[kWarps];
    int np[PER], sum = 0;
#pragma unroll
    for (int e = 0; e < PER; ++e) {
      const int i = tid * PER + e;                          // the service warp (tid >= 256) holds none
      const int n = (i < B && tid < kWarps * 32) ? max(__ldg(p.lens + i), 0) : 0;
      if (i < B && tid < kWarps * 32) slen[i] = n;
      np[e] = (n + 15) >> 4;
      sum += np[e];
    }
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(FULL, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane == 31 && warp < kWarps) warp_tot[warp] = incl;
    if (lane == 0 && warp < kWarps) {
      const uint32_t b0 = smem_u32(bars + warp * (kStages + 1));
      for (int s = 0; s <= kStages; ++s) mbar_init(b0 + 8 * s, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid == 0) { ctl->n_chunks = 0; ctl->exhausted = 0; ctl->lock = 0; ctl->ev_head = 0; ctl->ev_tail = 0; ctl->cons_done = 0; cum[0] = 0; }
    __syncthreads();
    int off = incl - sum;
    for (int w = 0; w < warp && w < kWarps; ++w) off += warp_tot[w];
#pragma unroll
    for (int e = 0; e < PER; ++e) {
      const int i = tid * PER + e;
      off += np[e];
      if (i < B && tid < kWarps * 32) cum[i + 1] = off;
    }
    __syncthreads();
    // reading S11: an empty context gives a zero output row (no tile ever touches it)
    for (int i = blockIdx.x * (kWarps * 32) + tid; i < B && tid < kWarps * 32; i += gridDim.x * (kWarps * 32))
      if (slen[i] == 0) {
        int4* row = reinterpret_cast<int4*>(p.out + (size_t)i * p.Hq * D);
        for (int e = 0; e < p.Hq * D / 8; ++e) row[e] = make_int4(0, 0, 0, 0);
      }
  }
  HX_STAMP(1);

  if (tid == 0) build_sched(sched, Hkv * cum[B], (int)gridDim.x);
  __syncthreads();

  // ---- service warp: finishes pairs that were split across chunks, off the consumers' path.  For
  // every queued event (request, kv head) it publishes this CTA's partial (fence + arrival counter)
  // and, when it is the last arriver, merges the pair's partials in chunk order (= token order, so
  // the result does not depend on who arrives last), normalises and writes the output (row A8).
  if (warp == kWarps) {
    const int tok0 = lane >> 2, hb = 2 * (lane & 3);
    int tail = 0;
    while (true) {
      int head = *(volatile int*)&ctl->ev_head;
      if (head == tail) {
        if (*(volatile int*)&ctl->cons_done == kWarps) {
          head = *(volatile int*)&ctl->ev_head;            // re-read: an event may precede the last exit
          if (head == tail) break;
        } else {
          __nanosleep(256);
          continue;
        }
      }
      __threadfence_block();
      const int i = ctl->ev[2 * (tail % kEvRing)], g = ctl->ev[2 * (tail % kEvRing) + 1];
      const int np = cum[i + 1] - cum[i];
      const int a = Hkv * cum[i] + g * np, b = a + np;      // the pair's tiles [a, b)
      const int id_a = chunk_of_tile(sched, a), id_b = chunk_of_tile(sched, b - 1);
      const int nseg = id_b - id_a + 1;                      // chunks that hold a part of the pair
      int last = 0;
      if (lane == 0) {
        int* counter = p.counters + i * Hkv + g;
        __threadfence();                                    // the CTA's partial slices, cumulatively
        const int old = atomicAdd(counter, 1);
        if (old == nseg - 1) { *counter = 0; last = 1; }    // leave the workspace clean for the next call
        __threadfence();
      }
      last = __shfl_sync(FULL, last, 0);
      if (last) {
        __half* orow = p.out + ((size_t)i * p.Hq + (size_t)g * G) * D;
        // slot of owner chunk id: its last segment if the pair starts inside it, else its first
        int st_a, sz_a;
        chunk_range(sched, id_a, st_a, sz_a);
        const int first_slot = st_a < a ? 2 * id_a + 1 : 2 * id_a;
        auto slot_ptr = [&](int e) -> const float* {
          return p.partials + (size_t)(e == 0 ? first_slot : 2 * (id_a + e)) * C::kSlotFloats;
        };
        // pass 1: running max per head over the owners (independent loads, 4 in flight)
        float mm[NT][2];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) mm[nt][0] = mm[nt][1] = -INFINITY;
        for (int e0 = 0; e0 < nseg; e0 += 4) {
          float2 mv[4][NT];
#pragma unroll
          for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
              mv[u][nt] = (e0 + u < nseg) ? __ldcg(reinterpret_cast<const float2*>(slot_ptr(e0 + u) + kSlices * 128 + nt * 16 + hb))
                                          : make_float2(-INFINITY, -INFINITY);
#pragma unroll
          for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) { mm[nt][0] = fmaxf(mm[nt][0], mv[u][nt].x); mm[nt][1] = fmaxf(mm[nt][1], mv[u][nt].y); }
        }
        // pass 2: owners in chunk order (= token order: deterministic); all slices of one owner in flight
        float ll[NT][2], acc[kSlices][4];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) ll[nt][0] = ll[nt][1] = 0.f;
#pragma unroll
        for (int sl = 0; sl < kSlices; ++sl) acc[sl][0] = acc[sl][1] = acc[sl][2] = acc[sl][3] = 0.f;
        for (int e = 0; e < nseg; ++e) {
          const float* gs = slot_ptr(e);
          float4 v[kSlices];
          float2 mv[NT], lv[NT];
#pragma unroll
          for (int sl = 0; sl < kSlices; ++sl) v[sl] = __ldcg(reinterpret_cast<const float4*>(gs) + sl * 32 + lane);
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            mv[nt] = __ldcg(reinterpret_cast<const float2*>(gs + kSlices * 128 + nt * 16 + hb));
            lv[nt] = __ldcg(reinterpret_cast<const float2*>(gs + kSlices * 128 + nt * 16 + 8 + hb));
          }
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            const float c0 = ex2(mv[nt].x - mm[nt][0]), c1 = ex2(mv[nt].y - mm[nt][1]);
            ll[nt][0] += lv[nt].x * c0; ll[nt][1] += lv[nt].y * c1;
#pragma unroll
            for (int mt = 0; mt < kMT; ++mt) {
              const int sl = nt * kMT + mt;
              acc[sl][0] += v[sl].x * c0; acc[sl][1] += v[sl].y * c1;
              acc[sl][2] += v[sl].z * c0; acc[sl][3] += v[sl].w * c1;
            }
          }
        }
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
          const float i0 = 1.f / ll[nt][0], i1 = 1.f / ll[nt][1];
          const int h0 = nt * 8 + hb;
#pragma unroll
          for (int mt = 0; mt < kMT; ++mt) {
            const int sl = nt * kMT + mt, d0 = 16 * mt + tok0;
            if (h0 < G) {
              orow[h0 * D + d0] = __float2half_rn(acc[sl][0] * i0);
              orow[h0 * D + d0 + 8] = __float2half_rn(acc[sl][2] * i0);
            }
            if (h0 + 1 < G) {
              orow[(h0 + 1) * D + d0] = __float2half_rn(acc[sl][1] * i1);
              orow[(h0 + 1) * D + d0 + 8] = __float2half_rn(acc[sl][3] * i1);
            }
          }
        }
      }
      ++tail;
      if (lane == 0) *(volatile int*)&ctl->ev_tail = tail;
    }
#ifdef HX_TRACE
    HX_STAMP(4);
    if (lane == 0) {
      unsigned long long* t = reinterpret_cast<unsigned long long*>(p.partials + (size_t)2 * kMaxChunks * C::kSlotFloats) + (size_t)(gridDim.x * kWarps + blockIdx.x) * 8;
      for (int e = 0; e < 5; ++e) t[e] = tr[e];
      t[5] = (unsigned long long)tail;
    }
#endif
    // leave the scheduler state clean: the last CTA of the grid zeroes the control words
    if (lane == 0) {
      const int old = atomicAdd(p.ctrl + 1, 1);
      if (old == (int)gridDim.x - 1) { p.ctrl[0] = 0; p.ctrl[1] = 0; }
    }
    return;
  }

  // chunk index n of this CTA's claim list: claimed on demand by whichever warp needs it first
  auto ensure = [&](int n) -> bool {
    while (true) {
      if (*(volatile int*)&ctl->n_chunks > n) return true;
      if (*(volatile int*)&ctl->exhausted) return false;
      if (lane == 0 && atomicCAS(&ctl->lock, 0, 1) == 0) {
        const int nc = *(volatile int*)&ctl->n_chunks;
        if (nc <= n && !*(volatile int*)&ctl->exhausted) {
          const int id = atomicAdd(p.ctrl, 1);
          int st, sz;
          chunk_range(sched, id, st, sz);
          if (sz == 0) {
            *(volatile int*)&ctl->exhausted = 1;
          } else {
            const int s = nc % kChunkRing;
            ctl->ch_start[s] = st; ctl->ch_size[s] = sz; ctl->ch_id[s] = id;
            __threadfence_block();
            *(volatile int*)&ctl->n_chunks = nc + 1;
          }
        }
        __threadfence_block();
        atomicExch(&ctl->lock, 0);
      }
      __syncwarp();
    }
  };
  auto own_count = [&](int size) -> int { return size > warp ? ((size - warp - 1) >> 3) + 1 : 0; };

  uint8_t* my_stage = smem + warp * kStages * C::kStage;
  const uint32_t stage_u32 = smem_u32(my_stage);
  uint8_t* my_q = q_base + warp * C::kQBytes;
  const uint32_t q_u32 = smem_u32(my_q);
  const uint32_t bar_u32 = smem_u32(bars + warp * (kStages + 1));
  const uint32_t qbar = bar_u32 + 8 * kStages;

  // ---- lookahead over this warp's own tiles (tile o of a chunk with o % 8 == warp): lane L < kRS of
  // round r describes own tile kRS*r + L: page id (global load), head part, Q row, "first own tile of
  // its segment".  Rounds r and r+1 are resident, so block-table loads run 4-8 own tiles ahead.
  int la_n = 0, la_u = 0;          // (chunk index, own offset) of own tile kRS * (cur_round + 2)
  auto load_round = [&](int& page, int& gpart, int& meta) {
    {  // warp-uniform: claim chunks until own tile la_u + kRS - 1 from chunk la_n exists (or none is left)
      int n = la_n, u = la_u + kRS - 1;
      while (ensure(n)) {
        const int cnt = own_count(*(volatile int*)&ctl->ch_size[n % kChunkRing]);
        if (u < cnt) break;
        u -= cnt; ++n;
      }
    }
    const int nc = *(volatile int*)&ctl->n_chunks;
    page = 0; gpart = 0; meta = -1;
    int n = la_n, u = la_u + lane;
    if (lane < kRS) {
      while (n < nc) {
        const int size = ctl->ch_size[n % kChunkRing];
        const int cnt = own_count(size);
        if (u < cnt) {
          const int o = warp + 8 * u;
          const Loc t = locate(ctl->ch_start[n % kChunkRing] + o, cum, B, Hkv);
          page = __ldg(p.bt + (size_t)t.i * p.bt_stride + t.j);
          gpart = t.g * 16;
          const int o_seg0 = o - min(t.j, o);                 // segment's first tile in this chunk
          const int fo = o_seg0 + ((warp - o_seg0) & 7);      // this warp's first own tile in it
          meta = ((t.i * p.Hq + t.g * G) << 1) | (o == fo ? 1 : 0);
          break;
        }
        u -= cnt; ++n;
      }
    }
    // advance the round base by kRS own tiles (warp-uniform)
    n = la_n; u = la_u + kRS;
    while (n < nc) {
      const int cnt = own_count(ctl->ch_size[n % kChunkRing]);
      if (u < cnt) break;
      u -= cnt; ++n;
    }
    la_n = n; la_u = u;
  };
  int page_cur, gpart_cur, meta_cur, page_nxt, gpart_nxt, meta_nxt;
  load_round(page_cur, gpart_cur, meta_cur);
  load_round(page_nxt, gpart_nxt, meta_nxt);
  int cur_round = 0;

  // fragment-address constants
  const int a_row = (lane & 7) + ((lane >> 3) & 1) * 8;   // K (A, non-trans): token row
  const int a_csel = lane >> 4;                           //   chunk select within the k-step
  const int v_row = (lane & 7) + (lane >> 4) * 8;         // V (A, trans): token row
  const int v_csel = (lane >> 3) & 1;
  const int tok0 = lane >> 2;
  const int hb = 2 * (lane & 3);

  uint32_t qb[NT][kKS][2];
  float o[NT][kMT][4];
  float m_run[NT][2], l_run[NT][2];
  int pm = 0, cm = 0, q_issued = 0, q_taken = 0;          // own tiles produced / consumed; Q loads

  for (int cidx = 0; ensure(cidx); ++cidx) {
    const int cslot = cidx % kChunkRing;
    const int cstart = ctl->ch_start[cslot], csize = ctl->ch_size[cslot], cid = ctl->ch_id[cslot];
    Loc c = locate(cstart, cum, B, Hkv);
    int cn = slen[c.i];
    int oseg = 0;                                          // chunk offset of the current segment
    while (oseg < csize) {
      const int seg_len = min(c.np - c.j, csize - oseg);
      const int fo = oseg + ((warp - oseg) & 7);
      const bool has_state = fo < oseg + seg_len;
      int last_stage = 0;
      bool wrote_smem = false;
      for (int oo = fo; oo < oseg + seg_len; oo += 8) {
        // ------------------------------------------ produce: keep kStages own tiles in flight
        while (pm < cm + kStages) {
          if (pm / kRS != cur_round) {
            page_cur = page_nxt; gpart_cur = gpart_nxt; meta_cur = meta_nxt;
            ++cur_round;
            load_round(page_nxt, gpart_nxt, meta_nxt);
          }
          const int src = pm % kRS;
          const int meta = __shfl_sync(FULL, meta_cur, src);
          if (meta < 0) break;                             // no tile left for this warp
          const bool segstart = meta & 1;
          if (segstart && q_issued != q_taken) break;      // Q slot still holds the running segment's Q
          const int page = __shfl_sync(FULL, page_cur, src);
          const int gpart = __shfl_sync(FULL, gpart_cur, src);
          const int stage = pm % kStages;
          if (lane == 0) {
            if (segstart) {
              mbar_expect_tx(qbar, (uint32_t)(G * D * 2));
              bulk_load(q_u32, p.q + (size_t)(meta >> 1) * D, (uint32_t)(G * D * 2), qbar);
            }
            const uint32_t full = bar_u32 + 8 * stage;
            const uint32_t dst = stage_u32 + stage * C::kStage;
            const int row = (int)(p.layer_row0 + (uint32_t)page * (uint32_t)(Hkv * 16) + (uint32_t)gpart);
            mbar_expect_tx(full, 2 * kTile);
            tma_tile_3d(dst, &tmK, 0, row, 0, full);
            tma_tile_3d(dst + kTile, &tmV, 0, row, 0, full);
          }
          if (segstart) ++q_issued;
          ++pm;
        }

        // ------------------------------------------ consume own tile cm = (chunk, offset oo)
        const int stage = cm % kStages;
        const int j = c.j + (oo - oseg);
        if (oo == fo) {                                    // first own tile of the segment
          mbar_wait(qbar, q_taken & 1);
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            const int head = nt * 8 + (lane >> 2);
            const uint8_t* qrow = my_q + head * (D * 2) + (lane & 3) * 4;
#pragma unroll
            for (int ks = 0; ks < kKS; ++ks) {
              const uint32_t b0 = *reinterpret_cast<const uint32_t*>(qrow + ks * 32);
              const uint32_t b1 = *reinterpret_cast<const uint32_t*>(qrow + ks * 32 + 16);
              qb[nt][ks][0] = head < G ? b0 : 0u;
              qb[nt][ks][1] = head < G ? b1 : 0u;
            }
#pragma unroll
            for (int mt = 0; mt < kMT; ++mt) o[nt][mt][0] = o[nt][mt][1] = o[nt][mt][2] = o[nt][mt][3] = 0.f;
            m_run[nt][0] = m_run[nt][1] = -INFINITY;
            l_run[nt][0] = l_run[nt][1] = 0.f;
          }
          __syncwarp();
          ++q_taken;
        }
        mbar_wait(bar_u32 + 8 * stage, (cm / kStages) & 1);
#ifdef HX_TRACE
        if (cm == 0) HX_STAMP(2);
        HX_STAMP(3);
#endif
        const uint32_t kb = stage_u32 + stage * C::kStage, vb = kb + kTile;
        const int valid = (j == c.np - 1) ? cn - 16 * (c.np - 1) : 16;
        if (valid < 16) {
          // tail slots may hold anything (NaN/Inf): P is 0 there, but 0 * Inf = NaN in the PV MMA,
          // so the V rows past the context end are zeroed in shared memory (reading S10).
          for (int e = lane; e < (16 - valid) * (D / 8); e += 32) {
            const int r = valid + e / (D / 8), ch = e % (D / 8);
            *reinterpret_cast<int4*>(my_stage + stage * C::kStage + kTile + (ch >> 3) * 2048 + r * 128 + (ch & 7) * 16) =
                make_int4(0, 0, 0, 0);
          }
          __syncwarp();
          wrote_smem = true;
        }

        // ---- S^T[16 tok x 8 heads] = K[16 x D] Q^T   (row A5)
        float sacc[NT][2][4];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int h = 0; h < 2; ++h) sacc[nt][h][0] = sacc[nt][h][1] = sacc[nt][h][2] = sacc[nt][h][3] = 0.f;
#pragma unroll
        for (int ks = 0; ks < kKS; ++ks) {
          const int cix = 2 * ks + a_csel;
          uint32_t a[4];
          ldsm_x4(kb + (cix >> 3) * 2048 + a_row * 128 + (((cix & 7) ^ (a_row & 7)) << 4), a);
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
            const float m_new = fmaxf(m_run[nt][e], mx);      // finite: every tile has >= 1 valid token
            corr[e] = ex2(m_run[nt][e] - m_new);              // -inf -> 0 on the first tile
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
          const int cix = 2 * mt + v_csel;
          uint32_t a[4];
          ldsm_x4_t(vb + (cix >> 3) * 2048 + v_row * 128 + (((cix & 7) ^ (v_row & 7)) << 4), a);
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) mma16816(o[nt][mt], a, pb[nt][0], pb[nt][1]);
        }
        __syncwarp();                                      // every lane is done reading this stage
        last_stage = stage;
        ++cm;
        if (wrote_smem && oo + 8 < oseg + seg_len) { fence_proxy_async(); __syncwarp(); wrote_smem = false; }
      }

      // -------------------------------------------- segment end: the 8 warps combine (row A8)
      const bool complete = (c.j == 0) && (seg_len == c.np);   // whole (request, kv head) in this chunk
      if (has_state) {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            float l = l_run[nt][e];
            l += __shfl_xor_sync(FULL, l, 4);
            l += __shfl_xor_sync(FULL, l, 8);
            l += __shfl_xor_sync(FULL, l, 16);
            l_run[nt][e] = l;
          }
          if (lane < 4) {
            float* w_ml = ml + warp * (NT * 16) + nt * 16;
            w_ml[hb] = m_run[nt][0]; w_ml[hb + 1] = m_run[nt][1];
            w_ml[8 + hb] = l_run[nt][0]; w_ml[8 + hb + 1] = l_run[nt][1];
          }
        }
        float4* sc = reinterpret_cast<float4*>(my_stage + last_stage * C::kStage);   // just-consumed stage
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int mt = 0; mt < kMT; ++mt)
            sc[(nt * kMT + mt) * 32 + lane] = make_float4(o[nt][mt][0], o[nt][mt][1], o[nt][mt][2], o[nt][mt][3]);
        if (lane == 0) sc_off[warp] = (warp * kStages + last_stage) * C::kStage;
        wrote_smem = true;
      } else if (lane < NT * 16) {
        ml[warp * (NT * 16) + lane] = ((lane & 8) == 0) ? -INFINITY : 0.f;            // m = -inf: no state
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");

      float* gslot = nullptr;
      if (!complete) gslot = p.partials + (size_t)(2 * cid + (oseg == 0 ? 0 : 1)) * C::kSlotFloats;
      __half* orow = p.out + ((size_t)c.i * p.Hq + (size_t)c.g * G) * D;
      for (int sl = warp; sl < kSlices; sl += kWarps) {
        const int nt = sl / kMT, mt = sl - nt * kMT;
        float mm0 = -INFINITY, mm1 = -INFINITY;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
          mm0 = fmaxf(mm0, ml[w * (NT * 16) + nt * 16 + hb]);
          mm1 = fmaxf(mm1, ml[w * (NT * 16) + nt * 16 + hb + 1]);
        }
        float l0 = 0.f, l1 = 0.f, acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {                  // fixed warp order: deterministic
          const float* w_ml = ml + w * (NT * 16) + nt * 16;
          if (w_ml[0] == -INFINITY) continue;               // warp w had no tile in this segment
          const float c0 = ex2(w_ml[hb] - mm0), c1 = ex2(w_ml[hb + 1] - mm1);
          l0 += w_ml[8 + hb] * c0; l1 += w_ml[8 + hb + 1] * c1;
          const float4 v = reinterpret_cast<const float4*>(smem + sc_off[w])[sl * 32 + lane];
          acc[0] += v.x * c0; acc[1] += v.y * c1; acc[2] += v.z * c0; acc[3] += v.w * c1;
        }
        if (complete) {
          const int d0 = 16 * mt + tok0, h0 = nt * 8 + hb;
          if (h0 < G) {
            orow[h0 * D + d0] = __float2half_rn(acc[0] / l0);
            orow[h0 * D + d0 + 8] = __float2half_rn(acc[2] / l0);
          }
          if (h0 + 1 < G) {
            orow[(h0 + 1) * D + d0] = __float2half_rn(acc[1] / l1);
            orow[(h0 + 1) * D + d0 + 8] = __float2half_rn(acc[3] / l1);
          }
        } else {
          __stcg(reinterpret_cast<float4*>(gslot) + sl * 32 + lane, make_float4(acc[0], acc[1], acc[2], acc[3]));
          if (mt == 0 && lane < 4) {
            float* g_ml = gslot + kSlices * 128 + nt * 16;
            __stcg(reinterpret_cast<float2*>(g_ml + hb), make_float2(mm0, mm1));
            __stcg(reinterpret_cast<float2*>(g_ml + 8 + hb), make_float2(l0, l1));
          }
        }
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");       // scratch stages free; partial slices stored
      if (!complete && tid == 0) {
        // the pair continues in other chunks: queue it for the service warp
        const int head = ctl->ev_head;
        while (head - *(volatile int*)&ctl->ev_tail >= kEvRing) __nanosleep(64);
        ctl->ev[2 * (head % kEvRing)] = c.i;
        ctl->ev[2 * (head % kEvRing) + 1] = c.g;
        __threadfence_block();
        *(volatile int*)&ctl->ev_head = head + 1;
      }
      if (wrote_smem) { fence_proxy_async(); __syncwarp(); }   // generic writes before the TMA refill

      // -------------------------------------------- next segment
      oseg += seg_len;
      c.j += seg_len;
      if (c.j == c.np) {
        c.j = 0;
        if (++c.g == Hkv) {
          c.g = 0;
          do { ++c.i; } while (c.i < B && cum[c.i + 1] == cum[c.i]);
          if (c.i < B) { c.np = cum[c.i + 1] - cum[c.i]; cn = slen[c.i]; }
        }
      }
    }
  }

  __syncwarp();
  if (lane == 0) { __threadfence_block(); atomicAdd(&ctl->cons_done, 1); }
#ifdef HX_TRACE
  HX_STAMP(4);
  if (lane == 0) {
    unsigned long long* t = reinterpret_cast<unsigned long long*>(p.partials + (size_t)2 * kMaxChunks * C::kSlotFloats) + (size_t)(blockIdx.x * kWarps + warp) * 8;
    for (int e = 0; e < 5; ++e) t[e] = tr[e];
    t[5] = (unsigned long long)cm;
    unsigned smid; asm volatile("mov.u32 %0, %%smid;" : "=r"(smid)); t[6] = smid;
  }
#endif
}

// ------------------------------------------------------------------------------------------
// Kernel "simple": one CTA per (request, query head), CUDA-core dot products, no split.
// ------------------------------------------------------------------------------------------
struct SimpleParams {
  const __half* q; __half* out; const __half* k; const __half* v;
  const int32_t* bt; const int32_t* lens;
  int32_t q_heads, kv_heads, bt_stride;
  float scale_log2;
};

template <int D>
__global__ void __launch_bounds__(128) attn_simple_kernel(const SimpleParams p) {
  constexpr int E = D / 32;
  const int h = blockIdx.x, i = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n = p.lens[i];
  const int g = h / (p.q_heads / p.kv_heads);
  const __half* qrow = p.q + ((size_t)i * p.q_heads + h) * D;
  __half* orow = p.out + ((size_t)i * p.q_heads + h) * D;
  float qf[E], acc[E];
#pragma unroll
  for (int e = 0; e < E; ++e) { qf[e] = __half2float(qrow[lane * E + e]); acc[e] = 0.f; }
  float m = -INFINITY, l = 0.f;
  for (int t = warp; t < n; t += 4) {
    const int page = p.bt[(size_t)i * p.bt_stride + (t >> 4)];
    const size_t off = (((size_t)page * p.kv_heads + g) * 16 + (t & 15)) * D + lane * E;
    float dot = 0.f;
#pragma unroll
    for (int e = 0; e < E; ++e) dot += qf[e] * __half2float(p.k[off + e]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
    const float s = dot * p.scale_log2;
    const float m_new = fmaxf(m, s);
    const float corr = exp2f(m - m_new), wgt = exp2f(s - m_new);
    l = l * corr + wgt;
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = acc[e] * corr + wgt * __half2float(p.v[off + e]);
    m = m_new;
  }
  __shared__ float sm_m[4], sm_l[4], sm_acc[4][D];
  if (lane == 0) { sm_m[warp] = m; sm_l[warp] = l; }
#pragma unroll
  for (int e = 0; e < E; ++e) sm_acc[warp][lane * E + e] = acc[e];
  __syncthreads();
  if (warp == 0) {
    const float mm = fmaxf(fmaxf(sm_m[0], sm_m[1]), fmaxf(sm_m[2], sm_m[3]));
    float ll = 0.f, o[E];
#pragma unroll
    for (int e = 0; e < E; ++e) o[e] = 0.f;
    for (int w = 0; w < 4; ++w) {
      const float c = (sm_m[w] == -INFINITY) ? 0.f : exp2f(sm_m[w] - mm);
      ll += sm_l[w] * c;
#pragma unroll
      for (int e = 0; e < E; ++e) o[e] += sm_acc[w][lane * E + e] * c;
    }
#pragma unroll
    for (int e = 0; e < E; ++e) orow[lane * E + e] = __float2half_rn(n > 0 ? o[e] / ll : 0.f);
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

template <int D, int NT>
int launch_stream(const AttnParams& a, const DeviceInfo& di, cudaStream_t stream) {
  using C = Cfg<D, NT>;
  static bool attr_set[64] = {false};
  if (!attr_set[di.device]) {
    if (C::kSmem > di.max_smem_optin) HX_FAIL(HX_ERR_UNSUPPORTED, "device offers %d B shared memory per CTA, kernel needs %d", di.max_smem_optin, C::kSmem);
    HX_CUDA_OK(cudaFuncSetAttribute(attn_stream_kernel<D, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmem));
    attr_set[di.device] = true;
  }
  const uint64_t rows_per_layer = (uint64_t)a.num_pages * a.kv_heads * 16;
  const uint64_t rows = rows_per_layer * a.layers;
  if (rows >= (1ull << 31)) HX_FAIL(HX_ERR_UNSUPPORTED, "cache too large for one tensor map (%llu rows)", (unsigned long long)rows);
  CUtensorMap tk, tv;
  int rc = get_tile_maps(a.k_base, a.v_base, rows, D, &tk, &tv);
  if (rc) return rc;

  int grid = di.sm_count < 256 ? di.sm_count : 256;       // one persistent CTA per SM
  char* ws = static_cast<char*>(a.workspace);
  const size_t ctrl_bytes = 64;
  const size_t counter_bytes = ((size_t)kBMax * a.kv_heads * sizeof(int32_t) + 15) & ~(size_t)15;
  for (int b0 = 0; b0 < a.batch; b0 += kBMax) {
    StreamParams p;
    p.B = (a.batch - b0 < kBMax) ? a.batch - b0 : kBMax;
    p.q = static_cast<const __half*>(a.q) + (size_t)b0 * a.q_heads * D;
    p.out = static_cast<__half*>(a.out) + (size_t)b0 * a.q_heads * D;
    p.bt = a.block_table + (size_t)b0 * a.bt_stride;
    p.lens = a.seq_lens + b0;
    p.ctrl = reinterpret_cast<int32_t*>(ws);
    p.counters = reinterpret_cast<int32_t*>(ws + ctrl_bytes);
    p.partials = reinterpret_cast<float*>(ws + ctrl_bytes + counter_bytes);
    p.Hq = a.q_heads; p.Hkv = a.kv_heads; p.G = a.q_heads / a.kv_heads; p.bt_stride = a.bt_stride;
    p.layer_row0 = (uint32_t)(rows_per_layer * a.layer);
    p.scale_log2 = a.sm_scale * kLog2e;
    attn_stream_kernel<D, NT><<<grid, kWarps * 32 + 32, C::kSmem, stream>>>(tk, tv, p);
    HX_CUDA_OK(cudaGetLastError());
  }
  return HX_OK;
}

template <int D>
int launch_simple(const AttnParams& a, cudaStream_t stream) {
  SimpleParams p;
  const size_t layer_elems = (size_t)a.num_pages * a.kv_heads * 16 * D;
  p.q = static_cast<const __half*>(a.q); p.out = static_cast<__half*>(a.out);
  p.k = static_cast<const __half*>(a.k_base) + layer_elems * a.layer;
  p.v = static_cast<const __half*>(a.v_base) + layer_elems * a.layer;
  p.bt = a.block_table; p.lens = a.seq_lens;
  p.q_heads = a.q_heads; p.kv_heads = a.kv_heads; p.bt_stride = a.bt_stride;
  p.scale_log2 = a.sm_scale * kLog2e;
  attn_simple_kernel<D><<<dim3(a.q_heads, a.batch), 128, 0, stream>>>(p);
  HX_CUDA_OK(cudaGetLastError());
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
  return 64 + counter_bytes + 2 * (size_t)kMaxChunks * slot;
}

int launch_attention(const AttnParams& a, cudaStream_t stream) {
  DeviceInfo di;
  int rc = device_info(&di);
  if (rc) return rc;
  static const bool simple = [] { const char* e = getenv("HX_ATTN_IMPL"); return e && !strcmp(e, "simple"); }();
  if (simple) return a.head_dim == 128 ? launch_simple<128>(a, stream) : launch_simple<64>(a, stream);
  const int G = a.q_heads / a.kv_heads;
  if (a.head_dim == 128) return G > 8 ? launch_stream<128, 2>(a, di, stream) : launch_stream<128, 1>(a, di, stream);
  return G > 8 ? launch_stream<64, 2>(a, di, stream) : launch_stream<64, 1>(a, di, stream);
}

}  // namespace hx
