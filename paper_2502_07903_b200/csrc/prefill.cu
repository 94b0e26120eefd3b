// hx_prefill_attention — causal, paged, multi-token attention on the 5th-generation tensor cores
// ("the prefill phase processes the request's input tokens all at
// once" and is compute-bound, PAPER.md:L110 integrates FlashAttention for it and gives no kernel:
// the design below is ours, for sm_100a).
//
// Roofline: tensor.  Algorithmic flops = 4 * D per (query row, visible kv token) pair (QK^T and PV),
// causal pairs only.  Unlike the decode path this IS a dense contraction: 128 query rows share every
// K/V tile, so it runs on tcgen05.mma with accumulators in TMEM.
//
// One CTA = one (request, kv head, tile of 128 query rows); a row is a (token, head-of-the-group)
// pair, so a GQA group of G heads packs 128/G tokens x G heads into one M = 128 tile and the K/V tile
// is read once for all of them.  Two CTAs share an SM (97 KiB of shared memory and 256 TMEM columns
// each): while one CTA's softmax runs, the tensor pipe works for the other.  Roles: 8 softmax warps
// (two threads per row), one MMA warp (warp-uniform code, one elected lane issues), one TMA loader warp.
// Per 128-token KV tile (8 pages):
//   TMA     K, V pages -> shared [D/64 halves][128 tokens][128 B], 128-byte swizzle; one K and one V tile,
//           each reloaded as soon as the MMAs that read it are done (a whole softmax before its next use)
//   UMMA 1  S[128 x 128] = Q K^T           (8 x tcgen05.mma M128 N128 K16, f16 in / f32 in TMEM cols 0..127)
//   softmax tcgen05.ld S; both threads of a row scan all 128 scores for the max (no exchange), then each
//           turns its 64 scores into weights: causal + length mask on diagonal tiles only, fp32 row sum of
//           the rounded weights, P -> fp16 -> tcgen05.st over the thread's OWN first 32 score columns
//   UMMA 2  O[128 x D] += P V              (P is the TMEM A operand, V the MN-major B operand straight from
//           the page layout; O stays in TMEM cols 128..255 for the whole CTA), then S of the next tile
//           over the same columns (the pipe runs in issue order)
//   rescale O and l only when a row max has moved by more than 2^8 since the scale was last set
//           (tcgen05.ld / st; rare): the stale scale cancels in O / l.
// Epilogue: tcgen05.ld O, O / l -> fp16 -> out.  The measured fraction of the tensor peak is reported by
// bench.py as it stands; DESIGN.md 6.4 has the history and what bounds it.
#include <cuda.h>
#include <cuda_fp16.h>

#include <cstring>
#include <mutex>

#include "hx_internal.h"

namespace hx {
namespace {

constexpr int kRows = 128;               // query rows per CTA (UMMA M)
constexpr int kKvTile = 128;             // kv tokens per tile (UMMA N of S, K of PV): 8 pages
constexpr int kHalfBytes = kRows * 128;  // Q: one [128 rows][128 B] swizzled region (64 fp16 wide)
constexpr int kKvHalfBytes = kKvTile * 128;      // K or V: one [128 tokens][128 B] region
// Sizes that depend on head_dim D (64 or 128): operands are stored as D/64 regions of [128 rows][128 B].
template <int D>
struct PfCfg {
  static constexpr int kHalves = D / 64;
  static constexpr int kQBytes = kHalves * kHalfBytes;       // Q tile, 128 rows x D fp16
  static constexpr int kKvBytes = kHalves * kKvHalfBytes;    // a K or V tile, 128 tokens x D fp16
  // Q + K + V tiles (96 KiB at D = 128) + the row-sum exchange + 5 mbarriers, the TMEM address: two CTAs per SM
  static constexpr int kSmem = kQBytes + 2 * kKvBytes + 1024 + 64;
  // UMMA instruction descriptor of O += P V: N = D, B operand MN-major
  static constexpr uint32_t kIdescPV = (1u << 4) | (1u << 16) | ((uint32_t)(D >> 3) << 17) | ((uint32_t)(kRows >> 4) << 24);
};
constexpr float kLog2e = 1.4426950408889634f;
constexpr int kIssuer = 8;               // warps 0..7: softmax (two threads per row); warp 8 issues tcgen05.mma, warp 9 TMA
constexpr int kLoader = 9;

struct PrefillParams {
  __half* out;
  const int32_t* bt;
  const int32_t* lens;
  const int32_t* qlens;
  const int32_t* cuq;
  int32_t B, Hq, Hkv, G, bt_stride;
  uint32_t layer_row0;
  float scale_log2;
};

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
__device__ __forceinline__ void tma_3d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_4d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
      ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ float max3(float a, float b, float c) {     // one FMNMX3 (sm_100)
  float r;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
  return r;
}

// ---- tcgen05 wrappers
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void umma_f16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// A operand from TMEM (128 lanes = rows, two fp16 per 32-bit column along K), B from shared memory
__device__ __forceinline__ void umma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {   // no wait
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
        "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
}
// Warp-uniform issue: every lane of the MMA warp executes these with identical operands and ONE elected
// lane issues.  With uniform control flow ptxas keeps the descriptors in uniform registers; under an
// `if (lane == 0)` it cannot prove uniformity and emits a waterfall loop (ELECT / R2UR.BROADCAST / BRA)
// of a dozen instructions around every UTCHMMA.
__device__ __forceinline__ uint32_t elect_one() {     // 1 in exactly one lane of a converged warp
  uint32_t pred;
  asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
  return pred;
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// 32 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int e = 0; e < 32; ++e) v[e] = __uint_as_float(r[e]);
}

__device__ __forceinline__ void tmem_ld32_issue(uint32_t taddr, uint32_t (&r)[32]) {   // no wait
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32]) {   // no wait
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
        "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]),
        "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]),
        "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]) : "memory");
}
// Shared-memory matrix descriptor (cute::UMMA::SmemDescriptor bit layout): start address >> 4 in
// [0,14), leading byte offset >> 4 in [16,30), stride byte offset >> 4 in [32,46), version 1 in
// [46,48), layout type in [61,64) (2 = 128-byte swizzle).
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((addr >> 4) & 0x3fff) | ((uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16) |
         ((uint64_t)((sbo_bytes >> 4) & 0x3fff) << 32) | (1ull << 46) | (2ull << 61);
}
// Instruction descriptor (cute::UMMA::InstrDescriptor): c_format f32 (1 << 4), a/b format f16 (0),
// a_major bit 15, b_major bit 16 (1 = MN-major), N >> 3 in [17,23), M >> 4 in [24,29).
constexpr uint32_t kIdescS = (1u << 4) | ((uint32_t)(kKvTile >> 3) << 17) | ((uint32_t)(kRows >> 4) << 24);

template <int D>
__global__ void __launch_bounds__(320, 2)
prefill_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
               const __grid_constant__ CUtensorMap tmV, const PrefillParams p) {
  using C = PfCfg<D>;
  constexpr int kHalves = C::kHalves;
  extern __shared__ __align__(1024) uint8_t smem[];
  if ((smem_u32(smem) & 1023u) != 0) __trap();   // the 128-byte swizzle needs 1 KiB-aligned regions
  uint8_t* sQ = smem;
  uint8_t* sK = smem + C::kQBytes;                // one K tile and one V tile: each is reloaded as soon as the
  uint8_t* sV = sK + C::kKvBytes;                 // MMAs that read it are done, a whole softmax before its next use
  float* lsum = reinterpret_cast<float*>(sV + C::kKvBytes);         // [2 column halves][128 rows] row sums (epilogue)
  uint64_t* bars = reinterpret_cast<uint64_t*>(lsum + 256);      // q, k, v, s, o
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 5);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int G = p.G, Hkv = p.Hkv;
  const int TQ = kRows / G;                          // query tokens per tile
  const int i = blockIdx.z, g = blockIdx.y;
  const int n = max(__ldg(p.lens + i), 0);
  const int m = min(__ldg(p.qlens + i), n);          // (q_lens > seq_lens breaks the contract: clamped, never a hang)
  const int qt = (int)gridDim.x - 1 - (int)blockIdx.x;   // heavy (late) tiles first
  if (qt * TQ >= m) return;
  const int r0 = qt * TQ;                            // first query token of the tile (within the request's m)
  const int row_tok0 = __ldg(p.cuq + i) + r0;        // its packed row in q / out
  const int pos0 = n - m + r0;                       // its position in the context
  const int pos_last = min(pos0 + TQ - 1, n - 1);
  const int nkv = pos_last / kKvTile + 1;            // causal: kv tiles 0..nkv-1
  const int np = (n + 15) >> 4;

  const uint32_t bar_q = smem_u32(bars), bar_k = bar_q + 8, bar_v = bar_q + 16, bar_s = bar_q + 24, bar_o = bar_q + 32;
  if (tid == 0) {
    for (int e = 0; e < 5; ++e) mbar_init(bar_q + 8 * e, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmQ) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmK) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmV) : "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"(smem_u32(tmem_slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t tS = tmem, tO = tmem + 128;       // S (and P over its first 64 columns) | O
  // 8 softmax warps: warp w and warp w + 4 share TMEM lanes 32 (w & 3) .. +31 (= rows) and split the columns
  const int row = tid & 127, ch_half = warp >> 2;
  const uint32_t lane_sel = (uint32_t)((warp & 3) * 32) << 16;

  float m_used = -INFINITY, l_run = 0.f;             // softmax threads' row state (see below)

  if (warp == kLoader) {
    // ===== loader warp: lane l < 8 owns page l of a 128-token tile; its block-table entry is fetched one
    // tile ahead.  K_{j+1} goes out when S_j is done, V_{j+1} when P V_j is done.
    auto load_page = [&](int t) -> int {
      const int pg = t * (kKvTile / 16) + lane;
      return (lane < kKvTile / 16 && t < nkv && pg < np) ? __ldg(p.bt + (size_t)i * p.bt_stride + pg) : 0;
    };
    auto issue_tile = [&](int t, bool is_v, int page) {
      const uint32_t bar = is_v ? bar_v : bar_k;
      const int npg = min(kKvTile / 16, np - t * (kKvTile / 16));
      if (lane == 0) mbar_expect_tx(bar, (uint32_t)(npg * 16 * D * 2));
      if (lane < npg) {
        uint8_t* dstb = (is_v ? sV : sK) + lane * 2048;
        const int rw = (int)(p.layer_row0 + (uint32_t)page * (uint32_t)(Hkv * 16) + (uint32_t)(g * 16));
#pragma unroll
        for (int h = 0; h < kHalves; ++h) tma_3d(smem_u32(dstb + h * kKvHalfBytes), is_v ? &tmV : &tmK, 0, rw, h, bar);
      }
      __syncwarp();
    };
    int pg_cur = load_page(0), pg_nxt = load_page(1);
    if (lane == 0) {
      mbar_expect_tx(bar_q, C::kQBytes);
#pragma unroll
      for (int h = 0; h < kHalves; ++h) tma_4d(smem_u32(sQ + h * kHalfBytes), &tmQ, 0, g * G, row_tok0, h, bar_q);
    }
    issue_tile(0, false, pg_cur);
    issue_tile(0, true, pg_cur);
    for (int j = 0; j + 1 < nkv; ++j) {
      const int pg_nn = load_page(j + 2);
      if (lane == 0) mbar_wait(bar_s, (uint32_t)j & 1);         // S_j done: the K tile is free
      __syncwarp();
      issue_tile(j + 1, false, pg_nxt);
      if (lane == 0) mbar_wait(bar_o, (uint32_t)j & 1);         // P V_j done: the V tile is free
      __syncwarp();
      issue_tile(j + 1, true, pg_nxt);
      pg_cur = pg_nxt; pg_nxt = pg_nn;
    }
  } else if (warp == kIssuer) {
    // ===== MMA warp (warp-uniform; one elected lane issues).  Per tile: P V_j after the step barrier, then
    // S_{j+1} over the same TMEM columns (the pipe runs in issue order, so P_j is read before it is
    // overwritten).  The other CTA of the SM keeps the pipe fed while this CTA's softmax runs.
    const uint32_t tmem_u = __shfl_sync(0xffffffffu, tmem, 0);  // the same value, provably warp-uniform
    auto issue_s = [&]() {
      tc_fence_after();
      if (elect_one()) {
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
          const uint32_t koff = (uint32_t)(ks & 3) * 32;
          umma_f16(tmem_u, smem_desc(smem_u32(sQ) + (uint32_t)(ks >> 2) * kHalfBytes + koff, 16, 1024),
                   smem_desc(smem_u32(sK) + (uint32_t)(ks >> 2) * kKvHalfBytes + koff, 16, 1024), kIdescS, ks > 0);
        }
        umma_commit(bar_s);
      }
      __syncwarp();
    };
    mbar_wait(bar_q, 0);
    mbar_wait(bar_k, 0);
    issue_s();
    for (int j = 0; j < nkv; ++j) {
      tc_fence_before();
      asm volatile("bar.sync 5, 288;" ::: "memory");             // P_j is in TMEM, V_j landed and its tail is cleared
      tc_fence_after();
      if (elect_one()) {
#pragma unroll
        for (int ks = 0; ks < kKvTile / 16; ++ks)
          umma_f16_ts(tmem_u + 128, tmem_u + (ks < 4 ? ks * 8 : 64 + (ks - 4) * 8), smem_desc(smem_u32(sV) + (uint32_t)ks * 2048, kKvHalfBytes, 1024), C::kIdescPV,
                      (j > 0 || ks > 0) ? 1u : 0u);
        umma_commit(bar_o);
      }
      __syncwarp();
      if (j + 1 < nkv) {
        mbar_wait(bar_k, (uint32_t)(j + 1) & 1);
        issue_s();
      }
    }
  } else {
    // ===== softmax warps: thread (row, ch_half) owns 64 of the row's 128 scores, handled 32 at a time.
    // O lives in TMEM (columns 128..255) across all tiles at the scale m_used, a STALE row max that is
    // moved (and O, l rescaled) only when the true max has run ahead of it by more than 2^8: the weights
    // 2^(s - m_used) then stay <= 256, exact in fp16's relative precision, and the result is the same
    // softmax average (the factor cancels in O / l).
    const int my_pos = min(pos0 + row / G, n - 1);     // rows past the request's last query are never stored
    for (int j = 0; j < nkv; ++j) {
      const int t0 = j * kKvTile;
      mbar_wait(bar_s, (uint32_t)j & 1);
      tc_fence_after();
      const bool need_mask = (t0 + kKvTile - 1 > pos0);          // some (row, token) of this tile is masked
      const int tk0 = t0 + ch_half * 64;                          // first kv token of this thread's columns
      // ---- pass 1: row max on the raw scores (the scale is positive).  Both threads of a row scan all
      // 128 scores (TMEM loads are cheap) instead of exchanging half-row maxima: no barrier, and both get
      // bit-identical scales.
      float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        float s[32];
        tmem_ld32(tS + c * 32 + lane_sel, s);
        if (need_mask) {
#pragma unroll
          for (int e = 0; e < 32; ++e) mx4[e & 3] = fmaxf(mx4[e & 3], (t0 + c * 32 + e <= my_pos) ? s[e] : -INFINITY);
        } else {
#pragma unroll
          for (int e = 0; e < 32; e += 2) mx4[(e >> 1) & 3] = max3(mx4[(e >> 1) & 3], s[e], s[e + 1]);
        }
      }
      const float m_tile = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * p.scale_log2;
      if (j == 0) {
        m_used = m_tile;                                         // finite: token 0 is visible to every row
      } else {
        const bool move = m_tile > m_used + 8.f;
        if (__any_sync(0xffffffffu, move)) {                      // rare after the first tiles
          mbar_wait(bar_o, (uint32_t)(j - 1) & 1);                // only the rescale touches O: P V_{j-1} must be done
          tc_fence_after();
          const float corr = move ? ex2(m_used - m_tile) : 1.f;
          if (move) m_used = m_tile;
          l_run *= corr;
#pragma unroll 1
          for (int c = 0; c < D / 64; ++c) {                      // this half's D/2 columns of O
            uint32_t r[32];
            tmem_ld32_issue(tO + lane_sel + ch_half * (D / 2) + c * 32, r);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int e = 0; e < 32; ++e) r[e] = __float_as_uint(__uint_as_float(r[e]) * corr);
            tmem_st32(tO + lane_sel + ch_half * (D / 2) + c * 32, r);
          }
        }
      }
      // ---- pass 2: weights -> fp16 -> P, 32 scores at a time.  A thread's P (32 packed columns) overwrites
      // the first half of ITS OWN 64 score columns, chunk by chunk after the chunk is in registers, so no
      // thread ever waits for another: P sits at columns [0,32) (tokens 0..63) and [64,96) (tokens 64..127),
      // and the MMA warp points each K = 16 step's A operand there.
      // (Pass 1 of the row's other thread reads these columns too: see the barrier note below.)
      float rs4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        float s[32];
        tmem_ld32(tS + ch_half * 64 + c * 32 + lane_sel, s);
        uint32_t pk[16];
#pragma unroll
        for (int e = 0; e < 32; e += 2) {
          float w0 = ex2(fmaf(s[e], p.scale_log2, -m_used)), w1 = ex2(fmaf(s[e + 1], p.scale_log2, -m_used));
          if (need_mask) {
            w0 = (tk0 + c * 32 + e <= my_pos) ? w0 : 0.f;
            w1 = (tk0 + c * 32 + e + 1 <= my_pos) ? w1 : 0.f;
          }
          const __half2 h2 = __floats2half2_rn(w0, w1);
          rs4[(e >> 1) & 3] += __low2float(h2) + __high2float(h2);  // the ROUNDED weights (reading S22)
          pk[e >> 1] = *reinterpret_cast<const uint32_t*>(&h2);
        }
        if (c == 0) asm volatile("bar.sync %0, 64;" ::"r"(1 + (warp & 3)) : "memory");   // the row's other thread has finished pass 1
        tmem_st16(tS + ch_half * 64 + c * 16 + lane_sel, pk);       // P_j: the TMEM A operand of P V_j
      }
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
      l_run += (rs4[0] + rs4[1]) + (rs4[2] + rs4[3]);
      // ---- V_j must have landed; clear what the MMA must not see (0 * Inf = NaN in P V): V rows of
      // slots past the context end and of pages that were not loaded (reading S10)
      mbar_wait(bar_v, (uint32_t)j & 1);
      if (t0 + kKvTile > n) {
        for (int e = tid; e < (t0 + kKvTile - n) * (D / 8); e += 256) {
          const int r = (n - t0) + e / (D / 8), ch = e % (D / 8);
          *reinterpret_cast<int4*>(sV + (ch >> 3) * kKvHalfBytes + r * 128 + (((ch & 7) ^ (r & 7)) << 4)) = make_int4(0, 0, 0, 0);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      }
      tc_fence_before();
      asm volatile("bar.sync 5, 288;" ::: "memory");
    }
  }
  mbar_wait(bar_o, (uint32_t)(nkv - 1) & 1);
  tc_fence_after();

  // ---- epilogue: thread (row, ch_half) -> D/2 columns of out[row_tok0 + row / G][g*G + row % G][:];
  // the two halves' row sums meet in shared memory
  {
    if (warp < kIssuer) lsum[ch_half * 128 + row] = l_run;
    __syncthreads();
    const float inv = 1.f / (lsum[row] + lsum[128 + row]);
    const bool store = warp < kIssuer && r0 + row / G < m;
    __half* dst = p.out + ((size_t)(row_tok0 + row / G) * p.Hq + (size_t)(g * G + row % G)) * D + ch_half * (D / 2);
#pragma unroll 1
    for (int c = 0; c < D / 64 && warp < kIssuer; ++c) {
      uint32_t r[32];
      tmem_ld32_issue(tO + lane_sel + ch_half * (D / 2) + c * 32, r);
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      if (store) {
#pragma unroll
        for (int e = 0; e < 32; e += 8) {
          __half2 h[4];
#pragma unroll
          for (int u = 0; u < 4; ++u)
            h[u] = __floats2half2_rn(__uint_as_float(r[e + 2 * u]) * inv, __uint_as_float(r[e + 2 * u + 1]) * inv);
          *reinterpret_cast<int4*>(dst + c * 32 + e) = *reinterpret_cast<const int4*>(h);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tmem) : "memory");
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int encode_fn(EncodeTiledFn* out) {
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

}  // namespace

template <int D>
static int launch_prefill_d(const PrefillArgs& a, cudaStream_t stream) {
  constexpr int kSmem = PfCfg<D>::kSmem;
  DeviceInfo di;
  int rc = device_info(&di);
  if (rc) return rc;
  {
    static std::mutex mu;
    static bool attr_set[64] = {false};
    std::lock_guard<std::mutex> lock(mu);
    if (!attr_set[di.device]) {
      if (kSmem > di.max_smem_optin) HX_FAIL(HX_ERR_UNSUPPORTED, "device offers %d B shared memory per CTA, kernel needs %d", di.max_smem_optin, kSmem);
      HX_CUDA_OK(cudaFuncSetAttribute(prefill_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
      attr_set[di.device] = true;
    }
  }
  EncodeTiledFn enc;
  rc = encode_fn(&enc);
  if (rc) return rc;
  const int G = a.q_heads / a.kv_heads;
  const uint64_t rows_per_layer = (uint64_t)a.num_pages * a.kv_heads * 16;
  const uint64_t rows = rows_per_layer * a.layers;
  if (rows >= (1ull << 31)) HX_FAIL(HX_ERR_UNSUPPORTED, "cache too large for one tensor map (%llu rows)", (unsigned long long)rows);
  CUtensorMap tq, tk, tv;
  {
    // K / V cache as [D/64 halves][rows][64]; box = one 64-wide half of one (page, head) tile
    cuuint64_t dims[3] = {64, rows, (cuuint64_t)(D / 64)};
    cuuint64_t strides[2] = {(cuuint64_t)D * 2, 128};
    cuuint32_t box[3] = {64, 16, 1};
    cuuint32_t es[3] = {1, 1, 1};
    for (int x = 0; x < 2; ++x) {
      CUresult r = enc(x ? &tv : &tk, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void*>(x ? a.v_base : a.k_base), dims,
                       strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                       CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (r != CUDA_SUCCESS) HX_FAIL(HX_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d) for the K/V cache", (int)r);
    }
  }
  {
    // Q as [64][Hq heads][Tq tokens][D/64 halves]; box {64, G, 128/G, 1} lands as [token][head][128 B]:
    // row = token * G + head, the M order of the tile.  Tokens past the end read as zeros.
    cuuint64_t dims[4] = {64, (cuuint64_t)a.q_heads, (cuuint64_t)a.total_q, (cuuint64_t)(D / 64)};
    cuuint64_t strides[3] = {(cuuint64_t)D * 2, (cuuint64_t)a.q_heads * D * 2, 128};
    cuuint32_t box[4] = {64, (cuuint32_t)G, (cuuint32_t)(kRows / G), 1};
    cuuint32_t es[4] = {1, 1, 1, 1};
    CUresult r = enc(&tq, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 4, const_cast<void*>(a.q), dims, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) HX_FAIL(HX_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d) for q", (int)r);
  }
  PrefillParams p;
  p.out = static_cast<__half*>(a.out);
  p.bt = a.block_table; p.lens = a.seq_lens; p.qlens = a.q_lens; p.cuq = a.cu_q_lens;
  p.B = a.batch; p.Hq = a.q_heads; p.Hkv = a.kv_heads; p.G = G; p.bt_stride = a.bt_stride;
  p.layer_row0 = (uint32_t)(rows_per_layer * a.layer);
  p.scale_log2 = a.sm_scale * kLog2e;
  const int TQ = kRows / G;
  const int qtiles = (a.max_q_len + TQ - 1) / TQ;
  for (int b0 = 0; b0 < a.batch; b0 += 65535) {
    PrefillParams pb = p;
    pb.B = (a.batch - b0 < 65535) ? a.batch - b0 : 65535;
    pb.bt = a.block_table + (size_t)b0 * a.bt_stride;
    pb.lens = a.seq_lens + b0; pb.qlens = a.q_lens + b0; pb.cuq = a.cu_q_lens + b0;
    prefill_kernel<D><<<dim3(qtiles, a.kv_heads, pb.B), 320, kSmem, stream>>>(tq, tk, tv, pb);
    HX_CUDA_OK(cudaGetLastError());
  }
  return HX_OK;
}

int launch_prefill(const PrefillArgs& a, cudaStream_t stream) {
  return a.head_dim == 128 ? launch_prefill_d<128>(a, stream) : launch_prefill_d<64>(a, stream);
}

}  // namespace hx
