// hx_prefill_attention — causal, paged, multi-token attention on the 5th-generation tensor cores
// ("the prefill phase processes the request's input tokens all at
// once" and is compute-bound, PAPER.md:L110 integrates FlashAttention for it and gives no kernel:
// the design below is ours, for sm_100a).
//
// Roofline: tensor.  Algorithmic flops = 4 * D per (query row, visible kv token) pair (QK^T and PV),
// causal pairs only.  Unlike the decode path this IS a dense contraction: 128 query rows share every
// K/V tile, so it runs on tcgen05.mma with accumulators in TMEM.
//
// A row is a (token, head-of-the-group) pair, so a GQA group of G heads packs 128/G tokens x G heads into one M = 128
// row tile and a K/V tile is read once for all of them.  Per 128-token KV tile (8 pages) and row tile:
//   TMA     K, V pages -> shared [D/64 halves][128 tokens][128 B], 128-byte swizzle
//   UMMA 1  S[128 x 128] = Q K^T           (8 x tcgen05.mma M128 N128 K16, f16 in / f32 in TMEM)
//   softmax tcgen05.ld S; row max; causal + length mask on diagonal tiles only; weights -> fp16 -> tcgen05.st over the
//           first 64 columns of the row's own S; fp32 row sum
//   UMMA 2  O[128 x D] += P V              (P is the TMEM A operand, V the MN-major B operand straight from the page
//           layout; O stays in TMEM for the whole row tile)
//   rescale O and l only when a row max has moved by more than 2^8 since the scale was last set
//           (tcgen05.ld / st; rare): the stale scale cancels in O / l.
// Epilogue: tcgen05.ld O, O / l -> fp16 -> out.  How the steps are arranged in time is the kernel's comment below;
// DESIGN.md 6.4 has the measurements behind it.
#include <cuda.h>
#include <cuda_fp16.h>

#include <cstring>
#include <mutex>

#include "hx_internal.h"

namespace hx {
namespace {

constexpr int kRows = 128;               // query rows per row tile (UMMA M)
constexpr int kKvTile = 128;             // kv tokens per tile (UMMA N of S, K of PV): 8 pages
constexpr int kHalfBytes = kRows * 128;  // Q: one [128 rows][128 B] swizzled region (64 fp16 wide)
constexpr int kKvHalfBytes = kKvTile * 128;      // K or V: one [128 tokens][128 B] region
constexpr float kLog2e = 1.4426950408889634f;

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
// 32 consecutive 32-bit columns of this thread's TMEM lane
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

// ============================================================================================================
// prefill_pp_kernel — the same contraction as prefill_kernel, restructured around what its profile and a per-warp
// timeline showed: per 128 x 128 score tile the tensor pipe needs 1024 cycles (S and P V) and the MUFU
// pipe 1024 (one ex2 per score), so the two must run side by side all the time; two independent CTAs per SM drift
// into the same phase, and every CTA boundary drains the pipe.  Here ONE persistent CTA per SM holds TWO row tiles,
// A and B (consecutive 128-row tiles of the same request and kv head, so they share every K/V tile), and its single
// MMA warp issues   P V_A(j), S_A(j+1), P V_B(j), S_B(j+1), ...   in that fixed order: while the tensor pipe works for
// A, B's softmax runs, and vice versa — anti-phase by construction.  One softmax thread per row (warps 0-3: tile A,
// warps 4-7: tile B; the row's 128 scores stay in registers between the max and the exponentials), so there is no
// exchange between threads.  K and V tiles are double-buffered and loaded once for both row tiles.
// The CTA walks a static list of work items (heavy diagonals first, round-robin over CTAs) WITHOUT draining: both row
// tiles run the same number of kv tiles per item (A's extra tile, if any, is fully masked), so after the last P V_X of
// an item the MMA warp issues S_X(0) of the NEXT item at once (its Q and first K tile were prefetched), and the
// softmax warps find it ready when their epilogue is done.  The epilogue converts O / l to fp16 into a swizzled
// shared-memory tile and ONE TMA tensor store writes it (a row per lane stores 32 lines per instruction otherwise).
// Tensor memory (all 512 columns): S_A | S_B | O_A | O_B, 128 columns each; P overwrites the first 64 of its S.
constexpr int kPpThreads = 352;          // warps 0-3 softmax A, 4-7 softmax B, 8 MMA issuer, 9 TMA loader, 10 TMA storer
constexpr int kPpIssuer = 8, kPpLoader = 9, kPpStorer = 10;
constexpr int kPpBlock = 32;             // (request, kv head) pairs whose row tiles are in flight together
template <int D>
struct PpCfg {
  static constexpr int kHalves = D / 64;
  static constexpr int kQBytes = kHalves * kHalfBytes;       // one Q tile (and one staged output tile), 128 rows x D fp16
  static constexpr int kKvBytes = kHalves * kKvHalfBytes;    // one K or V tile
  static constexpr int kBars = 24;
  static constexpr int kSmem = 3 * kQBytes + 4 * kKvBytes + kBars * 8 + 64;
  static constexpr uint32_t kIdescPV = (1u << 4) | (1u << 16) | ((uint32_t)(D >> 3) << 17) | ((uint32_t)(kRows >> 4) << 24);
};

struct PpRaw { int n, m, cu; };          // what an item needs from global memory (prefetched one item ahead)
struct PpItem {                          // one work item: two row tiles of (request i, kv head g)
  int i, g, n, np, m;
  int nkv;                               // kv tiles of the item (both row tiles run all of them)
  bool act[2], full[2];                  // the row tile exists / lies wholly inside the request's query rows
  int row_tok0[2], pos0[2], r0[2];
  bool any;
};

template <int D>
__global__ void __launch_bounds__(kPpThreads, 1)
prefill_pp_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                  const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmO, const PrefillParams p,
                  int qpairs, long long items) {
  using C = PpCfg<D>;
  constexpr int kHalves = C::kHalves;
  extern __shared__ __align__(1024) uint8_t smem[];
  if ((smem_u32(smem) & 1023u) != 0) __trap();
  uint8_t* sQ = smem;                                  // [2 row tiles]
  uint8_t* sK = smem + 2 * C::kQBytes;                 // [2 buffers]
  uint8_t* sV = sK + 2 * C::kKvBytes;                  // [2 buffers]
  uint8_t* sO = sV + 2 * C::kKvBytes;                  // staged output tile (one, shared by both row tiles)
  uint64_t* bars = reinterpret_cast<uint64_t*>(sO + C::kQBytes);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + C::kBars);
  const uint32_t b0 = smem_u32(bars);
  // mbarriers (all count 1): q_full[2] | q_free[2] | k_full[2] | k_free[2] | v_full[2] | v_free[2] | s_full[2] | o_full[2] | stage_free
  auto BAR = [&](int idx) -> uint32_t { return b0 + 8u * (uint32_t)idx; };
  enum { Q_FULL = 0, Q_FREE = 2, K_FULL = 4, K_FREE = 6, V_FULL = 8, V_FREE = 10, S_FULL = 12, O_FULL = 14, STAGE_FREE = 16 };
  // named barriers: 1 + X = P_X ready (128 softmax threads arrive, the MMA warp syncs), 3 + X = O_X drained by the epilogue
  // (same), 5 + X = output tile of X staged (128 softmax threads arrive, the storer warp syncs)

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int G = p.G, Hkv = p.Hkv;
  const int TQ = kRows / G;
  if (tid == 0) {
    for (int e = 0; e < 17; ++e) mbar_init(BAR(e), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmQ) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmK) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmV) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tmO) : "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  // item k -> (qp, i, g).  The (request, kv head) pairs are taken in blocks of kPpBlock; inside a block late (heavy)
  // row-tile pairs come first, then the block's pairs.  The CTAs of a wave thus work on a few (request, kv head)
  // pairs at a time, whose K/V stay in L2 for all their row tiles (ordering ALL pairs under each row-tile index
  // re-read K/V from DRAM for every index: 3.2 GB instead of 0.7 GB per launch), while the heavy-first order inside a
  // block still deals every CTA a similar sum.  The three global loads of an item are issued one item ahead (load_raw)
  // and only consumed when the item starts (make_item).
  const long long per_qp = (long long)p.B * Hkv;
  const long long per_block = (long long)kPpBlock * qpairs;
  auto item_coords = [&](long long k, int* qp, int* ig) {
    const long long blk = k / per_block;
    const int r = (int)(k - blk * per_block);
    const long long ig0 = blk * kPpBlock;
    const int pb = (int)(per_qp - ig0 < kPpBlock ? per_qp - ig0 : kPpBlock);      // pairs in this block
    *qp = qpairs - 1 - r / pb;
    *ig = (int)ig0 + r % pb;
  };
  auto load_raw = [&](long long k) -> PpRaw {
    PpRaw r = {0, 0, 0};
    if (k >= items) return r;
    int qp, ig;
    item_coords(k, &qp, &ig);
    const int i = ig / Hkv;
    r.n = __ldg(p.lens + i); r.m = __ldg(p.qlens + i); r.cu = __ldg(p.cuq + i);
    return r;
  };
  auto make_item = [&](long long k, const PpRaw& r) -> PpItem {
    PpItem it;
    it.any = false; it.i = it.g = it.n = it.np = it.m = it.nkv = 0;
    it.act[0] = it.act[1] = it.full[0] = it.full[1] = false;
    it.row_tok0[0] = it.row_tok0[1] = 0; it.pos0[0] = it.pos0[1] = 0; it.r0[0] = it.r0[1] = 0;
    if (k >= items) return it;
    int qp, rem;
    item_coords(k, &qp, &rem);
    it.i = rem / Hkv; it.g = rem - it.i * Hkv;
    it.n = max(r.n, 0);
    it.m = min(r.m, it.n);
    it.np = (it.n + 15) >> 4;
#pragma unroll
    for (int x = 0; x < 2; ++x) {
      it.r0[x] = (2 * qp + x) * TQ;
      it.row_tok0[x] = r.cu + it.r0[x];
      it.pos0[x] = it.n - it.m + it.r0[x];
      if (it.r0[x] < it.m) {
        const int pos_last = min(it.pos0[x] + TQ - 1, it.n - 1);
        it.nkv = max(it.nkv, pos_last / kKvTile + 1);
        it.act[x] = true;
        it.full[x] = it.r0[x] + TQ <= it.m;
        it.any = true;
      }
    }
    return it;
  };
  const long long k_step = gridDim.x;
  // the items this CTA walks: (k, it) current; `kn`, `raw_n` the candidate after it (loads already in flight)
  struct Walk { long long k, kn; PpItem it; PpRaw raw_n; bool valid; };
  auto walk_begin = [&]() -> Walk {
    Walk w;
    w.k = blockIdx.x;
    w.it = make_item(w.k, load_raw(w.k));
    while (w.k < items && !w.it.any) { w.k += k_step; w.it = make_item(w.k, load_raw(w.k)); }
    w.valid = w.k < items;
    w.kn = w.k + k_step;
    w.raw_n = load_raw(w.kn);
    return w;
  };
  // the next valid item after w (its loads were issued an item ago in the common case); prefetches the one after
  auto walk_peek = [&](const Walk& w, long long* kn_out, PpRaw* raw_nn) -> PpItem {
    long long kn = w.kn;
    PpItem nx = make_item(kn, w.raw_n);
    while (kn < items && !nx.any) { kn += k_step; nx = make_item(kn, load_raw(kn)); }
    *kn_out = kn;
    *raw_nn = load_raw(kn + k_step);
    return nx;
  };

  if (warp == kPpLoader) {
    // ===================================================== loader warp
    int cq[2] = {0, 0};                   // Q loads issued per row tile
    int ck = 0, cv = 0;                   // K / V tiles issued (buffer = count & 1)
    Walk w = walk_begin();
    while (w.valid) {
      long long kn; PpRaw raw_nn;
      const PpItem nx = walk_peek(w, &kn, &raw_nn);
      const PpItem& it = w.it;
      const int nkv = it.nkv;
      auto load_page = [&](int t) -> int {
        const int pg = t * (kKvTile / 16) + lane;
        return (lane < kKvTile / 16 && t < nkv && pg < it.np) ? __ldg(p.bt + (size_t)it.i * p.bt_stride + pg) : 0;
      };
      int pg_cur = load_page(0), pg_nxt = load_page(1);
#pragma unroll
      for (int x = 0; x < 2; ++x)
        if (it.act[x]) {
          if (lane == 0) {
            if (cq[x] > 0) mbar_wait(BAR(Q_FREE + x), (uint32_t)(cq[x] - 1) & 1);
            mbar_expect_tx(BAR(Q_FULL + x), C::kQBytes);
#pragma unroll
            for (int h = 0; h < kHalves; ++h)
              tma_4d(smem_u32(sQ + x * C::kQBytes + h * kHalfBytes), &tmQ, 0, it.g * G, it.row_tok0[x], h, BAR(Q_FULL + x));
          }
          ++cq[x];
        }
      auto issue_tile = [&](int t, bool is_v, int page) {
        int& cnt = is_v ? cv : ck;
        const int b = cnt & 1;
        const uint32_t full = BAR((is_v ? V_FULL : K_FULL) + b);
        const int npg = min(kKvTile / 16, it.np - t * (kKvTile / 16));
        if (lane == 0) {
          if (cnt >= 2) mbar_wait(BAR((is_v ? V_FREE : K_FREE) + b), (uint32_t)((cnt >> 1) - 1) & 1);
          mbar_expect_tx(full, (uint32_t)(npg * 16 * D * 2));
        }
        __syncwarp();
        if (lane < npg) {
          uint8_t* dstb = (is_v ? sV : sK) + b * C::kKvBytes + lane * 2048;
          const int rw = (int)(p.layer_row0 + (uint32_t)page * (uint32_t)(Hkv * 16) + (uint32_t)(it.g * 16));
#pragma unroll
          for (int h = 0; h < kHalves; ++h) tma_3d(smem_u32(dstb + h * kKvHalfBytes), is_v ? &tmV : &tmK, 0, rw, h, full);
        }
        __syncwarp();
        ++cnt;
      };
      for (int j = 0; j < nkv; ++j) {
        const int pg_nn = load_page(j + 2);
        issue_tile(j, false, pg_cur);
        issue_tile(j, true, pg_cur);
        pg_cur = pg_nxt; pg_nxt = pg_nn;
      }
      w.k = kn; w.it = nx; w.valid = kn < items; w.kn = kn + k_step; w.raw_n = raw_nn;
    }
  } else if (warp == kPpIssuer) {
    // ===================================================== MMA warp (warp-uniform; one elected lane issues)
    const uint32_t tmem_u = __shfl_sync(0xffffffffu, tmem, 0);
    int cq[2] = {0, 0}, ck = 0, cv = 0;   // Q tiles consumed; K / V tile index of the current item's tile 0
    bool had_prev[2] = {false, false};
    // S_X(j) of item `w`: K tile t (running index); commits S_FULL, and frees Q_X / the K buffer when this was their last use
    auto issue_s = [&](int x, int t, bool last_s_of_item, bool last_user) {
      const int b = t & 1;
      mbar_wait(BAR(K_FULL + b), (uint32_t)(t >> 1) & 1);
      tc_fence_after();
      if (elect_one()) {
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
          const uint32_t koff = (uint32_t)(ks & 3) * 32;
          umma_f16(tmem_u + (uint32_t)x * 128,
                   smem_desc(smem_u32(sQ) + (uint32_t)x * C::kQBytes + (uint32_t)(ks >> 2) * kHalfBytes + koff, 16, 1024),
                   smem_desc(smem_u32(sK) + (uint32_t)b * C::kKvBytes + (uint32_t)(ks >> 2) * kKvHalfBytes + koff, 16, 1024), kIdescS, ks > 0);
        }
        umma_commit(BAR(S_FULL + x));
        if (last_s_of_item) umma_commit(BAR(Q_FREE + x));
        if (last_user) umma_commit(BAR(K_FREE + b));
      }
      __syncwarp();
    };
    Walk w = walk_begin();
    if (w.valid) {
#pragma unroll
      for (int x = 0; x < 2; ++x)
        if (w.it.act[x]) {
          mbar_wait(BAR(Q_FULL + x), (uint32_t)cq[x] & 1); ++cq[x];
          issue_s(x, ck, w.it.nkv == 1, x == (w.it.act[1] ? 1 : 0));
        }
    }
    while (w.valid) {
      long long kn; PpRaw raw_nn;
      const PpItem nx = walk_peek(w, &kn, &raw_nn);
      const bool has_next = kn < items;
      const PpItem& it = w.it;
      const int nkv = it.nkv;
      const int last_x = it.act[1] ? 1 : 0;
      for (int j = 0; j < nkv; ++j) {
#pragma unroll
        for (int x = 0; x < 2; ++x) {
          if (!it.act[x]) {
            if (j == nkv - 1 && has_next && nx.act[x]) {       // the row tile sits this item out and comes back in the next
              mbar_wait(BAR(Q_FULL + x), (uint32_t)cq[x] & 1); ++cq[x];
              issue_s(x, ck + nkv, nx.nkv == 1, x == (nx.act[1] ? 1 : 0));
            }
            continue;
          }
          tc_fence_before();
          asm volatile("bar.sync %0, 160;" ::"r"(1 + x) : "memory");           // P_X(j) is in tensor memory
          if (j == 0 && had_prev[x]) asm volatile("bar.sync %0, 160;" ::"r"(3 + x) : "memory");   // previous O_X drained
          const int t = cv + j, b = t & 1;
          mbar_wait(BAR(V_FULL + b), (uint32_t)(t >> 1) & 1);
          tc_fence_after();
          if (elect_one()) {
#pragma unroll
            for (int ks = 0; ks < kKvTile / 16; ++ks)
              umma_f16_ts(tmem_u + 256 + (uint32_t)x * 128, tmem_u + (uint32_t)x * 128 + (uint32_t)ks * 8,
                          smem_desc(smem_u32(sV) + (uint32_t)b * C::kKvBytes + (uint32_t)ks * 2048, kKvHalfBytes, 1024), C::kIdescPV,
                          (j > 0 || ks > 0) ? 1u : 0u);
            umma_commit(BAR(O_FULL + x));
            if (x == last_x) umma_commit(BAR(V_FREE + b));
          }
          __syncwarp();
          if (j + 1 < nkv) {
            issue_s(x, ck + j + 1, j + 1 == nkv - 1, x == last_x);
          } else if (has_next && nx.act[x]) {
            // the item is done for this row tile: S_X(0) of the NEXT item goes out now (no drain between items)
            mbar_wait(BAR(Q_FULL + x), (uint32_t)cq[x] & 1); ++cq[x];
            issue_s(x, ck + nkv, nx.nkv == 1, x == (nx.act[1] ? 1 : 0));
          }
        }
      }
      ck += nkv; cv += nkv;
      had_prev[0] = had_prev[0] || it.act[0];
      had_prev[1] = had_prev[1] || it.act[1];
      w.k = kn; w.it = nx; w.valid = has_next; w.kn = kn + k_step; w.raw_n = raw_nn;
    }
  } else if (warp == kPpStorer) {
    // ===================================================== storer warp: one TMA tensor store per staged output tile.  A
    // bulk-group wait belongs to the thread that issued the copy, so a warp of its own does the waiting and the softmax
    // warps never block on the store.
    Walk w = walk_begin();
    while (w.valid) {
      long long kn; PpRaw raw_nn;
      const PpItem nx = walk_peek(w, &kn, &raw_nn);
      const PpItem& it = w.it;
#pragma unroll
      for (int x = 0; x < 2; ++x)
        if (it.act[x] && it.full[x]) {
          asm volatile("bar.sync %0, 160;" ::"r"(5 + x) : "memory");           // the tile is staged (and fenced for the async proxy)
          if (lane == 0) {
#pragma unroll
            for (int h = 0; h < kHalves; ++h)
              asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
                           ::"l"(&tmO), "r"(smem_u32(sO + h * kHalfBytes)), "r"(0), "r"(it.g * G), "r"(it.row_tok0[x]), "r"(h) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(BAR(STAGE_FREE)) : "memory");
          }
          __syncwarp();
        }
      w.k = kn; w.it = nx; w.valid = kn < items; w.kn = kn + k_step; w.raw_n = raw_nn;
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // the last store has landed
  } else {
    // ===================================================== softmax warps: thread = one row of row tile x
    const int x = warp >> 2;
    const int row = tid & 127;
    const uint32_t lane_sel = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tmem + (uint32_t)x * 128 + lane_sel, tO = tmem + 256 + (uint32_t)x * 128 + lane_sel;
    int cs = 0, co = 0, cv = 0;           // S tiles consumed, P V commits seen so far (this row tile), V tiles (both)
    int nstage = 0;                       // uses of the staged output tile so far (both row tiles)
    Walk w = walk_begin();
    while (w.valid) {
      long long kn; PpRaw raw_nn;
      const PpItem nx = walk_peek(w, &kn, &raw_nn);
      const PpItem& it = w.it;
      const int nkv = it.nkv;
      const int my_stage = nstage + ((x == 1 && it.act[0] && it.full[0]) ? 1 : 0);
      nstage += ((it.act[0] && it.full[0]) ? 1 : 0) + ((it.act[1] && it.full[1]) ? 1 : 0);
      if (it.act[x]) {
        const int my_pos = min(it.pos0[x] + row / G, it.n - 1);
        float m_used = -INFINITY, l_run = 0.f;
        for (int j = 0; j < nkv; ++j) {
          const int t0 = j * kKvTile;
          mbar_wait(BAR(S_FULL + x), (uint32_t)cs & 1);
          ++cs;
          tc_fence_after();
          // Two passes over the row's 128 scores, 32 at a time, both straight from tensor memory (a second read costs far
          // less than holding the row in registers: the step's code stays small enough for the instruction cache and
          // nothing spills).  Pass 1: the row max.
          const bool need_mask = (t0 + kKvTile - 1 > it.pos0[x]);
          float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll 1
          for (int c = 0; c < 4; c += 2) {
            uint32_t s0[32], s1[32];
            tmem_ld32_issue(tS + c * 32, s0);
            tmem_ld32_issue(tS + c * 32 + 32, s1);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (need_mask) {
#pragma unroll
              for (int e = 0; e < 32; ++e) {
                if (t0 + c * 32 + e > my_pos) s0[e] = 0xff800000u;              // -inf
                if (t0 + c * 32 + 32 + e > my_pos) s1[e] = 0xff800000u;
              }
            }
#pragma unroll
            for (int e = 0; e < 32; e += 2) {
              mx4[(e >> 1) & 1] = max3(mx4[(e >> 1) & 1], __uint_as_float(s0[e]), __uint_as_float(s0[e + 1]));
              mx4[2 + ((e >> 1) & 1)] = max3(mx4[2 + ((e >> 1) & 1)], __uint_as_float(s1[e]), __uint_as_float(s1[e + 1]));
            }
          }
          const float m_tile = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * p.scale_log2;
          if (j == 0) {
            m_used = m_tile;                                         // finite: token 0 is visible to every row
          } else {
            const bool move = m_tile > m_used + 8.f;                 // (a fully masked tile has m_tile = -inf: never)
            if (__any_sync(0xffffffffu, move)) {                     // rare after the first tiles
              mbar_wait(BAR(O_FULL + x), (uint32_t)(co + j - 1) & 1);   // only the rescale touches O: P V(j-1) must be done
              tc_fence_after();
              const float corr = move ? ex2(m_used - m_tile) : 1.f;
              if (move) m_used = m_tile;
              l_run *= corr;
#pragma unroll 1
              for (int c = 0; c < D / 32; ++c) {
                uint32_t r[32];
                tmem_ld32_issue(tO + c * 32, r);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int e = 0; e < 32; ++e) r[e] = __float_as_uint(__uint_as_float(r[e]) * corr);
                tmem_st32(tO + c * 32, r);
              }
            }
          }
          // Pass 2: weights -> fp16 -> P over the first 64 columns of this row's S (the TMEM A operand of P V).  Chunk c's
          // 16 packed columns land on columns [16c, 16c + 16), all of which lie in score chunks <= c, already read.
          unsigned long long rs2[2] = {0ull, 0ull};           // two packed pairs of fp32 partial row sums
#pragma unroll 1
          for (int c = 0; c < 4; ++c) {
            uint32_t sc[32];
            tmem_ld32_issue(tS + c * 32, sc);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (need_mask) {
#pragma unroll
              for (int e = 0; e < 32; ++e)
                if (t0 + c * 32 + e > my_pos) sc[e] = 0xff800000u;              // -inf -> weight 0
            }
            // Packed fp32 arithmetic (fma.rn.f32x2 / add.f32x2: two scores per instruction) for the scale-and-subtract and the
            // row sum: the warp scheduler, not a pipe, is what this loop saturates, so instructions are what to save.
            uint32_t pk[16];
            unsigned long long sc2, nm2, t2[16];
            asm("mov.b64 %0, {%1, %1};" : "=l"(sc2) : "f"(p.scale_log2));
            asm("mov.b64 %0, {%1, %1};" : "=l"(nm2) : "f"(-m_used));
#pragma unroll
            for (int i = 0; i < 16; ++i) {
              unsigned long long s2;
              asm("mov.b64 %0, {%1, %2};" : "=l"(s2) : "r"(sc[2 * i]), "r"(sc[2 * i + 1]));
              asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(t2[i]) : "l"(s2), "l"(sc2), "l"(nm2));
            }
#pragma unroll
            for (int i = 0; i < 16; ++i) {
              float ta, tb, wa, wb;
              asm("mov.b64 {%0, %1}, %2;" : "=f"(ta), "=f"(tb) : "l"(t2[i]));
              asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(wa) : "f"(ta));
              asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(wb) : "f"(tb));
              asm volatile("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(pk[i]) : "f"(wb), "f"(wa));
              unsigned long long w2;
              asm("mov.b64 %0, {%1, %2};" : "=l"(w2) : "f"(wa), "f"(wb));
              asm volatile("add.f32x2 %0, %0, %1;" : "+l"(rs2[i & 1]) : "l"(w2));
            }
            tmem_st16(tS + c * 16, pk);
          }
          asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
          {
            float r0, r1, r2, r3;
            asm("mov.b64 {%0, %1}, %2;" : "=f"(r0), "=f"(r1) : "l"(rs2[0]));
            asm("mov.b64 {%0, %1}, %2;" : "=f"(r2), "=f"(r3) : "l"(rs2[1]));
            l_run += (r0 + r1) + (r2 + r3);
          }
          if (t0 + kKvTile > it.n) {
            // V rows of slots past the context end / of pages that were not loaded must be zero (0 * Inf = NaN in P V;
            // reading S10).  Both row tiles' warps write the same zeros; each does so before ITS barrier arrival.
            const int t = cv + j, b = t & 1;
            mbar_wait(BAR(V_FULL + b), (uint32_t)(t >> 1) & 1);
            for (int e = row; e < (t0 + kKvTile - it.n) * (D / 8); e += 128) {
              const int r = (it.n - t0) + e / (D / 8), ch = e % (D / 8);
              *reinterpret_cast<int4*>(sV + b * C::kKvBytes + (ch >> 3) * kKvHalfBytes + r * 128 + (((ch & 7) ^ (r & 7)) << 4)) = make_int4(0, 0, 0, 0);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          }
          tc_fence_before();
          asm volatile("bar.arrive %0, 160;" ::"r"(1 + x) : "memory");
        }
        // ---- epilogue of this row tile: O / l -> fp16 -> out
        mbar_wait(BAR(O_FULL + x), (uint32_t)(co + nkv - 1) & 1);
        co += nkv;
        tc_fence_after();
        const float inv = 1.f / l_run;
        if (it.full[x]) {
          // through the staged tile: [half][row][128 B] with the 128-byte swizzle (the layout Q arrives in), one TMA store
          if (my_stage > 0) mbar_wait(BAR(STAGE_FREE), (uint32_t)(my_stage - 1) & 1);
#pragma unroll 1
          for (int c = 0; c < D / 32; ++c) {
            uint32_t r[32];
            tmem_ld32_issue(tO + c * 32, r);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int e = 0; e < 32; e += 8) {
              __half2 h[4];
#pragma unroll
              for (int u = 0; u < 4; ++u)
                h[u] = __floats2half2_rn(__uint_as_float(r[e + 2 * u]) * inv, __uint_as_float(r[e + 2 * u + 1]) * inv);
              const int ch = c * 4 + (e >> 3);                       // 16-byte chunk of the row
              *reinterpret_cast<int4*>(sO + (ch >> 3) * kHalfBytes + row * 128 + (((ch & 7) ^ (row & 7)) << 4)) = *reinterpret_cast<const int4*>(h);
            }
          }
          tc_fence_before();
          asm volatile("bar.arrive %0, 160;" ::"r"(3 + x) : "memory");           // O_X may be overwritten
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          asm volatile("bar.arrive %0, 160;" ::"r"(5 + x) : "memory");          // the storer warp takes it from here
        } else {
          // the request's last (partial) row tile: rows past its query rows must not be written; a row per lane
          const bool store = it.r0[x] + row / G < it.m;
          __half* dst = p.out + ((size_t)(it.row_tok0[x] + row / G) * p.Hq + (size_t)(it.g * G + row % G)) * D;
#pragma unroll 1
          for (int c = 0; c < D / 32; ++c) {
            uint32_t r[32];
            tmem_ld32_issue(tO + c * 32, r);
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
          tc_fence_before();
          asm volatile("bar.arrive %0, 160;" ::"r"(3 + x) : "memory");           // O_X may be overwritten
        }
      }
      cv += nkv;
      w.k = kn; w.it = nx; w.valid = kn < items; w.kn = kn + k_step; w.raw_n = raw_nn;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
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
  constexpr int kSmem = PpCfg<D>::kSmem;
  DeviceInfo di;
  int rc = device_info(&di);
  if (rc) return rc;
  {
    static std::mutex mu;
    static bool attr_set[64] = {false};
    std::lock_guard<std::mutex> lock(mu);
    if (!attr_set[di.device]) {
      if (kSmem > di.max_smem_optin) HX_FAIL(HX_ERR_UNSUPPORTED, "device offers %d B shared memory per CTA, kernel needs %d", di.max_smem_optin, kSmem);
      HX_CUDA_OK(cudaFuncSetAttribute(prefill_pp_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
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
  CUtensorMap tq, to, tk, tv;
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
    // q and out as [64][Hq heads][Tq tokens][D/64 halves]; box {64, G, 128/G, 1} is [token][head][128 B]:
    // row = token * G + head, the M order of a row tile.  q tokens past the end read as zeros; out is only stored
    // through its map for row tiles that lie wholly inside a request.
    cuuint64_t dims[4] = {64, (cuuint64_t)a.q_heads, (cuuint64_t)a.total_q, (cuuint64_t)(D / 64)};
    cuuint64_t strides[3] = {(cuuint64_t)D * 2, (cuuint64_t)a.q_heads * D * 2, 128};
    cuuint32_t box[4] = {64, (cuuint32_t)G, (cuuint32_t)(kRows / G), 1};
    cuuint32_t es[4] = {1, 1, 1, 1};
    for (int x = 0; x < 2; ++x) {
      CUresult r = enc(x ? &to : &tq, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 4, x ? a.out : const_cast<void*>(a.q), dims, strides, box, es,
                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                       CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (r != CUDA_SUCCESS) HX_FAIL(HX_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d) for %s", (int)r, x ? "out" : "q");
    }
  }
  PrefillParams p;
  p.out = static_cast<__half*>(a.out);
  p.bt = a.block_table; p.lens = a.seq_lens; p.qlens = a.q_lens; p.cuq = a.cu_q_lens;
  p.B = a.batch; p.Hq = a.q_heads; p.Hkv = a.kv_heads; p.G = G; p.bt_stride = a.bt_stride;
  p.layer_row0 = (uint32_t)(rows_per_layer * a.layer);
  p.scale_log2 = a.sm_scale * kLog2e;
  const int TQ = kRows / G;
  const int qtiles = (a.max_q_len + TQ - 1) / TQ;
  const int qpairs = (qtiles + 1) / 2;
  const long long items = (long long)qpairs * a.batch * a.kv_heads;      // (row-tile pair, request, kv head)
  const int grid = (int)(items < di.sm_count ? items : di.sm_count);
  prefill_pp_kernel<D><<<grid, kPpThreads, kSmem, stream>>>(tq, tk, tv, to, p, qpairs, items);
  HX_CUDA_OK(cudaGetLastError());
  return HX_OK;
}

int launch_prefill(const PrefillArgs& a, cudaStream_t stream) {
  return a.head_dim == 128 ? launch_prefill_d<128>(a, stream) : launch_prefill_d<64>(a, stream);
}

}  // namespace hx
