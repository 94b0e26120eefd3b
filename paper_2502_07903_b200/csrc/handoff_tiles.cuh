// The KV handoff as a TILE MOVER (SURVEY.md §8(a) rows A2 + A3): the same bit copy as the rows
// kernel of ingest.cu, moved by the copy engines instead of by registers.
//
// The destination of (layer, K|V, page, owned head) is one contiguous (page, head) tile of 16 tokens x D fp16 (4 KiB at
// D = 128); its source is 16 token rows of D*2 bytes, hs*D*2 bytes apart, in the shard that owns the head.  ONE WARP
// moves a tile with two instructions of one lane: a TMA tensor load (cp.async.bulk.tensor, box {D, 1 head, 16 tokens}
// of a map over the shard viewed as [layers*tokens][hs][D], no swizzle) lands the 16 rows as one contiguous tile in a
// buffer of the warp's ring, completion counted on an mbarrier; then ONE cp.async.bulk (shared -> global) of
// valid*D*2 bytes puts it into the page.  (16 row-sized bulk copies instead of the tensor load were measured first:
// 256-byte requests keep the copy engine below the rows kernel's rate.)  Nothing passes through registers, no thread
// waits on a load of its own, and a warp keeps two tiles landing while two drain: 16 KiB in flight per warp, so a
// handful of warps can draw what the per-thread kernel needs whole SMs for.  That is what lets the handoff ride in the
// decode-attention kernel's slack (attention.cu, HANDOFF): warps that have finished their attention range move tiles.
// A tile of a prompt's last page loads the rows past the prompt's end too (the next prompt's, or zeros past the end of
// the shard) and stores only the valid ones.
//
// Units.  The (request, page) slots of the handoff are enumerated block-table-shaped: slot = i * pages_per_req + j,
// pages_per_req = ceil(max_seq_len / 16); slots with j >= ceil(n_i / 16) are skipped.  A unit = (layer, K|V, slot,
// group of `hg` owned heads); units are handed to warps by `next_unit` (the fused kernel claims them from a global
// counter: its warps become free at different times).  A bit copy does not care who moves what.  A unit's three metadata loads
// (length, block-table entry, first token) are issued together one unit ahead, and the unit index two ahead, so that
// neither an atomic nor a dependent load ever sits on the warp's critical path; the block-table entry of a skipped
// slot is therefore READ (inside the row, below pages_per_req) but never used.
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>

#include "hx_internal.h"

namespace hx {

struct TileUnits {
  int32_t pages_per_req;   // ceil(max_seq_len / 16)
  int32_t hg;              // owned heads per unit (divides hd)
  long long units;         // layers * 2 * batch * pages_per_req * (hd / hg)
};

// Tensor maps of the source shards this destination rank reads: shard r_lo + e is maps k[e] / v[e].
constexpr int kMaxTileShards = 8;
struct alignas(64) TileMaps {
  CUtensorMap k[kMaxTileShards];
  CUtensorMap v[kMaxTileShards];
};

namespace tiles {

constexpr int kBufs = 4;     // tile buffers per warp (the fused kernel: a warp's 16 KiB attention ring)
constexpr int kAhead = 2;    // loads run this many tiles ahead of the stores

__device__ __forceinline__ void mbar_expect(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait_parity(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  } while (!done);
}
// the shards are read once: evict-first in L2
__device__ __forceinline__ void tile_load(uint32_t dst, const CUtensorMap* tm, int head, int row, uint32_t bar, uint64_t pol) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;"
      ::"r"(dst), "l"(tm), "r"(0), "r"(head), "r"(row), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ void tile_store(void* dst, uint32_t src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}

// One warp's share of the handoff.  buf_u32: kBufs tile buffers of 16*D*2 bytes (16-byte aligned) this warp owns;
// bar_u32: kBufs mbarriers (count 1) in phase 0 that nothing else uses.  Every lane must call with identical arguments;
// `next_unit()` returns this warp's next unit in LANE 0 (other lanes: anything; >= u.units when there is none left):
// it is broadcast one iteration after it was asked for.  On return every store of this warp has completed.
template <int D, int kBufs, int kAhead, class NextUnit>
__device__ __forceinline__ void move_tiles(const IngestParams& p, const TileUnits& u, const TileMaps& maps, uint32_t buf_u32,
                                           uint32_t bar_u32, NextUnit next_unit) {
  constexpr uint32_t kRow = D * 2, kTile = 16 * kRow;
  const int lane = threadIdx.x & 31;
  const int hgroups = p.hd / u.hg;
  const long long slots = (long long)p.batch * u.pages_per_req;
  const int r_lo = p.head0 / p.hs;                                         // first shard this rank reads
  const size_t dst_layer = (size_t)p.num_pages * p.hd * 16 * D;
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));

  // what a unit needs from global memory: three independent loads, issued one unit ahead of the unit's tiles
  struct Meta { int l, x, hg0, page, valid, tok0; };
  auto load_meta = [&](long long uu) -> Meta {
    Meta m = {0, 0, 0, 0, 0, 0};
    if (uu >= u.units) return m;
    const long long per_lx = slots * hgroups;
    const int lx = (int)(uu / per_lx);
    const long long rem = uu - (long long)lx * per_lx;
    const int slot = (int)(rem / hgroups);
    m.hg0 = (int)(rem - (long long)slot * hgroups) * u.hg;
    m.l = lx >> 1; m.x = lx & 1;
    const int i = slot / u.pages_per_req, j = slot - i * u.pages_per_req;
    m.valid = __ldg(p.seq_lens + i) - 16 * j;                             // > 16: a full page; <= 0: no such page
    m.page = __ldg(p.block_table + (size_t)i * p.bt_stride + j);          // (used only when valid > 0)
    m.tok0 = __ldg(p.cu_seqlens + i) + 16 * j;
    return m;
  };
  constexpr uint32_t FULLM = 0xffffffffu;
  long long raw_b = next_unit();               // lane 0 holds the index; broadcast when it is needed
  long long raw_c = next_unit();
  long long u_cur = __shfl_sync(FULLM, raw_b, 0);
  raw_b = raw_c;
  Meta m_cur = load_meta(u_cur);
  int t = 0;                                   // tiles issued by this warp
  __half* q_dst[kAhead];                       // destinations of the tiles whose loads are in flight (oldest first)
  uint32_t q_bytes[kAhead];
#pragma unroll
  for (int e = 0; e < kAhead; ++e) { q_dst[e] = nullptr; q_bytes[e] = 0; }
  auto retire = [&](int tt) {                  // tile tt has its loads issued kAhead tiles ago: wait for it, store it
    const int b = tt % kBufs;
    if (lane == 0) {
      mbar_wait_parity(bar_u32 + 8 * b, (uint32_t)(tt / kBufs) & 1u);
      tile_store(q_dst[0], buf_u32 + b * kTile, q_bytes[0]);
    }
  };
  while (u_cur < u.units) {
    raw_c = next_unit();
    const long long u_nxt = __shfl_sync(FULLM, raw_b, 0);
    const Meta m_nxt = load_meta(u_nxt);
    m_cur.valid = min(m_cur.valid, 16);
    if (m_cur.valid > 0) {
      for (int jh = 0; jh < u.hg; ++jh) {
        const int jd = m_cur.hg0 + jh;         // owned head (index in the destination rank)
        const int h = p.head0 + jd;            // global head
        const int r = h / p.hs;                // source shard
        const CUtensorMap* tm = m_cur.x ? &maps.v[r - r_lo] : &maps.k[r - r_lo];
        const int row = (m_cur.l + p.src_layer0) * p.total_tokens + m_cur.tok0;   // < 2^31 (host check)
        __half* dbase = static_cast<__half*>(m_cur.x ? p.dst_v : p.dst_k);
        __half* d = dbase + (size_t)(m_cur.l + p.dst_layer0) * dst_layer + ((size_t)m_cur.page * p.hd + jd) * (16 * D);
        const int b = t % kBufs;
        const uint32_t bar = bar_u32 + 8 * b;
        if (lane == 0) {
          // the store that last read this buffer (tile t - kBufs) must have finished reading it
          asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(kBufs - 1 - kAhead) : "memory");
          mbar_expect(bar, kTile);
          tile_load(buf_u32 + b * kTile, tm, h - r * p.hs, row, bar, pol);
        }
        if (t >= kAhead) retire(t - kAhead);
#pragma unroll
        for (int e = 0; e + 1 < kAhead; ++e) { q_dst[e] = q_dst[e + 1]; q_bytes[e] = q_bytes[e + 1]; }
        q_dst[kAhead - 1] = d; q_bytes[kAhead - 1] = (uint32_t)m_cur.valid * kRow;
        ++t;
      }
    }
    u_cur = u_nxt; raw_b = raw_c; m_cur = m_nxt;
  }
  // drain: the last min(t, kAhead) tiles
  for (int e = 0; e < kAhead; ++e) {
    const int tt = t - kAhead + e;
    if (tt >= 0) retire(tt);
#pragma unroll
    for (int s_ = 0; s_ + 1 < kAhead; ++s_) { q_dst[s_] = q_dst[s_ + 1]; q_bytes[s_] = q_bytes[s_ + 1]; }
  }
  if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  __syncwarp();
}

}  // namespace tiles
}  // namespace hx
