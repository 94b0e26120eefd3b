// hx_decode_attention kernels.
#include <cuda_fp16.h>

#include <cstdlib>

#include "hx_internal.h"

namespace hx {
namespace {

// ------------------------------------------------------------------------------------------
// Kernel "simple": one CTA per (request, query head), CUDA-core dot products, no split.
// Bring-up / fallback path for shapes the streaming kernel does not cover (head_dim 64).
// ------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(128) attn_simple_kernel(const AttnParams p) {
  constexpr int E = D / 32;                       // elements per lane
  const int h = blockIdx.x, i = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n = p.seq_lens[i];
  const int G = p.q_heads / p.kv_heads;
  const int g = h / G;
  const int ps = p.page_size;
  const __half* K = static_cast<const __half*>(p.k);
  const __half* V = static_cast<const __half*>(p.v);
  const __half* qrow = static_cast<const __half*>(p.q) + ((size_t)i * p.q_heads + h) * D;
  __half* orow = static_cast<__half*>(p.out) + ((size_t)i * p.q_heads + h) * D;

  float qf[E], acc[E];
#pragma unroll
  for (int e = 0; e < E; ++e) { qf[e] = __half2float(qrow[lane * E + e]); acc[e] = 0.f; }
  float m = -INFINITY, l = 0.f;
  const float scale_log2 = p.sm_scale * 1.4426950408889634f;

  for (int t = warp; t < n; t += 4) {
    const int page = p.block_table[(size_t)i * p.bt_stride + t / ps];
    const size_t off = (((size_t)page * p.kv_heads + g) * ps + (t % ps)) * D + lane * E;
    float dot = 0.f;
#pragma unroll
    for (int e = 0; e < E; ++e) dot += qf[e] * __half2float(K[off + e]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
    const float s = dot * scale_log2;
    const float m_new = fmaxf(m, s);
    const float corr = exp2f(m - m_new);          // m = -inf on first token -> 0
    const float w = exp2f(s - m_new);
    l = l * corr + w;
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = acc[e] * corr + w * __half2float(V[off + e]);
    m = m_new;
  }

  __shared__ float sm_m[4], sm_l[4], sm_acc[4][D];
  if (lane == 0) { sm_m[warp] = m; sm_l[warp] = l; }
#pragma unroll
  for (int e = 0; e < E; ++e) sm_acc[warp][lane * E + e] = acc[e];
  __syncthreads();
  if (warp == 0) {
    float mm = fmaxf(fmaxf(sm_m[0], sm_m[1]), fmaxf(sm_m[2], sm_m[3]));
    float ll = 0.f, o[E];
#pragma unroll
    for (int e = 0; e < E; ++e) o[e] = 0.f;
    for (int w = 0; w < 4; ++w) {                 // fixed order: deterministic
      const float c = (sm_m[w] == -INFINITY) ? 0.f : exp2f(sm_m[w] - mm);
      ll += sm_l[w] * c;
#pragma unroll
      for (int e = 0; e < E; ++e) o[e] += sm_acc[w][lane * E + e] * c;
    }
    const float inv = (n > 0) ? 1.f / ll : 0.f;
#pragma unroll
    for (int e = 0; e < E; ++e) orow[lane * E + e] = __float2half_rn(n > 0 ? o[e] * inv : 0.f);
  }
}

}  // namespace

size_t attn_workspace_bytes(int32_t batch, int32_t q_heads, int32_t kv_heads, int32_t head_dim,
                            int32_t max_seq_len, int32_t page_size) {
  (void)batch; (void)q_heads; (void)kv_heads; (void)head_dim; (void)max_seq_len; (void)page_size;
  return 0;
}

int launch_attention(const AttnParams& p, cudaStream_t stream) {
  dim3 grid(p.q_heads, p.batch);
  if (p.head_dim == 128) attn_simple_kernel<128><<<grid, 128, 0, stream>>>(p);
  else                   attn_simple_kernel<64><<<grid, 128, 0, stream>>>(p);
  HX_CUDA_OK(cudaGetLastError());
  return HX_OK;
}

}  // namespace hx
