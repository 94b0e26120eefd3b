/* hxo — the ORACLE for the hx decode-phase KV-cache path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU code.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may call it.  It shares no code, header,
 * table or helper with the CUDA path under paper_2502_07903_b200/csrc/, and is written from
 * the layout contract in DESIGN.md ("Data layout") and the definitions below, not from the
 * kernels.
 *
 * What it follows
 *  - Ingest: PAPER.md:L92 (§3.3: "each GPU containing the j-th layer within phi_i should
 *    transmit its KV cache to the matching GPU housing the j-th layer within delta_i") and
 *    PAPER.md:L110 (§4: async SendRecv/cudaMemcpy KV handoff, PagedAttention).  TP shards own
 *    contiguous head ranges (reading S4).  The equation is
 *      dst_X[l][ bt[i][t div ps] ][h mod hd][t mod ps][d] = src_X[r][l][cu[i]+t][h mod hs][d]
 *    with r = h div hs and destination rank q = h div hd.  Payload is an
 *    opaque 16-bit pattern (B_type = 2); no arithmetic touches it.
 *  - Attention: the paper only cites PagedAttention / FlashAttention; the
 *    definition is the textbook one (reading S1): out = softmax(scale * q.K^T) V over
 *    the request's n_i cached tokens, GQA head h -> kv head h div G (reading S3).  Two passes,
 *    float64 throughout, output NOT rounded.
 *
 * Pins (tests/test_oracle_pins.py): brute-force dense numpy float64, constant-V, n=1, q=0 mean,
 * page-permutation invariance, GQA==repeated-MHA, split-merge identity, stability under 8x
 * logits, NaN-poison masking, ingest/gather round trip for every (S,R), changed-element count,
 * all-65536-pattern fp16 decode vs numpy, Table-1 byte counts;
 * stage ingest: any cut of the model into prefill x decode stages == the one-call ingest, and an
 * independent numpy restatement; append: ingest of n-1 tokens + append == ingest of n tokens,
 * changed-element count, attention after append == dense softmax over the concatenation;
 * prefill: brute-force causal numpy/scipy, m = 1 == decode attention, first token returns v_0,
 * future tokens never matter, chunked (m < n) == the tail rows of the whole-prompt result.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* IEEE-754 binary16 -> double, exact, by the definition of the format. */
double hxo_half_to_double(uint16_t h) {
  int sign = (h >> 15) & 1;
  int e = (h >> 10) & 0x1f;
  int f = h & 0x3ff;
  double v;
  if (e == 0)       v = ldexp((double)f, -24);               /* zero / subnormal: f * 2^-24 */
  else if (e == 31) v = f ? NAN : INFINITY;
  else              v = ldexp((double)(f + 1024), e - 25);   /* (1 + f/1024) * 2^(e-15) */
  return sign ? -v : v;
}

void hxo_half_to_double_array(const uint16_t* in, double* out, int64_t n) {
  for (int64_t i = 0; i < n; ++i) out[i] = hxo_half_to_double(in[i]);
}

int hxo_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* Ingest for ONE destination rank q (SURVEY.md §8(c) equation).  src_k/src_v: array of S host
 * pointers, shard r is uint16 [L][T][hs][D].  dst_k/dst_v: uint16 [L][P][hd][ps][D].
 * gather != 0 runs the same equation right to left (dst -> src).  threads <= 0: all cores
 * (parallel over layers). */
int hxo_kv_ingest(uint16_t* const* src_k, uint16_t* const* src_v,
                  int layers, int total_tokens, int heads, int head_dim,
                  int src_tp, int dst_tp, int dst_rank,
                  uint16_t* dst_k, uint16_t* dst_v, int num_pages, int page_size,
                  const int32_t* block_table, int block_table_stride,
                  const int32_t* cu_seqlens, const int32_t* seq_lens, int batch,
                  int gather, int threads) {
  if (heads % src_tp || heads % dst_tp || dst_rank < 0 || dst_rank >= dst_tp) return 1;
  const int hs = heads / src_tp, hd = heads / dst_tp;
  const int64_t D = head_dim, T = total_tokens, P = num_pages, ps = page_size;
#ifdef _OPENMP
  if (threads <= 0) threads = omp_get_max_threads();
#pragma omp parallel for num_threads(threads) schedule(static)
#endif
  for (int l = 0; l < layers; ++l) {
    for (int i = 0; i < batch; ++i) {
      for (int t = 0; t < seq_lens[i]; ++t) {
        const int64_t page = block_table[(int64_t)i * block_table_stride + t / ps];
        const int64_t slot = t % ps;
        for (int h = dst_rank * hd; h < (dst_rank + 1) * hd; ++h) {
          const int r = h / hs;
          const int64_t s_off = ((((int64_t)l * T) + cu_seqlens[i] + t) * hs + (h % hs)) * D;
          const int64_t d_off = ((((int64_t)l * P + page) * hd + (h % hd)) * ps + slot) * D;
          for (int x = 0; x < 2; ++x) {
            uint16_t* s = (x ? src_v : src_k)[r] + s_off;
            uint16_t* d = (x ? dst_v : dst_k) + d_off;
            for (int e = 0; e < D; ++e) {
              if (gather) s[e] = d[e]; else d[e] = s[e];
            }
          }
        }
      }
    }
  }
  return 0;
}

/* Pipeline-stage ingest ("each GPU containing the j-th layer
 * within phi_i should transmit its KV cache to the matching GPU housing the j-th layer within
 * delta_i"; prefill and decode replicas cut the model into different
 * pipeline stages).  The source buffers hold `src_layers` layers of a prefill stage, the paged
 * cache holds `dst_layers` layers of a decode stage; `count` consecutive layers move, source
 * layer src_layer0 + c landing at cache layer dst_layer0 + c, c = 0..count-1.  Everything else
 * is the ingest equation above.  Written as its own loop nest (not by calling hxo_kv_ingest). */
int hxo_kv_ingest_stage(uint16_t* const* src_k, uint16_t* const* src_v,
                        int src_layers, int src_layer0, int dst_layers, int dst_layer0, int count,
                        int total_tokens, int heads, int head_dim,
                        int src_tp, int dst_tp, int dst_rank,
                        uint16_t* dst_k, uint16_t* dst_v, int num_pages, int page_size,
                        const int32_t* block_table, int block_table_stride,
                        const int32_t* cu_seqlens, const int32_t* seq_lens, int batch) {
  if (heads % src_tp || heads % dst_tp || dst_rank < 0 || dst_rank >= dst_tp) return 1;
  if (count < 0 || src_layer0 < 0 || dst_layer0 < 0 || src_layer0 + count > src_layers ||
      dst_layer0 + count > dst_layers) return 2;
  const int hs = heads / src_tp, hd = heads / dst_tp;
  const int64_t D = head_dim, T = total_tokens, P = num_pages, ps = page_size;
  for (int c = 0; c < count; ++c) {
    const int64_t ls = src_layer0 + c, ld = dst_layer0 + c;
    for (int i = 0; i < batch; ++i)
      for (int t = 0; t < seq_lens[i]; ++t)
        for (int h = dst_rank * hd; h < (dst_rank + 1) * hd; ++h)
          for (int x = 0; x < 2; ++x)
            for (int e = 0; e < D; ++e) {
              const int64_t page = block_table[(int64_t)i * block_table_stride + t / ps];
              const uint16_t* s = (x ? src_v : src_k)[h / hs];
              uint16_t* d = x ? dst_v : dst_k;
              d[((((ld * P) + page) * hd + (h % hd)) * ps + (t % ps)) * D + e] =
                  s[(((ls * T) + cu_seqlens[i] + t) * hs + (h % hs)) * D + e];
            }
  }
  return 0;
}

/* Append of the decode step's new token ("the decoding phase
 * generates subsequent tokens by one token at each step", each step's K/V joining the cache,
 * PAPER.md:L54).  seq_lens[i] = n_i counts the new token (reading S12), so it is
 * token t = n_i - 1:
 *     X[layer][ bt[i][(n_i-1) div ps] ][g][(n_i-1) mod ps][:] = x_new[i][g][:],  X in {K, V}
 * for every request with n_i >= 1 and every local kv head g.  n_i = 0: nothing is written.
 * k_new, v_new: uint16 [B][Hkv][D].  Nothing else in the cache changes. */
int hxo_kv_append(const uint16_t* k_new, const uint16_t* v_new, uint16_t* k, uint16_t* v,
                  int layer, int layers, int num_pages, int kv_heads, int page_size, int head_dim,
                  const int32_t* block_table, int block_table_stride, const int32_t* seq_lens,
                  int batch) {
  if (layer < 0 || layer >= layers) return 1;
  const int64_t D = head_dim, P = num_pages, ps = page_size;
  for (int i = 0; i < batch; ++i) {
    const int n = seq_lens[i];
    if (n <= 0) continue;
    const int t = n - 1;
    const int64_t page = block_table[(int64_t)i * block_table_stride + t / ps];
    for (int g = 0; g < kv_heads; ++g) {
      const int64_t d_off = ((((int64_t)layer * P + page) * kv_heads + g) * ps + (t % ps)) * D;
      const int64_t s_off = ((int64_t)i * kv_heads + g) * D;
      for (int e = 0; e < D; ++e) { k[d_off + e] = k_new[s_off + e]; v[d_off + e] = v_new[s_off + e]; }
    }
  }
  return 0;
}

/* One-token attention over a paged cache, float64, two passes (readings S1-S3, S11).
 * q: uint16 (fp16 bits) [B][Hq][D]; k, v: [layers][P][Hkv][ps][D]; out: double [B][Hq][D].
 * n_i = 0 -> zeros (S11).  scale is taken as given (caller passes (double)(float)sm_scale). */
int hxo_decode_attention(double* out, const uint16_t* q, const uint16_t* k, const uint16_t* v,
                         int layer, int num_pages, int kv_heads, int page_size, int head_dim,
                         int q_heads, const int32_t* block_table, int block_table_stride,
                         const int32_t* seq_lens, int batch, double scale, int threads) {
  if (kv_heads <= 0 || q_heads % kv_heads) return 1;
  const int G = q_heads / kv_heads;
  const int64_t D = head_dim, P = num_pages, ps = page_size;
#ifdef _OPENMP
  if (threads <= 0) threads = omp_get_max_threads();
#pragma omp parallel for num_threads(threads) schedule(dynamic, 1) collapse(2)
#endif
  for (int i = 0; i < batch; ++i) {
    for (int h = 0; h < q_heads; ++h) {
      const int n = seq_lens[i];
      double* o = out + ((int64_t)i * q_heads + h) * D;
      for (int e = 0; e < D; ++e) o[e] = 0.0;
      if (n <= 0) continue;
      const int g = h / G;
      const uint16_t* qh = q + ((int64_t)i * q_heads + h) * D;
      double* s = (double*)malloc(sizeof(double) * (size_t)n);
      /* pass 1: scores and their max */
      double m = -INFINITY;
      for (int t = 0; t < n; ++t) {
        const int64_t page = block_table[(int64_t)i * block_table_stride + t / ps];
        const uint16_t* kt = k + ((((int64_t)layer * P + page) * kv_heads + g) * ps + (t % ps)) * D;
        double dot = 0.0;
        for (int e = 0; e < D; ++e) dot += hxo_half_to_double(qh[e]) * hxo_half_to_double(kt[e]);
        s[t] = scale * dot;
        if (s[t] > m) m = s[t];
      }
      /* pass 2: weights, weighted sum, normalise */
      double l = 0.0;
      for (int t = 0; t < n; ++t) {
        const int64_t page = block_table[(int64_t)i * block_table_stride + t / ps];
        const uint16_t* vt = v + ((((int64_t)layer * P + page) * kv_heads + g) * ps + (t % ps)) * D;
        const double w = exp(s[t] - m);
        l += w;
        for (int e = 0; e < D; ++e) o[e] += w * hxo_half_to_double(vt[e]);
      }
      for (int e = 0; e < D; ++e) o[e] /= l;
      free(s);
    }
  }
  return 0;
}

/* Paged prefill (multi-token) attention, causal ("the prefill phase
 * processes the request's input tokens all at once", PAPER.md:L110 integrates FlashAttention for it;
 * the definition is the textbook causal one, reading S24).  Request i has n_i cached tokens
 * and m_i query tokens, which are its LAST m_i tokens: query r (0 <= r < m_i) sits at position
 * p = n_i - m_i + r and attends to the cached tokens t = 0..p:
 *     out[cu_q[i] + r][h] = sum_{t<=p} softmax_t(scale * <q[cu_q[i]+r][h], k_t>) v_t,   g = h div G.
 * m_i = n_i is a whole-prompt prefill; m_i = 1 is hx's decode attention.  m_i = 0: no rows.
 * q: uint16 [Tq][Hq][D] packed by request; out: double [Tq][Hq][D].  Two passes, float64. */
int hxo_prefill_attention(double* out, const uint16_t* q, const uint16_t* k, const uint16_t* v,
                          int layer, int num_pages, int kv_heads, int page_size, int head_dim,
                          int q_heads, const int32_t* block_table, int block_table_stride,
                          const int32_t* seq_lens, const int32_t* q_lens, const int32_t* cu_q,
                          int batch, double scale, int threads) {
  if (kv_heads <= 0 || q_heads % kv_heads) return 1;
  for (int i = 0; i < batch; ++i) if (q_lens[i] < 0 || q_lens[i] > seq_lens[i]) return 2;
  const int G = q_heads / kv_heads;
  const int64_t D = head_dim, P = num_pages, ps = page_size;
#ifdef _OPENMP
  if (threads <= 0) threads = omp_get_max_threads();
#pragma omp parallel for num_threads(threads) schedule(dynamic, 1)
#endif
  for (int i = 0; i < batch; ++i) {
    double* s = (double*)malloc(sizeof(double) * (size_t)(seq_lens[i] > 0 ? seq_lens[i] : 1));
    for (int r = 0; r < q_lens[i]; ++r) {
      const int p = seq_lens[i] - q_lens[i] + r;           /* position of this query token */
      for (int h = 0; h < q_heads; ++h) {
        const int g = h / G;
        const uint16_t* qh = q + (((int64_t)cu_q[i] + r) * q_heads + h) * D;
        double* o = out + (((int64_t)cu_q[i] + r) * q_heads + h) * D;
        double m = -INFINITY;
        for (int t = 0; t <= p; ++t) {
          const int64_t page = block_table[(int64_t)i * block_table_stride + t / ps];
          const uint16_t* kt = k + ((((int64_t)layer * P + page) * kv_heads + g) * ps + (t % ps)) * D;
          double dot = 0.0;
          for (int e = 0; e < D; ++e) dot += hxo_half_to_double(qh[e]) * hxo_half_to_double(kt[e]);
          s[t] = scale * dot;
          if (s[t] > m) m = s[t];
        }
        double l = 0.0;
        for (int e = 0; e < D; ++e) o[e] = 0.0;
        for (int t = 0; t <= p; ++t) {
          const int64_t page = block_table[(int64_t)i * block_table_stride + t / ps];
          const uint16_t* vt = v + ((((int64_t)layer * P + page) * kv_heads + g) * ps + (t % ps)) * D;
          const double w = exp(s[t] - m);
          l += w;
          for (int e = 0; e < D; ++e) o[e] += w * hxo_half_to_double(vt[e]);
        }
        for (int e = 0; e < D; ++e) o[e] /= l;
      }
    }
    free(s);
  }
  return 0;
}

/* Split-merge identity helper (FlashAttention online-softmax merge, cited PAPER.md:L110,
 * L204-L205): partial state (m, l, acc[D]) of a token range [t0, t1) for one (request, head). */
int hxo_partial_attention(double* m_out, double* l_out, double* acc, const uint16_t* q_row,
                          const uint16_t* k, const uint16_t* v, int layer, int num_pages,
                          int kv_heads, int g, int page_size, int head_dim,
                          const int32_t* bt_row, int t0, int t1, double scale) {
  const int64_t D = head_dim, P = num_pages, ps = page_size;
  double m = -INFINITY, l = 0.0;
  for (int e = 0; e < D; ++e) acc[e] = 0.0;
  for (int t = t0; t < t1; ++t) {
    const uint16_t* kt = k + ((((int64_t)layer * P + bt_row[t / ps]) * kv_heads + g) * ps + (t % ps)) * D;
    double dot = 0.0;
    for (int e = 0; e < D; ++e) dot += hxo_half_to_double(q_row[e]) * hxo_half_to_double(kt[e]);
    dot *= scale;
    if (dot > m) m = dot;
  }
  for (int t = t0; t < t1; ++t) {
    const uint16_t* kt = k + ((((int64_t)layer * P + bt_row[t / ps]) * kv_heads + g) * ps + (t % ps)) * D;
    const uint16_t* vt = v + ((((int64_t)layer * P + bt_row[t / ps]) * kv_heads + g) * ps + (t % ps)) * D;
    double dot = 0.0;
    for (int e = 0; e < D; ++e) dot += hxo_half_to_double(q_row[e]) * hxo_half_to_double(kt[e]);
    const double w = exp(scale * dot - m);
    l += w;
    for (int e = 0; e < D; ++e) acc[e] += w * hxo_half_to_double(vt[e]);
  }
  *m_out = m; *l_out = l;
  return 0;
}
