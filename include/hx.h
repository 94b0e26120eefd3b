/* hx.h — C ABI of libhx: the decode-phase KV-cache path of disaggregated LLM serving
 * (HexGen-2, arxiv 2502.07903), hand-written CUDA for sm_100a (B200).
 *
 * The path (§2, L92 §3.3, L110 §4): a prefill replica produces the KV cache,
 * sharded over its tensor-parallel (TP) group; it is handed, layer by layer, to the decode
 * replica, whose TP degree may differ (Table 2: TP in {1,2,4} on either
 * side); the decode replica keeps it in a paged cache (PagedAttention) and reads
 * all of it once per generated token ("HBM memory I/O-bound").
 *
 * Conventions (all entry points)
 *  - Payload is IEEE fp16 (B_type = 2).  fp32 accumulation inside attention.
 *  - DEVICE pointers are marked "device"; everything else is host memory.  The caller owns all
 *    device memory, including the workspace.  The library allocates no device memory and keeps no
 *    state on the device (one exception, part of the library's image rather than an allocation: the
 *    fixed scratch array behind hx_decode_attention_noalloc).  Its host-side state: (1) per device, one side stream and two events, created
 *    by the first hx_decode_step_host call that asks for an overlapped handoff and destroyed by
 *    hx_shutdown(); (2) caches of device properties and TMA descriptors.  hx_page_pool is
 *    the only heap object the caller owns (host).
 *  - No call's behaviour depends on which library calls came before it: what a launch may overlap is always an
 *    explicit argument (inputs_ready, behind_ingest, overlap_ingest).
 *  - Thread safety: every entry point may be called from several host threads (on different streams);
 *    hx_decode_step* serialise on one library mutex while they enqueue.  An hx_page_pool and an attention
 *    workspace each serve one caller at a time.
 *  - hx_kv_ingest / hx_kv_gather / hx_decode_attention only ENQUEUE work on `stream`
 *    (a cudaStream_t passed as void*, NULL = legacy default stream) and return.  They never
 *    synchronise and never read device memory from the host; this is why sizes that only
 *    shape the launch are also passed as host scalars.
 *  - Return value: an hx_status.  Nothing is launched unless every host-side check passes.
 *    hx_last_error() gives a thread-local detail string for the last non-OK return.
 *  - Device-side contract (not checkable from the host; undefined behaviour if violated):
 *    page ids in [0, num_pages); row i of the block table holds ceil(n_i/page_size) valid
 *    entries; cu_seqlens is the exclusive prefix sum of seq_lens; ingest destinations are
 *    pairwise distinct.  Attention may read a page shared by several requests.
 *  - Determinism: same inputs -> same bits, run to run, on a given GPU model (no floating-point
 *    atomics; the work partition depends only on seq_lens and the SM count; partial results are
 *    merged in a fixed order).
 *
 * Layouts (readings S4, S7, S8, S9)
 *  - Source shard r of a prefill TP group of degree S:  fp16 [layers][total_tokens][heads/S][head_dim]
 *    for K and, separately, for V.  Prompts are packed back to back on the token axis; prompt i
 *    owns rows [cu_seqlens[i], cu_seqlens[i+1]).  Shard r owns the contiguous global kv-head
 *    range [r*heads/S, (r+1)*heads/S)   (column-wise weight split).
 *  - Paged cache of ONE decode TP rank q of degree R:  fp16 [layers][num_pages][heads/R][page_size][head_dim]
 *    for K and, separately, for V.  Rank q owns global kv heads [q*heads/R, (q+1)*heads/R).
 *    A (page, head) tile is one contiguous page_size*head_dim*2-byte run (4 KiB at 16 x 128).
 *  - Block table: int32 [batch][block_table_stride]; entry j of row i is the physical page of
 *    tokens [j*page_size, (j+1)*page_size) of request i; the same table serves every layer,
 *    K and V, and every decode rank.  Entries at or past ceil(n_i/page_size) are never read.
 */
#ifndef HX_H_
#define HX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HX_VERSION 135 /* 0.1.3.5: hx_decode_attention_overlapped takes an explicit behind_ingest (no inferred state);
                          0.1.3.4: + hx_decode_attention_noalloc (built-in scratch, no workspace argument) */

typedef enum {
  HX_OK = 0,
  HX_ERR_INVALID_ARG = 1, /* NULL / misaligned pointer, negative size, indivisible heads, bad rank/layer/stride */
  HX_ERR_UNSUPPORTED = 2, /* head_dim not in {64,128}; page_size != 16; group size not in {1,2,4,8,16}; tp > heads */
  HX_ERR_WORKSPACE = 3,   /* workspace NULL or smaller than hx_decode_attention_workspace_bytes() */
  HX_ERR_CUDA = 4,        /* a CUDA call failed; text in hx_last_error() */
  HX_ERR_NO_PAGES = 5     /* hx_pool_alloc: not enough free pages, nothing was taken; hx_pool_create: out of host memory */
} hx_status;

int hx_version(void);
const char* hx_status_string(int status); /* static string, never NULL */
const char* hx_last_error(void);          /* thread-local, never NULL */

/* One decode-TP-rank's paged KV cache (caller-owned device memory). */
typedef struct {
  void* k;            /* device, fp16 [layers][num_pages][kv_heads][page_size][head_dim], 16-byte aligned */
  void* v;            /* device, same shape */
  int32_t layers;
  int32_t num_pages;
  int32_t kv_heads;   /* LOCAL kv heads = global heads / dst_tp */
  int32_t page_size;  /* 16 */
  int32_t head_dim;   /* 64 or 128 */
} hx_paged_cache;

/* Bytes of ONE tensor (k or v) of a paged cache; 0 on overflow / non-positive arguments. */
size_t hx_paged_cache_bytes(int32_t layers, int32_t num_pages, int32_t kv_heads,
                            int32_t page_size, int32_t head_dim);

/* ---- (a) KV handoff ingest -------------------------------------------------------------
 * PAPER.md:L92 (§3.3): "each GPU containing the j-th layer within phi_i should transmit its KV
 * cache to the matching GPU housing the j-th layer within delta_i"; PAPER.md:L110 (§4): KV
 * moved by asynchronous SendRecv/cudaMemcpy so that it overlaps compute.  This call is the
 * LANDING of that handoff on decode rank `dst_rank`: for every layer l < layers, request
 * i < batch, token t < seq_lens[i], owned global kv head h, tensor X in {K, V}:
 *
 *   dst->X[l][ block_table[i][t / ps] ][ h % hd ][ t % ps ][:] = src_X[h / hs][l][ cu_seqlens[i] + t ][ h % hs ][:]
 *
 * with hs = heads/src_tp, hd = heads/dst_tp, h in [dst_rank*hd, (dst_rank+1)*hd).  A bit copy:
 * no arithmetic touches the payload.  Nothing else in dst changes (tail slots of last pages,
 * unowned pages and other layers beyond `layers` keep their contents).
 *
 * src_k, src_v : HOST arrays of src_tp DEVICE pointers (16-byte aligned).  Entries for shards
 *                that hold none of dst_rank's heads may be NULL.  "Device pointer" = any address the
 *                GPU can load from: its own HBM, a peer GPU's memory (peer access enabled) or pinned
 *                host memory; the last two make the call a PULL-mode handoff (F2): the shard crosses
 *                the link once, straight into its pages.
 * layers       : layers present in the source buffers; they land at layers [0, layers) of dst
 *                (a pipeline stage = one call; dst->layers >= layers).
 * heads        : GLOBAL kv heads; must be divisible by src_tp and dst_tp; dst->kv_heads == heads/dst_tp.
 * block_table  : device int32 [batch][block_table_stride]; stride >= ceil(max_seq_len/ps).
 * cu_seqlens   : device int32 [batch+1].   seq_lens: device int32 [batch].
 * batch, total_tokens, max_seq_len : host copies, used for launch sizing and checks only.
 * Returns HX_OK without launching when batch == 0 or total_tokens == 0 or layers == 0.      */
int hx_kv_ingest(const void* const* src_k, const void* const* src_v,
                 int32_t layers, int32_t heads, int32_t head_dim,
                 int32_t src_tp, int32_t dst_tp, int32_t dst_rank,
                 const hx_paged_cache* dst,
                 const int32_t* block_table, int32_t block_table_stride,
                 const int32_t* cu_seqlens, const int32_t* seq_lens,
                 int32_t batch, int32_t total_tokens, int32_t max_seq_len,
                 void* stream);

/* Exact inverse of hx_kv_ingest (the same equation read right to left): writes dst_rank's
 * heads of every valid token back into the shard buffers.  src_k/src_v entries are written. */
int hx_kv_gather(void* const* src_k, void* const* src_v,
                 int32_t layers, int32_t heads, int32_t head_dim,
                 int32_t src_tp, int32_t dst_tp, int32_t dst_rank,
                 const hx_paged_cache* dst,
                 const int32_t* block_table, int32_t block_table_stride,
                 const int32_t* cu_seqlens, const int32_t* seq_lens,
                 int32_t batch, int32_t total_tokens, int32_t max_seq_len,
                 void* stream);

/* ---- (a') pipeline-stage ingest -------------------------------------
 * PAPER.md:L92 matches layers, not stages: "each GPU containing the j-th layer within phi_i should
 * transmit its KV cache to the matching GPU housing the j-th layer within delta_i", and prefill
 * and decode replicas cut the model into different pipeline stages (Table 2:
 * PP in {1,2,3,5}).  One call moves the layers that ONE prefill stage and
 * ONE decode stage have in common: the source buffers hold `src_layers` layers
 * (fp16 [src_layers][total_tokens][heads/src_tp][head_dim]); source layer src_layer0 + c lands at
 * cache layer dst_layer0 + c for c = 0..layers-1.  Everything else is hx_kv_ingest
 * (hx_kv_ingest == this with src_layers = layers, src_layer0 = dst_layer0 = 0).
 * HX_ERR_INVALID_ARG when [src_layer0, src_layer0+layers) leaves [0, src_layers) or
 * [dst_layer0, dst_layer0+layers) leaves [0, dst->layers).  hx_stage_overlap computes the three
 * numbers from the two stages' global layer ranges. */
int hx_kv_ingest_stage(const void* const* src_k, const void* const* src_v,
                       int32_t src_layers, int32_t src_layer0, int32_t dst_layer0, int32_t layers,
                       int32_t heads, int32_t head_dim,
                       int32_t src_tp, int32_t dst_tp, int32_t dst_rank,
                       const hx_paged_cache* dst,
                       const int32_t* block_table, int32_t block_table_stride,
                       const int32_t* cu_seqlens, const int32_t* seq_lens,
                       int32_t batch, int32_t total_tokens, int32_t max_seq_len,
                       void* stream);

/* Host helper: a prefill stage holds global layers [src_first, src_first + src_count), a decode
 * stage [dst_first, dst_first + dst_count).  Writes the arguments of hx_kv_ingest_stage for their
 * intersection; *layers = 0 when they share none.  Returns HX_ERR_INVALID_ARG on negative input
 * or NULL outputs. */
int hx_stage_overlap(int32_t src_first, int32_t src_count, int32_t dst_first, int32_t dst_count,
                     int32_t* src_layer0, int32_t* dst_layer0, int32_t* layers);

/* ---- (a'') append of the decode step's token -----------------------
 * "the decoding phase generates subsequent tokens by one token at each step"; the
 * token's K/V joins the request's cache.  seq_lens[i] = n_i COUNTS the new token
 * (reading S12), so it is token n_i - 1: for every request with n_i >= 1, local kv head g, X in {K,V}
 *
 *   cache->X[layer][ block_table[i][(n_i-1) / ps] ][g][(n_i-1) % ps][:] = x_new[i][g][:]
 *
 * A bit copy; n_i == 0 writes nothing; nothing else in the cache changes.
 * k_new, v_new : device fp16 [batch][kv_heads][head_dim], 16-byte aligned.
 * Device-side contract: the destination slots of different requests are distinct (the last page
 * of a request is not shared). */
int hx_kv_append(const void* k_new, const void* v_new,
                 const hx_paged_cache* cache, int32_t layer,
                 const int32_t* block_table, int32_t block_table_stride,
                 const int32_t* seq_lens, int32_t batch, int32_t max_seq_len,
                 void* stream);

/* ---- (b) paged decode attention ---------------------------------------------------------
 * PAPER.md:L110 (§4) integrates PagedAttention / FlashAttention and gives no formula; the
 * definition is the textbook one (reading S1).  For request i with n = seq_lens[i]
 * cached tokens (the current token included, already in the cache: reading S12), local query
 * head h, kv head g = h / (q_heads / cache->kv_heads):
 *
 *   s_t = sm_scale * <q[i][h], K[layer][bt[i][t/ps]][g][t%ps]>,   t = 0..n-1
 *   out[i][h] = sum_t softmax(s)_t * V[layer][bt[i][t/ps]][g][t%ps]
 *
 * fp16 in, fp32 accumulate, fp16 out.  n == 0 -> out row = zeros.  Tail slots and unowned
 * pages are never read into the result.
 *
 * out, q      : device fp16 [batch][q_heads][head_dim], 16-byte aligned.
 * sm_scale    : <= 0 means 1/sqrt(head_dim) rounded to fp32.
 * workspace   : device, 16-byte aligned, >= hx_decode_attention_workspace_bytes(...) bytes.
 *               It must be ZERO-FILLED once before its first use (cudaMemsetAsync) and then only
 *               be passed to hx_decode_attention* / hx_decode_step: every call leaves its counters at zero
 *               again (zero it again after a launch that failed with a CUDA error: an aborted kernel
 *               may leave them set).  One workspace serves one call at a time (calls on one stream are fine). */
size_t hx_decode_attention_workspace_bytes(int32_t batch, int32_t q_heads, int32_t kv_heads,
                                           int32_t head_dim, int32_t max_seq_len, int32_t page_size);

int hx_decode_attention(void* out, const void* q,
                        const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                        const int32_t* block_table, int32_t block_table_stride,
                        const int32_t* seq_lens,
                        int32_t batch, int32_t max_seq_len, float sm_scale,
                        void* workspace, size_t workspace_bytes,
                        void* stream);

/* hx_decode_attention that may OVERLAP the hx_kv_ingest enqueued just before it on `stream` (SURVEY.md §8(a) row
 * A9; "asynchronous ... to enable overlapping between computation and communication").  Same
 * arguments and result as hx_decode_attention, plus one explicit statement by the caller (the library keeps no
 * record of earlier calls and infers nothing):
 *   behind_ingest == 0: exactly hx_decode_attention.
 *   behind_ingest != 0: the CALLER asserts that (1) the kernel directly before this call on `stream` is the one an
 *                       hx_kv_ingest / hx_kv_ingest_stage call LAUNCHED (a call that returned without launching -
 *                       empty batch, no tokens, no layers - does not count), with nothing enqueued on `stream` in
 *                       between, and (2) this call reads nothing that ingest writes: the step's new prompts live in
 *                       pages disjoint from the active batch's.  The grid is then launched as a programmatic dependent
 *                       of the ingest kernel (which signals its dependents at once) and starts while the handoff is
 *                       still landing; every CTA executes griddepcontrol.wait before it exits, so the grid completes
 *                       only after the ingest has completed and its writes are visible: work enqueued after this
 *                       call is ordered after BOTH kernels.  If (1) is false because the predecessor is another kernel
 *                       of this library sharing `workspace` or `out`, the two race (undefined result); behind a kernel
 *                       of another library the call degrades to a plain launch. */
int hx_decode_attention_overlapped(void* out, const void* q,
                                   const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                                   const int32_t* block_table, int32_t block_table_stride,
                                   const int32_t* seq_lens,
                                   int32_t batch, int32_t max_seq_len, float sm_scale,
                                   void* workspace, size_t workspace_bytes,
                                   int32_t behind_ingest, void* stream);

/* ---- (b'') decode attention for callers that have no device memory to give ---------------------
 * Same operation, same kernel and same result as hx_decode_attention (definition above), without the
 * workspace argument: the partial results and counters live in an array that is part of libhx's device image.
 *
 * Who this is for.  hx_decode_attention needs ~17 MB of scratch from the caller.  Some callers have none and cannot get
 * any: a decode replica sizes its paged KV cache to fill the GPU at start-up (PAPER.md:L136 names out-of-memory as
 * what an overloaded replica dies of, so every spare byte becomes pages), which leaves a later cudaMalloc to fail; an attention backend plugged
 * into someone else's serving engine is handed tensors but no allocator, and a raw cudaMalloc from inside the engine's
 * step loop would also synchronise the whole device in the middle of a step; and code that runs while another
 * thread's stream capture is open must not call cudaMalloc at all.  For them the scratch is paid for once, when the
 * library's image is loaded onto a GPU, and this call allocates nothing: no cudaMalloc / cudaFree, no
 * stream-ordered allocation, no library routine that allocates behind the caller's back.
 *
 * The price and the limits.
 *  - Every GPU on which this process uses libhx holds HX_NOALLOC_SCRATCH_BYTES (20 MiB) of device memory from the
 *    moment the image is loaded there until the process exits, whether or not this call is ever made.
 *  - Shapes whose hx_decode_attention_workspace_bytes() exceeds HX_NOALLOC_SCRATCH_BYTES are refused with
 *    HX_ERR_WORKSPACE and a message naming both sizes (today: group size 16 at head_dim 128, or more than ~470 local
 *    kv heads); nothing is enqueued.  Those shapes need hx_decode_attention and a caller-owned workspace.
 *  - ONE array per GPU serves every call from every thread and stream.  Calls are safe one after another on one
 *    stream (or otherwise ordered so that one finishes before the next starts); two calls that can run on the GPU at
 *    the same time - different streams, different threads - write the same scratch and corrupt each other's result.
 *    The library does not detect this.
 *  - The array keeps whatever the previous call left in it, and where the counters sit depends on the shape, so
 *    each call first clears the counters it is about to use (one small cudaMemsetAsync on `stream`, ahead of the
 *    kernel).  Nothing needs zero-filling by the caller, also not after a launch that failed.
 *  - First call on each GPU: the library looks up the array's device address (cudaGetSymbolAddress, with that GPU
 *    current; this may load the library's device image) and remembers it per device.  Make that first call outside
 *    any stream capture, e.g. once at start-up on each GPU; later calls do no such look-up.
 * Arguments and errors otherwise exactly as hx_decode_attention.  Size checks run on the host before any CUDA call. */
#define HX_NOALLOC_SCRATCH_BYTES ((size_t)20 * 1024 * 1024)
int hx_decode_attention_noalloc(void* out, const void* q,
                                const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                                const int32_t* block_table, int32_t block_table_stride,
                                const int32_t* seq_lens,
                                int32_t batch, int32_t max_seq_len, float sm_scale,
                                void* stream);

/* Fused append-then-attend (F1): the same result, bit for bit, in the cache AND in `out`, as
 * hx_kv_append(k_new, v_new, ...) followed by hx_decode_attention(...), in ONE launch: the warp
 * that streams the last page of (request, kv head) overlays the new K/V row on the tile in shared
 * memory and stores it to the page.  Arguments as in the two calls. */
int hx_decode_attention_append(void* out, const void* q, const void* k_new, const void* v_new,
                               const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                               const int32_t* block_table, int32_t block_table_stride,
                               const int32_t* seq_lens,
                               int32_t batch, int32_t max_seq_len, float sm_scale,
                               void* workspace, size_t workspace_bytes,
                               void* stream);

/* ---- (c) paged prefill attention -------------------------------------
 * "the prefill phase processes the request's input tokens all at once" (compute-bound);
 * PAPER.md:L110 integrates FlashAttention for it.  Causal attention of the LAST q_lens[i] tokens of
 * request i over its paged context of seq_lens[i] tokens (reading S24): query r (0 <= r < q_lens[i])
 * sits at position p = seq_lens[i] - q_lens[i] + r and attends to cached tokens t = 0..p,
 *
 *   out[cu_q_lens[i] + r][h] = sum_{t<=p} softmax_t(sm_scale * <q[cu_q_lens[i]+r][h], K_t>) V_t
 *
 * with K_t, V_t read through the block table as in hx_decode_attention (kv head h / G).  q_lens ==
 * seq_lens is a whole-prompt prefill over a cache the prompt's K/V were already written to;
 * q_lens < seq_lens is a chunked prefill; q_lens == 1 equals hx_decode_attention.
 * Runs on tcgen05 tensor cores (fp16 in, fp32 accumulate in tensor memory, fp16 out).
 *
 * out, q       : device fp16 [total_q_tokens][q_heads][head_dim], rows packed by request, 16-byte aligned.
 * q_lens       : device int32 [batch], 0 <= q_lens[i] <= seq_lens[i] (device-side contract).
 * cu_q_lens    : device int32 [batch+1], exclusive prefix sums of q_lens.
 * total_q_tokens, max_q_len, max_seq_len : host copies for launch sizing and checks.
 * HX_ERR_UNSUPPORTED: head_dim not in {64,128}, group size not in {1,2,4,8,16}. */
int hx_prefill_attention(void* out, const void* q,
                         const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                         const int32_t* block_table, int32_t block_table_stride,
                         const int32_t* seq_lens, const int32_t* q_lens, const int32_t* cu_q_lens,
                         int32_t batch, int32_t total_q_tokens, int32_t max_q_len, int32_t max_seq_len,
                         float sm_scale, void* stream);

/* ---- (b') per-step plan for the layer calls of a decode step ------------------------------
 * A model calls hx_decode_attention once per layer (80 times per step for LLaMA-2-70B), every time with the SAME
 * seq_lens and block table (reading S9: one table serves every layer).  What the kernel derives from those two
 * alone - the page-count prefix sums, the work partition (row A4) and, per (request, kv head, page) tile, the cache
 * row to load - can be computed once per step: hx_decode_plan writes it into a caller-owned device buffer, and
 * hx_decode_attention_planned is hx_decode_attention reading that buffer instead of seq_lens / block_table (its
 * first K/V load is issued after one L2 round trip instead of a scan, a search and a table load).  Same work
 * partition, same arithmetic: the result is bit-identical to hx_decode_attention's.
 *
 * plan        : device, 16-byte aligned, >= hx_decode_plan_bytes(batch, cache->kv_heads, max_seq_len, page_size)
 *               bytes.  Valid for the (seq_lens, block_table, batch, q_heads, kv_heads) it was made from, on the
 *               device it was made on, until one of them changes; any number of layer calls may read it.
 * batch       : <= 2048 (HX_ERR_UNSUPPORTED above).
 * Device-side contract: the plan passed to hx_decode_attention_planned was written by hx_decode_plan with the same
 * batch and head counts (the kernel checks the plan's header and traps on a mismatch). */
size_t hx_decode_plan_bytes(int32_t batch, int32_t kv_heads, int32_t max_seq_len, int32_t page_size);

int hx_decode_plan(void* plan, size_t plan_bytes,
                   const hx_paged_cache* cache, int32_t q_heads,
                   const int32_t* block_table, int32_t block_table_stride,
                   const int32_t* seq_lens,
                   int32_t batch, int32_t max_seq_len,
                   void* stream);

int hx_decode_attention_planned(void* out, const void* q,
                                const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                                const void* plan, size_t plan_bytes,
                                int32_t batch, int32_t max_seq_len, float sm_scale,
                                void* workspace, size_t workspace_bytes,
                                void* stream);

/* hx_decode_attention_planned launched as a PROGRAMMATIC DEPENDENT of whatever kernel precedes it on `stream`
 * ("asynchronous ... to enable overlapping"; a model issues one attention call per layer, and a call of
 * configs[2]'s size is so short that its launch latency, set-up and the tail in which its last warps finish are a fifth
 * of it).  Same arguments and bit-identical result.  The grid may be placed on an SM as soon as the preceding kernel
 * has left it (this library's kernels release their dependents as soon as they start; any other kernel does when it
 * exits, which makes this a plain launch), and
 *   inputs_ready == 0: it reads nothing from device memory until the preceding kernel has completed and its writes are
 *                      visible (griddepcontrol.wait): safe behind ANY kernel, e.g. the projection that produced q and
 *                      the append that wrote this token's K/V; launch latency and barrier/descriptor set-up overlap.
 *   inputs_ready != 0: the CALLER asserts that nothing this call reads (q, the plan, this layer's K/V) is written by the
 *                      kernel directly before it on `stream`.  The grid then streams its first K/V ranges under that
 *                      kernel's tail; every global write (out, workspace) still waits for that kernel's completion, so
 *                      consecutive calls may share `workspace` and `out`.
 * In both modes every CTA waits for the preceding kernel before it exits: work enqueued after this call is ordered
 * after both.  Nothing may be enqueued on `stream` between the preceding kernel and this call for the overlap to
 * happen (an event record in between turns it into a plain launch; the result is the same). */
int hx_decode_attention_chained(void* out, const void* q,
                                const hx_paged_cache* cache, int32_t layer, int32_t q_heads,
                                const void* plan, size_t plan_bytes,
                                int32_t batch, int32_t max_seq_len, float sm_scale,
                                void* workspace, size_t workspace_bytes,
                                int32_t inputs_ready, void* stream);

/* ---- host page allocator (paging by citation PAPER.md:L110, OOM
 * remark PAPER.md:L136).  A free list of page ids; alloc is all-or-nothing.  Not thread-safe. */
typedef struct hx_page_pool hx_page_pool;
int     hx_pool_create(hx_page_pool** out, int32_t num_pages);
int     hx_pool_shuffle(hx_page_pool* pool, uint64_t seed);  /* randomise free-list order (deterministic in seed) */
int     hx_pool_alloc(hx_page_pool* pool, int32_t n, int32_t* out_page_ids /* host [n] */);
int     hx_pool_free(hx_page_pool* pool, const int32_t* page_ids /* host [n] */, int32_t n); /* double free / bad id -> INVALID_ARG, nothing freed */
int32_t hx_pool_num_free(const hx_page_pool* pool);
int32_t hx_pool_num_pages(const hx_page_pool* pool);
/* Allocate ceil(seq_lens[i]/page_size) pages for each of `batch` requests and write their rows
 * into a HOST block table [batch][stride] (unused entries = -1).  All or nothing. */
int     hx_pool_alloc_table(hx_page_pool* pool, const int32_t* seq_lens, int32_t batch,
                            int32_t page_size, int32_t* block_table, int32_t stride);
void    hx_pool_destroy(hx_page_pool* pool);

/* ---- whole decode step on DEVICE buffers (bench.py's timed step) --------
 * KV cache communication is asynchronous "to enable overlapping between computation and
 * communication".  One call = hx_kv_ingest of the step's new prompts (ing_* arguments; skipped when
 * ing_batch == 0) + hx_decode_attention over the active batch (skipped when batch == 0).  Every argument means
 * what it means in those two calls.
 * overlap_ingest == 0: ingest, then attention, in order on `stream` (the attention may read the new pages).
 * overlap_ingest != 0: the caller asserts that the attention does NOT read the pages this step ingests (the new
 * prompts join the batch in a later step).  Both parts are HBM-bound, so side by side they would only share the
 * bandwidth; what CAN be won is the slack of the attention's uneven finish (its warps end up to tens of microseconds
 * apart).  The step is therefore ONE kernel: the attention kernel carries the handoff, and every warp that has
 * finished its attention range moves (page, head) tiles of the new prompts with the copy engines (one TMA tensor load
 * of the tile's 16 token rows into the warp's shared-memory ring, one bulk store into the page), claiming units from
 * a counter until none are left.  Work enqueued on `stream` afterwards is ordered after both parts.  Uses the last 16
 * bytes of `workspace` (two counters that every call leaves at zero).  The fused kernel is used when batch <= 2048, the
 * handoff is not empty and at most 8 source shards hold this rank's heads; otherwise the two kernels run in order, which is
 * always allowed (hx_decode_step_is_fused tells which).  The shards may be in this device's memory, in pinned host memory
 * or in a peer GPU's memory with peer access enabled: in the last two cases the fused step is a PULL-mode handoff (F2;
 * PAPER.md:L110), the copy engines fetch each tile over the link straight into its page.
 * block-table rows of the handoff: entries [ceil(n_i/page_size), ceil(ing_max_seq_len/page_size)) of a row may be
 * READ by the fused kernel (they lie inside the row) but are never used.  ing_max_seq_len must not be smaller than
 * any ing_seq_lens[i] (device-side contract): the fused kernel enumerates a prompt's pages up to it.
 * Every host-side check of both calls runs first, size limits of the launches included; nothing is enqueued unless
 * all pass.  (The one check that needs the device - that it offers the shared memory per CTA the kernels use - runs
 * when the first kernel of a kind is launched on that device; it cannot fail on sm_100.)  Capturable in a CUDA graph. */
typedef struct {
  /* attention over the active batch (hx_decode_attention) */
  void*       out;               /* device fp16 [batch][q_heads][head_dim] */
  const void* q;                 /* device fp16 [batch][q_heads][head_dim] */
  const hx_paged_cache* cache;
  int32_t layer, q_heads;
  const int32_t* block_table; int32_t block_table_stride;   /* device */
  const int32_t* seq_lens;       /* device [batch] */
  int32_t batch, max_seq_len;
  float sm_scale;
  void* workspace; size_t workspace_bytes;
  /* handoff of the step's new prompts (hx_kv_ingest into `cache`, layers [0, ing_layers)) */
  const void* const* src_k; const void* const* src_v;       /* host arrays of src_tp device pointers */
  int32_t ing_layers, heads, src_tp, dst_tp, dst_rank;
  const int32_t* ing_block_table; int32_t ing_block_table_stride;   /* device [ing_batch][stride] */
  const int32_t* ing_cu_seqlens;  const int32_t* ing_seq_lens;      /* device */
  int32_t ing_batch, ing_total_tokens, ing_max_seq_len;
  int32_t overlap_ingest;
  /* optional timing: cudaEvent_t handles (or NULL) recorded directly before / after the ingest kernel and directly
   * before / after the attention kernel.  With overlap_ingest != 0 nothing may sit between the two launches, so both
   * "begin" events are recorded before the pair and both "end" events after it. */
  void* ev_ingest_begin; void* ev_ingest_end; void* ev_attention_begin; void* ev_attention_end;
} hx_step_args;
int hx_decode_step(const hx_step_args* args, void* stream);

/* Would hx_decode_step(args) run as the ONE fused kernel?  Runs the same checks and the same decision as the call itself
 * and enqueues nothing: *fused = 1 when overlap_ingest != 0, both halves have work and the copy engines can take the
 * handoff (see above), else 0 (the step then runs its two kernels in order).  Errors as hx_decode_step. */
int hx_decode_step_is_fused(const hx_step_args* args, int32_t* fused);

/* Destroys the library-owned side streams and events of every device (after synchronising them; only
 * hx_decode_step_host with overlap_ingest creates them).  Optional: call when no such call is in flight; a later
 * call re-creates them. */
int hx_shutdown(void);

/* ---- whole decode step with HOST inputs (bench.py "e2e") --------
 * Copies q, the new prompts' block-table rows / lengths and the source shards from (pinned)
 * host memory to caller-provided device staging buffers, runs hx_kv_ingest for the new
 * prompts then hx_decode_attention over the active batch on `stream`, and copies `out` back to
 * host.  Asynchronous like the rest; the caller synchronises `stream` before reading out_host.
 * See hx_step_host_args for the buffers. */
typedef struct {
  /* attention over the active batch */
  const void* q_host;            /* host fp16 [batch][q_heads][head_dim] */
  void*       out_host;          /* host fp16 [batch][q_heads][head_dim] */
  void*       q_dev;             /* device staging, same size */
  void*       out_dev;           /* device staging, same size */
  const hx_paged_cache* cache;
  int32_t layer, q_heads;
  const int32_t* block_table_dev; int32_t block_table_stride;   /* device, active batch */
  const int32_t* seq_lens_dev;    int32_t batch, max_seq_len;
  float sm_scale;
  void* workspace; size_t workspace_bytes;
  /* ingest of the step's new prompts (ing_batch == 0 -> skipped) */
  const void* const* src_k_host; const void* const* src_v_host; /* host arrays of src_tp HOST shard pointers */
  void* const* src_k_dev;        void* const* src_v_dev;        /* host arrays of src_tp DEVICE staging pointers */
  int32_t ing_layers, heads, src_tp, dst_tp, dst_rank;
  const int32_t* ing_block_table_host; int32_t ing_block_table_stride; /* host [ing_batch][stride] */
  const int32_t* ing_cu_seqlens_host;  const int32_t* ing_seq_lens_host;
  int32_t* ing_block_table_dev; int32_t* ing_cu_seqlens_dev; int32_t* ing_seq_lens_dev; /* device staging */
  int32_t ing_batch, ing_total_tokens, ing_max_seq_len;
  /* F2 pull mode ("asynchronous ... to enable overlapping"): non-zero =
   * do NOT stage the shards; hx_kv_ingest reads them through src_k_host/src_v_host directly, over
   * the link, fusing transfer + head regroup + page scatter in one kernel.  The pointers must then
   * be reachable from the device: pinned host memory (UVA) or a peer GPU's memory with peer access
   * enabled.  src_k_dev/src_v_dev are ignored. */
  int32_t pull_src;
  /* non-zero = the step's attention does NOT read the pages this step ingests (the new prompts join the
   * batch later; "asynchronous ... to enable overlapping between computation and
   * communication"): the shard transfer + ingest run on a library-owned side stream, forked from `stream`
   * at entry and joined to it before return (on every path, errors included), so PCIe and the ingest overlap
   * the attention.  0 = everything in order on `stream` (the attention may read the freshly ingested pages).
   * As in hx_decode_step, every host-side check runs before anything is enqueued. */
  int32_t overlap_ingest;
} hx_step_host_args;
int hx_decode_step_host(const hx_step_host_args* args, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* HX_H_ */
