/*
 * shuntstage.h — C-ABI of libshuntstage.so: the forward pass of ONE pipeline stage of ShuntServe
 * (arxiv/paper_2606_18600), hand-written CUDA for sm_100a.
 *
 * What a "stage" is: the contiguous range of decoder layers [l0,l1) that the paper's placement optimizer
 * assigns to one node (§2.3 "uneven layer partitioning"; Algorithm 1 line 9 `add_stage(i,
 * l_new)`).  Its input and output is the hidden-state tensor [tokens, H] of E-byte elements that
 * crosses stage boundaries (Eq. 2; E = 2, bf16).  The operations inside a layer
 * are the ones Table 2 costs: QKV projection, attention (prefill / decode), output
 * projection, up-and-gate projection, down projection, logits — "the de-facto standard of transformer-based
 * generative LLMs", i.e. the public Llama-3 / Qwen3 pre-norm decoder layer.  The two calls are
 *   - ss_stage_decode : one batched decode iteration over a paged GQA KV cache ("memory-bound decode",
 *                       PAPER.md:21, 96, 222);
 *   - ss_stage_prefill: causal prefill; this is also the compute of the paper's output-preserving request
 *                       migration, which re-runs "input sequence and already-generated output sequence" to
 *                       reconstruct the KV cache (§5.1).
 *
 * All pointers named "dev" are CUDA device pointers, all others are host pointers.  Nothing in this header is
 * a torch type.  A stage never allocates or frees device memory: weights, KV pool, workspace, inputs and
 * outputs are BORROWED from the caller (this mirrors the paper's engine, which attaches to tensors owned by the
 * Shared Tensor Store).  Borrowed pointers must stay valid and unchanged until ss_stage_destroy.
 * The one exception in the library is the store side of that mechanism itself: ss_store_alloc / ss_store_free wrap
 * cudaMalloc / cudaFree so that the arena is a whole allocation and therefore exportable over CUDA IPC.
 *
 * Calls enqueue work on the stage's CUDA stream and return; results are valid after the caller synchronises
 * that stream.  Errors that the host can detect are returned synchronously and nothing is enqueued.  A stage
 * is not thread-safe; distinct stages are independent.
 *
 * Environment variables read by the library (all at ss_stage_create, none afterwards; there are no others in a
 * product build — the GEMM tuning overrides exist only in builds compiled with -DSS_TUNE):
 *   SS_DEBUG=1    every call first runs the device-side contract checks described at ss_stage_debug_info and waits
 *                 for their verdict (one stream synchronisation per call);
 *   SS_NO_GRAPH=1 ss_stage_decode enqueues its kernels directly instead of replaying a captured CUDA graph;
 *   SS_NO_PDL=1   kernels are launched without programmatic dependent launch (plain stream order);
 *   SS_ATTN_LAZY=n (0..64, default 16) the prefill attention moves a row's running maximum only when a key tile exceeds
 *                 it by more than 2^n, and then rescales its accumulator in place; n changes rounding only (O / l is the
 *                 same quotient).  A test aid: with 0 every growth of the maximum takes the rescale path.
 * SS_NO_GRAPH and SS_NO_PDL change scheduling only, never results (tests compare them bit for bit).
 *
 * Readings of points the paper leaves open are listed in DESIGN.md ("Readings"), numbered A1..A22 after
 * SURVEY.md §8(c).
 */
#ifndef SHUNTSTAGE_H
#define SHUNTSTAGE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- error codes (0 = OK, negative = error) ------------------------------------------------------------ */
#define SS_OK                 0
#define SS_ERR_INVALID_ARG   -1  /* null / contradictory pointers, l0>=l1, both or neither of hidden/token_ids */
#define SS_ERR_UNSUPPORTED   -2  /* head_dim not in {64,128}, page_size != 16, n_q % n_kv != 0, G > 16,
                                    hidden/ffn/n_q*d not multiples of 8, hidden > 16384, misaligned pointers */
#define SS_ERR_CAPACITY      -3  /* tokens / seqs / max_blocks over the dims' maxima; pool or workspace too small */
#define SS_ERR_NO_PAGES      -4  /* ss_kv_alloc: fewer than n pages free — nothing was allocated */
#define SS_ERR_BAD_PAGE      -5  /* ss_kv_free: id out of range or already free — nothing was freed */
#define SS_ERR_CUDA          -6  /* a CUDA runtime/driver call failed; see ss_last_cuda_error */

typedef struct ss_stage ss_stage; /* opaque */

/* Model dimensions (Table 3 notation: H = hidden, H_kv = n_kv_heads*head_dim (reading A2),
 * H_ffn = ffn, V = vocab) and the capacity of one call. */
typedef struct {
  int32_t hidden;            /* H */
  int32_t n_q_heads;         /* query heads; Hq = n_q_heads*head_dim (may differ from H: Qwen3-32B, A4) */
  int32_t n_kv_heads;        /* KV heads; q heads [h*G,(h+1)*G) share kv head h, G = n_q/n_kv (A16) */
  int32_t head_dim;          /* d: 64 or 128 */
  int32_t ffn;               /* H_ffn */
  int32_t n_layers_total;    /* layers of the whole model; l1 <= n_layers_total */
  int32_t vocab;             /* V; used only when edge weights are given */
  float   rms_eps;           /* RMSNorm epsilon (also the per-head QK-norm epsilon) (A8) */
  float   rope_theta;        /* RoPE base; inv_freq[c] = theta^(-2c/d), rotate-half pairing (A10) */
  int32_t qk_norm;           /* 0 Llama; 1 Qwen3: per-head RMSNorm on q and k before RoPE, gain [d] (A11) */
  int32_t page_size;         /* tokens per KV page; must be 16 */
  int32_t max_pos;           /* RoPE table length: positions 0..max_pos-1 are legal */
  int32_t max_tokens;        /* capacity T of one prefill call (a decode call needs batch <= max_seqs) */
  int32_t max_seqs;          /* capacity: sequences per call */
  int32_t max_blocks_per_seq;/* capacity: block-table row length */
} ss_model_dims;

/* Per-layer weights: dev pointers, bf16, row-major [out_features, in_features] ("K-major": row n is the weight
 * vector of output feature n), no biases (A7).  Every pointer 16-byte aligned.  Borrowed. */
typedef struct {
  const void *ln1;     /* [H]        RMSNorm gain before attention                           (step S1) */
  const void *wq;      /* [Hq, H]    Table 2 "QKV Projection", PAPER.md:141-142              (S2) */
  const void *wk;      /* [Hkv, H] */
  const void *wv;      /* [Hkv, H] */
  const void *q_norm;  /* [d] or NULL when qk_norm == 0                                      (S3) */
  const void *k_norm;  /* [d] or NULL */
  const void *wo;      /* [H, Hq]    Table 2 "Output Projection", PAPER.md:145-146           (S7) */
  const void *ln2;     /* [H]        RMSNorm gain before the FFN                             (S8) */
  const void *w_gate;  /* [F, H]     Table 2 "Up and Gate Projection", PAPER.md:147-148      (S9) */
  const void *w_up;    /* [F, H] */
  const void *w_down;  /* [H, F]     Table 2 "Down Projection", PAPER.md:149-150             (S10) */
} ss_layer_weights;

/* Optional first-/last-stage weights (dev, bf16, borrowed).  Any member may be NULL. */
typedef struct {
  const void  *embed;       /* [V, H]: needed for token_ids input (stage 0 takes tokens)  (S0) */
  const void  *final_norm;  /* [H]                                                                     (S11) */
  const void  *lm_head;     /* [V, H]: Table 2 "Logits Calculation", PAPER.md:151-152                   (S11) */
  const float *inv_freq;    /* HOST pointer, [d/2] fp32, or NULL -> theta^(-2c/d); read at create only */
} ss_edge_weights;

/* Bytes of caller-allocated device workspace a stage with these dims and layer range needs. 0 on bad dims. */
size_t ss_stage_workspace_bytes(const ss_model_dims *dims, int l0, int l1);

/* Bytes of one KV page over all layers of the stage: (l1-l0) * 2 * n_kv_heads * 16 * head_dim * 2. */
size_t ss_kv_page_bytes(const ss_model_dims *dims, int l0, int l1);

/*
 * Create a stage for layers [l0,l1).  `layers` is a HOST array of l1-l0 structs (copied).  `edge` may be NULL.
 * kv_pool: dev, 256-byte aligned, layout (bf16, contiguous; part of the contract because page contents are
 * compared bit for bit):
 *     pool[layer - l0][kv in {0:K,1:V}][page][h_kv][slot 0..15][c 0..d-1]
 * with num_pages = kv_pool_bytes / ss_kv_page_bytes(); the token at position p of a sequence whose block-table
 * row is bt lives in page bt[p >> 4], slot p & 15 (paged KV cache: PAPER.md:265, 271; [31] PAPER.md:540).
 * workspace: dev, 256-byte aligned, >= ss_stage_workspace_bytes().  cuda_stream: a cudaStream_t (may be 0).
 * The call uploads the RoPE table and builds TMA descriptors; it synchronises the stream once.
 */
int ss_stage_create(ss_stage **out, const ss_model_dims *dims, int l0, int l1,
                    const ss_layer_weights *layers, const ss_edge_weights *edge,
                    void *kv_pool, size_t kv_pool_bytes,
                    void *workspace, size_t workspace_bytes,
                    void *cuda_stream);
int ss_stage_destroy(ss_stage *st);

/* Page pool (host-side free list over page ids 0..num_pages-1; no device work). */
int ss_kv_num_pages(const ss_stage *st);
int ss_kv_num_free(const ss_stage *st);
int ss_kv_alloc(ss_stage *st, int n, int32_t *out_page_ids /* host, [n] */);   /* all-or-nothing */
int ss_kv_free(ss_stage *st, int n, const int32_t *page_ids /* host, [n] */);  /* all-or-nothing */

/* The same page allocator stand-alone: host-only, no device and no stage needed (a scheduler can size and drive a
 * pool before any stage exists; the stage's ss_kv_* calls run this code on its own pool).  LIFO free list;
 * ss_pool_alloc hands out n distinct free ids or nothing (SS_ERR_NO_PAGES); ss_pool_free returns n ids or nothing
 * (SS_ERR_BAD_PAGE on an id out of range, already free, or repeated within the call).  Paged KV: PAPER.md:265, 271. */
typedef struct ss_pool ss_pool;
int ss_pool_create(ss_pool **out, int num_pages);
int ss_pool_destroy(ss_pool *p);
int ss_pool_num_pages(const ss_pool *p);
int ss_pool_num_free(const ss_pool *p);
int ss_pool_alloc(ss_pool *p, int n, int32_t *out_page_ids /* host, [n] */);
int ss_pool_free(ss_pool *p, int n, const int32_t *page_ids /* host, [n] */);

/*
 * Causal prefill of n_seqs packed sequences (steps S0-S11 of DESIGN.md; migration recompute).
 * Token i of sequence s sits in packed row cu_q[s]+i and at global position ctx_before[s]+i; it attends keys
 * 0..ctx_before[s]+i, which are read from the pages (including those this call appends).  Rows with q_len = 1
 * are legal, so a mixed decode+prefill iteration is one call (A19: decode rows first).
 *   hidden_bf16 XOR token_ids: dev [T,H] bf16, or dev [T] int32 (needs edge->embed and l0 == 0).
 *   cu_q: dev int32 [n_seqs+1], cu_q[0] = 0, cu_q[n_seqs] = total_tokens.  ctx_before: dev int32 [n_seqs].
 *   block_tables: dev int32 [n_seqs, max_blocks]; pages for positions [0, ctx_before+q_len) must be listed.
 *   out_hidden_bf16: dev [T,H] or NULL (every token: the next stage needs all of them to build its KV).
 *   out_logits: dev fp32 [n_seqs,V] or NULL; out_argmax: dev int32 [n_seqs] or NULL — for the LAST token of
 *   each sequence; need edge->final_norm and edge->lm_head.  argmax ties resolve to the lowest index.
 */
int ss_stage_prefill(ss_stage *st, int n_seqs,
                     const void *hidden_bf16, const int32_t *token_ids,
                     const int32_t *cu_q, const int32_t *ctx_before,
                     const int32_t *block_tables, int max_blocks, int total_tokens,
                     void *out_hidden_bf16, float *out_logits, int32_t *out_argmax);

/* Mixed iteration of online serving (continuous batching: decode requests and prefill chunks share one pass over the
 * weights; the paper's online experiments; BASELINE.json configs[4]).  Same arguments, semantics
 * and errors as ss_stage_prefill, plus one HOST hint: the first n_decode_rows sequences of the batch are decode
 * requests, i.e. have q_len == 1 (cu_q[s+1] - cu_q[s] == 1 for s < n_decode_rows; "decode rows first").  Their
 * attention then runs in the page-balanced GQA decode kernel instead of one 64-row causal tile per (row, head).
 * Results are those of ss_stage_prefill on the same arguments.  A hint that does not hold is undefined behaviour.
 * n_decode_rows = 0 is ss_stage_prefill; n_decode_rows = n_seqs = total_tokens is a decode step expressed through
 * cu_q.  SS_ERR_INVALID_ARG if n_decode_rows < 0 or > n_seqs. */
int ss_stage_mixed(ss_stage *st, int n_decode_rows, int n_seqs,
                   const void *hidden_bf16, const int32_t *token_ids, const int32_t *cu_q,
                   const int32_t *ctx_before, const int32_t *block_tables, int max_blocks, int total_tokens,
                   void *out_hidden_bf16, float *out_logits, int32_t *out_argmax);

/*
 * One decode iteration for `batch` sequences, one new token each (Table 2 "Decode" rows).
 * context_lens[b] = tokens already cached (A20); the new token's K/V are appended at that position by the
 * attention kernel itself and attended to.  The page bt[b][context_lens[b] >> 4] must exist.
 *   hidden_bf16 XOR token_ids: dev [B,H] bf16 / dev [B] int32.   block_tables: dev int32 [B, max_blocks].
 *   out_hidden_bf16 dev [B,H] or NULL; out_logits dev fp32 [B,V] or NULL; out_argmax dev int32 [B] or NULL.
 * The kernel sequence of a decode call is captured into a CUDA graph per (batch, max_blocks, output kind) and
 * replayed; user pointers are passed through a small device-side argument block, so they may change per call.
 */
int ss_stage_decode(ss_stage *st, int batch,
                    const void *hidden_bf16, const int32_t *token_ids,
                    const int32_t *block_tables, int max_blocks, const int32_t *context_lens,
                    void *out_hidden_bf16, float *out_logits, int32_t *out_argmax);

/* Number of kernels the stage launched (directly or inside replayed graphs) since creation. */
int64_t ss_stage_launch_count(const ss_stage *st);

/* Batch-invariant mode (the paper's migration is OUTPUT-PRESERVING: recomputing prompt + generated
 * tokens must reconstruct the KV cache the incremental decode built).  In the default mode the GPU reproduces that only
 * up to the summation order of its kernels (a stream-K cut, an attention split and a reduction tree that depend on how
 * many rows a call has: KV equal or within 2 bf16 ulp).  With on != 0 every reduction of a token row is done in an order
 * that depends on that row alone — projections: every output tile's whole K by one CTA, k-blocks in order, one
 * accumulator; RMSNorm: one reduction tree; attention: each (row, kv head) walked from page 0 to its last page by one
 * warp of the decode kernel, prefill tokens included, no split and no merge — so ss_stage_prefill over prompt + generated
 * tokens leaves KV pages and next-token hidden states BIT-IDENTICAL to prefill of the prompt followed by ss_stage_decode
 * steps, whatever the batch composition or chunking (tests/test_gpu_parity.py).  It is an opt-in exactness mode: the
 * projections lose stream-K's load balance and prefill attention re-reads the keys per token (cost in DESIGN.md).
 * Switching synchronises the stream and drops the captured decode graphs. */
int ss_stage_set_batch_invariant(ss_stage *st, int on);

/* Tensor parallelism inside a stage.  A rank of a D_TP-way stage is an
 * ordinary ss_stage created with that rank's SHARD: dims.n_q_heads, n_kv_heads and ffn divided by D_TP (hidden
 * unchanged), wq/wk/wv and w_gate/w_up = the rank's rows, wo = the rank's columns [H, Hq/D_TP] and w_down = [H, F/D_TP]
 * (each a contiguous matrix), norms replicated, and its own KV pool holding only its kv heads.  Once an all-reduce is
 * registered here the O and down projections produce fp32 partials [T, H] and the stage calls
 *     fn(partial, T * H, user, cuda_stream)
 * twice per layer (the two all-reduces of Eq. 3) — fn must enqueue, on `cuda_stream`, an in-place SUM of `partial`
 * across the ranks (e.g. ncclAllReduce) and return 0 without synchronising — then adds the sum to the fp32 residual.
 * A non-zero return aborts the call: nothing further is enqueued and the stage call returns SS_ERR_CUDA.
 * Decode steps are not graph-captured in this mode.  fn = NULL returns the stage to single-GPU operation. */
typedef int (*ss_allreduce_fn)(float *partial_dev, size_t count, void *user, void *cuda_stream);
int ss_stage_set_allreduce(ss_stage *st, ss_allreduce_fn fn, void *user);

/* The same all-reduce FUSED into the projections (Eq. 3), for decode-sized calls
 * (tokens <= 128), with no collective library call and no host callback, so the decode step stays one CUDA graph:
 *   gather  — the O / down projection's epilogue warps store every stream-K piece of their accumulator into the
 *             exchange buffer of EVERY rank (plain stores to peer-mapped memory: over NVLink for the other ranks), then
 *             each CTA raises, with system scope, one arrival counter per rank;
 *   wait    — each rank's STREAM waits until all ranks' counters in its own buffer have reached the grid size
 *             (cuStreamWaitValue32) and re-arms them; no kernel ever spins on another rank;
 *   reduce  — the consumer kernel that runs next anyway (residual add + RMSNorm) adds the pieces of all ranks in
 *             (rank, CTA) order: every rank gets the same bits, and each value crosses the link exactly once per peer.
 * Every rank allocates one exchange buffer of ss_tp_xchg_bytes(tp_size) bytes (device, 256-byte aligned; across
 * processes a whole allocation made by ss_store_alloc, handed over with ss_store_export / ss_store_attach; with peer
 * access enabled) and passes the device addresses of ALL ranks' buffers, indexed by rank, as xchg_dev (HOST array of
 * tp_size pointers; xchg_dev[rank] is its own).  The call zeroes this rank's counters: no rank may start its first step
 * before every rank has returned from it.  Two buffers alternate inside (O, down), which is enough because a rank cannot
 * run more than one all-reduce point ahead of another.  Calls with more than 128 tokens (prefill) use the callback of
 * ss_stage_set_allreduce, which a shard with tp_size > 1 must also register.  size = 0 switches the mode off.
 * SS_ERR_INVALID_ARG (rank / size / null or misaligned pointers), SS_ERR_UNSUPPORTED (no stream memory operations). */
size_t ss_tp_xchg_bytes(int tp_size);
int ss_stage_set_tp_fused(ss_stage *st, int rank, int size, void *const *xchg_dev);

/* Migration by KV transfer (the alternative to recomputation the paper measures; SURVEY
 * 8(f) NEXT-4).  ss_kv_export gathers the n pages `page_ids_dev[0..n)` (DEVICE int32) of every layer of the stage into
 * the caller's contiguous DEVICE buffer, laid out [layer][K/V][i][h_kv][16][d] bf16 (n * ss_kv_page_bytes() bytes) —
 * the message a GPU-to-GPU copy carries; ss_kv_import scatters such a buffer into the pages `page_ids_dev` of this
 * stage's pool (ids chosen by the importing side, e.g. from ss_kv_alloc).  Byte-exact copies, enqueued on the stage's
 * stream.  Errors: SS_ERR_INVALID_ARG (null / n <= 0), SS_ERR_UNSUPPORTED (buffer not 16-byte aligned),
 * SS_ERR_CAPACITY (buffer too small).  Page ids out of range are undefined behaviour. */
int ss_kv_export(ss_stage *st, int n, const int32_t *page_ids_dev, void *buf_dev, size_t buf_bytes);
int ss_kv_import(ss_stage *st, int n, const int32_t *page_ids_dev, const void *buf_dev, size_t buf_bytes);

/* Number of decode CUDA graphs the stage has captured so far (0 while SS_NO_GRAPH=1 or while an all-reduce CALLBACK is
 * in use; the fused tensor-parallel mode keeps its graphs). */
int64_t ss_stage_graph_count(const ss_stage *st);

/* Device-side contract checks: block tables, context lengths, cu_q and token ids live in
 * device memory, so the host cannot validate them, and in a normal run a violation is undefined behaviour (a page id
 * out of range writes outside the pool).  In a stage created while SS_DEBUG=1 is set, ss_stage_prefill / mixed / decode
 * and ss_kv_export / import first run a checking kernel and synchronise: every listed page id of positions
 * [0, ctx + q_len) must lie in [0, num_pages); ctx >= 0; ctx + q_len <= max_blocks * 16 and <= dims.max_pos; cu_q[0] = 0,
 * cu_q[n_seqs] = total_tokens, q_len >= 1 (= 1 for the decode rows of a mixed call); token ids in [0, vocab).  On a
 * violation the call returns SS_ERR_INVALID_ARG, nothing else is enqueued (pool and workspace untouched), and
 * ss_stage_debug_info reports the first violation found: out = {code, sequence (-1: none), index, offending value} with
 * code 1 page id out of range (index = block-table column, or position in page_ids for export / import), 2 ctx + q_len
 * beyond the listed pages, 3 beyond max_pos, 4 token id out of range (index = token), 5 malformed cu_q, 6 negative
 * context.  Returns 1 if the stage runs with the checks on, 0 if not, SS_ERR_INVALID_ARG on null arguments. */
int ss_stage_debug_info(const ss_stage *st, int32_t out[4]);

/* Debug aid: device address and size of one of the stage's workspace tensors, as the last call left it (valid after the
 * caller synchronises the stream).  Names: "x" fp32 [T,H] residual stream (after a call: the stage output before the
 * bf16 hand-off); "h" bf16 [T,H] last RMSNorm output; "qkv" fp32 [T,Hq+2Hkv] last QKV projection (S2); "q" bf16 [T,Hq]
 * last layer's queries after QK-norm + RoPE (S3, S4); "attn" bf16 [T,Hq] last attention output (S6); "a" bf16 [T,F] last
 * SwiGLU output (S9).  Used by the per-step parity tests.  SS_ERR_INVALID_ARG on an unknown name. */
int ss_stage_debug_tap(const ss_stage *st, const char *name, void **dev_ptr_out, size_t *bytes_out);

/* ---- op-level entry points (the same kernels the stage uses; for per-kernel parity tests and profiling) -- */

/* Scratch (dev, 256-byte aligned) the op-level GEMMs need for the stream-K fix-up: >= this many bytes, whose first
 * 1024 bytes must be ZERO before the first call (the kernel leaves them zero). */
size_t ss_op_gemm_scratch_bytes(void);

/* Debug aid.  `host_mapped_u64x4` is pinned, device-mapped HOST memory of 4 x uint64 (or NULL to disable).  Every
 * wait inside the GEMM kernel is bounded; when one expires the kernel stores {site id, block<<32|thread,
 * info<<32|parity} there and traps (the call then fails with SS_ERR_CUDA), so a protocol bug is a located error and
 * never a hung GPU.  Returns SS_OK or SS_ERR_CUDA. */
int ss_debug_buffer(void *host_mapped_u64x4);

/* C[T, N] (fp32, row-major, ld = N) = X[T, K] (bf16, row-major) * W[N, K]^T (bf16) through the persistent
 * tcgen05/TMEM GEMM.  K % 8 == 0.  Asynchronous on cuda_stream. */
int ss_op_gemm_bf16(const void *x_dev, const void *w_dev, float *c_dev, int T, int N, int K,
                    void *scratch_dev, size_t scratch_bytes, void *cuda_stream);

/* Fused gate/up GEMM + SwiGLU: A[T, F] (bf16) = silu(X Wg^T) * (X Wu^T). */
int ss_op_gemm_swiglu_bf16(const void *x_dev, const void *wg_dev, const void *wu_dev, void *a_dev,
                           int T, int F, int K, void *scratch_dev, size_t scratch_bytes, void *cuda_stream);

/* The same GEMM for callers that may NOT allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): C[T, N] (fp32, row-major, ld = N) = X[T, K] (bf16) * W[N, K]^T (bf16), as
 * ss_op_gemm_bf16 (same kernel, same launch plan, bit-identical result), but the stream-K fix-up scratch is a fixed
 * __device__ array inside the library instead of a caller buffer.  The call allocates nothing: no cudaMalloc / cudaFree
 * and no allocating library routine; on the stream it enqueues one 1 KiB memset node (the fix-up flags) and the kernel.
 *   Limit: T <= SS_OP_GEMM_STATIC_MAX_T (decode batches); any N, K with K % 8 == 0; x_dev / w_dev 16-byte aligned.
 *   Cost: SS_OP_GEMM_STATIC_SCRATCH_BYTES of device memory on EVERY GPU that loads the library, held until exit.
 *   Sharing: every call on a device uses the same array.  Calls that overlap on the GPU (two streams, two host
 *   threads, a captured graph replayed while another call is in flight) RACE on it and give wrong sums or trip the
 *   kernel's bounded waits; serialise them on one stream or with events.  Nothing else is kept between calls.
 * Errors: SS_ERR_INVALID_ARG (null pointer, non-positive size), SS_ERR_UNSUPPORTED (K % 8, alignment),
 * SS_ERR_CAPACITY (T > SS_OP_GEMM_STATIC_MAX_T: refused, never clipped; ss_last_cuda_error says so), SS_ERR_CUDA.
 * The device address of the array is looked up once per device on the first call made with that device current
 * (cudaGetSymbolAddress; not an allocation): make one call outside graph capture first. */
#define SS_OP_GEMM_STATIC_MAX_T 128
#define SS_OP_GEMM_STATIC_SCRATCH_BYTES (1024 + 256 * 128 * 128 * 4) /* flags + 256 CTAs x (128 x 128 fp32) = 16 MiB + 1 KiB */
int ss_op_gemm_bf16_static(const void *x_dev, const void *w_dev, float *c_dev, int T, int N, int K, void *cuda_stream);

/* Shared Tensor Store attach (Section 5.2 "Concurrent initialization", Figure 7).  The paper keeps
 * the weight tensors and the KV-cache space in a separate per-node process and shares them with the inference engine
 * "in a zero-copy manner through CUDA IPC handles", so that a replacement engine can be initialised beside the serving
 * one without a second copy of either.  These calls are that mechanism and nothing more (plain cudaMalloc / cudaIpc*;
 * no kernel): the STORE process allocates one arena with ss_store_alloc (a whole cudaMalloc allocation, hence
 * exportable), fills it (ss_store_upload, or any device copy) and hands the 64-byte handle of ss_store_export to the
 * engines by whatever channel it likes; every ENGINE process calls ss_store_attach, which maps the same physical
 * memory and returns its device address in that process, carves weights and KV pool out of it at the offsets the store
 * published, and passes those pointers to ss_stage_create (all of whose device inputs are borrowed).  An engine must
 * ss_stage_destroy before ss_store_detach; the store must outlive every attachment.  `handle` is HOST memory of
 * SS_IPC_HANDLE_BYTES.  A handle cannot be opened by the process that exported it (CUDA's rule).  Errors:
 * SS_ERR_INVALID_ARG (null argument / zero bytes), SS_ERR_CUDA (see ss_last_cuda_error). */
#define SS_IPC_HANDLE_BYTES 64
int ss_store_alloc(void **dev_ptr_out, size_t bytes);
int ss_store_free(void *dev_ptr);
int ss_store_upload(void *dst_dev, const void *src_host, size_t bytes);   /* synchronous host -> arena copy */
int ss_store_export(const void *dev_ptr, void *handle_out /* host, SS_IPC_HANDLE_BYTES */);
int ss_store_attach(const void *handle /* host, SS_IPC_HANDLE_BYTES */, void **dev_ptr_out);
int ss_store_detach(void *dev_ptr);

const char *ss_strerror(int code);
const char *ss_last_cuda_error(void); /* text of the last CUDA error seen by this thread ("" if none) */
const char *ss_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SHUNTSTAGE_H */
