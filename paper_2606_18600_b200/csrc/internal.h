// internal.h — host-side declarations shared by the translation units of libshuntstage.so (not installed).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace ss {

// ---------------------------------------------------------------------------------------------------------------
// tcgen05 GEMM (gemm_tcgen05.cu).  Orientation ("swap-AB", used for every shape): the UMMA M dimension (128 TMEM
// lanes) runs over OUTPUT FEATURES, i.e. rows of the weight matrix W[N,K]; the UMMA N dimension (TMEM columns,
// bn in {32,64,128,256}) runs over TOKENS, rows of X[T,K].  out[t][n] = sum_k X[t,k] W[n,k].
// Persistent: gridDim.x CTAs (<= #SMs, one per SM) walk a work list.  Two schedules:
//   SCHED_STREAMK (few tiles, the HBM-bound decode case): the flattened (tile, k-block) units are cut into gridDim.x
//     equal contiguous ranges; a tile cut between CTAs is fixed up in-kernel (the CTA holding the tile's first
//     k-blocks adds the others' fp32 partials, in CTA order, then runs the epilogue) — every SM streams the same
//     number of weight bytes whatever the tile count;
//   SCHED_TILES (many tiles, the tensor-bound prefill case): whole tiles, round-robin, rasterised in bands of
//     `band` weight-row tiles so that concurrently running CTAs share weight and activation tiles in L2.
// ---------------------------------------------------------------------------------------------------------------
constexpr int GEMM_BM = 128;  // weight rows per tile
constexpr int GEMM_BK = 64;   // K elements per stage (= one 128-byte swizzle row of bf16)
constexpr int GEMM_MAX_STAGES = 12;
constexpr int SS_TP_MAX = 8;   // tensor-parallel degree of the fused all-reduce (ss_stage_set_tp_fused)

enum GemmEpilogue {
  EPI_F32 = 0,          // out_f32[t][col] = acc
  EPI_SWIGLU_BF16 = 1,  // dual: out_bf16[t][col] = silu(acc_gate) * acc_up
  EPI_RESID_F32 = 2,    // out_f32[t][col] += acc   (residual stream updated in place; each element once)
  EPI_PARTIAL = 3       // stream-K, one token tile: every work item dumps its raw fp32 accumulator to slot
                        // 2 * cta + item of fix_slots ([token column][tile row], bn * 128 floats); the CONSUMER kernel
                        // (qkv_post, residual_rmsnorm) adds a tile's pieces in CTA order (GemmPartials below)
};
enum GemmSchedule { SCHED_STREAMK = 0, SCHED_TILES = 1 };

struct GemmParams {
  int n_seg;            // 1..3 weight segments laid side by side in the output (q | k | v)
  int seg_rows[3];      // rows (output features) of each segment
  int seg_tile0[3];     // first row-tile index of each segment
  int seg_col[3];       // output column of each segment's row 0
  int n_row_tiles;      // sum of the segments' row tiles
  int n_t_tiles;        // ceil(T / bn)
  int T, K;             // tokens, reduction length
  int bn;               // tokens per tile (UMMA N)
  int stages;           // smem pipeline depth
  int w_policy;         // L2 policy of the weight loads: 0 evict_first, 1 evict_normal, 2 evict_last
  int x_policy;         // pair kernel: L2 policy of the activation loads (same encoding)
  int single_buf;       // debug: 1 = never double-buffer the TMEM accumulators
  int issuers;          // MMA-issuing threads (2 on the HBM-bound schedule, see gemm_tcgen05.cu)
  int sched;            // GemmSchedule
  int band;             // SCHED_TILES: row tiles per raster band
  int epi;              // GemmEpilogue
  int ld_out;           // leading dimension (elements) of the output
  float *out_f32;
  void *out_bf16;
  int tp_size;          // > 0 (EPI_PARTIAL only): every piece is stored into the exchange buffer of EVERY rank
  float *tp_slots[SS_TP_MAX];     // rank d's region for pieces coming from THIS rank (peer-mapped for d != this rank)
  unsigned *tp_flags[SS_TP_MAX];  // rank d's arrival counter for this rank's pieces: += 1 per CTA, system scope
  float *fix_slots;     // SCHED_STREAMK: gridDim.x partial-accumulator slots of (dual ? 2 : 1) * bn * 128 floats
  unsigned long long *trace;  // profiling builds (-DSS_GEMM_TRACE): [grid][64] globaltimer stamps, else null
  int *fix_flags;       // SCHED_STREAMK: gridDim.x flags, zero between launches (consumers reset them)
};

// What the consumer of an EPI_PARTIAL projection needs to put a tile together again.  Row tile i of the projection
// was held by the `count` consecutive CTAs starting at `first_cta`; CTA c's piece is slot 2 * c + (c == first_cta ?
// first_item : 0)  (a CTA range spans at most two tiles: the tail of one, then the head of the next).  The pieces are
// added in CTA order, which is the order the in-kernel fix-up uses, so both give the same bits.
struct PartialTile {
  int32_t first_cta, count, first_item, pad;
};
struct GemmPartials {
  const float *slots;         // null: the projection's result is in its ordinary output buffer
  const PartialTile *tiles;   // [n_row_tiles] (device)
  int slot_floats;            // bn * 128
  int n_src;                  // 1, or the tensor-parallel degree: the pieces of EVERY rank are added, rank-major
  long long src_stride;       // floats between two ranks' slot regions
};

// Fused tensor-parallel all-reduce (ss_stage_set_tp_fused): exchange buffer layout, identical on every rank:
//   [buffer 0 = O projection | buffer 1 = down projection][source rank][TP_SLOTS slots of TP_SLOT_FLOATS floats],
//   then one 128-byte flag line per (buffer, source rank).
constexpr int TP_SLOTS = 320;                    // 2 items x up to 160 CTAs
constexpr int TP_SLOT_FLOATS = 128 * GEMM_BM;    // token tiles up to 128 columns
inline size_t tp_region_floats() { return (size_t)TP_SLOTS * TP_SLOT_FLOATS; }
inline size_t tp_flags_offset(int size) { return 2 * (size_t)size * tp_region_floats() * sizeof(float); }
inline size_t tp_xchg_bytes(int size) { return tp_flags_offset(size) + 2 * (size_t)size * 128; }

struct GemmLaunch {
  const CUtensorMap *a[3];  // weight maps, box {64, 128}; dual (SwiGLU): a[0] = gate, a[1] = up, n_seg = 1
  const CUtensorMap *b;     // activation map, box {64, bn}
  bool dual;
  bool pair;                // set by gemm_plan: run on CTA pairs (gemm_pair_kernel; b must be the 128-row activation map)
  bool invariant;           // batch-invariant mode: whole-K tiles, one issuer (the K order of an element never depends on T)
  bool no_pdl;              // weights may have been written by the preceding kernel (op-level entry points)
  int grid;                 // persistent CTAs
  GemmParams p;
  cudaStream_t stream;
};

// Encode a 2-D bf16 row-major [rows, cols] tensor map with box {64 cols, box_rows}, SWIZZLE_128B.
int make_tmap_bf16_2d(CUtensorMap *out, const void *base, uint64_t rows, uint64_t cols, uint32_t box_rows,
                      bool weight_like);
// Fills sched / band / stages / n_*_tiles / grid from the problem shape; fix buffers must be set by the caller.
void gemm_plan(GemmLaunch &g, int n_sm);
// true if this planned launch may run with EPI_PARTIAL (stream-K, one token tile, no CTA range spanning > 2 tiles)
bool gemm_partial_ok(const GemmLaunch &g);
// host: the PartialTile table of a planned stream-K launch (n_row_tiles entries)
void gemm_partial_table(const GemmLaunch &g, PartialTile *out);
cudaError_t gemm_launch(const GemmLaunch &g);
// stage.cu: record the text that ss_last_cuda_error returns (thread-local) and hand back the code to return
int note_cuda_error(cudaError_t e, const char *where);  // -> SS_ERR_CUDA
int note_error(int code, const char *text);             // -> code
cudaError_t gemm_init();  // sets max dynamic smem attributes once
cudaError_t gemm_set_debug_buffer(unsigned long long *host_mapped);  // see gemm_tcgen05.cu wait_expired()
int gemm_pick_bn(int T);  // 32 for T <= 32, else the narrowest multiple of 32 covering T in ceil(T / 256) token tiles
int gemm_pick_stages(int bn, bool dual);
size_t gemm_smem_bytes(int bn, bool dual, int stages);
constexpr int GEMM_MAX_GRID = 256;                       // upper bound on persistent CTAs (sizes the fix buffers)
constexpr size_t GEMM_FIX_FLAG_BYTES = 1024;             // GEMM_MAX_GRID ints
constexpr size_t GEMM_FIX_SLOT_BYTES = 2 * 256 * 128 * 4;  // worst case: dual, bn = 256 (or two plain items of a CTA)
inline size_t gemm_fix_bytes() { return GEMM_FIX_FLAG_BYTES + GEMM_MAX_GRID * GEMM_FIX_SLOT_BYTES; }

// ---------------------------------------------------------------------------------------------------------------
// element-wise / reduction kernels (elementwise.cu)
// ---------------------------------------------------------------------------------------------------------------
struct CallArgs {  // device-resident block of user pointers, rewritten before every call (graph-replay safe)
  const void *hidden_in;       // bf16 [T,H] or null
  const int32_t *token_ids;    // [T] or null
  const int32_t *block_tables; // [n_seqs,max_blocks]
  const int32_t *ctx;          // decode: context_lens[B]; prefill: ctx_before[n_seqs]
  const int32_t *cu_q;         // prefill only
  void *out_hidden;            // bf16 [T,H] or null
  float *out_logits;           // [n_seqs,V] or null
  int32_t *out_argmax;         // [n_seqs] or null
  int32_t n_seqs, T, max_blocks, pad;
};

// x[t,:] = widen(input row t) (bf16 hidden or embedding gather); h[t,:] = bf16(rmsnorm(x[t,:]) * w)
cudaError_t launch_input_rmsnorm(const CallArgs *args, const void *embed, const void *ln_w, float eps, int H,
                                 int T, float *x, void *h, cudaStream_t s);
// x[t,:] += sum_{s<splits} part[s][t,:]; then (w != null) h = bf16(rmsnorm(x) * w); (out_from_args) the bf16 of
// x goes to args->out_hidden when that is non-null.
// gp.slots != null: additionally x[t,:] += the pieces of an EPI_PARTIAL projection (added in CTA order first).
// fixed_shape: always the 1024-threads-per-row variant (batch-invariant mode: the reduction tree of a row must not
// depend on how many rows the call has)
cudaError_t launch_residual_rmsnorm(float *x, const float *part, int splits, long long split_stride,
                                    const GemmPartials &gp, const void *ln_w, float eps, int H, int T, void *h,
                                    const CallArgs *args, bool write_out_hidden, cudaStream_t s, bool fixed_shape = false,
                                    bool pdl = true);
// gather the last row of each sequence: hl[s,:] = bf16(rmsnorm(x[last(s),:]) * wf)
cudaError_t launch_final_norm_rows(const float *x, const CallArgs *args, bool decode, const void *wf, float eps,
                                   int H, int n_seqs, void *hl, cudaStream_t s);
// logits -> args->out_logits (when non-null) and argmax (lowest index among maxima) -> args->out_argmax;
// part_max / part_idx: n_rows * 16 scratch entries each
cudaError_t launch_logits_argmax(const float *logits, int V, int n_rows, float *part_max, int *part_idx,
                                 const CallArgs *args, cudaStream_t s);

struct QkvPostParams {
  GemmPartials gp;         // slots != null: the QKV projection's tiles are in pieces (EPI_PARTIAL) instead of qkv_part
  int tile0_k, tile0_v;    // first row tile of the k and v segments (q starts at tile 0)
  const float *qkv_part;   // [splits][T][Hq+2Hkv]
  int splits;
  long long split_stride;
  int T, n_q, n_kv, d;
  int qk_norm;
  float eps;
  const void *q_norm, *k_norm;  // bf16 [d]
  const float *rope;            // [max_pos][d/2][2] (cos, sin)
  void *q_out;                  // bf16 [T,Hq]
  void *kv_new;                 // decode: bf16 [T,2*Hkv] (k | v), appended by the attention kernel
  void *kpool, *vpool;          // prefill: this layer's pools, appended here
  int n_pages;
  const int32_t *tok_seq;       // prefill: [T] sequence of each token
  const int32_t *tok_pos;       // prefill: [T] global position of each token
  const CallArgs *args;
  int decode;
};
cudaError_t launch_qkv_post(const QkvPostParams &p, cudaStream_t s);

// ---------------------------------------------------------------------------------------------------------------
// attention (attn_decode.cu, attn_prefill.cu)
// ---------------------------------------------------------------------------------------------------------------
struct DecodePlan {          // device buffers in the workspace
  int32_t *cum_pages;        // [max_seqs+1] prefix sum of pages per sequence (pages = (ctx+1+15)/16)
  int32_t *meta;             // [4]: total flattened pages (x n_kv), pages per worker warp, n_workers
};
cudaError_t launch_decode_plan(const CallArgs *args, int batch, int n_kv, int n_workers, DecodePlan plan,
                               cudaStream_t s);
struct DecodeAttnParams {
  const void *q;             // bf16 [B,Hq]
  const void *kv_new;        // bf16 [B,2*Hkv]
  void *kpool, *vpool;       // this layer
  const CUtensorMap *kv_map; // this layer's pool as a 2-D bf16 tensor [2 * n_pages * n_kv * 16 rows, d], box {64, 16}
  int n_pages;
  int batch, n_q, n_kv, d;
  DecodePlan plan;
  float *part_o;             // [n_slots][16][d]  (rows >= G unused)
  float *part_ml;            // [n_slots][16][2]
  void *out;                 // bf16 [B,Hq]
  const CallArgs *args;
  int n_workers;             // worker warps in the grid
  int append;                // 1: write kv_new into the last page (decode step); 0: the token is already in the pool
  int warps_per_cta;
  // batch-invariant mode (ss_stage_set_batch_invariant): worker w = one (row, kv head) pair, walked from page 0 to the
  // last by ONE warp, result normalised and written by that warp (no split, no merge kernel): the summation order of a
  // row depends on its own context only.  row_seq / row_pos (prefill rows: the plan's tok_seq / tok_pos) replace
  // args->ctx and the row's own block-table row; null for a decode step.
  int per_pair;
  int n_rows;
  const int32_t *row_seq, *row_pos;
};
cudaError_t launch_decode_attn(const DecodeAttnParams &p, cudaStream_t s);
cudaError_t launch_decode_merge(const DecodeAttnParams &p, cudaStream_t s);
cudaError_t attn_init();
int decode_attn_warps_per_cta();
int decode_attn_default_ctas_per_sm();

struct PrefillPlan {
  int32_t *tok_seq;          // [max_tokens]
  int32_t *tok_pos;          // [max_tokens]
  int32_t *tile_cum;         // [max_seqs+1] prefix sum of 128-row query tiles per sequence
  int32_t *tile_order;       // [2 * max_tiles]: tile -> launch slot, heaviest (most keys) first; second half = sort keys
  int32_t *tile_desc;        // [max_tiles][4]: per launch slot {first packed row, rows, first position, sequence}
  int max_tiles;             // capacity: max_tokens / 64 + max_seqs + 1
};
// seq0: the first seq0 sequences get no query tiles (mixed batches: their attention runs in the decode kernel)
cudaError_t launch_prefill_plan(const CallArgs *args, int n_seqs, int seq0, PrefillPlan plan, cudaStream_t s);
struct PrefillAttnParams {
  const CUtensorMap *q_map;  // q bf16 [max_tokens, Hq] as a 2-D tensor, box {64 columns, 128 rows}
  const CUtensorMap *kv_map; // this layer's pool, as in DecodeAttnParams
  int n_pages;
  int n_seqs, T, n_q, n_kv, d;
  PrefillPlan plan;
  void *out;                 // bf16 [T,Hq]
  const CallArgs *args;
  int max_tiles;             // upper bound on query tiles = ceil(T / prefill_attn_tile_rows()) + n_seqs
  int n_sm;                  // SMs of the device: the kernel is persistent, one CTA per SM
  float lazy;                // log2 threshold of the lazy running maximum (16; SS_ATTN_LAZY overrides: a test aid)
};
int prefill_attn_tile_rows();
cudaError_t launch_prefill_attn(const PrefillAttnParams &p, cudaStream_t s);
cudaError_t prefill_attn_init();

// gather (to_buffer) / scatter n pages of every layer between the pool and a contiguous [L][2][n][n_kv][16][d] buffer
cudaError_t launch_kv_pages_copy(void *pool, void *buf, const int32_t *page_ids, int n, int n_layers, int n_pages_pool,
                                 int piece_bytes, bool to_buffer, cudaStream_t s);

// SS_DEBUG=1 contract checks (elementwise.cu): codes of the device error word, mirrored in include/shuntstage.h
enum { SS_DBG_BAD_PAGE = 1, SS_DBG_BEYOND_PAGES = 2, SS_DBG_BEYOND_MAX_POS = 3, SS_DBG_BAD_TOKEN = 4, SS_DBG_BAD_CU_Q = 5,
       SS_DBG_BAD_CTX = 6 };
struct DebugCheck {
  int decode;          // 1: ss_stage_decode (q_len == 1 everywhere, cu_q unused)
  int n_decode_rows;   // mixed call: the first rows must have q_len == 1
  int num_pages, max_pos, vocab;
};
cudaError_t launch_debug_validate(const CallArgs *args, const DebugCheck &c, int32_t *err /* dev [4], zeroed */, cudaStream_t s);
cudaError_t launch_debug_validate_pages(const int32_t *ids, int n, int num_pages, int32_t *err, cudaStream_t s);

void count_launch(int n = 1);  // stage.cu: per-thread launch counter hook
bool pdl_enabled();            // stage.cu: false when SS_NO_PDL=1

// Launch with the programmatic-stream-serialization attribute (PDL; see common.cuh) and count it.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl_if(bool allow, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem,
                                 cudaStream_t s, Args &&...args) {
  cudaLaunchConfig_t cfg;
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (allow && pdl_enabled()) ? 1 : 0;
  count_launch();
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                              Args &&...args) {
  return launch_pdl_if(true, kernel, grid, block, smem, s, static_cast<Args &&>(args)...);
}

}  // namespace ss
