// stage.cu — host runtime and C-ABI of libshuntstage.so (include/shuntstage.h): argument validation, workspace
// carving, TMA descriptors, the per-layer kernel sequence of ss_stage_decode / ss_stage_prefill (steps S0-S11 of
// DESIGN.md; Table 2 of the paper), CUDA-graph capture of the decode step, and the host-side
// page allocator.  A stage never allocates device memory (the paper's engine attaches to tensors owned by
// the Shared Tensor Store); the only cudaMalloc in the library is ss_store_alloc, the store side of
// that mechanism.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <map>
#include <string>
#include <vector>

#include "../../include/shuntstage.h"
#include "internal.h"

namespace ss {

static thread_local int64_t g_launches = 0;
static thread_local std::string g_cuda_err;
void count_launch(int n) { g_launches += n; }
bool pdl_enabled() {
  static int v = -1;
  if (v < 0) {
    const char *e = getenv("SS_NO_PDL");
    v = (e && atoi(e) != 0) ? 0 : 1;
  }
  return v == 1;
}

static int cuda_fail(cudaError_t e, const char *where) {
  g_cuda_err = std::string(where) + ": " + cudaGetErrorString(e);
  cudaGetLastError();  // reported through the return code: do not leave a non-sticky error for the caller's next CUDA call
  return SS_ERR_CUDA;
}
// for the other translation units of the library (op_static.cu): record the text ss_last_cuda_error returns
int note_cuda_error(cudaError_t e, const char *where) { return cuda_fail(e, where); }
int note_error(int code, const char *text) {
  g_cuda_err = text;
  return code;
}
#define CK(call)                                          \
  do {                                                    \
    cudaError_t e__ = (call);                             \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
  } while (0)

constexpr int PTAB_STRIDE = 512;    // row tiles per table: (16384 + 2 * 16384) / 128 = 384 at most, see dims_ok
constexpr int MAX_WORKERS = 4096;  // upper bound on decode-attention worker warps (sizes the partial buffers)

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// stream-ordered wait / write on a 32-bit word in device memory (driver API, resolved at run time): the cross-rank
// synchronisation of the fused tensor-parallel all-reduce is done by the STREAM, never by a spinning kernel
typedef CUresult (*PFN_streamValue32)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
static PFN_streamValue32 g_wait32 = nullptr, g_write32 = nullptr;
static bool load_stream_memops() {
  if (g_wait32 && g_write32) return true;
  void *fw = nullptr, *fr = nullptr;
  cudaDriverEntryPointQueryResult q1, q2;
  if (cudaGetDriverEntryPoint("cuStreamWaitValue32", &fw, cudaEnableDefault, &q1) != cudaSuccess || !fw ||
      q1 != cudaDriverEntryPointSuccess)
    return false;
  if (cudaGetDriverEntryPoint("cuStreamWriteValue32", &fr, cudaEnableDefault, &q2) != cudaSuccess || !fr ||
      q2 != cudaDriverEntryPointSuccess)
    return false;
  g_wait32 = (PFN_streamValue32)fw;
  g_write32 = (PFN_streamValue32)fr;
  return true;
}

struct Carve {  // byte offsets into the workspace
  size_t args, err, ptab, rope, x, h, qkv_part, q, kv_new, attn_out, fix, a, part_o, part_ml, cum_pages, meta, tp_part, am_part, tok_seq,
      tok_pos, tile_cum, tile_order, tile_desc, hl, logits, total;
};

static bool dims_ok(const ss_model_dims *d, int l0, int l1, int *why) {
  *why = SS_ERR_INVALID_ARG;
  if (!d || l0 < 0 || l0 >= l1 || l1 > d->n_layers_total) return false;
  if (d->hidden <= 0 || d->n_q_heads <= 0 || d->n_kv_heads <= 0 || d->ffn <= 0 || d->max_tokens <= 0 ||
      d->max_seqs <= 0 || d->max_blocks_per_seq <= 0 || d->max_pos <= 0)
    return false;
  *why = SS_ERR_UNSUPPORTED;
  if (d->head_dim != 64 && d->head_dim != 128) return false;
  if (d->page_size != 16) return false;
  if (d->n_q_heads % d->n_kv_heads != 0 || d->n_q_heads / d->n_kv_heads > 16) return false;
  if (d->hidden % 8 != 0 || d->ffn % 8 != 0 || d->hidden > 16384) return false;
  if ((long long)d->n_q_heads * d->head_dim > 16384) return false;
  return true;
}

static Carve carve(const ss_model_dims *d) {
  Carve c;
  const size_t Tm = (size_t)(d->max_tokens > d->max_seqs ? d->max_tokens : d->max_seqs);
  const size_t H = d->hidden, Hq = (size_t)d->n_q_heads * d->head_dim, Hkv = (size_t)d->n_kv_heads * d->head_dim;
  const size_t F = d->ffn, Nqkv = Hq + 2 * Hkv;
  const size_t n_slots = (size_t)MAX_WORKERS + (size_t)d->max_seqs * d->n_kv_heads;
  size_t o = 0;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o = align_up(o + bytes, 1024);
    return at;
  };
  c.args = take(sizeof(CallArgs));
  c.err = take(16);  // SS_DEBUG device error word {code, sequence, index, value}
  // EPI_PARTIAL tile tables of the QKV, O and down projections (internal.h PartialTile), PTAB_STRIDE entries each
  c.ptab = take(3 * PTAB_STRIDE * sizeof(PartialTile));
  c.rope = take((size_t)d->max_pos * (d->head_dim / 2) * 2 * sizeof(float));
  c.x = take(Tm * H * 4);
  c.h = take(Tm * H * 2);
  c.qkv_part = take(Tm * Nqkv * 4);
  c.q = take(Tm * Hq * 2);
  c.kv_new = take((size_t)d->max_seqs * 2 * Hkv * 2);
  c.attn_out = take(Tm * Hq * 2);
  c.fix = take(gemm_fix_bytes());  // stream-K fix-up flags + partial-accumulator slots
  c.a = take(Tm * F * 2);
  c.part_o = take(n_slots * 16 * d->head_dim * 4);
  c.part_ml = take(n_slots * 32 * 4);
  c.cum_pages = take(((size_t)d->max_seqs + 1) * 4);
  c.meta = take(16);
  c.am_part = take((size_t)d->max_seqs * 16 * 8);  // argmax partials: 16 (max, index) pairs per row
  c.tp_part = take(Tm * H * 4);  // tensor-parallel mode: fp32 partial of the O / down projection
  c.tok_seq = take(Tm * 4);
  c.tok_pos = take(Tm * 4);
  c.tile_cum = take(((size_t)d->max_seqs + 1) * 4);
  c.tile_order = take(2 * (Tm / 64 + (size_t)d->max_seqs + 1) * 4);
  c.tile_desc = take(4 * (Tm / 64 + (size_t)d->max_seqs + 1) * 4);
  c.hl = take((size_t)d->max_seqs * H * 2);
  c.logits = take(d->vocab > 0 ? (size_t)d->max_seqs * d->vocab * 4 : 0);
  c.total = o;
  return c;
}

struct LayerMaps {
  CUtensorMap wq, wk, wv, wo, wg, wu, wd;
  CUtensorMap kv;  // this layer's K and V pools: [2 * num_pages * n_kv * 16 rows, head_dim], box {64, 16}
};

struct Graph {
  cudaGraphExec_t exec = nullptr;
  int64_t kernels = 0;
};

}  // namespace ss

using namespace ss;

// Host-side page allocator of the paged KV cache: a LIFO free list + a state byte per page.
// All-or-nothing semantics; never touches the device.
struct ss_pool {
  int num_pages = 0;
  std::vector<int32_t> free_list;
  std::vector<uint8_t> is_free;
  void init(int n) {
    num_pages = n;
    free_list.resize(n);
    for (int i = 0; i < n; ++i) free_list[i] = n - 1 - i;  // pop gives 0,1,2,...
    is_free.assign(n, 1);
  }
  int alloc(int n, int32_t *out) {
    if (n < 0 || (n > 0 && !out)) return SS_ERR_INVALID_ARG;
    if ((size_t)n > free_list.size()) return SS_ERR_NO_PAGES;
    for (int i = 0; i < n; ++i) {
      const int32_t id = free_list.back();
      free_list.pop_back();
      is_free[id] = 0;
      out[i] = id;
    }
    return SS_OK;
  }
  int release(int n, const int32_t *ids) {
    if (n < 0 || (n > 0 && !ids)) return SS_ERR_INVALID_ARG;
    int bad = -1;  // validate first (all-or-nothing); 2 marks "seen in this call" so duplicates are caught in O(n)
    for (int i = 0; i < n; ++i) {
      const int32_t id = ids[i];
      if (id < 0 || id >= num_pages || is_free[id] != 0) {
        bad = i;
        break;
      }
      is_free[id] = 2;
    }
    if (bad >= 0) {
      for (int i = 0; i < bad; ++i) is_free[ids[i]] = 0;
      return SS_ERR_BAD_PAGE;
    }
    for (int i = 0; i < n; ++i) {
      is_free[ids[i]] = 1;
      free_list.push_back(ids[i]);
    }
    return SS_OK;
  }
};

struct ss_stage {
  ss_model_dims d;
  int l0, l1, L;
  std::vector<ss_layer_weights> lw;
  ss_edge_weights edge;
  bool has_edge;
  uint8_t *pool;
  size_t pool_bytes;
  int num_pages;
  uint8_t *ws;
  Carve c;
  cudaStream_t stream;
  int n_sm;
  int n_workers;
  std::vector<LayerMaps> maps;
  CUtensorMap lm_map;
  CUtensorMap q_map;   // q [Tm, Hq] bf16, box {64, 128}: the prefill attention's query tiles
  CUtensorMap b_h[9], b_attn[9], b_a[9], b_hl[9];  // activation maps for bn = 16 and 32, 64, ..., 256 (index bn / 32)
  bool ptab_ok[3];  // the QKV / O / down projection may leave its tiles in pieces at decode-sized calls
  ss_pool pages;
  int64_t launches;
  std::map<int, Graph> graphs;  // key = batch*2 + tail
  bool use_graph;
  bool invariant;      // ss_stage_set_batch_invariant
  int64_t graph_captures;  // decode graphs captured so far (ss_stage_graph_count)
  ss_allreduce_fn allreduce;  // non-null: tensor-parallel shard (ss_stage_set_allreduce)
  void *allreduce_user;
  int tp_rank, tp_size;       // ss_stage_set_tp_fused: > 0 ranks, this stage's rank
  uint8_t *tp_xchg[SS_TP_MAX];  // every rank's exchange buffer (own and peer-mapped), internal.h layout
  CallArgs *h_args;    // pinned host staging for the argument block (+ 4 ints behind it: the SS_DEBUG error word)
  cudaEvent_t args_ev; // the last H2D copy out of h_args (the host must not overwrite the block before it has run)
  bool debug;          // SS_DEBUG=1 at create: every call validates its device-side arguments first
  float attn_lazy;     // prefill attention: log2 threshold of the lazy running maximum (SS_ATTN_LAZY, default 16)
  int32_t dbg_info[4]; // last violation {code, sequence, index, value}
  int32_t *h_err() const { return (int32_t *)(h_args + 1); }

  size_t layer_kv_elems() const { return (size_t)num_pages * d.n_kv_heads * 16 * d.head_dim; }
  __nv_bfloat16 *kpool(int l) const { return (__nv_bfloat16 *)pool + (size_t)l * 2 * layer_kv_elems(); }
  __nv_bfloat16 *vpool(int l) const { return kpool(l) + layer_kv_elems(); }
  template <typename T>
  T *at(size_t off) const { return (T *)(ws + off); }
};


static int env_int(const char *name, int dflt) {
  const char *e = getenv(name);
  return e ? atoi(e) : dflt;
}

extern "C" {

const char *ss_strerror(int code) {
  switch (code) {
    case SS_OK: return "ok";
    case SS_ERR_INVALID_ARG: return "invalid argument";
    case SS_ERR_UNSUPPORTED: return "unsupported configuration";
    case SS_ERR_CAPACITY: return "capacity exceeded";
    case SS_ERR_NO_PAGES: return "not enough free KV pages";
    case SS_ERR_BAD_PAGE: return "bad KV page id";
    case SS_ERR_CUDA: return "CUDA error";
    default: return "unknown error";
  }
}
const char *ss_last_cuda_error(void) { return g_cuda_err.c_str(); }
const char *ss_version(void) { return "shuntstage 0.1 (sm_100a)"; }

size_t ss_stage_workspace_bytes(const ss_model_dims *dims, int l0, int l1) {
  int why;
  if (!dims_ok(dims, l0, l1, &why)) return 0;
  return carve(dims).total;
}

size_t ss_kv_page_bytes(const ss_model_dims *dims, int l0, int l1) {
  int why;
  if (!dims_ok(dims, l0, l1, &why)) return 0;
  return (size_t)(l1 - l0) * 2 * dims->n_kv_heads * 16 * dims->head_dim * 2;
}

int ss_stage_create(ss_stage **out, const ss_model_dims *dims, int l0, int l1, const ss_layer_weights *layers,
                    const ss_edge_weights *edge, void *kv_pool, size_t kv_pool_bytes, void *workspace,
                    size_t workspace_bytes, void *cuda_stream) {
  int why;
  if (!out) return SS_ERR_INVALID_ARG;
  *out = nullptr;
  if (!dims_ok(dims, l0, l1, &why)) return why;
  if (!layers || !kv_pool || !workspace) return SS_ERR_INVALID_ARG;
  if (((uintptr_t)kv_pool & 255) || ((uintptr_t)workspace & 255)) return SS_ERR_UNSUPPORTED;
  const int L = l1 - l0;
  for (int l = 0; l < L; ++l) {
    const ss_layer_weights &w = layers[l];
    const void *req[] = {w.ln1, w.wq, w.wk, w.wv, w.wo, w.ln2, w.w_gate, w.w_up, w.w_down};
    for (const void *p : req) {
      if (!p) return SS_ERR_INVALID_ARG;
      if ((uintptr_t)p & 15) return SS_ERR_UNSUPPORTED;
    }
    if (dims->qk_norm && (!w.q_norm || !w.k_norm)) return SS_ERR_INVALID_ARG;
  }
  if (edge && edge->lm_head && (!edge->final_norm || dims->vocab <= 0)) return SS_ERR_INVALID_ARG;
  Carve c = carve(dims);
  if (workspace_bytes < c.total) return SS_ERR_CAPACITY;
  const size_t page_bytes = ss_kv_page_bytes(dims, l0, l1);
  if (kv_pool_bytes < page_bytes) return SS_ERR_CAPACITY;

  ss_stage *st = new ss_stage();
  st->d = *dims;
  st->l0 = l0; st->l1 = l1; st->L = L;
  st->lw.assign(layers, layers + L);
  st->has_edge = edge != nullptr;
  if (edge) st->edge = *edge; else memset(&st->edge, 0, sizeof(st->edge));
  st->pool = (uint8_t *)kv_pool;
  st->pool_bytes = kv_pool_bytes;
  st->num_pages = (int)(kv_pool_bytes / page_bytes);
  st->ws = (uint8_t *)workspace;
  st->c = c;
  st->stream = (cudaStream_t)cuda_stream;
  st->launches = 0;
  st->use_graph = (cuda_stream != nullptr) && env_int("SS_NO_GRAPH", 0) == 0;
  st->invariant = false;
  st->graph_captures = 0;
  st->h_args = nullptr;
  st->args_ev = nullptr;
  st->debug = env_int("SS_DEBUG", 0) != 0;
  {
    const int lz = env_int("SS_ATTN_LAZY", 16);
    st->attn_lazy = (float)(lz < 0 ? 0 : (lz > 64 ? 64 : lz));
  }
  memset(st->dbg_info, 0, sizeof(st->dbg_info));
  st->allreduce = nullptr;
  st->allreduce_user = nullptr;
  st->tp_rank = 0;
  st->tp_size = 0;
  memset(st->tp_xchg, 0, sizeof(st->tp_xchg));

  auto fail = [&](int code) {
    if (st->h_args) cudaFreeHost(st->h_args);
    if (st->args_ev) cudaEventDestroy(st->args_ev);
    delete st;
    return code;
  };
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(cuda_fail(e, "cudaGetDevice"));
  e = cudaDeviceGetAttribute(&st->n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return fail(cuda_fail(e, "cudaDeviceGetAttribute"));
  int ctas_per_sm = decode_attn_default_ctas_per_sm();
  if (ctas_per_sm < 1) ctas_per_sm = 1;
  const int wpc = decode_attn_warps_per_cta();
  st->n_workers = st->n_sm * ctas_per_sm * wpc;
  if (st->n_workers > MAX_WORKERS) st->n_workers = MAX_WORKERS / wpc * wpc;
  if ((e = gemm_init()) != cudaSuccess) return fail(cuda_fail(e, "gemm_init"));
  if ((e = attn_init()) != cudaSuccess) return fail(cuda_fail(e, "attn_init"));
  if ((e = prefill_attn_init()) != cudaSuccess) return fail(cuda_fail(e, "prefill_attn_init"));
  if ((e = cudaMallocHost((void **)&st->h_args, sizeof(CallArgs) + 16)) != cudaSuccess)
    return fail(cuda_fail(e, "cudaMallocHost"));
  if ((e = cudaEventCreateWithFlags(&st->args_ev, cudaEventDisableTiming)) != cudaSuccess)
    return fail(cuda_fail(e, "cudaEventCreate"));

  // RoPE table: cos/sin in double, stored fp32 (reading A10)
  {
    const int half = dims->head_dim / 2;
    std::vector<float> tab((size_t)dims->max_pos * half * 2);
    for (int c2 = 0; c2 < half; ++c2) {
      const double f = (edge && edge->inv_freq) ? (double)edge->inv_freq[c2]
                                                : pow((double)dims->rope_theta, -2.0 * (double)c2 / dims->head_dim);
      for (int p = 0; p < dims->max_pos; ++p) {
        const double ang = (double)p * f;
        tab[((size_t)p * half + c2) * 2 + 0] = (float)cos(ang);
        tab[((size_t)p * half + c2) * 2 + 1] = (float)sin(ang);
      }
    }
    e = cudaMemcpyAsync(st->ws + c.rope, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice, st->stream);
    if (e != cudaSuccess) return fail(cuda_fail(e, "rope upload"));
    e = cudaMemsetAsync(st->ws + c.fix, 0, GEMM_FIX_FLAG_BYTES, st->stream);  // stream-K flags start (and stay) zero
    if (e != cudaSuccess) return fail(cuda_fail(e, "fix flags memset"));
    e = cudaStreamSynchronize(st->stream);
    if (e != cudaSuccess) return fail(cuda_fail(e, "rope upload sync"));
  }

  // TMA descriptors
  const uint64_t H = dims->hidden, Hq = (uint64_t)dims->n_q_heads * dims->head_dim,
                 Hkv = (uint64_t)dims->n_kv_heads * dims->head_dim, F = dims->ffn;
  const uint64_t Tm = (uint64_t)(dims->max_tokens > dims->max_seqs ? dims->max_tokens : dims->max_seqs);
  int rc = 0;
  st->maps.resize(L);
  for (int l = 0; l < L && rc == 0; ++l) {
    const ss_layer_weights &w = layers[l];
    LayerMaps &m = st->maps[l];
    rc |= make_tmap_bf16_2d(&m.wq, w.wq, Hq, H, GEMM_BM, true);
    rc |= make_tmap_bf16_2d(&m.wk, w.wk, Hkv, H, GEMM_BM, true);
    rc |= make_tmap_bf16_2d(&m.wv, w.wv, Hkv, H, GEMM_BM, true);
    rc |= make_tmap_bf16_2d(&m.wo, w.wo, H, Hq, GEMM_BM, true);
    rc |= make_tmap_bf16_2d(&m.wg, w.w_gate, F, H, GEMM_BM, true);
    rc |= make_tmap_bf16_2d(&m.wu, w.w_up, F, H, GEMM_BM, true);
    rc |= make_tmap_bf16_2d(&m.wd, w.w_down, H, F, GEMM_BM, true);
    rc |= make_tmap_bf16_2d(&m.kv, st->kpool(l), (uint64_t)2 * st->num_pages * dims->n_kv_heads * 16,
                            (uint64_t)dims->head_dim, 16, true);
  }
  rc |= make_tmap_bf16_2d(&st->q_map, st->ws + c.q, Tm, Hq, 128, false);
  if (rc == 0 && edge && edge->lm_head)
    rc |= make_tmap_bf16_2d(&st->lm_map, edge->lm_head, (uint64_t)dims->vocab, H, GEMM_BM, true);
  const int bns[9] = {16, 32, 64, 96, 128, 160, 192, 224, 256};
  for (int i = 0; i < 9 && rc == 0; ++i) {
    rc |= make_tmap_bf16_2d(&st->b_h[i], st->ws + c.h, Tm, H, bns[i], false);
    rc |= make_tmap_bf16_2d(&st->b_attn[i], st->ws + c.attn_out, Tm, Hq, bns[i], false);
    rc |= make_tmap_bf16_2d(&st->b_a[i], st->ws + c.a, Tm, F, bns[i], false);
    rc |= make_tmap_bf16_2d(&st->b_hl[i], st->ws + c.hl, (uint64_t)dims->max_seqs, H, bns[i], false);
  }
  if (rc != 0) {
    g_cuda_err = "cuTensorMapEncodeTiled failed (code " + std::to_string(rc) + ")";
    return fail(SS_ERR_CUDA);
  }

  {  // EPI_PARTIAL tile tables: the stream-K cut of a one-token-tile launch depends on the shape only, not on T
    std::vector<PartialTile> tab(3 * PTAB_STRIDE);
    const int rows[3][3] = {{(int)Hq, (int)Hkv, (int)Hkv}, {(int)H, 0, 0}, {(int)H, 0, 0}};
    const int nseg[3] = {3, 1, 1}, Ks[3] = {(int)H, (int)Hq, (int)F};
    for (int i = 0; i < 3; ++i) {
      GemmLaunch g;
      memset(&g, 0, sizeof(g));
      g.p.n_seg = nseg[i];
      for (int j = 0; j < 3; ++j) g.p.seg_rows[j] = rows[i][j];
      g.p.T = 1;
      g.p.K = Ks[i];
      gemm_plan(g, st->n_sm);
      st->ptab_ok[i] = gemm_partial_ok(g) && g.p.n_row_tiles <= PTAB_STRIDE;
      if (st->ptab_ok[i]) gemm_partial_table(g, tab.data() + (size_t)i * PTAB_STRIDE);
    }
    e = cudaMemcpyAsync(st->ws + c.ptab, tab.data(), tab.size() * sizeof(PartialTile), cudaMemcpyHostToDevice, st->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st->stream);
    if (e != cudaSuccess) return fail(cuda_fail(e, "partial tables upload"));
  }

  st->pages.init(st->num_pages);
  *out = st;
  return SS_OK;
}

int ss_stage_destroy(ss_stage *st) {
  if (!st) return SS_ERR_INVALID_ARG;
  for (auto &g : st->graphs)
    if (g.second.exec) cudaGraphExecDestroy(g.second.exec);
  if (st->h_args) cudaFreeHost(st->h_args);
  if (st->args_ev) cudaEventDestroy(st->args_ev);
  delete st;
  return SS_OK;
}

// ---- page pool --------------------------------------------------------------------------------------------------
int ss_kv_num_pages(const ss_stage *st) { return st ? st->num_pages : SS_ERR_INVALID_ARG; }
int ss_kv_num_free(const ss_stage *st) { return st ? (int)st->pages.free_list.size() : SS_ERR_INVALID_ARG; }
int ss_kv_alloc(ss_stage *st, int n, int32_t *out_page_ids) {
  return st ? st->pages.alloc(n, out_page_ids) : SS_ERR_INVALID_ARG;
}
int ss_kv_free(ss_stage *st, int n, const int32_t *page_ids) {
  return st ? st->pages.release(n, page_ids) : SS_ERR_INVALID_ARG;
}

// the same allocator stand-alone (no device, no stage): what a scheduler sizing a pool ahead of a stage uses, and
// what the CPU property tests drive
int ss_pool_create(ss_pool **out, int num_pages) {
  if (!out || num_pages < 0) return SS_ERR_INVALID_ARG;
  ss_pool *p = new ss_pool();
  p->init(num_pages);
  *out = p;
  return SS_OK;
}
int ss_pool_destroy(ss_pool *p) {
  if (!p) return SS_ERR_INVALID_ARG;
  delete p;
  return SS_OK;
}
int ss_pool_num_pages(const ss_pool *p) { return p ? p->num_pages : SS_ERR_INVALID_ARG; }
int ss_pool_num_free(const ss_pool *p) { return p ? (int)p->free_list.size() : SS_ERR_INVALID_ARG; }
int ss_pool_alloc(ss_pool *p, int n, int32_t *out_page_ids) { return p ? p->alloc(n, out_page_ids) : SS_ERR_INVALID_ARG; }
int ss_pool_free(ss_pool *p, int n, const int32_t *page_ids) { return p ? p->release(n, page_ids) : SS_ERR_INVALID_ARG; }

// ---- Shared Tensor Store attach: plain cudaMalloc + CUDA IPC, no kernel ------------------------
static_assert(sizeof(cudaIpcMemHandle_t) == SS_IPC_HANDLE_BYTES, "handle size");
int ss_store_alloc(void **dev_ptr_out, size_t bytes) {
  if (!dev_ptr_out || bytes == 0) return SS_ERR_INVALID_ARG;
  CK(cudaMalloc(dev_ptr_out, bytes));
  return SS_OK;
}
int ss_store_free(void *dev_ptr) {
  if (!dev_ptr) return SS_ERR_INVALID_ARG;
  CK(cudaFree(dev_ptr));
  return SS_OK;
}
int ss_store_upload(void *dst_dev, const void *src_host, size_t bytes) {
  if (!dst_dev || !src_host) return SS_ERR_INVALID_ARG;
  if (bytes) CK(cudaMemcpy(dst_dev, src_host, bytes, cudaMemcpyHostToDevice));
  return SS_OK;
}
int ss_store_export(const void *dev_ptr, void *handle_out) {
  if (!dev_ptr || !handle_out) return SS_ERR_INVALID_ARG;
  cudaIpcMemHandle_t h;
  CK(cudaIpcGetMemHandle(&h, const_cast<void *>(dev_ptr)));
  memcpy(handle_out, &h, sizeof(h));
  return SS_OK;
}
int ss_store_attach(const void *handle, void **dev_ptr_out) {
  if (!handle || !dev_ptr_out) return SS_ERR_INVALID_ARG;
  cudaIpcMemHandle_t h;
  memcpy(&h, handle, sizeof(h));
  CK(cudaIpcOpenMemHandle(dev_ptr_out, h, cudaIpcMemLazyEnablePeerAccess));
  return SS_OK;
}
int ss_store_detach(void *dev_ptr) {
  if (!dev_ptr) return SS_ERR_INVALID_ARG;
  CK(cudaIpcCloseMemHandle(dev_ptr));
  return SS_OK;
}

int64_t ss_stage_launch_count(const ss_stage *st) { return st ? st->launches : 0; }

int64_t ss_stage_graph_count(const ss_stage *st) { return st ? st->graph_captures : 0; }

int ss_stage_debug_info(const ss_stage *st, int32_t out[4]) {
  if (!st || !out) return SS_ERR_INVALID_ARG;
  memcpy(out, st->dbg_info, 16);
  return st->debug ? 1 : 0;
}

int ss_stage_debug_tap(const ss_stage *st, const char *name, void **dev_ptr_out, size_t *bytes_out) {
  if (!st || !name || !dev_ptr_out || !bytes_out) return SS_ERR_INVALID_ARG;
  const ss_model_dims &d = st->d;
  const size_t Tm = (size_t)(d.max_tokens > d.max_seqs ? d.max_tokens : d.max_seqs);
  const size_t H = d.hidden, Hq = (size_t)d.n_q_heads * d.head_dim, Hkv = (size_t)d.n_kv_heads * d.head_dim;
  const struct { const char *n; size_t off, bytes; } taps[] = {
      {"x", st->c.x, Tm * H * 4},       {"h", st->c.h, Tm * H * 2},
      {"qkv", st->c.qkv_part, Tm * (Hq + 2 * Hkv) * 4}, {"q", st->c.q, Tm * Hq * 2},
      {"attn", st->c.attn_out, Tm * Hq * 2}, {"a", st->c.a, Tm * (size_t)d.ffn * 2}};
  for (const auto &t : taps)
    if (strcmp(t.n, name) == 0) {
      *dev_ptr_out = st->ws + t.off;
      *bytes_out = t.bytes;
      return SS_OK;
    }
  return SS_ERR_INVALID_ARG;
}

int ss_stage_set_batch_invariant(ss_stage *st, int on) {
  if (!st) return SS_ERR_INVALID_ARG;
  if (st->invariant != (on != 0)) {  // the captured decode graphs hold the other mode's kernels
    cudaError_t e = cudaStreamSynchronize(st->stream);
    if (e != cudaSuccess) return cuda_fail(e, "ss_stage_set_batch_invariant");
    for (auto &g : st->graphs)
      if (g.second.exec) cudaGraphExecDestroy(g.second.exec);
    st->graphs.clear();
    st->invariant = on != 0;
  }
  return SS_OK;
}

size_t ss_tp_xchg_bytes(int tp_size) {
  return (tp_size >= 1 && tp_size <= SS_TP_MAX) ? tp_xchg_bytes(tp_size) : 0;
}

int ss_stage_set_tp_fused(ss_stage *st, int rank, int size, void *const *xchg_dev) {
  if (!st) return SS_ERR_INVALID_ARG;
  if (size == 0) {  // off
    st->tp_size = 0;
  } else {
    if (size < 1 || size > SS_TP_MAX || rank < 0 || rank >= size || !xchg_dev) return SS_ERR_INVALID_ARG;
    for (int i = 0; i < size; ++i)
      if (!xchg_dev[i] || ((uintptr_t)xchg_dev[i] & 255)) return SS_ERR_INVALID_ARG;
    if (!load_stream_memops()) {
      g_cuda_err = "cuStreamWaitValue32 / cuStreamWriteValue32 not available";
      return SS_ERR_UNSUPPORTED;
    }
    st->tp_rank = rank;
    st->tp_size = size;
    for (int i = 0; i < size; ++i) st->tp_xchg[i] = (uint8_t *)xchg_dev[i];
    // this rank's arrival counters start at zero (the caller must not start any rank's first call before every rank
    // has returned from this function: the counters are written by the peers' first projection)
    CK(cudaMemsetAsync(st->tp_xchg[rank] + tp_flags_offset(size), 0, 2 * (size_t)size * 128, st->stream));
    CK(cudaStreamSynchronize(st->stream));
  }
  CK(cudaStreamSynchronize(st->stream));
  for (auto &g : st->graphs)
    if (g.second.exec) cudaGraphExecDestroy(g.second.exec);
  st->graphs.clear();
  return SS_OK;
}

int ss_stage_set_allreduce(ss_stage *st, ss_allreduce_fn fn, void *user) {
  if (!st) return SS_ERR_INVALID_ARG;
  st->allreduce = fn;
  st->allreduce_user = user;
  return SS_OK;
}

namespace ss { static int debug_fetch(ss_stage *st); }
static int kv_copy(ss_stage *st, int n, const int32_t *page_ids_dev, void *buf, size_t buf_bytes, bool to_buffer) {
  if (!st || n <= 0 || !page_ids_dev || !buf) return SS_ERR_INVALID_ARG;
  if ((uintptr_t)buf & 15) return SS_ERR_UNSUPPORTED;
  const size_t piece = (size_t)st->d.n_kv_heads * 16 * st->d.head_dim * 2;
  if (buf_bytes < (size_t)st->L * 2 * n * piece) return SS_ERR_CAPACITY;
  if (st->debug) {
    CK(cudaMemsetAsync(st->ws + st->c.err, 0, 16, st->stream));
    const int64_t b0 = g_launches;
    CK(launch_debug_validate_pages(page_ids_dev, n, st->num_pages, st->at<int32_t>(st->c.err), st->stream));
    st->launches += g_launches - b0;
    const int rc = debug_fetch(st);
    if (rc != SS_OK) return rc;
  }
  const int64_t before = g_launches;
  cudaError_t e = launch_kv_pages_copy(st->pool, buf, page_ids_dev, n, st->L, st->num_pages, (int)piece, to_buffer,
                                       st->stream);
  st->launches += g_launches - before;
  return e == cudaSuccess ? SS_OK : cuda_fail(e, "ss_kv_export/import");
}
int ss_kv_export(ss_stage *st, int n, const int32_t *page_ids_dev, void *buf_dev, size_t buf_bytes) {
  return kv_copy(st, n, page_ids_dev, buf_dev, buf_bytes, true);
}
int ss_kv_import(ss_stage *st, int n, const int32_t *page_ids_dev, const void *buf_dev, size_t buf_bytes) {
  return kv_copy(st, n, page_ids_dev, const_cast<void *>(buf_dev), buf_bytes, false);
}

}  // extern "C"

// ===================================================================================================================
// the forward pass
// ===================================================================================================================
namespace ss {

// one projection through the persistent tcgen05 GEMM
// the fused tensor-parallel all-reduce applies to a decode-sized projection whose pieces fit the exchange slots
static bool tp_fused_ok(const ss_stage *st, int T, int grid) {
  return st->tp_size > 0 && T <= 128 && 2 * grid <= TP_SLOTS;
}
// ... and a call uses it only if BOTH its O and down projections will (the batch-invariant mode runs whole tiles, which
// leave no pieces: it falls back to the all-reduce callback)
static bool tp_fused_eligible(const ss_stage *st, int T) {
  return st->tp_size > 0 && T <= 128 && !st->invariant && st->ptab_ok[1] && st->ptab_ok[2] && 2 * st->n_sm <= TP_SLOTS;
}

// `piece` (0 QKV, 1 O, 2 down; -1 none): if the planned launch allows it, the projection leaves its tiles in pieces
// (EPI_PARTIAL) and *gp tells the consumer kernel where; otherwise gp->slots = null and `epi` is used as given.
static cudaError_t run_gemm(const ss_stage *st, const CUtensorMap *const a[3], int n_seg, const int rows[3],
                            bool dual, const CUtensorMap bmaps[5], int T, int K, int epi, float *out_f32,
                            void *out_bf16, int ld_out, int piece = -1, GemmPartials *gp = nullptr) {
  GemmLaunch g;
  memset(&g, 0, sizeof(g));
  GemmParams &p = g.p;
  p.n_seg = n_seg;
  for (int i = 0; i < 3; ++i) {
    g.a[i] = a[i];
    p.seg_rows[i] = i < n_seg ? rows[i] : 0;
  }
  p.T = T;
  p.K = K;
  p.epi = epi;
  p.ld_out = ld_out;
  p.out_f32 = out_f32;
  p.out_bf16 = out_bf16;
  p.fix_flags = st->at<int>(st->c.fix);
  p.fix_slots = (float *)(st->ws + st->c.fix + GEMM_FIX_FLAG_BYTES);
  g.dual = dual;
  g.invariant = st->invariant;
  g.stream = st->stream;
  gemm_plan(g, st->n_sm);
  g.b = &bmaps[(g.pair ? 128 : p.bn) / 32];  // a CTA pair loads the token tile in two 128-row halves
  if (gp) {
    gp->slots = nullptr;
    gp->n_src = 1;
    gp->src_stride = 0;
    if (piece >= 0 && st->ptab_ok[piece] && gemm_partial_ok(g)) {
      p.epi = EPI_PARTIAL;
      gp->slots = p.fix_slots;
      gp->tiles = st->at<PartialTile>(st->c.ptab) + (size_t)piece * PTAB_STRIDE;
      gp->slot_floats = p.bn * GEMM_BM;
      if (piece >= 1 && tp_fused_ok(st, T, g.grid)) {
        // fused all-reduce (Eq. 3): the pieces go to every rank's exchange buffer (O: buffer 0, down:
        // buffer 1; a rank is never more than one all-reduce point ahead of another), the consumer adds all ranks'
        const int buf = piece - 1, size = st->tp_size;
        p.tp_size = size;
        for (int d = 0; d < size; ++d) {
          p.tp_slots[d] = (float *)st->tp_xchg[d] + ((size_t)buf * size + st->tp_rank) * tp_region_floats();
          p.tp_flags[d] = (unsigned *)(st->tp_xchg[d] + tp_flags_offset(size) + ((size_t)buf * size + st->tp_rank) * 128);
        }
        gp->slots = (const float *)st->tp_xchg[st->tp_rank] + (size_t)buf * size * tp_region_floats();
        gp->n_src = size;
        gp->src_stride = (long long)tp_region_floats();
        cudaError_t e = gemm_launch(g);
        if (e != cudaSuccess) return e;
        // wait (stream-ordered) until every rank's CTAs have arrived on this rank's counters, then re-arm them
        for (int q = 0; q < size; ++q) {
          const CUdeviceptr flag = (CUdeviceptr)(st->tp_xchg[st->tp_rank] + tp_flags_offset(size) + ((size_t)buf * size + q) * 128);
          if (g_wait32((CUstream)st->stream, flag, (cuuint32_t)g.grid, CU_STREAM_WAIT_VALUE_GEQ) != CUDA_SUCCESS ||
              g_write32((CUstream)st->stream, flag, 0u, CU_STREAM_WRITE_VALUE_DEFAULT) != CUDA_SUCCESS)
            return cudaErrorUnknown;
        }
        return cudaSuccess;
      }
    }
  }
  return gemm_launch(g);
}

#define CKE(call)                      \
  do {                                 \
    cudaError_t e__ = (call);          \
    if (e__ != cudaSuccess) return e__; \
  } while (0)

// enqueue every kernel of one call; `decode` selects the q_len == 1 fast path
// `n_dec` (prefill calls only): the first n_dec sequences are decode rows (q_len == 1) whose attention runs in the
// decode kernel (mixed batches, reading A19)
static cudaError_t enqueue_forward(ss_stage *st, bool decode, int n_seqs, int T, bool tail, int n_dec = 0) {
  const ss_model_dims &d = st->d;
  const int H = d.hidden, dh = d.head_dim, Hq = d.n_q_heads * dh, Hkv = d.n_kv_heads * dh, F = d.ffn;
  const int Nqkv = Hq + 2 * Hkv;
  const Carve &c = st->c;
  const CallArgs *args = st->at<CallArgs>(c.args);
  float *x = st->at<float>(c.x);
  void *h = st->at<void>(c.h);
  float *qkv_part = st->at<float>(c.qkv_part);
  cudaStream_t s = st->stream;

  // tensor-parallel shard: the fused exchange for decode-sized calls, else the caller's all-reduce callback
  const bool fused = tp_fused_eligible(st, T);
  const bool tp = !fused && (st->allreduce != nullptr || st->tp_size > 1);
  if (tp && !st->allreduce) return cudaErrorNotSupported;  // a TP shard's large calls need ss_stage_set_allreduce
  float *tp_part = st->at<float>(c.tp_part);
  DecodePlan dplan{st->at<int32_t>(c.cum_pages), st->at<int32_t>(c.meta)};
  PrefillPlan pplan{st->at<int32_t>(c.tok_seq), st->at<int32_t>(c.tok_pos), st->at<int32_t>(c.tile_cum),
                    st->at<int32_t>(c.tile_order), st->at<int32_t>(c.tile_desc),
                    (int)(d.max_tokens / 64 + d.max_seqs + 1)};
  if (decode)
    CKE(launch_decode_plan(args, n_seqs, d.n_kv_heads, st->n_workers, dplan, s));
  else {
    CKE(launch_prefill_plan(args, n_seqs, n_dec, pplan, s));
    if (n_dec > 0) CKE(launch_decode_plan(args, n_dec, d.n_kv_heads, st->n_workers, dplan, s));
  }
  CKE(launch_input_rmsnorm(args, st->edge.embed, st->lw[0].ln1, d.rms_eps, H, T, x, h, s));

  for (int l = 0; l < st->L; ++l) {
    const ss_layer_weights &w = st->lw[l];
    const LayerMaps &m = st->maps[l];
    GemmPartials gp_qkv, gp_o, gp_d;
    const GemmPartials gp_none{nullptr, nullptr, 0, 1, 0};
    {  // S2: QKV projection -> fp32 [T][Hq+2Hkv] (or pieces, added by qkv_post)
      const CUtensorMap *a[3] = {&m.wq, &m.wk, &m.wv};
      const int rows[3] = {Hq, Hkv, Hkv};
      CKE(run_gemm(st, a, 3, rows, false, st->b_h, T, H, EPI_F32, qkv_part, nullptr, Nqkv, 0, &gp_qkv));
    }
    QkvPostParams qp;
    memset(&qp, 0, sizeof(qp));
    qp.gp = gp_qkv;
    qp.tile0_k = (Hq + GEMM_BM - 1) / GEMM_BM;
    qp.tile0_v = qp.tile0_k + (Hkv + GEMM_BM - 1) / GEMM_BM;
    qp.qkv_part = qkv_part;
    qp.splits = 1;
    qp.split_stride = 0;
    qp.T = T; qp.n_q = d.n_q_heads; qp.n_kv = d.n_kv_heads; qp.d = dh;
    qp.qk_norm = d.qk_norm;
    qp.eps = d.rms_eps;
    qp.q_norm = w.q_norm; qp.k_norm = w.k_norm;
    qp.rope = st->at<float>(c.rope);
    qp.q_out = st->at<void>(c.q);
    qp.kv_new = st->at<void>(c.kv_new);
    qp.kpool = st->kpool(l); qp.vpool = st->vpool(l);
    qp.n_pages = st->num_pages;
    qp.tok_seq = pplan.tok_seq; qp.tok_pos = pplan.tok_pos;
    qp.args = args;
    qp.decode = decode ? 1 : 0;
    CKE(launch_qkv_post(qp, s));  // S3, S4 (+S5 in prefill)

    if (st->invariant) {
      // batch-invariant mode: every row (decode rows and prefill tokens alike) is one (row, kv head) walk of the decode
      // kernel from page 0 to its last page by one warp — the same arithmetic in the same order whatever the call
      DecodeAttnParams ap;
      memset(&ap, 0, sizeof(ap));
      ap.q = st->at<void>(c.q);
      ap.kv_new = st->at<void>(c.kv_new);
      ap.kpool = st->kpool(l); ap.vpool = st->vpool(l);
      ap.kv_map = &st->maps[l].kv;
      ap.n_pages = st->num_pages;
      ap.batch = 0; ap.n_q = d.n_q_heads; ap.n_kv = d.n_kv_heads; ap.d = dh;
      ap.plan = dplan;
      ap.out = st->at<void>(c.attn_out);
      ap.args = args;
      ap.warps_per_cta = decode_attn_warps_per_cta();
      ap.per_pair = 1;
      ap.n_rows = T;
      ap.append = decode ? 1 : 0;  // prefill: qkv_post has appended every token already
      ap.row_seq = decode ? nullptr : pplan.tok_seq;
      ap.row_pos = decode ? nullptr : pplan.tok_pos;
      CKE(launch_decode_attn(ap, s));
    } else {
      if (decode || n_dec > 0) {  // S5 + S6a (mixed call: the decode rows' K/V were appended by qkv_post already)
        DecodeAttnParams ap;
        memset(&ap, 0, sizeof(ap));
        ap.q = st->at<void>(c.q);
        ap.kv_new = st->at<void>(c.kv_new);
        ap.kpool = st->kpool(l); ap.vpool = st->vpool(l);
        ap.kv_map = &st->maps[l].kv;
        ap.n_pages = st->num_pages;
        ap.batch = decode ? n_seqs : n_dec; ap.n_q = d.n_q_heads; ap.n_kv = d.n_kv_heads; ap.d = dh;
        ap.plan = dplan;
        ap.part_o = st->at<float>(c.part_o);
        ap.part_ml = st->at<float>(c.part_ml);
        ap.out = st->at<void>(c.attn_out);
        ap.args = args;
        ap.n_workers = st->n_workers;
        ap.warps_per_cta = decode_attn_warps_per_cta();
        ap.append = decode ? 1 : 0;
        CKE(launch_decode_attn(ap, s));
        CKE(launch_decode_merge(ap, s));
      }
      if (!decode && n_dec < n_seqs) {  // S6b
        PrefillAttnParams ap;
        memset(&ap, 0, sizeof(ap));
        ap.q_map = &st->q_map;
        ap.kv_map = &st->maps[l].kv;
        ap.n_pages = st->num_pages;
        ap.n_seqs = n_seqs; ap.T = T; ap.n_q = d.n_q_heads; ap.n_kv = d.n_kv_heads; ap.d = dh;
        ap.plan = pplan;
        ap.out = st->at<void>(c.attn_out);
        ap.args = args;
        ap.max_tiles = (T - n_dec + prefill_attn_tile_rows() - 1) / prefill_attn_tile_rows() + (n_seqs - n_dec);
        ap.n_sm = st->n_sm;
        ap.lazy = st->attn_lazy;
        CKE(launch_prefill_attn(ap, s));
      }
    }
    {  // S7: output projection, then S8: x1 = x + o Wo^T ; h2 = rmsnorm(x1; ln2)
      const CUtensorMap *a[3] = {&m.wo, nullptr, nullptr};
      const int rows[3] = {H, 0, 0};
      if (!tp) {
        CKE(run_gemm(st, a, 1, rows, false, st->b_attn, T, Hq, EPI_RESID_F32, x, nullptr, H, 1, &gp_o));
        CKE(launch_residual_rmsnorm(x, nullptr, 0, 0, gp_o, w.ln2, d.rms_eps, H, T, h, args, false, s, st->invariant, gp_o.n_src == 1));
      } else {  // this rank's partial over its heads -> all-reduce -> x += sum (two per layer)
        CKE(run_gemm(st, a, 1, rows, false, st->b_attn, T, Hq, EPI_F32, tp_part, nullptr, H));
        if (st->allreduce(tp_part, (size_t)T * H, st->allreduce_user, (void *)s) != 0) return cudaErrorLaunchFailure;
        CKE(launch_residual_rmsnorm(x, tp_part, 1, 0, gp_none, w.ln2, d.rms_eps, H, T, h, args, false, s, st->invariant));
      }
    }
    {  // S9: gate/up + SwiGLU fused -> a bf16 [T,F]
      const CUtensorMap *a[3] = {&m.wg, &m.wu, nullptr};
      const int rows[3] = {F, 0, 0};
      CKE(run_gemm(st, a, 1, rows, true, st->b_h, T, H, EPI_SWIGLU_BF16, nullptr, st->at<void>(c.a), F));
    }
    {  // S10: down projection + residual, then the next layer's RMSNorm-1 (or the stage output)
      const CUtensorMap *a[3] = {&m.wd, nullptr, nullptr};
      const int rows[3] = {H, 0, 0};
      const bool last = (l == st->L - 1);
      const void *next_ln = last ? nullptr : st->lw[l + 1].ln1;
      if (!tp) {
        CKE(run_gemm(st, a, 1, rows, false, st->b_a, T, F, EPI_RESID_F32, x, nullptr, H, 2, &gp_d));
        CKE(launch_residual_rmsnorm(x, nullptr, 0, 0, gp_d, next_ln, d.rms_eps, H, T, h, args, last, s, st->invariant, gp_d.n_src == 1));
      } else {
        CKE(run_gemm(st, a, 1, rows, false, st->b_a, T, F, EPI_F32, tp_part, nullptr, H));
        if (st->allreduce(tp_part, (size_t)T * H, st->allreduce_user, (void *)s) != 0) return cudaErrorLaunchFailure;
        CKE(launch_residual_rmsnorm(x, tp_part, 1, 0, gp_none, next_ln, d.rms_eps, H, T, h, args, last, s, st->invariant));
      }
    }
  }
  if (tail) {  // S11: final norm of each sequence's last row, lm_head, argmax
    CKE(launch_final_norm_rows(x, args, decode, st->edge.final_norm, d.rms_eps, H, n_seqs, st->at<void>(c.hl), s));
    const CUtensorMap *a[3] = {&st->lm_map, nullptr, nullptr};
    const int rows[3] = {d.vocab, 0, 0};
    CKE(run_gemm(st, a, 1, rows, false, st->b_hl, n_seqs, H, EPI_F32, st->at<float>(c.logits), nullptr, d.vocab));
    CKE(launch_logits_argmax(st->at<float>(c.logits), d.vocab, n_seqs, st->at<float>(c.am_part),
                             (int *)(st->ws + c.am_part + (size_t)d.max_seqs * 16 * 4), args, s));
  }
  return cudaSuccess;
}

static int common_checks(ss_stage *st, int n_seqs, int T, const void *hidden, const int32_t *ids,
                         const int32_t *bt, int max_blocks, const int32_t *ctx, float *out_logits,
                         int32_t *out_argmax) {
  if (!st || n_seqs <= 0 || T <= 0 || !bt || !ctx || max_blocks <= 0) return SS_ERR_INVALID_ARG;
  if ((hidden == nullptr) == (ids == nullptr)) return SS_ERR_INVALID_ARG;
  if (ids && (!st->edge.embed || st->l0 != 0)) return SS_ERR_INVALID_ARG;
  if ((out_logits || out_argmax) && !st->edge.lm_head) return SS_ERR_INVALID_ARG;
  if (n_seqs > st->d.max_seqs || max_blocks > st->d.max_blocks_per_seq) return SS_ERR_CAPACITY;
  if (hidden && ((uintptr_t)hidden & 15)) return SS_ERR_UNSUPPORTED;
  return SS_OK;
}

static int upload_args(ss_stage *st, const CallArgs &a) {
  // the previous call's copy may still be in flight from the same pinned block: the stream orders the copies,
  // but the host must not overwrite the block before the previous copy has read it
  CK(cudaEventSynchronize(st->args_ev));  // a never-recorded event is complete
  *st->h_args = a;
  CK(cudaMemcpyAsync(st->ws + st->c.args, st->h_args, sizeof(CallArgs), cudaMemcpyHostToDevice, st->stream));
  CK(cudaEventRecord(st->args_ev, st->stream));
  return SS_OK;
}

// SS_DEBUG=1: run the device-side contract checks of this call and wait for their verdict; nothing else has been
// enqueued yet, so a violation leaves the pool and the workspace untouched.
static int debug_fetch(ss_stage *st) {
  CK(cudaMemcpyAsync(st->h_err(), st->ws + st->c.err, 16, cudaMemcpyDeviceToHost, st->stream));
  CK(cudaStreamSynchronize(st->stream));
  if (st->h_err()[0] != 0) {
    memcpy(st->dbg_info, st->h_err(), 16);
    return SS_ERR_INVALID_ARG;
  }
  return SS_OK;
}
static int debug_check(ss_stage *st, bool decode, int n_dec) {
  if (!st->debug) return SS_OK;
  CK(cudaMemsetAsync(st->ws + st->c.err, 0, 16, st->stream));
  DebugCheck c{decode ? 1 : 0, n_dec, st->num_pages, st->d.max_pos, st->d.vocab};
  const int64_t before = g_launches;
  CK(launch_debug_validate(st->at<CallArgs>(st->c.args), c, st->at<int32_t>(st->c.err), st->stream));
  st->launches += g_launches - before;
  return debug_fetch(st);
}

}  // namespace ss

extern "C" {

int ss_stage_prefill(ss_stage *st, int n_seqs, const void *hidden_bf16, const int32_t *token_ids,
                     const int32_t *cu_q, const int32_t *ctx_before, const int32_t *block_tables, int max_blocks,
                     int total_tokens, void *out_hidden_bf16, float *out_logits, int32_t *out_argmax) {
  return ss_stage_mixed(st, 0, n_seqs, hidden_bf16, token_ids, cu_q, ctx_before, block_tables, max_blocks,
                        total_tokens, out_hidden_bf16, out_logits, out_argmax);
}

int ss_stage_mixed(ss_stage *st, int n_decode_rows, int n_seqs, const void *hidden_bf16, const int32_t *token_ids,
                   const int32_t *cu_q, const int32_t *ctx_before, const int32_t *block_tables, int max_blocks,
                   int total_tokens, void *out_hidden_bf16, float *out_logits, int32_t *out_argmax) {
  if (n_decode_rows < 0 || n_decode_rows > n_seqs || n_decode_rows > total_tokens) return SS_ERR_INVALID_ARG;
  int rc = common_checks(st, n_seqs, total_tokens, hidden_bf16, token_ids, block_tables, max_blocks, ctx_before,
                         out_logits, out_argmax);
  if (rc != SS_OK) return rc;
  if (!cu_q) return SS_ERR_INVALID_ARG;
  if (total_tokens > st->d.max_tokens) return SS_ERR_CAPACITY;
  CallArgs a;
  memset(&a, 0, sizeof(a));
  a.hidden_in = hidden_bf16; a.token_ids = token_ids; a.block_tables = block_tables; a.ctx = ctx_before;
  a.cu_q = cu_q; a.out_hidden = out_hidden_bf16; a.out_logits = out_logits; a.out_argmax = out_argmax;
  a.n_seqs = n_seqs; a.T = total_tokens; a.max_blocks = max_blocks;
  if ((rc = upload_args(st, a)) != SS_OK) return rc;
  if ((rc = debug_check(st, false, n_decode_rows)) != SS_OK) return rc;
  const int64_t before = g_launches;
  cudaError_t e = enqueue_forward(st, false, n_seqs, total_tokens, out_logits || out_argmax, n_decode_rows);
  st->launches += g_launches - before;
  if (e != cudaSuccess) return cuda_fail(e, "ss_stage_mixed");
  return SS_OK;
}

int ss_stage_decode(ss_stage *st, int batch, const void *hidden_bf16, const int32_t *token_ids,
                    const int32_t *block_tables, int max_blocks, const int32_t *context_lens,
                    void *out_hidden_bf16, float *out_logits, int32_t *out_argmax) {
  int rc = common_checks(st, batch, batch, hidden_bf16, token_ids, block_tables, max_blocks, context_lens,
                         out_logits, out_argmax);
  if (rc != SS_OK) return rc;
  CallArgs a;
  memset(&a, 0, sizeof(a));
  a.hidden_in = hidden_bf16; a.token_ids = token_ids; a.block_tables = block_tables; a.ctx = context_lens;
  a.out_hidden = out_hidden_bf16; a.out_logits = out_logits; a.out_argmax = out_argmax;
  a.n_seqs = batch; a.T = batch; a.max_blocks = max_blocks;
  if ((rc = upload_args(st, a)) != SS_OK) return rc;
  if ((rc = debug_check(st, true, 0)) != SS_OK) return rc;
  const bool tail = out_logits || out_argmax;
  const bool tp_callback = (st->allreduce || st->tp_size > 1) && !tp_fused_eligible(st, batch);
  if (!st->use_graph || tp_callback) {  // the all-reduce CALLBACK calls back into the caller: never captured
    const int64_t before = g_launches;
    cudaError_t e = enqueue_forward(st, true, batch, batch, tail);
    st->launches += g_launches - before;
    if (e != cudaSuccess) return cuda_fail(e, "ss_stage_decode");
    return SS_OK;
  }
  const int key = batch * 2 + (tail ? 1 : 0);
  auto it = st->graphs.find(key);
  if (it == st->graphs.end()) {
    // capture the kernel sequence once; user pointers are reached through the device-side CallArgs block
    cudaGraph_t graph = nullptr;
    const int64_t before = g_launches;
    CK(cudaStreamBeginCapture(st->stream, cudaStreamCaptureModeThreadLocal));
    cudaError_t e = enqueue_forward(st, true, batch, batch, tail);
    cudaError_t e2 = cudaStreamEndCapture(st->stream, &graph);
    const int64_t n_kernels = g_launches - before;
    if (e != cudaSuccess || e2 != cudaSuccess) {
      if (graph) cudaGraphDestroy(graph);
      return cuda_fail(e != cudaSuccess ? e : e2, "decode graph capture");
    }
    st->graph_captures += 1;
    Graph gr;
    e = cudaGraphInstantiate(&gr.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGraphInstantiate");
    gr.kernels = n_kernels;
    it = st->graphs.emplace(key, gr).first;
  }
  CK(cudaGraphLaunch(it->second.exec, st->stream));
  st->launches += it->second.kernels;
  return SS_OK;
}

}  // extern "C"

// ===================================================================================================================
// op-level entry points: the same GEMM kernel, stand-alone (per-kernel parity tests, profiling)
// ===================================================================================================================
namespace ss {
static int device_sms() {  // of the current device (a process may drive several)
  int dev = 0, n = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return 0;
  return n;
}

static int op_gemm(const void *x_dev, const void *w0, const void *w1, float *c_f32, void *c_bf16, int T, int N, int K,
                   bool dual, void *scratch_dev, size_t scratch_bytes, void *cuda_stream) {
  if (!x_dev || !w0 || (dual && !w1) || (!c_f32 && !c_bf16) || T <= 0 || N <= 0 || K <= 0 || !scratch_dev)
    return SS_ERR_INVALID_ARG;
  if (K % 8 != 0 || ((uintptr_t)x_dev & 15) || ((uintptr_t)w0 & 15) || (dual && ((uintptr_t)w1 & 15)) ||
      ((uintptr_t)scratch_dev & 255))
    return SS_ERR_UNSUPPORTED;
  if (scratch_bytes < gemm_fix_bytes()) return SS_ERR_CAPACITY;
  cudaError_t e = gemm_init();
  if (e != cudaSuccess) return cuda_fail(e, "gemm_init");
  const int n_sm = device_sms();
  if (n_sm <= 0) return cuda_fail(cudaErrorNoDevice, "device_sms");
  CUtensorMap ta, tu, tb;
  GemmLaunch g;
  memset(&g, 0, sizeof(g));
  GemmParams &p = g.p;
  p.n_seg = 1;
  p.seg_rows[0] = N;
  p.T = T;
  p.K = K;
  p.epi = dual ? EPI_SWIGLU_BF16 : EPI_F32;
  p.ld_out = N;
  p.out_f32 = c_f32;
  p.out_bf16 = c_bf16;
  p.fix_flags = (int *)scratch_dev;
#ifdef SS_GEMM_TRACE
  p.trace = (unsigned long long *)((uint8_t *)scratch_dev + gemm_fix_bytes());  // profiling build: caller over-allocates
#endif
  p.fix_slots = (float *)((uint8_t *)scratch_dev + GEMM_FIX_FLAG_BYTES);
  g.dual = dual;
  // the caller's weights may come straight out of a preceding kernel, so the weight ring must not be primed before
  // that kernel has finished: no programmatic dependent launch here
  g.no_pdl = true;
  g.stream = (cudaStream_t)cuda_stream;
  gemm_plan(g, n_sm);
  if (make_tmap_bf16_2d(&ta, w0, (uint64_t)N, (uint64_t)K, GEMM_BM, true) != 0 ||
      (dual && make_tmap_bf16_2d(&tu, w1, (uint64_t)N, (uint64_t)K, GEMM_BM, true) != 0) ||
      make_tmap_bf16_2d(&tb, x_dev, (uint64_t)T, (uint64_t)K, (uint32_t)(g.pair ? 128 : p.bn), false) != 0) {
    g_cuda_err = "cuTensorMapEncodeTiled failed";
    return SS_ERR_CUDA;
  }
  g.a[0] = &ta;
  g.a[1] = dual ? &tu : nullptr;
  g.b = &tb;
  e = gemm_launch(g);
  if (e != cudaSuccess) return cuda_fail(e, "gemm_launch");
  return SS_OK;
}
}  // namespace ss

extern "C" {

size_t ss_op_gemm_scratch_bytes(void) { return gemm_fix_bytes(); }

int ss_debug_buffer(void *host_mapped_u64x4) {
  cudaError_t e = gemm_set_debug_buffer((unsigned long long *)host_mapped_u64x4);
  return e == cudaSuccess ? SS_OK : cuda_fail(e, "ss_debug_buffer");
}

int ss_op_gemm_bf16(const void *x_dev, const void *w_dev, float *c_dev, int T, int N, int K, void *scratch_dev,
                    size_t scratch_bytes, void *cuda_stream) {
  return op_gemm(x_dev, w_dev, nullptr, c_dev, nullptr, T, N, K, false, scratch_dev, scratch_bytes, cuda_stream);
}

int ss_op_gemm_swiglu_bf16(const void *x_dev, const void *wg_dev, const void *wu_dev, void *a_dev, int T, int F,
                           int K, void *scratch_dev, size_t scratch_bytes, void *cuda_stream) {
  return op_gemm(x_dev, wg_dev, wu_dev, nullptr, a_dev, T, F, K, true, scratch_dev, scratch_bytes, cuda_stream);
}

}  // extern "C"
