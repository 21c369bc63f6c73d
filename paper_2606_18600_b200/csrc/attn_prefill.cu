// attn_prefill.cu — step S6b: causal varlen prefill attention over the paged KV cache, with prior context
// (Table 2 "Attention / Prefill"; this is the attention of the migration recompute, PAPER.md:247,
// 259, and of chunked prefill in mixed iterations).  Query i of sequence s sits at global position
// p = ctx_before[s] + i and attends keys 0..p, ALL read from the pages (the keys of this call were appended by
// qkv_post before this kernel runs), which is what makes prefill == incremental decode.
//
// Both products are dense contractions, so they run on the tcgen05 tensor cores with the accumulators in tensor memory:
//   S = Q K^T   UMMA M = 128 query rows x N = 128 keys, K = d; Q and K tiles in smem (TMA, SWIZZLE_128B, K-major)
//   O += P V    UMMA M = 128 x N = d, K = 128 keys; P (bf16) is read from TENSOR MEMORY, where the softmax warps wrote it
//               over the S tile it came from; V tile in smem as TMA wrote it ([key][d]: the MN-major B operand)
// CTA = one 128-row query tile of one (sequence, q head); 8 warps, one role each:
//   warp 0  TMA producer: the Q tile once, then per key tile 8 pages of K and of V (16 tokens x d, one 2-D box per 64
//           columns; the layer's pool is one 2-D tensor), 3-stage ring
//   warp 1  issues the S MMAs (one lane) into a DOUBLE-buffered S so that S_{j+1} is computed while tile j is in softmax
//   warp 2  issues the P.V MMAs (one lane); a separate issuing thread because one tcgen05.mma occupies its issuer
//           ~128 cycles whatever its shape
//   warps 4-7  softmax: thread = query row = TMEM lane, so row max / row sum need no shuffle; tcgen05.ld of the S row,
//           exp2 in fp32, P -> bf16 -> tcgen05.st; the running maximum is only moved when it grows by more than 2^8
//           (then, rarely, the O accumulator is rescaled in place), else P simply is up to 2^8 larger — the final
//           O / l is unchanged
// The 8 q heads of a GQA group are adjacent in blockIdx.x so their K/V re-reads hit L2.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "common.cuh"
#include "internal.h"

namespace ss {

constexpr int TA_BM = 128;      // query rows per CTA = UMMA M = TMEM lanes
constexpr int TA_BN = 128;      // keys per tile
constexpr int TA_STAGES = 3;    // K/V ring depth
constexpr int TA_THREADS = 256;
constexpr int TA_PAGES = TA_BN / 16;
constexpr float TA_LAZY = 8.0f; // the running maximum (log2 units) is moved only when exceeded by more than this

// ---- plan: token -> (sequence, position) and the prefix sum of query tiles --------------------------------------
__global__ void prefill_plan_kernel(const CallArgs *__restrict__ args, int n_seqs, int seq0, PrefillPlan plan) {
  pdl_launch_dependents();
  pdl_wait();
  if (blockIdx.x == 0) {
    __shared__ int n_tiles_s;
    if (threadIdx.x == 0) {
      int acc = 0;
      plan.tile_cum[0] = 0;
      for (int s = 0; s < n_seqs; ++s) {
        if (s >= seq0) acc += (args->cu_q[s + 1] - args->cu_q[s] + TA_BM - 1) / TA_BM;
        plan.tile_cum[s + 1] = acc;
      }
      n_tiles_s = acc;
    }
    __syncthreads();
    // launch order = heaviest tile first (keys attended = context + causal prefix): the grid is dispatched in
    // blockIdx order, and a causal batch in natural order would start its most expensive tiles last
    const int n = min(n_tiles_s, plan.max_tiles);
    int32_t *key = plan.tile_order + plan.max_tiles;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      int lo = 0, hi = n_seqs;
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (plan.tile_cum[mid] <= i) lo = mid; else hi = mid;
      }
      const int q_len = args->cu_q[lo + 1] - args->cu_q[lo];
      key[i] = args->ctx[lo] + min(q_len, (i - plan.tile_cum[lo] + 1) * TA_BM);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x) {  // rank sort (stable): n is a few hundred, once per call
      const int k = key[i];
      int rank = 0;
      for (int j = 0; j < n; ++j) {
        const int kj = key[j];
        rank += (kj > k || (kj == k && j < i)) ? 1 : 0;
      }
      plan.tile_order[rank] = i;
    }
  }
  for (int s = blockIdx.x; s < n_seqs; s += gridDim.x) {
    const int t0 = args->cu_q[s], t1 = args->cu_q[s + 1], c = args->ctx[s];
    for (int t = t0 + threadIdx.x; t < t1; t += blockDim.x) {
      plan.tok_seq[t] = s;
      plan.tok_pos[t] = c + (t - t0);
    }
  }
}

cudaError_t launch_prefill_plan(const CallArgs *args, int n_seqs, int seq0, PrefillPlan plan, cudaStream_t s) {
  int blocks = n_seqs < 1 ? 1 : (n_seqs > 1024 ? 1024 : n_seqs);
  return launch_pdl(prefill_plan_kernel, dim3(blocks), dim3(256), 0, s, args, n_seqs, seq0, plan);
}
int prefill_attn_tile_rows() { return TA_BM; }

template <int D>
__global__ void __launch_bounds__(TA_THREADS, 1)
prefill_attn_kernel(const __grid_constant__ CUtensorMap q_map, const __grid_constant__ CUtensorMap kv_map,
                    const PrefillAttnParams p) {
  constexpr int NH = D / 64;                     // 64-column halves of a row (one 128-byte swizzle row each)
  constexpr uint32_t HALF_BYTES = TA_BM * 128;   // [128 rows][64 bf16]
  constexpr uint32_t TILE_BYTES = NH * HALF_BYTES;
  constexpr uint32_t S_COLS = TA_BN;             // fp32 S tile; P (bf16) lives in its first 64 columns
  constexpr uint32_t O_COL = 2 * S_COLS;
  constexpr uint32_t TMEM_COLS = 512;
  extern __shared__ uint8_t smem_raw[];
  uint8_t *base = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t *q_s = base;
  uint8_t *k_s = q_s + TILE_BYTES;                       // [TA_STAGES][TILE_BYTES]
  uint8_t *v_s = k_s + (size_t)TA_STAGES * TILE_BYTES;   // [TA_STAGES][TILE_BYTES]
  uint64_t *bars = (uint64_t *)(v_s + (size_t)TA_STAGES * TILE_BYTES);
  uint64_t *q_full = bars;
  uint64_t *k_full = bars + 1, *v_full = k_full + TA_STAGES, *kv_empty = v_full + TA_STAGES;
  uint64_t *s_full = kv_empty + TA_STAGES, *p_full = s_full + 2, *pv_done = p_full + 2;
  uint32_t *tmem_slot = (uint32_t *)(pv_done + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  pdl_launch_dependents();
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&q_map);
    tma_prefetch_desc(&kv_map);
    mbar_init(q_full, 1);
    for (int i = 0; i < TA_STAGES; ++i) {
      mbar_init(&k_full[i], 1);
      mbar_init(&v_full[i], 1);
      mbar_init(&kv_empty[i], 2);  // the S issuer's and the P.V issuer's commits
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&s_full[i], 1);
      mbar_init(&p_full[i], 128);  // every softmax thread
      mbar_init(&pv_done[i], 1);
    }
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc_dyn(tmem_slot, TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait();  // q, the pools and the plan are written by earlier kernels of this call

  // ---- which tile
  const int head = blockIdx.x;
  const int32_t *tile_cum = p.plan.tile_cum;
  const bool live = (int)blockIdx.y < tile_cum[p.n_seqs];
  int n_kt = 0, s = 0, q_begin = 0, i0 = 0, rows = 0, p0 = 0, kv_len = 0, hk = 0;
  const CallArgs *args = p.args;
  if (live) {
    const int slot = p.plan.tile_order[blockIdx.y];
    int lo = 0, hi = p.n_seqs;  // tile_cum[lo] <= slot < tile_cum[hi]
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (tile_cum[mid] <= slot) lo = mid; else hi = mid;
    }
    s = lo;
    q_begin = args->cu_q[s];
    const int q_len = args->cu_q[s + 1] - q_begin;
    i0 = (slot - tile_cum[s]) * TA_BM;
    rows = min(TA_BM, q_len - i0);
    p0 = args->ctx[s] + i0;      // global position of the tile's first query
    kv_len = p0 + rows;          // keys 0..kv_len-1 are needed by this tile
    n_kt = (kv_len + TA_BN - 1) / TA_BN;
    hk = head / (p.n_q / p.n_kv);
  }
  const int n_pages_seq = (kv_len + 15) >> 4;

  if (warp == 0) {
    if (lane == 0 && live) {
      // ---------------- TMA producer ----------------
      const uint64_t pol_q = l2_policy_evict_first(), pol_kv = l2_policy_evict_last();  // K/V: re-read by the group's heads
      mbar_expect_tx(q_full, TILE_BYTES);
#pragma unroll
      for (int h = 0; h < NH; ++h) tma_load_2d(q_s + h * HALF_BYTES, &q_map, q_full, head * D + h * 64, q_begin + i0, pol_q);
      const int32_t *bt = args->block_tables + (size_t)s * args->max_blocks;
      const int v_row0 = p.n_pages * p.n_kv * 16;
      for (int j = 0; j < n_kt; ++j) {
        const int st = j % TA_STAGES;
        mbar_wait(&kv_empty[st], (((uint32_t)(j / TA_STAGES)) & 1u) ^ 1u);
        const int n_pg = min(TA_PAGES, n_pages_seq - j * TA_PAGES);  // pages past the sequence's end are never touched
        uint8_t *kd = k_s + (size_t)st * TILE_BYTES, *vd = v_s + (size_t)st * TILE_BYTES;
        mbar_expect_tx(&k_full[st], (uint32_t)n_pg * NH * 2048u);
        mbar_expect_tx(&v_full[st], (uint32_t)n_pg * NH * 2048u);
        int rowv[TA_PAGES];
#pragma unroll
        for (int pg = 0; pg < TA_PAGES; ++pg)
          rowv[pg] = pg < n_pg ? (bt[j * TA_PAGES + pg] * p.n_kv + hk) * 16 : 0;
#pragma unroll
        for (int pg = 0; pg < TA_PAGES; ++pg)
          if (pg < n_pg) {
#pragma unroll
            for (int h = 0; h < NH; ++h)
              tma_load_2d(kd + h * HALF_BYTES + pg * 2048, &kv_map, &k_full[st], h * 64, rowv[pg], pol_kv);
          }
#pragma unroll
        for (int pg = 0; pg < TA_PAGES; ++pg)
          if (pg < n_pg) {
#pragma unroll
            for (int h = 0; h < NH; ++h)
              tma_load_2d(vd + h * HALF_BYTES + pg * 2048, &kv_map, &v_full[st], h * 64, v_row0 + rowv[pg], pol_kv);
          }
      }
    }
  } else if (warp == 1) {
    if (lane == 0 && live) {
      // ---------------- S = Q K^T issuer ----------------
      const uint32_t idesc = umma_idesc_bf16(TA_BM, TA_BN);
      mbar_wait(q_full, 0);
      for (int j = 0; j < n_kt; ++j) {
        const int st = j % TA_STAGES, b = j & 1;
        if (j >= 2) mbar_wait(&pv_done[b], ((uint32_t)((j - 2) >> 1)) & 1u);  // P_{j-2} (in this S buffer) was consumed
        mbar_wait(&k_full[st], ((uint32_t)(j / TA_STAGES)) & 1u);
        tc_fence_after();
        const uint32_t qa = smem_u32(q_s), ka = smem_u32(k_s + (size_t)st * TILE_BYTES);
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
          const uint32_t off = (uint32_t)(ks >> 2) * HALF_BYTES + (uint32_t)(ks & 3) * 32u;
          umma_bf16(tmem_base + (uint32_t)b * S_COLS, umma_desc_k_sw128(qa + off), umma_desc_k_sw128(ka + off), idesc,
                    ks > 0 ? 1u : 0u);
        }
        umma_commit(&s_full[b]);
        umma_commit(&kv_empty[st]);
      }
    }
  } else if (warp == 2) {
    if (lane == 0 && live) {
      // ---------------- O += P V issuer ----------------
      const uint32_t idesc = umma_idesc_bf16_b_mn(TA_BM, D);
      for (int j = 0; j < n_kt; ++j) {
        const int st = j % TA_STAGES, b = j & 1;
        mbar_wait(&p_full[b], ((uint32_t)(j >> 1)) & 1u);
        mbar_wait(&v_full[st], ((uint32_t)(j / TA_STAGES)) & 1u);
        tc_fence_after();
        const uint32_t va = smem_u32(v_s + (size_t)st * TILE_BYTES);
        const int n_pg = min(TA_PAGES, n_pages_seq - j * TA_PAGES);  // one k-step = one page of 16 keys
        for (int ks = 0; ks < n_pg; ++ks)
          umma_bf16_ts(tmem_base + O_COL, tmem_base + (uint32_t)b * S_COLS + (uint32_t)ks * 8u,
                       umma_desc_mn_sw128(va + (uint32_t)ks * 2048u, HALF_BYTES, 1024u), idesc, (j > 0 || ks > 0) ? 1u : 0u);
        umma_commit(&kv_empty[st]);
        umma_commit(&pv_done[b]);
      }
    }
  } else if (warp >= 4 && live) {
    // ---------------- softmax: thread = query row ----------------
    const int quad = warp & 3;
    const int r = quad * 32 + lane;
    const uint32_t lane_base = tmem_base + ((uint32_t)(quad * 32) << 16);
    const float sl2 = 1.4426950408889634f / sqrtf((float)D);  // log2(e) / sqrt(d)
    const int qpos = p0 + r;
    float m_used = -INFINITY, l_run = 0.f;  // m_used in log2 units (score * sl2)
    for (int j = 0; j < n_kt; ++j) {
      const int b = j & 1, st = j % TA_STAGES;
      mbar_wait(&s_full[b], ((uint32_t)(j >> 1)) & 1u);
      tc_fence_after();
      uint32_t v[TA_BN];
#pragma unroll
      for (int c = 0; c < TA_BN / 32; ++c)
        tmem_ld_32x32(lane_base + (uint32_t)b * S_COLS + (uint32_t)c * 32u, *reinterpret_cast<uint32_t(*)[32]>(&v[c * 32]));
      tmem_ld_wait();
      const int jbase = j * TA_BN;
      if (jbase + TA_BN - 1 > p0) {  // the tile reaches past the first query's position: causal mask
#pragma unroll
        for (int c = 0; c < TA_BN; ++c)
          if (jbase + c > qpos) v[c] = 0xff800000u;  // -inf
      }
      float mx = -INFINITY;
#pragma unroll
      for (int c = 0; c < TA_BN; ++c) mx = fmaxf(mx, __uint_as_float(v[c]));
      mx *= sl2;
      // lazy maximum: move it only when the tile's maximum exceeds it by more than TA_LAZY (P then stays <= 2^TA_LAZY)
      const bool move = mx > m_used + TA_LAZY;   // also true on the first tile (m_used = -inf; key 0 is visible to all)
      float alpha = 1.0f;
      if (move) {
        alpha = fast_exp2(m_used - mx);  // 0 on the first tile
        m_used = mx;
        l_run *= alpha;
      }
      if (j > 0 && __any_sync(0xffffffffu, move)) {
        // rescale the O accumulator in place (rare): P.V of tile j-1 must have completed first
        mbar_wait(&pv_done[(j - 1) & 1], ((uint32_t)((j - 1) >> 1)) & 1u);
        tc_fence_after();
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
          uint32_t o[32];
          tmem_ld_32x32(lane_base + O_COL + (uint32_t)c * 32u, o);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
          tmem_st_32x32(lane_base + O_COL + (uint32_t)c * 32u, o);
        }
      }
      float rs = 0.f;
      uint32_t pk[TA_BN / 2];
      const float neg_m = -m_used;
#pragma unroll
      for (int c = 0; c < TA_BN; c += 2) {
        const float e0 = fast_exp2(fmaf(__uint_as_float(v[c]), sl2, neg_m));
        const float e1 = fast_exp2(fmaf(__uint_as_float(v[c + 1]), sl2, neg_m));
        rs += e0 + e1;
        pk[c >> 1] = pack_bf16x2(e0, e1);
      }
      l_run += rs;
#pragma unroll
      for (int c = 0; c < TA_BN / 64; ++c)
        tmem_st_32x32(lane_base + (uint32_t)b * S_COLS + (uint32_t)c * 32u, *reinterpret_cast<uint32_t(*)[32]>(&pk[c * 32]));
      if (j == n_kt - 1 && (kv_len & 15) != 0) {
        // the sequence's last page holds slots past its end with whatever the pool held: zero those V rows so that
        // 0 * garbage (possibly NaN) cannot reach the output (their P is exactly 0: the causal mask covers them)
        mbar_wait(&v_full[st], ((uint32_t)(j / TA_STAGES)) & 1u);
        const int k0 = kv_len - jbase, k1 = (n_pages_seq - j * TA_PAGES) * 16;  // rows [k0, k1) of the tile
        uint8_t *vd = v_s + (size_t)st * TILE_BYTES;
        for (int idx = r; idx < (k1 - k0) * NH * 8; idx += 128) {
          const int row = k0 + idx / (NH * 8), rem = idx % (NH * 8);
          *reinterpret_cast<uint4 *>(vd + (rem >> 3) * HALF_BYTES + row * 128 + (rem & 7) * 16) = make_uint4(0u, 0u, 0u, 0u);
        }
        fence_proxy_async();
      }
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(&p_full[b]);
    }
    // ---- normalise and store
    mbar_wait(&pv_done[(n_kt - 1) & 1], ((uint32_t)((n_kt - 1) >> 1)) & 1u);
    tc_fence_after();
    const float inv = 1.0f / l_run;
    __nv_bfloat16 *og = (__nv_bfloat16 *)p.out + ((size_t)(q_begin + i0 + r) * p.n_q + head) * D;
#pragma unroll
    for (int c = 0; c < D / 32; ++c) {
      uint32_t o[32];
      tmem_ld_32x32(lane_base + O_COL + (uint32_t)c * 32u, o);
      tmem_ld_wait();
      if (r < rows) {
#pragma unroll
        for (int i = 0; i < 32; i += 8) {
          uint4 w;
          w.x = pack_bf16x2(__uint_as_float(o[i]) * inv, __uint_as_float(o[i + 1]) * inv);
          w.y = pack_bf16x2(__uint_as_float(o[i + 2]) * inv, __uint_as_float(o[i + 3]) * inv);
          w.z = pack_bf16x2(__uint_as_float(o[i + 4]) * inv, __uint_as_float(o[i + 5]) * inv);
          w.w = pack_bf16x2(__uint_as_float(o[i + 6]) * inv, __uint_as_float(o[i + 7]) * inv);
          *reinterpret_cast<uint4 *>(og + c * 32 + i) = w;
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_dyn(tmem_base, TMEM_COLS);
  }
}

static size_t prefill_smem(int d) {
  return 1024 + (size_t)(1 + 2 * TA_STAGES) * (d / 64) * TA_BM * 128 + 8 * (1 + 3 * TA_STAGES + 6) + 16;
}

cudaError_t prefill_attn_init() {  // per device: called from ss_stage_create
  cudaError_t e = cudaFuncSetAttribute(prefill_attn_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)prefill_smem(128));
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(prefill_attn_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)prefill_smem(64));
}

cudaError_t launch_prefill_attn(const PrefillAttnParams &p, cudaStream_t s) {
  dim3 grid(p.n_q, p.max_tiles);
  if (p.d == 128)
    return launch_pdl(prefill_attn_kernel<128>, dim3(grid), dim3(TA_THREADS), prefill_smem(128), s, *p.q_map, *p.kv_map, p);
  return launch_pdl(prefill_attn_kernel<64>, dim3(grid), dim3(TA_THREADS), prefill_smem(64), s, *p.q_map, *p.kv_map, p);
}

}  // namespace ss
