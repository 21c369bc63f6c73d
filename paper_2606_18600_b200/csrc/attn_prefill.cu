// attn_prefill.cu — step S6b: causal varlen prefill attention over the paged KV cache, with prior context
// (Table 2 "Attention / Prefill"; this is the attention of the migration recompute, PAPER.md:247,
// 259, and of chunked prefill in mixed iterations).  Query i of sequence s sits at global position
// p = ctx_before[s] + i and attends keys 0..p, ALL read from the pages (the keys of this call were appended by
// qkv_post before this kernel runs), which is what makes prefill == incremental decode.
//
// Both products are dense contractions, so they run on the tcgen05 tensor cores with the accumulators in tensor memory:
//   S = Q K^T   UMMA M = 128 query rows x N = 64 keys, K = d; Q and K tiles in smem (TMA, SWIZZLE_128B, K-major)
//   O += P V    UMMA M = 128 x N = d, K = 64 keys; P (bf16) is read from TENSOR MEMORY, where the softmax warps wrote it
//               over the S tile it came from; V tile in smem as TMA wrote it ([key][d]: the MN-major B operand)
// CTA = the same 128 query positions of TWO q heads of one GQA group ("tile A", "tile B": they attend the same keys, so
// one K/V ring serves both and every K/V byte fetched from L2 feeds 256 query rows); 12 warps, one role each:
//   warps 0, 3  TMA producers of K and of V: both Q tiles per item (warp 0), then per key tile 4 pages (16 tokens x d, one 2-D
//               box per 64 columns; the layer's pool is one 2-D tensor) into a 5-stage ring.  Two threads because one
//               cp.async.bulk.tensor occupies its issuer ~100 cycles (clock64 stamps: 16 boxes per stage = 1,650 cycles)
//   warps 1, 2  issue ALL MMAs of tile A / tile B (one lane each): S_j into DOUBLE-buffered S tiles, then P.V of stage
//               j - 1, so S_j is computed while tile j - 1 is in softmax.  One thread per tile because one tcgen05.mma
//               occupies its issuer 75-150 cycles whatever its shape (a single P.V thread for both tiles was busy
//               ~2,000 cycles per stage); the MMAs of one thread execute in issue order, so S_j cannot overtake the
//               P.V_{j-2} that still reads the P stored over that S buffer
//   warps 4-7 / 8-11  softmax of tile A / B: thread = query row = TMEM lane, so row max / row sum need no shuffle;
//               tcgen05.ld of the S row, exp2 in fp32, P -> bf16 -> tcgen05.st; the running maximum is only moved when it
//               grows by more than 2^16 (then, rarely, the O accumulator is rescaled in place), else P simply is up to
//               2^16 larger — the final O / l is unchanged (at 2^8 the maximum still moved in 13% of the stages)
// TMEM (512 columns): S_A0 S_A1 S_B0 S_B1 (64 each), O_A, O_B (d each).
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "common.cuh"
#include "internal.h"

namespace ss {

constexpr int TA_BM = 128;      // query rows per tile = UMMA M = TMEM lanes
constexpr int TA_BN = 64;       // keys per ring stage (4 pages)
constexpr int TA_STAGES = 5;    // K/V ring depth: 320 keys in flight per CTA
constexpr int TA_THREADS = 384;
constexpr int TA_PAGES = TA_BN / 16;
// (the running maximum, in log2 units, is moved only when exceeded by more than PrefillAttnParams::lazy = 16)

// ---- plan: token -> (sequence, position), the prefix sum of query tiles and one descriptor per launch slot ---------
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
    auto seq_of = [&](int i) {
      int lo = 0, hi = n_seqs;  // tile_cum[lo] <= i < tile_cum[hi]
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (plan.tile_cum[mid] <= i) lo = mid; else hi = mid;
      }
      return lo;
    };
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      const int s = seq_of(i);
      const int q_len = args->cu_q[s + 1] - args->cu_q[s];
      key[i] = args->ctx[s] + min(q_len, (i - plan.tile_cum[s] + 1) * TA_BM);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x) {  // rank sort (stable): n is a few hundred, once per call
      const int k = key[i];
      int rank = 0;
      for (int j = 0; j < n; ++j) {
        const int kj = key[j];
        rank += (kj > k || (kj == k && j < i)) ? 1 : 0;
      }
      plan.tile_order[i] = rank;   // launch slot of tile i
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      const int s = seq_of(i);
      const int q_begin = args->cu_q[s], q_len = args->cu_q[s + 1] - q_begin;
      const int i0 = (i - plan.tile_cum[s]) * TA_BM;
      int4 d;
      d.x = q_begin + i0;              // first packed row of the tile
      d.y = min(TA_BM, q_len - i0);    // its rows
      d.z = args->ctx[s] + i0;         // global position of its first query
      d.w = s;
      reinterpret_cast<int4 *>(plan.tile_desc)[plan.tile_order[i]] = d;
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
  return launch_pdl(prefill_plan_kernel, dim3(blocks), dim3(1024), 0, s, args, n_seqs, seq0, plan);
}
int prefill_attn_tile_rows() { return TA_BM; }

template <int D>
__global__ void __launch_bounds__(TA_THREADS, 1)
prefill_attn_kernel(const __grid_constant__ CUtensorMap q_map, const __grid_constant__ CUtensorMap kv_map,
                    const PrefillAttnParams p) {
  constexpr int NH = D / 64;                     // 64-column halves of a row (one 128-byte swizzle row each)
  constexpr uint32_t QHALF_BYTES = TA_BM * 128;  // Q: [128 rows][64 bf16] per half
  constexpr uint32_t QTILE_BYTES = NH * QHALF_BYTES;
  constexpr uint32_t HALF_BYTES = TA_BN * 128;   // K, V: [TA_BN keys][64 bf16] per half
  constexpr uint32_t TILE_BYTES = NH * HALF_BYTES;
  constexpr uint32_t S_COLS = TA_BN;             // fp32 S tile; P (bf16) lives in its first TA_BN / 2 columns
  constexpr uint32_t O_COL = 4 * S_COLS;         // S_A0 S_A1 S_B0 S_B1 | O_A O_B
  constexpr uint32_t TMEM_COLS = 512;
  static_assert(O_COL + 2 * D <= TMEM_COLS, "TMEM budget");
  extern __shared__ uint8_t smem_raw[];
  uint8_t *base = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t *q_s = base;                                   // [2 tiles][QTILE_BYTES]
  uint8_t *k_s = q_s + 2 * QTILE_BYTES;                  // [TA_STAGES][TILE_BYTES]
  uint8_t *v_s = k_s + (size_t)TA_STAGES * TILE_BYTES;   // [TA_STAGES][TILE_BYTES]
  uint64_t *bars = (uint64_t *)(v_s + (size_t)TA_STAGES * TILE_BYTES);
  uint64_t *q_full = bars, *q_empty = bars + 1;
  uint64_t *k_full = bars + 2, *v_full = k_full + TA_STAGES, *kv_empty = v_full + TA_STAGES;
  uint64_t *s_full = kv_empty + TA_STAGES;  // [tile][buffer]
  uint64_t *p_full = s_full + 4, *pv_done = p_full + 4;
  uint64_t *o_free = pv_done + 4;           // [tile]
  uint32_t *tmem_slot = (uint32_t *)(o_free + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  pdl_launch_dependents();
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&q_map);
    tma_prefetch_desc(&kv_map);
    mbar_init(q_full, 1);
    mbar_init(q_empty, 2);         // one commit per issuing thread, after its last S of the item
    for (int i = 0; i < TA_STAGES; ++i) {
      mbar_init(&k_full[i], 1);
      mbar_init(&v_full[i], 1);
      mbar_init(&kv_empty[i], 2);  // one commit per tile's MMA-issuing thread, after its P.V of the stage
    }
    for (int i = 0; i < 4; ++i) {
      mbar_init(&s_full[i], 1);
      mbar_init(&p_full[i], 4);    // one arrival per softmax warp of the tile (32 arrivals of a warp on one barrier serialise)
      mbar_init(&pv_done[i], 1);
    }
    mbar_init(&o_free[0], 4);      // per softmax warp: every thread has read its O row out of tensor memory
    mbar_init(&o_free[1], 4);
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc_dyn(tmem_slot, TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait();  // q, the pools and the plan are written by earlier kernels of this call

  // ---- work items: (launch slot y of a query tile, heaviest first; x = (kv head, pair of its q heads)), dealt to the
  // persistent CTAs in snake order (round r runs left to right, r + 1 right to left) so that the sums stay level.
  // Every role walks the same list; all ring / buffer phases run on counters that continue across items:
  //   g    key stages so far (K/V ring slot g % TA_STAGES)       gt  the same for tile t alone (S buffer gt & 1)
  const int G = p.n_q / p.n_kv, pairs = (G + 1) >> 1, n_x = p.n_kv * pairs;
  const int n_items = min(p.plan.tile_cum[p.n_seqs], p.max_tiles) * n_x;
  const CallArgs *args = p.args;
  struct Item {
    int row0, rows, p0, s, hk, head_a, n_kt, n_pages_seq, kv_len;
    bool has_b;
  };
  auto get_item = [&](int k, Item &w) -> bool {
    const int idx = k * (int)gridDim.x + ((k & 1) ? (int)gridDim.x - 1 - (int)blockIdx.x : (int)blockIdx.x);
    if (idx >= n_items) return false;
    const int y = idx / n_x, x = idx - y * n_x;
    const int4 d = reinterpret_cast<const int4 *>(p.plan.tile_desc)[y];
    w.row0 = d.x; w.rows = d.y; w.p0 = d.z; w.s = d.w;
    w.hk = x / pairs;
    const int pi = x - w.hk * pairs;
    w.head_a = w.hk * G + 2 * pi;
    w.has_b = 2 * pi + 1 < G;            // an odd group leaves its last head alone
    w.kv_len = w.p0 + w.rows;            // keys 0..kv_len-1 are needed by this tile
    w.n_kt = (w.kv_len + TA_BN - 1) / TA_BN;
    w.n_pages_seq = (w.kv_len + 15) >> 4;
    return true;
  };
  Item w;

  // (whole-warp roles, issue under elect_one(): see gemm_tcgen05.cu)
  if (warp == 0 || warp == 3) {
    // ---------------- TMA producers: warp 0 = Q and K, warp 3 = V ----------------
    const bool is_k = warp == 0;
    const uint64_t pol_q = l2_policy_evict_first(), pol_kv = l2_policy_evict_last();  // K/V: re-read by other tiles
    const int row_off = is_k ? 0 : p.n_pages * p.n_kv * 16;   // the V rows follow the K rows in the layer's tensor
    uint8_t *ring = is_k ? k_s : v_s;
    uint64_t *full = is_k ? k_full : v_full;
    uint32_t g = 0;
    for (int k = 0; get_item(k, w); ++k) {
      if (is_k) {
        if (k > 0) mbar_wait(q_empty, (uint32_t)(k - 1) & 1u);  // the previous item's S MMAs have read its Q tiles
        if (elect_one()) {
          mbar_expect_tx(q_full, (w.has_b ? 2u : 1u) * QTILE_BYTES);
          for (int t = 0; t < (w.has_b ? 2 : 1); ++t)
#pragma unroll
            for (int h = 0; h < NH; ++h)
              tma_load_2d(q_s + t * QTILE_BYTES + h * QHALF_BYTES, &q_map, q_full, (w.head_a + t) * D + h * 64, w.row0, pol_q);
        }
        __syncwarp();
      }
      const int32_t *bt = args->block_tables + (size_t)w.s * args->max_blocks;
      // page ids: lane l holds the id of page 32 * blk + l of the sequence, fetched one block of 32 pages (8 stages)
      // ahead, so that no global-load latency sits in the per-stage loop (it was ~half of this warp's time per stage)
      int ids_next = lane < w.n_pages_seq ? bt[lane] : 0, ids = 0;
      for (int j = 0; j < w.n_kt; ++j, ++g) {
        if ((j & 7) == 0) {
          ids = ids_next;
          const int nx = (j + 8) * TA_PAGES + lane;
          ids_next = nx < w.n_pages_seq ? bt[nx] : 0;
        }
        const int st = (int)(g % TA_STAGES);
        const int n_pg = min(TA_PAGES, w.n_pages_seq - j * TA_PAGES);  // pages past the sequence's end are never touched
        int rowv[TA_PAGES];
#pragma unroll
        for (int pg = 0; pg < TA_PAGES; ++pg)
          rowv[pg] = (__shfl_sync(0xffffffffu, ids, (j & 7) * TA_PAGES + pg) * p.n_kv + w.hk) * 16 + row_off;
        mbar_wait(&kv_empty[st], ((g / TA_STAGES) & 1u) ^ 1u);
        uint8_t *dst = ring + (size_t)st * TILE_BYTES;
        if (elect_one()) {
          mbar_expect_tx(&full[st], (uint32_t)n_pg * NH * 2048u);
#pragma unroll
          for (int pg = 0; pg < TA_PAGES; ++pg)
            if (pg < n_pg) {
#pragma unroll
              for (int h = 0; h < NH; ++h)
                tma_load_2d(dst + h * HALF_BYTES + pg * 2048, &kv_map, &full[st], h * 64, rowv[pg], pol_kv);
            }
        }
        __syncwarp();
      }
    }
  } else if (warp == 1 || warp == 2) {
    // ---------------- MMA issuer of tile t: S of stage g, then P.V of stage g - 1 ----------------
    const int t = warp - 1;
    const uint32_t idesc_s = umma_idesc_bf16(TA_BM, TA_BN), idesc_pv = umma_idesc_bf16_b_mn(TA_BM, D);
    uint32_t g = 0, gt = 0, it_t = 0;
    // the P.V that is still owed: of the previous stage (possibly the previous item's last)
    bool pend = false, pend_on = false, pend_first = false;
    int pend_st = 0, pend_npg = 0;
    uint32_t pend_b = 0, pend_pp = 0, pend_vp = 0, pend_op = 0;
    auto flush_pv = [&]() {
      if (!pend) return;
      if (pend_on) {
        mbar_wait(&p_full[t * 2 + pend_b], pend_pp);
        if (pend_first && it_t > 0) mbar_wait(&o_free[t], pend_op);  // the previous item's O has been read out
      }
      mbar_wait(&v_full[pend_st], pend_vp);
      if (pend_on && elect_one()) {
        tc_fence_after();
        const uint32_t va = smem_u32(v_s + (size_t)pend_st * TILE_BYTES);
        for (int ks = 0; ks < pend_npg; ++ks)  // one k-step = one page of 16 keys
          umma_bf16_ts(tmem_base + O_COL + (uint32_t)t * D, tmem_base + (uint32_t)(t * 2 + pend_b) * S_COLS + (uint32_t)ks * 8u,
                       umma_desc_mn_sw128(va + (uint32_t)ks * 2048u, HALF_BYTES, 1024u), idesc_pv,
                       (!pend_first || ks > 0) ? 1u : 0u);
        umma_commit(&pv_done[t * 2 + pend_b]);
      }
      if (elect_one()) umma_commit(&kv_empty[pend_st]);  // this thread's S and P.V of the stage have read it (absent tile B: at once)
      __syncwarp();
      pend = false;
    };
    for (int k = 0; get_item(k, w); ++k) {
      const bool on = t == 0 || w.has_b;
      flush_pv();  // the previous item's last P.V goes first: this item's Q may still be in flight
      if (on) mbar_wait(q_full, (uint32_t)k & 1u);
      for (int j = 0; j < w.n_kt; ++j) {
        const int st = (int)(g % TA_STAGES);
        const uint32_t b = gt & 1u;
        mbar_wait(&k_full[st], (g / TA_STAGES) & 1u);
        if (elect_one()) {
          if (on) {
            // (S buffer b still holds P of stage gt - 2: that P.V was issued by this thread before, and executes before this)
            tc_fence_after();
            const uint32_t qa = smem_u32(q_s + t * QTILE_BYTES), ka = smem_u32(k_s + (size_t)st * TILE_BYTES);
            const uint32_t acc = tmem_base + (uint32_t)(t * 2 + b) * S_COLS;
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
              const uint32_t in_row = (uint32_t)(ks & 3) * 32u;
              umma_bf16(acc, umma_desc_k_sw128(qa + (uint32_t)(ks >> 2) * QHALF_BYTES + in_row),
                        umma_desc_k_sw128(ka + (uint32_t)(ks >> 2) * HALF_BYTES + in_row), idesc_s, ks > 0 ? 1u : 0u);
            }
            umma_commit(&s_full[t * 2 + b]);
          }
          if (j == w.n_kt - 1) umma_commit(q_empty);  // the item's Q tiles may be overwritten once these S MMAs are done
        }
        __syncwarp();
        if (j >= 1) flush_pv();
        pend = true; pend_on = on; pend_first = j == 0; pend_st = st; pend_b = b;
        pend_npg = min(TA_PAGES, w.n_pages_seq - j * TA_PAGES);
        pend_pp = (gt >> 1) & 1u; pend_vp = (g / TA_STAGES) & 1u; pend_op = (it_t - 1u) & 1u;
        ++g;
        if (on) ++gt;
      }
      if (on) ++it_t;
    }
    flush_pv();
  } else if (warp >= 4) {
    // ---------------- softmax of tile t: thread = query row ----------------
    const int t = warp >= 8 ? 1 : 0;
    const int quad = warp & 3;
    const int r = quad * 32 + lane;
    const uint32_t lane_base = tmem_base + ((uint32_t)(quad * 32) << 16);
    const uint32_t o_addr = lane_base + O_COL + (uint32_t)t * D;
    const float sl2 = 1.4426950408889634f / sqrtf((float)D);  // log2(e) / sqrt(d)
    uint32_t g = 0, gt = 0;
    for (int k = 0; get_item(k, w); ++k) {
      if (t == 1 && !w.has_b) {
        g += (uint32_t)w.n_kt;
        continue;
      }
      const int qpos = w.p0 + r, n_kt = w.n_kt;
      float m_used = -INFINITY, l_run = 0.f;  // m_used in log2 units (score * sl2)
      for (int j = 0; j < n_kt; ++j, ++g, ++gt) {
        const uint32_t b = gt & 1u;
        const int st = (int)(g % TA_STAGES);
        const uint32_t s_addr = lane_base + (uint32_t)(t * 2 + b) * S_COLS;
        mbar_wait(&s_full[t * 2 + b], (gt >> 1) & 1u);
        tc_fence_after();
        uint32_t v[TA_BN];
#pragma unroll
        for (int c = 0; c < TA_BN / 32; ++c) tmem_ld_32x32(s_addr + (uint32_t)c * 32u, *reinterpret_cast<uint32_t(*)[32]>(&v[c * 32]));
        tmem_ld_wait();
        const int jbase = j * TA_BN;
        if (jbase + TA_BN - 1 > w.p0) {  // the tile reaches past the first query's position: causal mask
#pragma unroll
          for (int c = 0; c < TA_BN; ++c)
            if (jbase + c > qpos) v[c] = 0xff800000u;  // -inf
        }
        float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};  // four independent chains
#pragma unroll
        for (int c = 0; c < TA_BN; ++c) mx4[c & 3] = fmaxf(mx4[c & 3], __uint_as_float(v[c]));
        const float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * sl2;
        // lazy maximum: move it only when the tile's maximum exceeds it by more than p.lazy (P then stays <= 2^lazy)
        const bool move = mx > m_used + p.lazy;    // also true on the first tile (m_used = -inf; key 0 is visible to all)
        float alpha = 1.0f;
        if (move) {
          alpha = fast_exp2(m_used - mx);  // 0 on the first tile
          m_used = mx;
          l_run *= alpha;
        }
        if (j > 0 && __any_sync(0xffffffffu, move)) {
          // rescale the O accumulator in place (rare): P.V of the previous stage must have completed first
          mbar_wait(&pv_done[t * 2 + ((gt - 1u) & 1u)], ((gt - 1u) >> 1) & 1u);
          tc_fence_after();
#pragma unroll
          for (int c = 0; c < D / 32; ++c) {
            uint32_t o[32];
            tmem_ld_32x32(o_addr + (uint32_t)c * 32u, o);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
            tmem_st_32x32(o_addr + (uint32_t)c * 32u, o);
          }
        }
        float rs4[4] = {0.f, 0.f, 0.f, 0.f};
        uint32_t pk[TA_BN / 2];
        const float neg_m = -m_used;
#pragma unroll
        for (int c = 0; c < TA_BN; c += 2) {
          const float e0 = fast_exp2(fmaf(__uint_as_float(v[c]), sl2, neg_m));
          const float e1 = fast_exp2(fmaf(__uint_as_float(v[c + 1]), sl2, neg_m));
          rs4[(c >> 1) & 3] += e0 + e1;
          pk[c >> 1] = pack_bf16x2(e0, e1);
        }
        l_run += (rs4[0] + rs4[1]) + (rs4[2] + rs4[3]);
        tmem_st_32x32(s_addr, pk);
        if (j == n_kt - 1 && (w.kv_len & 15) != 0) {
          // the sequence's last page holds slots past its end with whatever the pool held: zero those V rows so that
          // 0 * garbage (possibly NaN) cannot reach the output (their P is exactly 0: the causal mask covers them).
          // Done by BOTH tiles' warps (the same zeros), each before it publishes its own P to its own issuer.
          mbar_wait(&v_full[st], (g / TA_STAGES) & 1u);
          const int k0 = w.kv_len - jbase, k1 = (w.n_pages_seq - j * TA_PAGES) * 16;  // rows [k0, k1) of the tile
          uint8_t *vd = v_s + (size_t)st * TILE_BYTES;
          for (int idx = r; idx < (k1 - k0) * NH * 8; idx += 128) {
            const int row = k0 + idx / (NH * 8), rem = idx % (NH * 8);
            *reinterpret_cast<uint4 *>(vd + (rem >> 3) * HALF_BYTES + row * 128 + (rem & 7) * 16) = make_uint4(0u, 0u, 0u, 0u);
          }
          fence_proxy_async();
        }
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&p_full[t * 2 + b]);
      }
      // ---- normalise and store; the O accumulator is handed back (o_free) as soon as this row has left tensor memory
      mbar_wait(&pv_done[t * 2 + ((gt - 1u) & 1u)], ((gt - 1u) >> 1) & 1u);
      tc_fence_after();
      const float inv = 1.0f / l_run;
      __nv_bfloat16 *og = (__nv_bfloat16 *)p.out + ((size_t)(w.row0 + r) * p.n_q + w.head_a + t) * D;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32];
        tmem_ld_32x32(o_addr + (uint32_t)c * 32u, o);
        tmem_ld_wait();
        if (c == D / 32 - 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&o_free[t]);
        }
        if (r < w.rows) {
#pragma unroll
          for (int i = 0; i < 32; i += 8) {
            uint4 q4;
            q4.x = pack_bf16x2(__uint_as_float(o[i]) * inv, __uint_as_float(o[i + 1]) * inv);
            q4.y = pack_bf16x2(__uint_as_float(o[i + 2]) * inv, __uint_as_float(o[i + 3]) * inv);
            q4.z = pack_bf16x2(__uint_as_float(o[i + 4]) * inv, __uint_as_float(o[i + 5]) * inv);
            q4.w = pack_bf16x2(__uint_as_float(o[i + 6]) * inv, __uint_as_float(o[i + 7]) * inv);
            *reinterpret_cast<uint4 *>(og + c * 32 + i) = q4;
          }
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
  return 1024 + (size_t)(d / 64) * (2 * TA_BM + 2 * TA_STAGES * TA_BN) * 128 + 8 * (2 + 3 * TA_STAGES + 12 + 2) + 16;
}

cudaError_t prefill_attn_init() {  // per device: called from ss_stage_create
  cudaError_t e = cudaFuncSetAttribute(prefill_attn_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)prefill_smem(128));
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(prefill_attn_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)prefill_smem(64));
}

cudaError_t launch_prefill_attn(const PrefillAttnParams &p, cudaStream_t s) {
  const int G = p.n_q / p.n_kv;
  const long long items = (long long)p.n_kv * ((G + 1) / 2) * p.max_tiles;  // upper bound; the live count is on the device
  dim3 grid((unsigned)(items < p.n_sm ? items : p.n_sm));                   // persistent: one CTA per SM
  if (p.d == 128)
    return launch_pdl(prefill_attn_kernel<128>, dim3(grid), dim3(TA_THREADS), prefill_smem(128), s, *p.q_map, *p.kv_map, p);
  return launch_pdl(prefill_attn_kernel<64>, dim3(grid), dim3(TA_THREADS), prefill_smem(64), s, *p.q_map, *p.kv_map, p);
}

}  // namespace ss
