// attn_decode.cu — step S6a (+S5): paged GQA decode attention with split-K over the context and a fused KV append
// (Table 2 "Attention / Decode"; "memory-bound decode"; paged KV cache,
// PAPER.md:265, 271).  HBM-bound: every cached K/V byte is read exactly once per step.
//
// Work partition.  The (sequence b, kv head h, page) triples of the batch are flattened in that order into
// P_total = n_kv * sum_b pages_b items of one 16-token page (K 16xd + V 16xd bf16, each a contiguous block of the
// pool).  Each worker WARP takes a contiguous range of ceil(P_total / n_workers) items, so the load is balanced
// to one page whatever the length mix (the paper's workloads have lognormal lengths).  A range is cut
// at (b,h) boundaries into segments; each segment yields one partial (m, l, O[G x d]) in slot `worker + pair`,
// which is unique and monotone along the flattened order.  decode_merge combines the segments of a pair.
//
// A warp is an independent pipeline: one lane issues the TMA loads of whole pages (2-D boxes of 16 rows x 64
// columns, SWIZZLE_128B) into the warp's private smem ring, completion on the warp's own mbarriers (no block
// barrier anywhere), ldmatrix + mma.sync m16n8k16 with the G query heads of the group as the M rows
// (each K/V byte feeds all G heads), online softmax in fp32 with quad shuffles.  The warp that owns a sequence's
// last page writes the new token's K/V (bf16, post-RoPE, from qkv_post) into that page — in smem for its own use
// and in the pool — which is the fused append of step S5.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdlib.h>

#include "common.cuh"
#include "internal.h"

namespace ss {

#ifndef SS_DA_WARPS
#define SS_DA_WARPS 4
#endif
#ifndef SS_DA_STAGES
#define SS_DA_STAGES 2
#endif
// Measured (same-box A/B, cfg-2 / cfg-3 step): the kernel is bound by the latency of each warp's dependent chain
// (QK mma -> softmax -> PV mma per page), not by bytes in flight or by the load instructions: 8 warps/SM with 3-stage
// rings 7.57 / 5.34 ms; 12 warps/SM with 2-stage rings (4 warps x 3 CTAs, register-limited) 7.43 / 5.21 ms; fewer,
// deeper rings (7x4, 6x4, 5x5) slower.
constexpr int DA_WARPS = SS_DA_WARPS;    // independent warp pipelines per CTA
constexpr int DA_STAGES = SS_DA_STAGES;  // pages (K 4 KB + V 4 KB at d = 128) per warp ring
int decode_attn_warps_per_cta() { return DA_WARPS; }
int decode_attn_default_ctas_per_sm() { return (int)((size_t)228 * 1024 / (1024 + (size_t)DA_WARPS * DA_STAGES * (2 * 16 * 128 * 2 + 8))); }

// ---- plan: prefix sum of pages per sequence --------------------------------------------------------------------
__global__ void decode_plan_kernel(const CallArgs *__restrict__ args, int batch, int n_kv, int n_workers,
                                   DecodePlan plan) {
  pdl_launch_dependents();
  pdl_wait();
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    int acc = 0;
    plan.cum_pages[0] = 0;
    for (int b = 0; b < batch; ++b) {
      acc += (args->ctx[b] + 1 + 15) >> 4;
      plan.cum_pages[b + 1] = acc;
    }
    const int total = acc * n_kv;
    plan.meta[0] = total;
    plan.meta[1] = (total + n_workers - 1) / n_workers;
  }
}

cudaError_t launch_decode_plan(const CallArgs *args, int batch, int n_kv, int n_workers, DecodePlan plan,
                               cudaStream_t s) {
  return launch_pdl(decode_plan_kernel, dim3(1), dim3(32), 0, s, args, batch, n_kv, n_workers, plan);
}

struct Cursor {
  int b, h, pg, pages_b;
};

// smem image of one K (or V) page as TMA writes it: D/64 halves of [16 rows][128 B], SWIZZLE_128B inside each half
// (16-byte chunk c of row r sits at chunk c ^ (r & 7)): byte offset of chunk `ch` (0 .. D/8-1) of row `row`
__device__ __forceinline__ int page_off(int row, int ch) {
  return (ch >> 3) * 2048 + row * 128 + (((ch & 7) ^ (row & 7)) << 4);
}

// HI: the GQA group has more than 8 query heads, i.e. rows 8-15 of the 16-row MMA tile are live too.  The paper's
// models have G = 8: with HI = false the accumulators, query fragments and softmax statistics of rows 8-15 do not
// exist (about 45 registers fewer: more resident warps, which is what bounds this kernel).
template <int D, bool HI>
__global__ void __launch_bounds__(DA_WARPS * 32)
decode_attn_kernel(const __grid_constant__ CUtensorMap kv_map, const DecodeAttnParams p) {
  pdl_launch_dependents();
  pdl_wait();
  constexpr int ROW_BYTES = D * 2;
  constexpr int CHUNKS = ROW_BYTES / 16;       // 16-byte chunks per row: 16 (d=128) or 8 (d=64)
  constexpr int PAGE_BYTES = 16 * ROW_BYTES;   // one K (or V) page of one head
  constexpr int KSTEPS = D / 16;
  constexpr int NT = D / 8;                    // output n-tiles
  extern __shared__ __align__(1024) uint8_t smem[];   // swizzle atoms are 1 KB: the rings start 1 KB-aligned
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int w = blockIdx.x * DA_WARPS + warp;
  uint8_t *ring = smem + (size_t)warp * DA_STAGES * 2 * PAGE_BYTES;
  // one mbarrier per ring slot of each warp, behind the rings
  uint64_t *bars = (uint64_t *)(smem + (size_t)DA_WARPS * DA_STAGES * 2 * PAGE_BYTES) + warp * DA_STAGES;
  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < DA_STAGES; ++i) mbar_init(&bars[i], 1);
    mbar_fence_init();
    tma_prefetch_desc(&kv_map);
  }
  __syncwarp();

  const int n_kv = p.n_kv, G = p.n_q / p.n_kv;
  const int32_t *cum = p.plan.cum_pages;
  const CallArgs *args = p.args;
  const int max_blocks = args->max_blocks;
  // batch-invariant mode: this warp owns ONE (row, kv head) pair, all its pages, and writes the row's result itself
  const bool per_pair = p.per_pair != 0;
  int g0, g1, pp_ctx = 0;
  const int32_t *bt = args->block_tables;
  if (per_pair) {
    if (w >= p.n_rows * n_kv) return;
    const int row = w / n_kv;
    pp_ctx = p.row_pos ? p.row_pos[row] : args->ctx[row];
    bt += (size_t)(p.row_seq ? p.row_seq[row] : row) * max_blocks;  // the row's block-table row
    g0 = 0;
    g1 = (pp_ctx + 16) >> 4;
  } else {
    const int total = p.plan.meta[0], quota = p.plan.meta[1];
    g0 = w * quota;
    g1 = min(g0 + quota, total);
    if (g0 >= g1) return;
  }

  // locate g0: largest b with cum[b]*n_kv <= g0
  Cursor lc;
  if (per_pair) {
    lc.b = w / n_kv;
    lc.h = w - lc.b * n_kv;
    lc.pg = 0;
    lc.pages_b = g1;
  } else {
    int lo = 0, hi = p.batch;  // invariant: cum[lo]*n_kv <= g0 < cum[hi]*n_kv
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (cum[mid] * n_kv <= g0) lo = mid; else hi = mid;
    }
    lc.b = lo;
    lc.pages_b = cum[lo + 1] - cum[lo];
    const int r = g0 - cum[lo] * n_kv;
    lc.h = r / lc.pages_b;
    lc.pg = r - lc.h * lc.pages_b;
  }
  Cursor cc = lc;

  auto advance = [&](Cursor &c) {
    if (++c.pg == c.pages_b) {
      c.pg = 0;
      if (++c.h == n_kv) {
        c.h = 0;
        ++c.b;
        c.pages_b = (c.b < p.batch) ? cum[c.b + 1] - cum[c.b] : 1;
      }
    }
  };
  // one page = K tile + V tile of one (page, kv head): D/64 TMA boxes of {64 columns, 16 rows} each, issued by one
  // lane; the pool of this layer is one 2-D tensor [K rows | V rows] x D (rows = (page * n_kv + head) * 16 + slot)
  const uint64_t pol = l2_policy_evict_first();  // every K/V byte is read once per step
  const int v_row0 = p.n_pages * n_kv * 16;
  auto issue_load = [&](const Cursor &c, int slot) {
    if (elect_one()) {  // (not `lane == 0`: only under elect does nvcc issue UTMALDG straight from uniform registers)
      const int page = bt[(per_pair ? (size_t)0 : (size_t)c.b * max_blocks) + c.pg];
      const int row = (page * n_kv + c.h) * 16;
      uint8_t *kd = ring + (size_t)slot * 2 * PAGE_BYTES;
      fence_proxy_async();  // the slot's previous contents were read through the generic proxy (ldmatrix)
      mbar_expect_tx(&bars[slot], 2 * PAGE_BYTES);
#pragma unroll
      for (int hf = 0; hf < D / 64; ++hf) {
        tma_load_2d(kd + hf * 2048, &kv_map, &bars[slot], hf * 64, row, pol);
        tma_load_2d(kd + PAGE_BYTES + hf * 2048, &kv_map, &bars[slot], hf * 64, v_row0 + row, pol);
      }
    }
  };

  const int n = g1 - g0;
#pragma unroll
  for (int i = 0; i < DA_STAGES - 1; ++i) {
    if (i < n) {
      issue_load(lc, i);
      advance(lc);
    }
  }

  const float sl2 = 1.4426950408889634f / sqrtf((float)D);  // log2(e) / sqrt(d)
  constexpr int RW = HI ? 2 : 1;   // live 8-row groups
  uint32_t qf[KSTEPS][2 * RW];     // [ks][rowgroup * 2 + khalf]
  float o[NT][2 * RW];             // [n-tile][rowgroup * 2 + col]
  float m_run[RW], l_run[RW];
  bool seg_open = false;
  const int qrow = lane >> 2, qcol = (lane & 3) * 2;

  for (int i = 0; i < n; ++i) {
    if (i + DA_STAGES - 1 < n) {  // the slot was drained in iteration i - 1 (its trailing __syncwarp)
      issue_load(lc, (i + DA_STAGES - 1) % DA_STAGES);
      advance(lc);
    }
    mbar_wait(&bars[i % DA_STAGES], (uint32_t)(i / DA_STAGES) & 1u);

    const int ctx = per_pair ? pp_ctx : args->ctx[cc.b];
    if (!seg_open) {
      // new (b,h) segment: query fragments of the G heads of kv head h (rows >= G are zero)
      const __nv_bfloat16 *qb = (const __nv_bfloat16 *)p.q + (size_t)cc.b * p.n_q * D + (size_t)cc.h * G * D;
#pragma unroll
      for (int ks = 0; ks < KSTEPS; ++ks) {
        const int c = ks * 16 + qcol;
        qf[ks][0] = (qrow < G) ? *reinterpret_cast<const uint32_t *>(qb + (size_t)qrow * D + c) : 0u;
        qf[ks][1] = (qrow < G) ? *reinterpret_cast<const uint32_t *>(qb + (size_t)qrow * D + c + 8) : 0u;
        if (HI) {
          qf[ks][2] = (qrow + 8 < G) ? *reinterpret_cast<const uint32_t *>(qb + (size_t)(qrow + 8) * D + c) : 0u;
          qf[ks][3] = (qrow + 8 < G) ? *reinterpret_cast<const uint32_t *>(qb + (size_t)(qrow + 8) * D + c + 8) : 0u;
        }
      }
#pragma unroll
      for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int e = 0; e < 2 * RW; ++e) o[t][e] = 0.f;
#pragma unroll
      for (int r = 0; r < RW; ++r) {
        m_run[r] = -INFINITY;
        l_run[r] = 0.f;
      }
      seg_open = true;
    }

    uint8_t *ksm = ring + (size_t)(i % DA_STAGES) * 2 * PAGE_BYTES;
    uint8_t *vsm = ksm + PAGE_BYTES;
    const int last_pg = ctx >> 4;
    int n_valid = 16;
    if (cc.pg == last_pg) {
      // fused KV append (step S5): slot ctx & 15 of the sequence's last page <- bf16 k', v' of the new token
      n_valid = (ctx & 15) + 1;
      const int r = ctx & 15;
      const int page = bt[(per_pair ? (size_t)0 : (size_t)cc.b * max_blocks) + cc.pg];
      const uint8_t *src = (const uint8_t *)p.kv_new + ((size_t)cc.b * 2 * n_kv * D + (size_t)cc.h * D) * 2;
      const size_t goff = (((size_t)page * n_kv + cc.h) * 16 + r) * ROW_BYTES;
      for (int idx = lane; idx < (p.append ? 2 * CHUNKS : 0); idx += 32) {
        const int isv = idx / CHUNKS, ch = idx % CHUNKS;
        const uint4 val = *reinterpret_cast<const uint4 *>(src + (size_t)isv * n_kv * D * 2 + ch * 16);
        uint8_t *sdst = (isv ? vsm : ksm) + page_off(r, ch);
        *reinterpret_cast<uint4 *>(sdst) = val;
        uint8_t *gdst = (uint8_t *)(isv ? p.vpool : p.kpool) + goff + ch * 16;
        *reinterpret_cast<uint4 *>(gdst) = val;
      }
      // slots past the sequence end hold whatever the pool held: zero their V rows so that 0 * garbage (possibly
      // NaN) cannot reach the output; their scores are overwritten with -inf below
      for (int idx = lane; idx < (15 - r) * CHUNKS; idx += 32) {
        const int rr2 = r + 1 + idx / CHUNKS, ch = idx % CHUNKS;
        *reinterpret_cast<uint4 *>(vsm + page_off(rr2, ch)) = make_uint4(0u, 0u, 0u, 0u);
      }
      __syncwarp();
    }

    // ---- S = Q K^T for the 16 tokens of the page: two n-tiles of 8 tokens; s[tile][rowgroup * 2 + col]
    float sc[2][2 * RW];
#pragma unroll
    for (int e = 0; e < 2 * RW; ++e) sc[0][e] = sc[1][e] = 0.f;
    auto mma_rows = [&](float (&d)[2 * RW], const uint32_t (&a)[2 * RW], uint32_t b0, uint32_t b1) {
      if constexpr (HI) {
        const uint32_t af[4] = {a[0], a[2], a[1], a[3]};  // PTX order: (row, k-lo), (row+8, k-lo), (row, k-hi), (row+8, k-hi)
        float df[4] = {d[0], d[1], d[2], d[3]};
        mma_bf16_16816(df, af, b0, b1);
        d[0] = df[0]; d[1] = df[1]; d[2] = df[2]; d[3] = df[3];
      } else {
        mma_bf16_16816_lo(d, a[0], a[1], b0, b1);
      }
    };
    {
      const int mtx = lane >> 3, rr = lane & 7;
      const int tok = (mtx >> 1) * 8 + rr;
      const uint32_t kbase = smem_u32(ksm);
#pragma unroll
      for (int ks = 0; ks < KSTEPS; ++ks) {
        const int ch = ks * 2 + (mtx & 1);
        uint32_t kb[4];
        ldmatrix_x4(kb, kbase + page_off(tok, ch));
        mma_rows(sc[0], qf[ks], kb[0], kb[1]);
        mma_rows(sc[1], qf[ks], kb[2], kb[3]);
      }
    }
    // mask tokens past the sequence end (only on the last page)
    if (n_valid < 16) {
#pragma unroll
      for (int r = 0; r < RW; ++r) {
        if (qcol >= n_valid) sc[0][2 * r] = -INFINITY;
        if (qcol + 1 >= n_valid) sc[0][2 * r + 1] = -INFINITY;
        if (qcol + 8 >= n_valid) sc[1][2 * r] = -INFINITY;
        if (qcol + 9 >= n_valid) sc[1][2 * r + 1] = -INFINITY;
      }
    }
    // ---- online softmax per live row group, statistics across the quad
    float alpha[RW];
    uint32_t pa[2 * RW];  // [rowgroup * 2 + khalf] : P as the A fragment of the PV product (k = the 16 tokens)
#pragma unroll
    for (int r = 0; r < RW; ++r) {
      float mx = fmaxf(fmaxf(sc[0][2 * r], sc[0][2 * r + 1]), fmaxf(sc[1][2 * r], sc[1][2 * r + 1]));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
      const float mn = fmaxf(m_run[r], mx);
      alpha[r] = exp2f((m_run[r] - mn) * sl2);
      m_run[r] = mn;
      const float p00 = exp2f((sc[0][2 * r] - mn) * sl2), p01 = exp2f((sc[0][2 * r + 1] - mn) * sl2);
      const float p10 = exp2f((sc[1][2 * r] - mn) * sl2), p11 = exp2f((sc[1][2 * r + 1] - mn) * sl2);
      float rs = p00 + p01 + p10 + p11;
      rs += __shfl_xor_sync(0xffffffffu, rs, 1);
      rs += __shfl_xor_sync(0xffffffffu, rs, 2);
      l_run[r] = l_run[r] * alpha[r] + rs;
      pa[2 * r] = pack_bf16x2(p00, p01);      // tokens 0-7 (k-lo)
      pa[2 * r + 1] = pack_bf16x2(p10, p11);  // tokens 8-15 (k-hi)
    }
    // ---- O = O * alpha + P V
    {
      const int mtx = lane >> 3, rr = lane & 7;
      const int tok = (mtx & 1) * 8 + rr;
      const uint32_t vbase = smem_u32(vsm);
#pragma unroll
      for (int t2 = 0; t2 < NT / 2; ++t2) {
        const int ch = t2 * 2 + (mtx >> 1);
        uint32_t vb[4];
        ldmatrix_x4_trans(vb, vbase + page_off(tok, ch));
#pragma unroll
        for (int r = 0; r < RW; ++r) {
          o[2 * t2][2 * r] *= alpha[r]; o[2 * t2][2 * r + 1] *= alpha[r];
          o[2 * t2 + 1][2 * r] *= alpha[r]; o[2 * t2 + 1][2 * r + 1] *= alpha[r];
        }
        mma_rows(o[2 * t2], pa, vb[0], vb[1]);
        mma_rows(o[2 * t2 + 1], pa, vb[2], vb[3]);
      }
    }

    // ---- segment end?  (next item belongs to another (b,h), or this was the warp's last item)
    const bool seg_end = (i == n - 1) || (cc.pg + 1 == cc.pages_b);
    if (seg_end && per_pair) {
      // the pair's only segment: out = O / l, exactly what decode_merge computes for one segment (weight 2^0 = 1)
      __nv_bfloat16 *ob = (__nv_bfloat16 *)p.out + (size_t)cc.b * p.n_q * D + (size_t)cc.h * G * D;
      if (qrow < G) {
        const float inv = 1.0f / l_run[0];
#pragma unroll
        for (int t = 0; t < NT; ++t)
          *reinterpret_cast<uint32_t *>(ob + (size_t)qrow * D + t * 8 + qcol) = pack_bf16x2(o[t][0] * inv, o[t][1] * inv);
      }
      if constexpr (HI) {
        if (qrow + 8 < G) {
          const float inv = 1.0f / l_run[1];
#pragma unroll
          for (int t = 0; t < NT; ++t)
            *reinterpret_cast<uint32_t *>(ob + (size_t)(qrow + 8) * D + t * 8 + qcol) = pack_bf16x2(o[t][2] * inv, o[t][3] * inv);
        }
      }
      seg_open = false;
    } else if (seg_end) {
      const int slot = w + cc.b * n_kv + cc.h;
      float *po = p.part_o + (size_t)slot * 16 * D;
      float *pml = p.part_ml + (size_t)slot * 32;
      if (qrow < G) {
#pragma unroll
        for (int t = 0; t < NT; ++t)
          *reinterpret_cast<float2 *>(po + (size_t)qrow * D + t * 8 + qcol) = make_float2(o[t][0], o[t][1]);
        if ((lane & 3) == 0) *reinterpret_cast<float2 *>(pml + qrow * 2) = make_float2(m_run[0], l_run[0]);
      }
      if constexpr (HI) {
        if (qrow + 8 < G) {
#pragma unroll
          for (int t = 0; t < NT; ++t)
            *reinterpret_cast<float2 *>(po + (size_t)(qrow + 8) * D + t * 8 + qcol) = make_float2(o[t][2], o[t][3]);
          if ((lane & 3) == 0) *reinterpret_cast<float2 *>(pml + (qrow + 8) * 2) = make_float2(m_run[1], l_run[1]);
        }
      }
      seg_open = false;
    }
    advance(cc);
    __syncwarp();
  }
}

// ---- merge the segments of each (b, kv head): out[b][hq][:] = sum_i w_i O_i / sum_i w_i l_i, w_i = 2^((m_i-M) sl2)
// One CTA per (b, kv head); D/4 threads per q head, each owning 4 output columns, so all segment loads of a thread
// are independent 16-byte reads (no serial chain over heads).
constexpr int MERGE_THREADS = 256;
template <int D>
__global__ void __launch_bounds__(MERGE_THREADS) decode_merge_kernel(const DecodeAttnParams p) {
  pdl_launch_dependents();
  pdl_wait();
  constexpr int LANES = D / 4;                  // threads per q head
  constexpr int HEADS_PER_PASS = MERGE_THREADS / LANES;
  const int pair = blockIdx.x;
  const int b = pair / p.n_kv, h = pair % p.n_kv;
  const int G = p.n_q / p.n_kv;
  const int32_t *cum = p.plan.cum_pages;
  const int quota = p.plan.meta[1];
  const int pages_b = cum[b + 1] - cum[b];
  const int start = cum[b] * p.n_kv + h * pages_b;
  const int w_first = start / quota, w_last = (start + pages_b - 1) / quota;
  const float sl2 = 1.4426950408889634f / sqrtf((float)D);
  const int c = (threadIdx.x % LANES) * 4;
  for (int g = threadIdx.x / LANES; g < G; g += HEADS_PER_PASS) {
    float M = -INFINITY;
#pragma unroll 4
    for (int w = w_first; w <= w_last; ++w) M = fmaxf(M, p.part_ml[(size_t)(w + pair) * 32 + g * 2]);
    float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
    float den = 0.f;
#pragma unroll 4
    for (int w = w_first; w <= w_last; ++w) {
      const size_t slot = (size_t)(w + pair);
      const float2 ml = *reinterpret_cast<const float2 *>(p.part_ml + slot * 32 + g * 2);
      const float4 o = *reinterpret_cast<const float4 *>(p.part_o + slot * 16 * D + (size_t)g * D + c);
      const float wt = exp2f((ml.x - M) * sl2);
      num.x += wt * o.x; num.y += wt * o.y; num.z += wt * o.z; num.w += wt * o.w;
      den += wt * ml.y;
    }
    const float inv = 1.0f / den;
    uint2 r;
    r.x = pack_bf16x2(num.x * inv, num.y * inv);
    r.y = pack_bf16x2(num.z * inv, num.w * inv);
    *reinterpret_cast<uint2 *>((__nv_bfloat16 *)p.out + (size_t)b * p.n_q * D + (size_t)(h * G + g) * D + c) = r;
  }
}

static size_t decode_smem(int d) { return (size_t)DA_WARPS * DA_STAGES * (2 * 16 * d * 2 + 8); }  // rings + mbarriers

template <int D, bool HI>
static cudaError_t set_smem() {
  cudaError_t e = cudaFuncSetAttribute(decode_attn_kernel<D, HI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)decode_smem(D));
  if (e != cudaSuccess) return e;
  // several CTAs per SM are the point of this kernel: ask for the largest shared-memory carve-out
  return cudaFuncSetAttribute(decode_attn_kernel<D, HI>, cudaFuncAttributePreferredSharedMemoryCarveout,
                              cudaSharedmemCarveoutMaxShared);
}

cudaError_t attn_init() {
  cudaError_t e;
  if ((e = set_smem<128, false>()) != cudaSuccess) return e;
  if ((e = set_smem<128, true>()) != cudaSuccess) return e;
  if ((e = set_smem<64, false>()) != cudaSuccess) return e;
  return set_smem<64, true>();
}

cudaError_t launch_decode_attn(const DecodeAttnParams &p, cudaStream_t s) {
  const int ctas = p.per_pair ? (p.n_rows * p.n_kv + DA_WARPS - 1) / DA_WARPS : p.n_workers / DA_WARPS;
  const bool hi = p.n_q / p.n_kv > 8;
  const dim3 g(ctas), b(DA_WARPS * 32);
  if (p.d == 128)
    return hi ? launch_pdl(decode_attn_kernel<128, true>, g, b, decode_smem(128), s, *p.kv_map, p)
              : launch_pdl(decode_attn_kernel<128, false>, g, b, decode_smem(128), s, *p.kv_map, p);
  return hi ? launch_pdl(decode_attn_kernel<64, true>, g, b, decode_smem(64), s, *p.kv_map, p)
            : launch_pdl(decode_attn_kernel<64, false>, g, b, decode_smem(64), s, *p.kv_map, p);
}

cudaError_t launch_decode_merge(const DecodeAttnParams &p, cudaStream_t s) {
  if (p.d == 128)
    return launch_pdl(decode_merge_kernel<128>, dim3(p.batch * p.n_kv), dim3(MERGE_THREADS), 0, s, p);
  else
    return launch_pdl(decode_merge_kernel<64>, dim3(p.batch * p.n_kv), dim3(MERGE_THREADS), 0, s, p);
}

}  // namespace ss
