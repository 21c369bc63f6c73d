// attn_prefill.cu — step S6b: causal varlen prefill attention over the paged KV cache, with prior context
// (Table 2 "Attention / Prefill"; this is the attention of the migration recompute, PAPER.md:247,
// 259, and of chunked prefill in mixed iterations).  Query i of sequence s sits at global position
// p = ctx_before[s] + i and attends keys 0..p, ALL read from the pages (the keys of this call were appended by
// qkv_post before this kernel runs), which is what makes prefill == incremental decode.
//
// Flash-style: CTA = 4 warps = one 64-row query tile of one (sequence, q head); K/V tiles of 64 tokens (4 pages)
// double-buffered through cp.async into XOR-swizzled smem; mma.sync m16n8k16 bf16 with fp32 online softmax.
// The 8 q heads of a GQA group are adjacent in blockIdx.x so their K/V re-reads hit L2.  Attention is ~1.6% of the
// prefill FLOPs at the paper's lengths, so this kernel is sized for correctness and decent speed; the
// tensor-bound work is in gemm_tcgen05.cu.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "common.cuh"
#include "internal.h"

namespace ss {

constexpr int PA_WARPS = 4;
constexpr int PA_BM = 64;  // query rows per CTA
constexpr int PA_BN = 64;  // keys per tile

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
        if (s >= seq0) acc += (args->cu_q[s + 1] - args->cu_q[s] + PA_BM - 1) / PA_BM;
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
      key[i] = args->ctx[lo] + min(q_len, (i - plan.tile_cum[lo] + 1) * PA_BM);
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

template <int D>
__global__ void __launch_bounds__(PA_WARPS * 32, 3) prefill_attn_kernel(const PrefillAttnParams p) {
  pdl_launch_dependents();
  pdl_wait();
  constexpr int ROW_BYTES = D * 2;
  constexpr int CHUNKS = ROW_BYTES / 16;
  constexpr int TILE_BYTES = PA_BN * ROW_BYTES;
  constexpr int KSTEPS = D / 16;
  constexpr int NT = D / 8;
  extern __shared__ __align__(128) uint8_t smem[];
  // smem = 2 x (K tile, V tile).  The Q tile is staged once through the SECOND buffer (free until the prefetch of
  // key tile 1) and then lives in registers, so a CTA needs 64 KB and three fit on an SM (occupancy, not
  // bandwidth, bounds this kernel: ncu showed 8 warps/SM with 56% of the cycles without an eligible warp).
  uint8_t *kv_s = smem;
  uint8_t *q_s = smem + 2 * TILE_BYTES;      // [PA_BM][D], aliases buffer 1

  const int head = blockIdx.x;
  const int32_t *tile_cum = p.plan.tile_cum;
  if ((int)blockIdx.y >= tile_cum[p.n_seqs]) return;
  const int slot = p.plan.tile_order[blockIdx.y];
  int lo = 0, hi = p.n_seqs;  // tile_cum[lo] <= slot < tile_cum[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (tile_cum[mid] <= slot) lo = mid; else hi = mid;
  }
  const int s = lo;
  const CallArgs *args = p.args;
  const int q_begin = args->cu_q[s], q_len = args->cu_q[s + 1] - q_begin;
  const int ctx0 = args->ctx[s];
  const int i0 = (slot - tile_cum[s]) * PA_BM;
  const int rows = min(PA_BM, q_len - i0);
  const int p0 = ctx0 + i0;          // global position of the tile's first query
  const int kv_len = p0 + rows;      // keys 0..kv_len-1 are needed by this tile
  const int n_kt = (kv_len + PA_BN - 1) / PA_BN;
  const int G = p.n_q / p.n_kv, hk = head / G;
  const int32_t *bt = args->block_tables + (size_t)s * args->max_blocks;
  const __nv_bfloat16 *kpool = (const __nv_bfloat16 *)p.kpool;
  const __nv_bfloat16 *vpool = (const __nv_bfloat16 *)p.vpool;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  // ---- Q tile -> smem (rows past the tile's end are zero-filled)
  {
    const __nv_bfloat16 *qg = (const __nv_bfloat16 *)p.q + ((size_t)(q_begin + i0) * p.n_q + head) * D;
    for (int idx = tid; idx < PA_BM * CHUNKS; idx += PA_WARPS * 32) {
      const int r = idx / CHUNKS, ch = idx % CHUNKS;
      const bool ok = r < rows;
      const void *src = ok ? (const void *)(qg + (size_t)r * p.n_q * D + ch * 8) : (const void *)p.q;
      cp_async16_zfill(q_s + r * ROW_BYTES + ((ch ^ (r & 7)) << 4), src, ok ? 16u : 0u);
    }
  }
  auto load_kv = [&](int kt, int buf) {
    uint8_t *kd = kv_s + (size_t)buf * 2 * TILE_BYTES;
    uint8_t *vd = kd + TILE_BYTES;
    for (int idx = tid; idx < PA_BN * CHUNKS; idx += PA_WARPS * 32) {
      const int r = idx / CHUNKS, ch = idx % CHUNKS;
      const int j = kt * PA_BN + r;
      const bool ok = j < kv_len;
      size_t off = 0;
      if (ok) {
        const int page = bt[j >> 4];
        off = (((size_t)page * p.n_kv + hk) * 16 + (size_t)(j & 15)) * D + ch * 8;
      }
      const int dst = r * ROW_BYTES + ((ch ^ (r & 7)) << 4);
      cp_async16_zfill(kd + dst, kpool + off, ok ? 16u : 0u);
      cp_async16_zfill(vd + dst, vpool + off, ok ? 16u : 0u);
    }
  };
  load_kv(0, 0);
  cp_async_commit();

  const float sl2 = 1.4426950408889634f / sqrtf((float)D);
  const int qrow = lane >> 2, qcol = (lane & 3) * 2;
  const int qpos0 = p0 + warp * 16 + qrow, qpos1 = qpos0 + 8;
  uint32_t qf[KSTEPS][4];
  float o[NT][4];
#pragma unroll
  for (int t = 0; t < NT; ++t) o[t][0] = o[t][1] = o[t][2] = o[t][3] = 0.f;
  float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};

  {  // Q tile -> registers, then its smem (buffer 1) is free for the prefetch of key tile 1
    cp_async_wait<0>();
    __syncthreads();
    const int mtx = lane >> 3, rr = lane & 7;
    const int r = warp * 16 + (mtx & 1) * 8 + rr;
    const uint32_t qb = smem_u32(q_s) + r * ROW_BYTES;
#pragma unroll
    for (int ks = 0; ks < KSTEPS; ++ks) ldmatrix_x4(qf[ks], qb + (((ks * 2 + (mtx >> 1)) ^ (r & 7)) << 4));
    __syncthreads();
  }
  for (int kt = 0; kt < n_kt; ++kt) {
    if (kt + 1 < n_kt) load_kv(kt + 1, (kt + 1) & 1);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();
    const uint8_t *ksm = kv_s + (size_t)(kt & 1) * 2 * TILE_BYTES;
    const uint8_t *vsm = ksm + TILE_BYTES;

    // ---- S = Q K^T : 16 rows x 64 keys per warp
    float sc[PA_BN / 8][4];
#pragma unroll
    for (int t = 0; t < PA_BN / 8; ++t) sc[t][0] = sc[t][1] = sc[t][2] = sc[t][3] = 0.f;
    {
      const int mtx = lane >> 3, rr = lane & 7;
#pragma unroll
      for (int t2 = 0; t2 < PA_BN / 16; ++t2) {
        const int tok = t2 * 16 + (mtx >> 1) * 8 + rr;
        const uint32_t kb_addr = smem_u32(ksm) + tok * ROW_BYTES;
#pragma unroll
        for (int ks = 0; ks < KSTEPS; ++ks) {
          uint32_t kb[4];
          ldmatrix_x4(kb, kb_addr + (((ks * 2 + (mtx & 1)) ^ (tok & 7)) << 4));
          mma_bf16_16816(sc[2 * t2], qf[ks], kb[0], kb[1]);
          mma_bf16_16816(sc[2 * t2 + 1], qf[ks], kb[2], kb[3]);
        }
      }
    }
    // ---- causal mask (keys beyond the query's position); only tiles that reach past the first query need it
    const int jbase = kt * PA_BN;
    if (jbase + PA_BN - 1 > p0 + warp * 16) {
#pragma unroll
      for (int t = 0; t < PA_BN / 8; ++t) {
        const int j = jbase + t * 8 + qcol;
        if (j > qpos0) sc[t][0] = -INFINITY;
        if (j + 1 > qpos0) sc[t][1] = -INFINITY;
        if (j > qpos1) sc[t][2] = -INFINITY;
        if (j + 1 > qpos1) sc[t][3] = -INFINITY;
      }
    }
    // ---- online softmax
    float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
    for (int t = 0; t < PA_BN / 8; ++t) {
      mx0 = fmaxf(mx0, fmaxf(sc[t][0], sc[t][1]));
      mx1 = fmaxf(mx1, fmaxf(sc[t][2], sc[t][3]));
    }
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
    const float mn0 = fmaxf(m_run[0], mx0), mn1 = fmaxf(m_run[1], mx1);
    // key 0 is visible to every query, so after tile 0 the running max is finite
    const float a0 = exp2f((m_run[0] - mn0) * sl2), a1 = exp2f((m_run[1] - mn1) * sl2);
    m_run[0] = mn0;
    m_run[1] = mn1;
    float rs0 = 0.f, rs1 = 0.f;
    uint32_t pa[PA_BN / 16][4];
#pragma unroll
    for (int t = 0; t < PA_BN / 8; ++t) {
      const float e0 = exp2f((sc[t][0] - mn0) * sl2), e1 = exp2f((sc[t][1] - mn0) * sl2);
      const float e2 = exp2f((sc[t][2] - mn1) * sl2), e3 = exp2f((sc[t][3] - mn1) * sl2);
      rs0 += e0 + e1;
      rs1 += e2 + e3;
      pa[t >> 1][(t & 1) * 2 + 0] = pack_bf16x2(e0, e1);
      pa[t >> 1][(t & 1) * 2 + 1] = pack_bf16x2(e2, e3);
    }
    rs0 += __shfl_xor_sync(0xffffffffu, rs0, 1);
    rs0 += __shfl_xor_sync(0xffffffffu, rs0, 2);
    rs1 += __shfl_xor_sync(0xffffffffu, rs1, 1);
    rs1 += __shfl_xor_sync(0xffffffffu, rs1, 2);
    l_run[0] = l_run[0] * a0 + rs0;
    l_run[1] = l_run[1] * a1 + rs1;
    // the running maxima settle after the first few key tiles: skip the 64 multiplies when no row of the warp moved
    // (alpha == 1 exactly then, so skipping changes no bit)
    if (__any_sync(0xffffffffu, a0 != 1.0f || a1 != 1.0f)) {
#pragma unroll
      for (int t = 0; t < NT; ++t) {
        o[t][0] *= a0; o[t][1] *= a0; o[t][2] *= a1; o[t][3] *= a1;
      }
    }
    // ---- O += P V
    {
      const int mtx = lane >> 3, rr = lane & 7;
#pragma unroll
      for (int kk = 0; kk < PA_BN / 16; ++kk) {
        const int tok = kk * 16 + (mtx & 1) * 8 + rr;
        const uint32_t vb_addr = smem_u32(vsm) + tok * ROW_BYTES;
#pragma unroll
        for (int t2 = 0; t2 < NT / 2; ++t2) {
          uint32_t vb[4];
          ldmatrix_x4_trans(vb, vb_addr + (((t2 * 2 + (mtx >> 1)) ^ (tok & 7)) << 4));
          mma_bf16_16816(o[2 * t2], pa[kk], vb[0], vb[1]);
          mma_bf16_16816(o[2 * t2 + 1], pa[kk], vb[2], vb[3]);
        }
      }
    }
    __syncthreads();
  }
  cp_async_wait<0>();

  // ---- normalise and store
  __nv_bfloat16 *og = (__nv_bfloat16 *)p.out + ((size_t)(q_begin + i0) * p.n_q + head) * D;
  const int r0 = warp * 16 + qrow, r1 = r0 + 8;
  const float inv0 = 1.0f / l_run[0], inv1 = 1.0f / l_run[1];
#pragma unroll
  for (int t = 0; t < NT; ++t) {
    if (r0 < rows)
      *reinterpret_cast<uint32_t *>(og + (size_t)r0 * p.n_q * D + t * 8 + qcol) =
          pack_bf16x2(o[t][0] * inv0, o[t][1] * inv0);
    if (r1 < rows)
      *reinterpret_cast<uint32_t *>(og + (size_t)r1 * p.n_q * D + t * 8 + qcol) =
          pack_bf16x2(o[t][2] * inv1, o[t][3] * inv1);
  }
}

static size_t prefill_smem(int d) { return (size_t)(4 * PA_BN) * d * 2; }  // Q aliases the second K/V buffer

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
    return launch_pdl(prefill_attn_kernel<128>, dim3(grid), dim3(PA_WARPS * 32), prefill_smem(128), s, p);
  else
    return launch_pdl(prefill_attn_kernel<64>, dim3(grid), dim3(PA_WARPS * 32), prefill_smem(64), s, p);
}

}  // namespace ss
