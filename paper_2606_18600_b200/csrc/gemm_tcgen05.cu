// gemm_tcgen05.cu — the bf16 projections of a decoder layer (Table 2 rows "QKV Projection", "Output Projection",
// "Up and Gate Projection", "Down Projection", "Logits Calculation") as ONE tcgen05/TMEM GEMM
// kernel fed by TMA, for sm_100a.
//
// out[t][n] = sum_k X[t,k] * W[n,k]     X: activations [T,K] bf16 row-major, W: weights [N,K] bf16 row-major.
//
// Orientation: the 128 TMEM lanes (UMMA M) run over weight rows n, the TMEM columns (UMMA N = bn) over tokens t.
// At decode (T = 64..128) this streams every weight byte exactly once through full-width 128-row MMAs (the
// HBM-bound case); at prefill (bn = 256) the same kernel is a 128x256 compute tile.
//
// CTA = 6 warps: warp 0 = TMA producer (one lane), warp 1 = TMEM allocator + MMA issuer (one lane), warps 2-5 =
// epilogue (one TMEM lane quadrant each).  smem ring of `stages` x {A tile 128x64 (x2 when DUAL), B tile bn x 64},
// SWIZZLE_128B, full/empty mbarriers; accumulator(s) in TMEM; K-split over gridDim.z with fp32 partial outputs
// reduced in fixed order by the consumer kernel.  DUAL = gate and up tiles share the B tile and the epilogue
// writes silu(g)*u as bf16 (step S9), so [T,2F] never reaches HBM.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdlib.h>

#include "common.cuh"
#include "internal.h"

namespace ss {

constexpr int A_TILE_BYTES = GEMM_BM * GEMM_BK * 2;  // 16 KB

template <bool DUAL>
__global__ void __launch_bounds__(192)
gemm_kernel(const __grid_constant__ CUtensorMap ta0, const __grid_constant__ CUtensorMap ta1,
            const __grid_constant__ CUtensorMap ta2, const __grid_constant__ CUtensorMap tb, const GemmParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *base = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const int bn = p.bn;
  const uint32_t b_bytes = (uint32_t)bn * 128u;
  const uint32_t stage_bytes = A_TILE_BYTES * (DUAL ? 2 : 1) + b_bytes;
  const int stages = p.stages;
  uint64_t *full = (uint64_t *)(base + (size_t)stages * stage_bytes);
  uint64_t *empty = full + stages;
  uint64_t *acc_full = empty + stages;
  uint32_t *tmem_slot = (uint32_t *)(acc_full + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // tile -> (segment, first row)
  int seg = 0;
#pragma unroll
  for (int i = 1; i < 3; ++i)
    if (i < p.n_seg && (int)blockIdx.x >= p.seg_tile0[i]) seg = i;
  const int row0 = ((int)blockIdx.x - p.seg_tile0[seg]) * GEMM_BM;
  const int t0 = blockIdx.y * bn;
  const int nkb = (p.K + GEMM_BK - 1) / GEMM_BK;
  const int kb0 = blockIdx.z * p.kb_per_split;
  const int kb1 = min(nkb, kb0 + p.kb_per_split);

  const uint32_t tmem_cols_needed = (uint32_t)bn * (DUAL ? 2u : 1u);
  uint32_t tmem_cols = 32;
  while (tmem_cols < tmem_cols_needed) tmem_cols <<= 1;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(seg == 0 ? &ta0 : (seg == 1 ? &ta1 : &ta2));
    if (DUAL) tma_prefetch_desc(&ta1);
    tma_prefetch_desc(&tb);
    for (int i = 0; i < stages; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    mbar_init(acc_full, 1);
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc_dyn(tmem_slot, tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {
      // ---------------- TMA producer ----------------
      const uint64_t pol_w = l2_policy_evict_first();  // weights are streamed once
      const uint64_t pol_x = l2_policy_evict_last();   // activations are re-read by every CTA
      const CUtensorMap *ta = DUAL ? &ta0 : (seg == 0 ? &ta0 : (seg == 1 ? &ta1 : &ta2));
      int i = 0;
      for (int kb = kb0; kb < kb1; ++kb, ++i) {
        const int s = i % stages;
        const uint32_t ph = (uint32_t)(i / stages) & 1u;
        mbar_wait(&empty[s], ph ^ 1u);
        uint8_t *st = base + (size_t)s * stage_bytes;
        mbar_expect_tx(&full[s], stage_bytes);
        tma_load_2d(st, ta, &full[s], kb * GEMM_BK, row0, pol_w);
        if (DUAL) tma_load_2d(st + A_TILE_BYTES, &ta1, &full[s], kb * GEMM_BK, row0, pol_w);
        tma_load_2d(st + A_TILE_BYTES * (DUAL ? 2 : 1), &tb, &full[s], kb * GEMM_BK, t0, pol_x);
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      // ---------------- MMA issuer ----------------
      const uint32_t idesc = umma_idesc_bf16(GEMM_BM, (uint32_t)bn);
      int i = 0;
      for (int kb = kb0; kb < kb1; ++kb, ++i) {
        const int s = i % stages;
        const uint32_t ph = (uint32_t)(i / stages) & 1u;
        mbar_wait(&full[s], ph);
        tc_fence_after();
        const uint32_t st = smem_u32(base + (size_t)s * stage_bytes);
        const uint64_t da = umma_desc_k_sw128(st);
        const uint64_t db = umma_desc_k_sw128(st + A_TILE_BYTES * (DUAL ? 2 : 1));
#pragma unroll
        for (int k = 0; k < GEMM_BK / 16; ++k) {
          const uint32_t acc = (kb > kb0 || k > 0) ? 1u : 0u;
          umma_bf16(tmem_base, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, acc);
          if (DUAL) {
            const uint64_t da1 = umma_desc_k_sw128(st + A_TILE_BYTES);
            umma_bf16(tmem_base + (uint32_t)bn, da1 + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, acc);
          }
        }
        umma_commit(&empty[s]);  // frees the smem slot when these MMAs have read it
      }
      umma_commit(acc_full);
    }
  } else {
    // ---------------- epilogue: TMEM -> registers -> global ----------------
    const int quad = warp & 3;
    const int r = quad * 32 + lane;  // row of the tile = TMEM lane
    const int row_in_seg = row0 + r;
    const bool row_ok = row_in_seg < p.seg_rows[seg];
    const int col = p.seg_col[seg] + row_in_seg;
    mbar_wait(acc_full, 0);
    tc_fence_after();
    const uint32_t tq = tmem_base + ((uint32_t)(quad * 32) << 16);
    if (p.epi == EPI_F32) {
      float *o = p.out_f32 + (long long)blockIdx.z * p.split_stride + col;
      if (bn >= 32) {
        for (int c = 0; c < bn; c += 32) {
          uint32_t v[32];
          tmem_ld_32x32(tq + (uint32_t)c, v);
          tmem_ld_wait();
          if (row_ok) {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const int t = t0 + c + j;
              if (t < p.T) o[(size_t)t * p.ld_out] = __uint_as_float(v[j]);
            }
          }
        }
      } else {
        uint32_t v[16];
        tmem_ld_32x16(tq, v);
        tmem_ld_wait();
        if (row_ok) {
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            const int t = t0 + j;
            if (t < p.T) o[(size_t)t * p.ld_out] = __uint_as_float(v[j]);
          }
        }
      }
    } else if (DUAL) {  // EPI_SWIGLU_BF16: a = g / (1 + exp(-g)) * u
      __nv_bfloat16 *o = (__nv_bfloat16 *)p.out_bf16 + col;
      const int step = bn >= 32 ? 32 : 16;
      for (int c = 0; c < bn; c += step) {
        uint32_t g[32], u[32];
        if (step == 32) {
          tmem_ld_32x32(tq + (uint32_t)c, g);
          tmem_ld_32x32(tq + (uint32_t)(bn + c), u);
        } else {
          uint32_t g16[16], u16[16];
          tmem_ld_32x16(tq, g16);
          tmem_ld_32x16(tq + (uint32_t)bn, u16);
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            g[j] = g16[j];
            u[j] = u16[j];
          }
        }
        tmem_ld_wait();
        if (row_ok) {
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            const int t = t0 + c + j;
            if (j < step && t < p.T) {
              const float gv = __uint_as_float(g[j]), uv = __uint_as_float(u[j]);
              const float a = gv / (1.0f + __expf(-gv)) * uv;
              o[(size_t)t * p.ld_out] = __float2bfloat16_rn(a);
            }
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_dyn(tmem_base, tmem_cols);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                    CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                    CUtensorMapFloatOOBfill);
static PFN_encodeTiled g_encode = nullptr;

int make_tmap_bf16_2d(CUtensorMap *out, const void *base, uint64_t rows, uint64_t cols, uint32_t box_rows,
                      bool weight_like) {
  if (!g_encode) {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess)
      return -1;
    g_encode = (PFN_encodeTiled)fn;
  }
  cuuint64_t gdim[2] = {cols, rows};
  cuuint64_t gstride[1] = {cols * 2};
  cuuint32_t box[2] = {(cuuint32_t)GEMM_BK, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = g_encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), gdim, gstride, box,
                        estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                        weight_like ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B : CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? 0 : -(int)r - 1000;
}

int gemm_pick_bn(int T) {
  const int c[5] = {16, 32, 64, 128, 256};
  for (int i = 0; i < 5; ++i)
    if (T <= c[i]) return c[i];
  return 256;
}

size_t gemm_smem_bytes(int bn, bool dual, int stages) {
  size_t stage = (size_t)A_TILE_BYTES * (dual ? 2 : 1) + (size_t)bn * 128;
  return 1024 + stage * stages + 8 * (2 * stages + 1) + 16;
}

int gemm_pick_stages(int bn, bool dual) {
  static int env = -1;
  if (env < 0) {
    const char *e = getenv("SS_GEMM_STAGES");
    env = e ? atoi(e) : 0;
  }
  size_t stage = (size_t)A_TILE_BYTES * (dual ? 2 : 1) + (size_t)bn * 128;
  // small stages: aim at two co-resident CTAs per SM (their prologues/epilogues overlap); big stages: one CTA
  size_t budget = stage >= 32 * 1024 ? 200 * 1024 : 100 * 1024;
  int st = (int)(budget / stage);
  if (env > 0) st = env;
  if (st > 8) st = 8;
  while (st > 2 && gemm_smem_bytes(bn, dual, st) > 227 * 1024) --st;
  if (st < 2) st = 2;
  return st;
}

cudaError_t gemm_init() {
  cudaError_t e = cudaFuncSetAttribute(gemm_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(gemm_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
}

cudaError_t gemm_launch(const GemmLaunch &g) {
  const GemmParams &p = g.p;
  int tiles = 0;
  for (int i = 0; i < p.n_seg; ++i) tiles += (p.seg_rows[i] + GEMM_BM - 1) / GEMM_BM;
  dim3 grid(tiles, (p.T + p.bn - 1) / p.bn, g.splits);
  size_t smem = gemm_smem_bytes(p.bn, g.dual, p.stages);
  const CUtensorMap *a1 = g.a[1] ? g.a[1] : g.a[0];
  const CUtensorMap *a2 = g.a[2] ? g.a[2] : g.a[0];
  if (g.dual)
    gemm_kernel<true><<<grid, 192, smem, g.stream>>>(*g.a[0], *a1, *a2, *g.b, p);
  else
    gemm_kernel<false><<<grid, 192, smem, g.stream>>>(*g.a[0], *a1, *a2, *g.b, p);
  count_launch();
  return cudaGetLastError();
}

}  // namespace ss
