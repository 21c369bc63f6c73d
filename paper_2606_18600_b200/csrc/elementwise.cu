// elementwise.cu — the HBM-bound glue steps of a decoder layer, fused around the GEMMs' fp32 split-K partials:
//   S0/S1  input_rmsnorm      : widen the stage input (or gather embeddings) into the fp32 residual + RMSNorm-1
//   S3/S4  qkv_post           : split-K reduce + per-head QK RMSNorm (Qwen3) + RoPE; q -> bf16; k,v -> bf16 to the
//                               decode staging buffer (appended by the attention kernel) or, in prefill, to pages (S5)
//   S7/S8, S10/S1' residual_rmsnorm : residual += sum of split-K partials (fixed order), then the next RMSNorm
//   S11    final_norm_rows, logits_argmax
// The paper costs none of these (Table 2 has no norm / RoPE row); their math is readings A1,
// A8, A10, A11 of DESIGN.md.  All statistics and the residual stream are fp32.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "common.cuh"
#include "internal.h"

namespace ss {

constexpr int EW_THREADS = 256;

__device__ __forceinline__ float block_sum(float v, float *red /* [32] */) {
  v = warp_sum(v);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) red[warp] = v;
  __syncthreads();
  const int nw = (blockDim.x + 31) >> 5;
  float r = (lane < nw) ? red[lane] : 0.f;
  r = warp_sum(r);
  __syncthreads();
  return r;
}

// ---- S0 + S1 -------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(EW_THREADS)
input_rmsnorm_kernel(const CallArgs *__restrict__ args, const __nv_bfloat16 *__restrict__ embed,
                     const __nv_bfloat16 *__restrict__ w, float eps, int H, float *__restrict__ x,
                     __nv_bfloat16 *__restrict__ h) {
  pdl_launch_dependents();
  pdl_wait();
  __shared__ float red[32];
  const int t = blockIdx.x;
  const __nv_bfloat16 *src;
  if (args->hidden_in)
    src = (const __nv_bfloat16 *)args->hidden_in + (size_t)t * H;
  else
    src = embed + (size_t)args->token_ids[t] * H;
  float *xr = x + (size_t)t * H;
  float ss = 0.f;
  for (int j = threadIdx.x * 8; j < H; j += EW_THREADS * 8) {
    const uint4 v = *reinterpret_cast<const uint4 *>(src + j);
    float f[8] = {bf16_lo(v.x), bf16_hi(v.x), bf16_lo(v.y), bf16_hi(v.y),
                  bf16_lo(v.z), bf16_hi(v.z), bf16_lo(v.w), bf16_hi(v.w)};
#pragma unroll
    for (int i = 0; i < 8; ++i) ss += f[i] * f[i];
    *reinterpret_cast<float4 *>(xr + j) = make_float4(f[0], f[1], f[2], f[3]);
    *reinterpret_cast<float4 *>(xr + j + 4) = make_float4(f[4], f[5], f[6], f[7]);
  }
  ss = block_sum(ss, red);
  const float inv = 1.0f / sqrtf(ss / (float)H + eps);
  for (int j = threadIdx.x * 8; j < H; j += EW_THREADS * 8) {
    const uint4 v = *reinterpret_cast<const uint4 *>(src + j);
    const uint4 g = *reinterpret_cast<const uint4 *>(w + j);
    uint4 o;
    o.x = pack_bf16x2(bf16_lo(v.x) * inv * bf16_lo(g.x), bf16_hi(v.x) * inv * bf16_hi(g.x));
    o.y = pack_bf16x2(bf16_lo(v.y) * inv * bf16_lo(g.y), bf16_hi(v.y) * inv * bf16_hi(g.y));
    o.z = pack_bf16x2(bf16_lo(v.z) * inv * bf16_lo(g.z), bf16_hi(v.z) * inv * bf16_hi(g.z));
    o.w = pack_bf16x2(bf16_lo(v.w) * inv * bf16_lo(g.w), bf16_hi(v.w) * inv * bf16_hi(g.w));
    *reinterpret_cast<uint4 *>(h + (size_t)t * H + j) = o;
  }
}

cudaError_t launch_input_rmsnorm(const CallArgs *args, const void *embed, const void *ln_w, float eps, int H,
                                 int T, float *x, void *h, cudaStream_t s) {
  return launch_pdl(input_rmsnorm_kernel, dim3(T), dim3(EW_THREADS), 0, s, args, (const __nv_bfloat16 *)embed, (const __nv_bfloat16 *)ln_w, eps, H, x, (__nv_bfloat16 *)h);
}

// ---- pieces of an EPI_PARTIAL projection (internal.h GemmPartials): rows [r, r + 4) of row tile `tile`, token column
// `tok`, added in CTA order.  The loads of up to four pieces are issued together (independent L2 round trips). --------
__device__ __forceinline__ float4 gemm_partial_sum4(const GemmPartials &gp, int tile, int tok, int r) {
  const PartialTile pt = gp.tiles[tile];
  const float *base = gp.slots + (size_t)tok * GEMM_BM + r;
  // piece q of source rank q / count (one rank unless the fused tensor-parallel all-reduce is on), rank-major, CTA order
  const int n = pt.count * gp.n_src;
  auto piece = [&](int q) {
    const int src = q / pt.count, c = q - src * pt.count;
    const int slot = 2 * (pt.first_cta + c) + (c == 0 ? pt.first_item : 0);
    return __ldcg(reinterpret_cast<const float4 *>(base + (size_t)src * gp.src_stride + (size_t)slot * gp.slot_floats));
  };
  float4 y = piece(0);
  for (int q = 1; q < n; q += 4) {
    float4 z[4];
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (q + u < n) z[u] = piece(q + u);
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (q + u < n) {
        y.x += z[u].x; y.y += z[u].y; y.z += z[u].z; y.w += z[u].w;
      }
  }
  return y;
}

__device__ __forceinline__ float2 gemm_partial_sum2(const GemmPartials &gp, int tile, int tok, int r) {
  const PartialTile pt = gp.tiles[tile];
  const float *base = gp.slots + (size_t)tok * GEMM_BM + r;
  float2 y = make_float2(0.f, 0.f);
  for (int q = 0; q < pt.count; ++q) {
    const int slot = 2 * (pt.first_cta + q) + (q == 0 ? pt.first_item : 0);
    const float2 z = __ldcg(reinterpret_cast<const float2 *>(base + (size_t)slot * gp.slot_floats));
    y.x = q == 0 ? z.x : y.x + z.x;
    y.y = q == 0 ? z.y : y.y + z.y;
  }
  return y;
}

// ---- residual += sum_s part[s]; optional RMSNorm -> h; optional bf16 stage output -----------------------------
// One CTA of 1024 threads per token row; the whole row lives in registers (IT float4 per thread, H <= IT*4096), all
// loads are issued before any use, and x is read and written exactly once.
// Few rows (decode): 1024 threads per row for latency.  Many rows (prefill): 256 threads per row, so 8 rows are in
// flight per SM and the block reduction is two warps deep instead of 32.
template <int IT, int RN_THREADS, bool PARTS>  // PARTS = false: nothing to add to x (no partial sums, no stream-K pieces)
__global__ void __launch_bounds__(RN_THREADS)
residual_rmsnorm_kernel(float *__restrict__ x, const float *__restrict__ part, int splits, long long split_stride,
                        const GemmPartials gp, const __nv_bfloat16 *__restrict__ w, float eps, int H,
                        __nv_bfloat16 *__restrict__ h, const CallArgs *__restrict__ args, int write_out) {
  pdl_launch_dependents();
  pdl_wait();
  __shared__ float red[32];
  const int t = blockIdx.x;
  float *xr = x + (size_t)t * H;
  const float *pr = part + (size_t)t * H;
  __nv_bfloat16 *outp = nullptr;
  if (write_out && args->out_hidden) outp = (__nv_bfloat16 *)args->out_hidden + (size_t)t * H;
  float4 v[IT];
#pragma unroll
  for (int i = 0; i < IT; ++i) {
    const int j = (i * RN_THREADS + threadIdx.x) * 4;
    v[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (j < H) v[i] = *reinterpret_cast<const float4 *>(xr + j);
  }
  if constexpr (PARTS) {
    float4 y[IT];
#pragma unroll
    for (int i = 0; i < IT; ++i) {
      const int j = (i * RN_THREADS + threadIdx.x) * 4;
      y[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (j < H && splits > 0) y[i] = *reinterpret_cast<const float4 *>(pr + j);
    }
    if (gp.slots) {
      // the projection left its tiles in pieces (EPI_PARTIAL, internal.h): y = the tile's pieces added in CTA order
#pragma unroll
      for (int i = 0; i < IT; ++i) {
        const int j = (i * RN_THREADS + threadIdx.x) * 4;
        if (j < H) y[i] = gemm_partial_sum4(gp, j >> 7, t, j & 127);
      }
    }
    for (int s = 1; s < splits; ++s) {
#pragma unroll
      for (int i = 0; i < IT; ++i) {
        const int j = (i * RN_THREADS + threadIdx.x) * 4;
        if (j < H) {
          const float4 q = *reinterpret_cast<const float4 *>(pr + (size_t)s * split_stride + j);
          y[i].x += q.x; y[i].y += q.y; y[i].z += q.z; y[i].w += q.w;
        }
      }
    }
#pragma unroll
    for (int i = 0; i < IT; ++i) {
      v[i].x += y[i].x; v[i].y += y[i].y; v[i].z += y[i].z; v[i].w += y[i].w;
    }
  }
  float ss = 0.f;
#pragma unroll
  for (int i = 0; i < IT; ++i) {
    const int j = (i * RN_THREADS + threadIdx.x) * 4;
    if (j < H) {
      if (PARTS) *reinterpret_cast<float4 *>(xr + j) = v[i];  // otherwise x already holds the sum
      ss += v[i].x * v[i].x + v[i].y * v[i].y + v[i].z * v[i].z + v[i].w * v[i].w;
      if (outp) {
        uint2 o;
        o.x = pack_bf16x2(v[i].x, v[i].y);
        o.y = pack_bf16x2(v[i].z, v[i].w);
        *reinterpret_cast<uint2 *>(outp + j) = o;
      }
    }
  }
  if (w == nullptr) return;
  ss = block_sum(ss, red);
  const float inv = 1.0f / sqrtf(ss / (float)H + eps);
#pragma unroll
  for (int i = 0; i < IT; ++i) {
    const int j = (i * RN_THREADS + threadIdx.x) * 4;
    if (j < H) {
      const uint2 g = *reinterpret_cast<const uint2 *>(w + j);
      uint2 o;
      o.x = pack_bf16x2(v[i].x * inv * bf16_lo(g.x), v[i].y * inv * bf16_hi(g.x));
      o.y = pack_bf16x2(v[i].z * inv * bf16_lo(g.y), v[i].w * inv * bf16_hi(g.y));
      *reinterpret_cast<uint2 *>(h + (size_t)t * H + j) = o;
    }
  }
}

cudaError_t launch_residual_rmsnorm(float *x, const float *part, int splits, long long split_stride,
                                    const GemmPartials &gp, const void *ln_w, float eps, int H, int T, void *h,
                                    const CallArgs *args, bool write_out_hidden, cudaStream_t s, bool fixed_shape, bool pdl) {
  const __nv_bfloat16 *w = (const __nv_bfloat16 *)ln_w;
  __nv_bfloat16 *hh = (__nv_bfloat16 *)h;
  const int wo = write_out_hidden ? 1 : 0;
  const bool parts = splits > 0 || gp.slots != nullptr;
  auto go = [&](auto kernel, int threads) {
    return launch_pdl_if(pdl, kernel, dim3(T), dim3(threads), 0, s, x, part, splits, split_stride, gp, w, eps, H, hh, args, wo);
  };
#define SS_RN(IT, TH) (parts ? go(residual_rmsnorm_kernel<IT, TH, true>, TH) : go(residual_rmsnorm_kernel<IT, TH, false>, TH))
  if (!fixed_shape && T >= 512 && H <= 16 * 256 * 4) {  // many rows: 256 threads each
    const int it = (H + 1023) / 1024;
    if (it <= 2) return SS_RN(2, 256);
    if (it <= 4) return SS_RN(4, 256);
    if (it <= 8) return SS_RN(8, 256);
    return SS_RN(16, 256);
  }
  const int it = (H + 4095) / 4096;
  if (it <= 1) return SS_RN(1, 1024);
  if (it <= 2) return SS_RN(2, 1024);
  if (it <= 4) return SS_RN(4, 1024);
#undef SS_RN
  return cudaErrorInvalidValue;  // hidden > 16384 is rejected at create
}

// ---- S11a: final RMSNorm of the last row of each sequence -----------------------------------------------------
__global__ void __launch_bounds__(EW_THREADS)
final_norm_rows_kernel(const float *__restrict__ x, const CallArgs *__restrict__ args, int decode,
                       const __nv_bfloat16 *__restrict__ wf, float eps, int H, __nv_bfloat16 *__restrict__ hl) {
  pdl_launch_dependents();
  pdl_wait();
  __shared__ float red[32];
  const int s = blockIdx.x;
  const int row = decode ? s : (args->cu_q[s + 1] - 1);
  const float *xr = x + (size_t)row * H;
  float ss = 0.f;
  for (int j = threadIdx.x; j < H; j += EW_THREADS) ss += xr[j] * xr[j];
  ss = block_sum(ss, red);
  const float inv = 1.0f / sqrtf(ss / (float)H + eps);
  for (int j = threadIdx.x; j < H; j += EW_THREADS)
    hl[(size_t)s * H + j] = __float2bfloat16_rn(xr[j] * inv * __bfloat162float(wf[j]));
}

cudaError_t launch_final_norm_rows(const float *x, const CallArgs *args, bool decode, const void *wf, float eps,
                                   int H, int n_seqs, void *hl, cudaStream_t s) {
  return launch_pdl(final_norm_rows_kernel, dim3(n_seqs), dim3(EW_THREADS), 0, s, x, args, decode ? 1 : 0, (const __nv_bfloat16 *)wf, eps, H, (__nv_bfloat16 *)hl);
}

// ---- S11b: copy the logits out and argmax (lowest index among maxima), two passes: AM_SPLITS CTAs per row scan a
// slice of the vocabulary each (64 rows x 128,256 fp32 = 33 MB: one CTA per row would leave most SMs idle), then one
// warp per row combines the slices' (max, index) pairs in slice order.
constexpr int AM_SPLITS = 16;
__device__ __forceinline__ void argmax_combine(float &best, int &bi, float ob, int oi) {
  if (ob > best || (ob == best && oi < bi)) {
    best = ob;
    bi = oi;
  }
}

__global__ void __launch_bounds__(1024)
logits_argmax_part_kernel(const float *__restrict__ logits, int V, const CallArgs *__restrict__ args,
                          float *__restrict__ part_max, int *__restrict__ part_idx) {
  pdl_launch_dependents();
  pdl_wait();
  __shared__ float smax[32];
  __shared__ int sidx[32];
  const int r = blockIdx.x, sp = blockIdx.y;
  const int per = (V + AM_SPLITS - 1) / AM_SPLITS;
  const int j0 = sp * per, j1 = min(V, j0 + per);
  float *outl = args->out_logits ? args->out_logits + (size_t)r * V : nullptr;
  float best = -INFINITY;
  int bi = 0x7fffffff;
  for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
    const float v = logits[(size_t)r * V + j];
    if (outl) outl[j] = v;
    if (v > best) {  // j ascending per thread: strict > keeps the lowest index
      best = v;
      bi = j;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1)
    argmax_combine(best, bi, __shfl_xor_sync(0xffffffffu, best, o), __shfl_xor_sync(0xffffffffu, bi, o));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) {
    smax[warp] = best;
    sidx[warp] = bi;
  }
  __syncthreads();
  if (warp == 0) {
    const int nw = blockDim.x >> 5;
    best = lane < nw ? smax[lane] : -INFINITY;
    bi = lane < nw ? sidx[lane] : 0x7fffffff;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
      argmax_combine(best, bi, __shfl_xor_sync(0xffffffffu, best, o), __shfl_xor_sync(0xffffffffu, bi, o));
    if (lane == 0) {
      part_max[r * AM_SPLITS + sp] = best;
      part_idx[r * AM_SPLITS + sp] = bi;
    }
  }
}

__global__ void __launch_bounds__(32)
logits_argmax_final_kernel(const float *__restrict__ part_max, const int *__restrict__ part_idx,
                           const CallArgs *__restrict__ args) {
  pdl_launch_dependents();
  pdl_wait();
  const int r = blockIdx.x, lane = threadIdx.x;
  float best = lane < AM_SPLITS ? part_max[r * AM_SPLITS + lane] : -INFINITY;
  int bi = lane < AM_SPLITS ? part_idx[r * AM_SPLITS + lane] : 0x7fffffff;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1)
    argmax_combine(best, bi, __shfl_xor_sync(0xffffffffu, best, o), __shfl_xor_sync(0xffffffffu, bi, o));
  if (lane == 0 && args->out_argmax) args->out_argmax[r] = bi;
}

cudaError_t launch_logits_argmax(const float *logits, int V, int n_rows, float *part_max, int *part_idx,
                                 const CallArgs *args, cudaStream_t s) {
  cudaError_t e = launch_pdl(logits_argmax_part_kernel, dim3(n_rows, AM_SPLITS), dim3(1024), 0, s, logits, V, args,
                             part_max, part_idx);
  if (e != cudaSuccess) return e;
  return launch_pdl(logits_argmax_final_kernel, dim3(n_rows), dim3(32), 0, s, (const float *)part_max,
                    (const int *)part_idx, args);
}

// ---- S3 + S4 (+ S5 in prefill): one HALF-warp per (token, head) -------------------------------------------------
// Lane l of the half-warp owns V = d/32 consecutive elements of the low half, [V*l, V*l + V), and their rotation
// partners in the high half (c + d/2), so every access is one vector load / store (16 B at d = 128) and RoPE is
// thread-local; the per-head RMSNorm statistic is a 4-step shuffle inside the half-warp.
template <int V>  // V = d / 32: 4 (d = 128) or 2 (d = 64)
__global__ void __launch_bounds__(EW_THREADS) qkv_post_kernel(const QkvPostParams p) {
  pdl_launch_dependents();
  pdl_wait();
  const int hw = threadIdx.x >> 4, l = threadIdx.x & 15;
  const int n_heads = p.n_q + 2 * p.n_kv;
  const int head = blockIdx.y * (EW_THREADS / 16) + hw;
  const int t = blockIdx.x;
  const bool active = head < n_heads;
  const int d = p.d, half = d >> 1;
  const int c = V * l;
  float lo[V], hi[V];
#pragma unroll
  for (int i = 0; i < V; ++i) lo[i] = hi[i] = 0.f;
  const int ldq = n_heads * d;
  if (active && p.gp.slots) {
    // the QKV projection left its tiles in pieces (EPI_PARTIAL): this head's d rows lie inside one 128-row tile of its
    // segment (d divides 128), the low half at row r0 + c, the rotation partners d/2 rows further
    const int seg = head < p.n_q ? 0 : (head < p.n_q + p.n_kv ? 1 : 2);
    const int row = (head - (seg == 0 ? 0 : (seg == 1 ? p.n_q : p.n_q + p.n_kv))) * d;
    const int tile = (seg == 0 ? 0 : (seg == 1 ? p.tile0_k : p.tile0_v)) + (row >> 7);
    const int r0 = (row & 127) + c;
    if (V == 4) {
      const float4 a = gemm_partial_sum4(p.gp, tile, t, r0), b = gemm_partial_sum4(p.gp, tile, t, r0 + half);
      lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; lo[3] = a.w;
      hi[0] = b.x; hi[1] = b.y; hi[2] = b.z; hi[3] = b.w;
    } else {
      const float2 a = gemm_partial_sum2(p.gp, tile, t, r0), b = gemm_partial_sum2(p.gp, tile, t, r0 + half);
      lo[0] = a.x; lo[1] = a.y;
      hi[0] = b.x; hi[1] = b.y;
    }
  } else if (active) {
    const float *src = p.qkv_part + (size_t)t * ldq + (size_t)head * d;
    for (int s = 0; s < p.splits; ++s) {
      const float *sp = src + (size_t)s * p.split_stride;
      if (V == 4) {
        const float4 a = *reinterpret_cast<const float4 *>(sp + c), b = *reinterpret_cast<const float4 *>(sp + c + half);
        lo[0] += a.x; lo[1] += a.y; lo[2] += a.z; lo[3] += a.w;
        hi[0] += b.x; hi[1] += b.y; hi[2] += b.z; hi[3] += b.w;
      } else {
        const float2 a = *reinterpret_cast<const float2 *>(sp + c), b = *reinterpret_cast<const float2 *>(sp + c + half);
        lo[0] += a.x; lo[1] += a.y;
        hi[0] += b.x; hi[1] += b.y;
      }
    }
  }
  const bool is_q = head < p.n_q;
  const bool is_k = !is_q && head < p.n_q + p.n_kv;
  int pos = 0, seq = 0;
  if (active) {
    if (p.decode) {
      seq = t;
      pos = p.args->ctx[t];
    } else {
      seq = p.tok_seq[t];
      pos = p.tok_pos[t];
    }
  }
  if (p.qk_norm) {  // every lane takes part in the shuffles; the result is used by q / k heads only
    float ss = 0.f;
#pragma unroll
    for (int i = 0; i < V; ++i) ss += lo[i] * lo[i] + hi[i] * hi[i];
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    if (active && (is_q || is_k)) {
      const float inv = 1.0f / sqrtf(ss / (float)d + p.eps);
      const __nv_bfloat16 *g = (const __nv_bfloat16 *)(is_q ? p.q_norm : p.k_norm);
#pragma unroll
      for (int i = 0; i < V; ++i) {
        lo[i] = lo[i] * inv * __bfloat162float(g[c + i]);
        hi[i] = hi[i] * inv * __bfloat162float(g[c + half + i]);
      }
    }
  }
  if (!active) return;
  if (is_q || is_k) {
    const float2 *rt = reinterpret_cast<const float2 *>(p.rope) + (size_t)pos * half + c;
#pragma unroll
    for (int i = 0; i < V; ++i) {
      const float2 cs = rt[i];
      const float a = lo[i], b = hi[i];
      lo[i] = a * cs.x - b * cs.y;
      hi[i] = b * cs.x + a * cs.y;
    }
  }
  __nv_bfloat16 *dst;
  if (is_q) {
    dst = (__nv_bfloat16 *)p.q_out + (size_t)t * p.n_q * d + (size_t)head * d;
  } else {
    const int hk = is_k ? head - p.n_q : head - p.n_q - p.n_kv;
    if (p.decode) {
      dst = (__nv_bfloat16 *)p.kv_new + (size_t)t * 2 * p.n_kv * d + (size_t)(is_k ? 0 : p.n_kv * d) +
            (size_t)hk * d;
    } else {
      const int page = p.args->block_tables[(size_t)seq * p.args->max_blocks + (pos >> 4)];
      __nv_bfloat16 *pool = (__nv_bfloat16 *)(is_k ? p.kpool : p.vpool);
      dst = pool + (((size_t)page * p.n_kv + hk) * 16 + (size_t)(pos & 15)) * d;
    }
  }
  if (V == 4) {
    *reinterpret_cast<uint2 *>(dst + c) = make_uint2(pack_bf16x2(lo[0], lo[1]), pack_bf16x2(lo[2], lo[3]));
    *reinterpret_cast<uint2 *>(dst + c + half) = make_uint2(pack_bf16x2(hi[0], hi[1]), pack_bf16x2(hi[2], hi[3]));
  } else {
    *reinterpret_cast<uint32_t *>(dst + c) = pack_bf16x2(lo[0], lo[1]);
    *reinterpret_cast<uint32_t *>(dst + c + half) = pack_bf16x2(hi[0], hi[1]);
  }
}

cudaError_t launch_qkv_post(const QkvPostParams &p, cudaStream_t s) {
  const int n_heads = p.n_q + 2 * p.n_kv;
  const int per_block = EW_THREADS / 16;
  dim3 grid(p.T, (n_heads + per_block - 1) / per_block);
  if (p.d == 128) return launch_pdl(qkv_post_kernel<4>, dim3(grid), dim3(EW_THREADS), 0, s, p);
  return launch_pdl(qkv_post_kernel<2>, dim3(grid), dim3(EW_THREADS), 0, s, p);
}

// ---- KV migration by transfer (NEXT-4): gather a request's pages out of the layer-major pool into one contiguous
// buffer [L][K/V][n][n_kv][16][d] (what a GPU-to-GPU copy would carry), and the reverse scatter.  One (layer, K/V,
// page) piece is n_kv * 16 * d contiguous bf16 (32 KB at the paper's shapes); pure HBM copy, 16 bytes per thread. ----
__global__ void __launch_bounds__(256)
kv_pages_copy_kernel(uint4 *__restrict__ pool, uint4 *__restrict__ buf, const int32_t *__restrict__ page_ids, int n,
                     int n_pages_pool, int piece_vec /* uint4 per piece */, int to_buffer) {
  pdl_launch_dependents();
  pdl_wait();
  const int piece = blockIdx.x;              // = (layer * 2 + kv) * n + i
  const int lk = piece / n, i = piece - lk * n;
  uint4 *pp = pool + ((size_t)lk * n_pages_pool + page_ids[i]) * piece_vec;
  uint4 *bp = buf + (size_t)piece * piece_vec;
  for (int v = threadIdx.x; v < piece_vec; v += 256) {
    if (to_buffer) bp[v] = pp[v]; else pp[v] = bp[v];
  }
}

cudaError_t launch_kv_pages_copy(void *pool, void *buf, const int32_t *page_ids, int n, int n_layers, int n_pages_pool,
                                 int piece_bytes, bool to_buffer, cudaStream_t s) {
  return launch_pdl(kv_pages_copy_kernel, dim3(n_layers * 2 * n), dim3(256), 0, s, (uint4 *)pool, (uint4 *)buf, page_ids,
                    n, n_pages_pool, piece_bytes / 16, to_buffer ? 1 : 0);
}

// ---- SS_DEBUG=1: device-side contract checks (SURVEY.md section 8(b) "Errors"; include/shuntstage.h) -----------------
// One CTA walks the call's sequences before anything else is enqueued: ctx >= 0, q_len >= 1 (== 1 for the decode rows),
// cu_q consistent with T, ctx + q_len within the listed pages (max_blocks * 16) and within the RoPE table, every page id
// of positions [0, ctx + q_len) inside the pool, token ids inside the vocabulary.  The FIRST violation (lowest thread
// wins the CAS) is recorded as err = {code, sequence, index, value}.
__global__ void __launch_bounds__(256)
debug_validate_kernel(const CallArgs *__restrict__ args, DebugCheck c, int32_t *__restrict__ err) {
  auto fail = [&](int code, int seq, int idx, int val) {
    if (atomicCAS(err, 0, code) == 0) {
      err[1] = seq;
      err[2] = idx;
      err[3] = val;
    }
  };
  const int n = args->n_seqs;
  if (threadIdx.x == 0 && !c.decode) {
    if (args->cu_q[0] != 0) fail(SS_DBG_BAD_CU_Q, 0, 0, args->cu_q[0]);
    if (args->cu_q[n] != args->T) fail(SS_DBG_BAD_CU_Q, n, n, args->cu_q[n]);
  }
  for (int s = 0; s < n; ++s) {
    const int ctx = args->ctx[s];
    const int q_len = c.decode ? 1 : args->cu_q[s + 1] - args->cu_q[s];
    if (threadIdx.x == 0) {
      if (ctx < 0) fail(SS_DBG_BAD_CTX, s, 0, ctx);
      if (q_len < 1 || (s < c.n_decode_rows && q_len != 1)) fail(SS_DBG_BAD_CU_Q, s, s, q_len);
      if ((long long)ctx + q_len > (long long)args->max_blocks * 16) fail(SS_DBG_BEYOND_PAGES, s, args->max_blocks, ctx + q_len);
      if ((long long)ctx + q_len > (long long)c.max_pos) fail(SS_DBG_BEYOND_MAX_POS, s, c.max_pos, ctx + q_len);
    }
    if (ctx < 0 || q_len < 1) continue;
    long long need = ((long long)ctx + q_len + 15) >> 4;
    if (need > args->max_blocks) need = args->max_blocks;
    const int32_t *bt = args->block_tables + (size_t)s * args->max_blocks;
    for (int i = threadIdx.x; i < (int)need; i += blockDim.x) {
      const int pg = bt[i];
      if (pg < 0 || pg >= c.num_pages) fail(SS_DBG_BAD_PAGE, s, i, pg);
    }
  }
  if (args->token_ids)
    for (int t = threadIdx.x; t < args->T; t += blockDim.x) {
      const int id = args->token_ids[t];
      if (id < 0 || id >= c.vocab) fail(SS_DBG_BAD_TOKEN, -1, t, id);
    }
}

cudaError_t launch_debug_validate(const CallArgs *args, const DebugCheck &c, int32_t *err, cudaStream_t s) {
  count_launch();
  debug_validate_kernel<<<1, 256, 0, s>>>(args, c, err);
  return cudaGetLastError();
}

__global__ void __launch_bounds__(256)
debug_validate_pages_kernel(const int32_t *__restrict__ ids, int n, int num_pages, int32_t *__restrict__ err) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const int pg = ids[i];
    if ((pg < 0 || pg >= num_pages) && atomicCAS(err, 0, SS_DBG_BAD_PAGE) == 0) {
      err[1] = -1;
      err[2] = i;
      err[3] = pg;
    }
  }
}

cudaError_t launch_debug_validate_pages(const int32_t *ids, int n, int num_pages, int32_t *err, cudaStream_t s) {
  count_launch();
  debug_validate_pages_kernel<<<(n + 255) / 256 > 64 ? 64 : (n + 255) / 256, 256, 0, s>>>(ids, n, num_pages, err);
  return cudaGetLastError();
}

}  // namespace ss
