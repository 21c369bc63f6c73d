// gemm_tcgen05.cu — the bf16 projections of a decoder layer (Table 2 rows "QKV Projection", "Output Projection",
// "Up and Gate Projection", "Down Projection", "Logits Calculation") as persistent tcgen05/TMEM GEMM
// kernels fed by TMA, for sm_100a.
//
// out[t][n] = sum_k X[t,k] * W[n,k]     X: activations [T,K] bf16 row-major, W: weights [N,K] bf16 row-major.
//
// Orientation: the 128 TMEM lanes (UMMA M) run over weight rows n, the TMEM columns (UMMA N = bn) over tokens t.
// At decode (T = 64..128) this streams every weight byte exactly once through full-width 128-row MMAs (the
// HBM-bound case).
//
// gemm_kernel (one CTA per SM; every decode shape, T <= 512, the batch-invariant mode).  CTA = 11 warps: warp 0 = TMA
// producer (one lane), warps 1 and 6 = MMA issuers (one lane each; warp 1 also allocates TMEM), warps 2-5 and 7-10 =
// epilogue (two per TMEM lane quadrant).  ONE smem ring of up to 12 stages {weight tile 128x64 (x2 when DUAL), activation
// tile bn x 64}, SWIZZLE_128B, full/empty mbarriers; accumulators in TMEM, double-buffered when they fit so the epilogue
// of one work item overlaps the MMAs of the next; the producer primes the ring with weights before it waits for the
// predecessor kernel (PDL).  Schedules: see internal.h (stream-K for the decode shapes — in-kernel fix-up, or EPI_PARTIAL:
// every piece left to the consumer kernel, optionally stored into every tensor-parallel rank's exchange buffer —,
// band-rasterised whole tiles otherwise).  DUAL = gate and up tiles share the B tile and the epilogue writes silu(g)*u as
// bf16 (step S9), so [T,2F] never reaches HBM.  EPI_RESID_F32 adds the projection straight into the fp32 residual stream.
//
// gemm_pair_kernel (further down): the tensor-bound prefill shapes on CTA pairs (tcgen05.mma.cta_group::2).
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdlib.h>

#include "common.cuh"
#include "internal.h"

namespace ss {

constexpr int A_TILE_BYTES = GEMM_BM * GEMM_BK * 2;  // 16 KB
constexpr int GEMM_THREADS = 352;  // warp 0: TMA producer, 1: MMA issuer 0, 6: MMA issuer 1, 2-5 and 7-10: epilogue
constexpr int EPI_WARPS = 8;       // two warps per TMEM lane quadrant, taking alternate 32-column chunks

struct WorkItem {
  int row_tile, t_tile, kb0, kb1;
};

// Per-CTA work list.  All roles of a CTA construct the same iterator and see the same items in the same order.
struct WorkIter {
  int sched, nkb, n_row_tiles, n_t_tiles, band, G, c;
  uint32_t u, u_end;   // stream-K: unit cursor / end of this CTA's range (units = (tile, k-block); < 2^31, gemm_plan)
  uint32_t uq, ur;     // U / G, U % G
  int idx, n_tiles;    // tiles: next tile index

  // 32-bit arithmetic only: every role runs this before its first instruction of real work, and a 64-bit divide is
  // a ~200-cycle subroutine (the producer issued its first TMA load ~1 us after the CTA's setup was done)
  __device__ WorkIter(const GemmParams &p, int cta, int grid) {
    sched = p.sched;
    nkb = (p.K + GEMM_BK - 1) / GEMM_BK;
    n_row_tiles = p.n_row_tiles;
    n_t_tiles = p.n_t_tiles;
    band = p.band;
    G = grid;
    c = cta;
    n_tiles = n_row_tiles * n_t_tiles;
    const uint32_t U = (uint32_t)n_tiles * (uint32_t)nkb;
    uq = U / (uint32_t)G;
    ur = U - uq * (uint32_t)G;
    u = range_start(c);
    u_end = range_start(c + 1);
    idx = c;
  }
  // first unit of CTA cc's stream-K range = floor(cc * U / G)
  __device__ uint32_t range_start(int cc) const { return (uint32_t)cc * uq + ((uint32_t)cc * ur) / (uint32_t)G; }

  __device__ bool next(WorkItem &w) {
    if (sched == SCHED_STREAMK) {
      if (u >= u_end) return false;
      const uint32_t tile = u / (uint32_t)nkb;
      w.kb0 = (int)(u - tile * (uint32_t)nkb);
      const uint32_t left = u_end - u;
      w.kb1 = (int)min((uint32_t)w.kb0 + left, (uint32_t)nkb);
      w.t_tile = (int)tile / n_row_tiles;
      w.row_tile = (int)tile - w.t_tile * n_row_tiles;
      u += (uint32_t)(w.kb1 - w.kb0);
      return true;
    }
    if (idx >= n_tiles) return false;
    const int per_band = band * n_t_tiles;
    const int b = idx / per_band, rem = idx - b * per_band;
    const int rb = min(band, n_row_tiles - b * band);
    w.t_tile = rem / rb;
    w.row_tile = b * band + (rem - w.t_tile * rb);
    w.kb0 = 0;
    w.kb1 = nkb;
    idx += G;
    return true;
  }
};

__device__ __forceinline__ int ld_acquire(const int *p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// Debug aid: when a bounded wait expires, the site is recorded in host-mapped memory (if ss_debug_buffer() was
// given one) before the trap, so that a protocol bug can be located without a debugger.
__device__ unsigned long long *g_dbg = nullptr;
__device__ __noinline__ void wait_expired(int site, uint32_t a, uint32_t b) {
  if (g_dbg) {
    g_dbg[1] = ((unsigned long long)blockIdx.x << 32) | threadIdx.x;
    g_dbg[2] = ((unsigned long long)a << 32) | b;
    g_dbg[0] = (unsigned long long)site;
    __threadfence_system();
  }
  __trap();
}
__device__ __forceinline__ void mbar_wait_site(uint64_t *bar, uint32_t parity, int site, uint32_t info) {
  uint32_t polls = 0;
  unsigned long long t0 = 0;
  while (!mbar_try_wait(bar, parity)) {
    if (wait_expired_ns(polls, t0)) wait_expired(site, info, parity);
  }
}
// Optional timeline (profiling builds only: -DSS_GEMM_TRACE): globaltimer stamps per CTA into p.trace[cta*64 + slot].
#ifdef SS_GEMM_TRACE
__device__ __forceinline__ void trace(const GemmParams &p, int slot) {
  if (p.trace && slot < 64) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    p.trace[(size_t)blockIdx.x * 64 + slot] = t;
  }
}
#else
__device__ __forceinline__ void trace(const GemmParams &, int) {}
#endif
__device__ __forceinline__ void epi_bar() { asm volatile("bar.sync 1, 256;" ::: "memory"); }

template <bool DUAL>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_kernel(const __grid_constant__ CUtensorMap ta0, const __grid_constant__ CUtensorMap ta1,
            const __grid_constant__ CUtensorMap ta2, const __grid_constant__ CUtensorMap tb, const GemmParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *base = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const int bn = p.bn;
  constexpr uint32_t a_bytes = A_TILE_BYTES * (DUAL ? 2 : 1);
  const uint32_t b_bytes = (uint32_t)bn * 128u;
  const uint32_t stage_bytes = a_bytes + b_bytes;
  const int stages = p.stages;
  uint64_t *full = (uint64_t *)(base + (size_t)stages * stage_bytes);
  uint64_t *empty = full + stages;
  uint64_t *tfull = empty + stages;   // [2]
  uint64_t *tempty = tfull + 2;       // [2]
  uint32_t *tmem_slot = (uint32_t *)(tempty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cta = blockIdx.x, grid = gridDim.x;

  // One tcgen05.mma (M=128, K=16, operands in smem) occupies its issuing thread for ~128 cycles whatever N is
  // (measured in round 1 with a clock64 probe), i.e. 4 KB of weights per 128 cycles: a single issuer
  // cannot keep up with HBM at bn <= 128.  The HBM-bound schedule therefore runs TWO issuers (warps 1 and 6), each
  // into its own accumulator; the epilogue adds the two.  Issuer (slot & 1) owns ring slot `slot` for the whole
  // kernel: an mbarrier's single phase bit is only safe when all waits on it come, in order, from one thread (with
  // k-blocks dealt alternately and an odd ring size a slot changed hands every round, a fast issuer could take a
  // stale phase for its own and read a tile still in flight).
  const uint32_t acc_cols = (uint32_t)bn * (DUAL ? 2u : 1u);
  const int n_iss = p.issuers;
  const uint32_t acc_stride = acc_cols * (uint32_t)n_iss;  // TMEM columns per buffer
  const int nbuf = (p.single_buf == 0 && 2 * acc_stride <= 512) ? 2 : 1;
  uint32_t tmem_cols = 32;
  while (tmem_cols < acc_stride * nbuf) tmem_cols <<= 1;

  pdl_launch_dependents();
  if (threadIdx.x == 0) trace(p, 0);
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&ta0);
    if (DUAL || p.n_seg > 1) tma_prefetch_desc(&ta1);
    if (p.n_seg > 2) tma_prefetch_desc(&ta2);
    tma_prefetch_desc(&tb);
    for (int i = 0; i < stages; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1u);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&tfull[i], (uint32_t)n_iss);
      mbar_init(&tempty[i], EPI_WARPS);  // one arrival per epilogue warp
    }
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc_dyn(tmem_slot, tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  if (threadIdx.x == 0) trace(p, 7);

  // The single-thread roles run their loops on the WHOLE warp (uniform control flow: every lane waits on the barriers
  // and walks the same items) and issue under elect_one(): under `if (lane == 0)` nvcc cannot keep the TMA / MMA operands
  // in uniform registers and wraps every UTMALDG / UTCHMMA in an ELECT + 5 x R2UR.BROADCAST + BRA.U.ANY loop, which is
  // what made one issue cost ~100-130 cycles whatever its shape.
  if (warp == 0) {
    {
      // ---------------- TMA producer ----------------
      // Weights are never written by the stage, so the first `stages` weight tiles are requested BEFORE waiting for
      // the predecessor kernel (PDL): the ring is full of weights by the time the activations exist.
      // (No integer division in the per-k-block loops of the single-thread roles: they are latency-bound, and a
      // u32 divide by a runtime value cost ~0.1 us per k-block.)
      // stream-K (decode): weights are streamed once, activations are re-read by every CTA.  Tiles (prefill): a
      // weight tile is re-read by every token tile of its band, so it must stay in L2 as well.
      const uint64_t pol_w = p.w_policy == 0 ? l2_policy_evict_first()
                                             : (p.w_policy == 1 ? l2_policy_evict_normal() : l2_policy_evict_last());
      const uint64_t pol_x = l2_policy_evict_last();
      WorkIter it(p, cta, grid);
      WorkItem w;
      int n = 0;        // running k-block counter across items (saturating use: only compared with `stages`)
      int s = 0;        // = n % stages
      uint32_t ph = 0;  // = (n / stages) & 1
      bool waited = false;
      int pend_kb[GEMM_MAX_STAGES], pend_t0[GEMM_MAX_STAGES];
      while (it.next(w)) {
        int seg = 0;
#pragma unroll
        for (int i = 1; i < 3; ++i)
          if (i < p.n_seg && w.row_tile >= p.seg_tile0[i]) seg = i;
        const int row0 = (w.row_tile - p.seg_tile0[seg]) * GEMM_BM;
        const int t0 = w.t_tile * bn;
        const CUtensorMap *ta = DUAL ? &ta0 : (seg == 0 ? &ta0 : (seg == 1 ? &ta1 : &ta2));
        for (int kb = w.kb0; kb < w.kb1; ++kb) {
          if (!waited && n == stages) {  // ring primed with weights: now the activations of those k-blocks
            pdl_wait();
            waited = true;
            if (elect_one())
              for (int i = 0; i < stages; ++i)
                tma_load_2d(base + (size_t)i * stage_bytes + a_bytes, &tb, &full[i], pend_kb[i] * GEMM_BK, pend_t0[i],
                            pol_x);
            __syncwarp();
          }
          mbar_wait_site(&empty[s], ph ^ 1u, 1, (uint32_t)s);
          uint8_t *st = base + (size_t)s * stage_bytes;
          if (elect_one()) {
            mbar_expect_tx(&full[s], stage_bytes);
            tma_load_2d(st, ta, &full[s], kb * GEMM_BK, row0, pol_w);
            if (n == 0) trace(p, 8);
            if (DUAL) tma_load_2d(st + A_TILE_BYTES, &ta1, &full[s], kb * GEMM_BK, row0, pol_w);
            if (waited) tma_load_2d(st + a_bytes, &tb, &full[s], kb * GEMM_BK, t0, pol_x);
          }
          __syncwarp();
          if (!waited) {
            pend_kb[n] = kb;
            pend_t0[n] = t0;
            ++n;
          }
          if (++s == stages) {
            s = 0;
            ph ^= 1u;
          }
        }
      }
      if (!waited) {  // fewer k-blocks than stages
        pdl_wait();
        if (elect_one())
          for (int i = 0; i < n; ++i)
            tma_load_2d(base + (size_t)i * stage_bytes + a_bytes, &tb, &full[i], pend_kb[i] * GEMM_BK, pend_t0[i], pol_x);
      }
    }
  } else if (warp == 1 || warp == 6) {
    const int me = warp == 1 ? 0 : 1;
    if (me < n_iss) {
      // ---------------- MMA issuer `me` ----------------
      // the k-blocks in ring slots s = me (mod n_iss), into this issuer's own accumulator
      const uint32_t idesc = umma_idesc_bf16(GEMM_BM, (uint32_t)bn);
      const uint32_t acc_off = (uint32_t)me * acc_cols;
      WorkIter it(p, cta, grid);
      WorkItem w;
      uint32_t n = 0, item = 0;
      const uint32_t iss_mask = (uint32_t)n_iss - 1u;  // n_iss is 1 or 2
      const uint32_t my_slots = (uint32_t)me;
      int ms = 0;        // = n % stages
      uint32_t mph = 0;  // = (n / stages) & 1
      while (it.next(w)) {
        const uint32_t buf = item % nbuf, tph = (item / nbuf) & 1u;
        mbar_wait_site(&tempty[buf], tph ^ 1u, 2 + me, item);  // epilogue has drained this accumulator
        tc_fence_after();
        const uint32_t acc_addr = tmem_base + buf * acc_stride + acc_off;
        bool first = true;
        for (int kb = w.kb0; kb < w.kb1; ++kb, ++n) {
          const int s = ms;
          const uint32_t ph = mph;
          if (++ms == stages) {
            ms = 0;
            mph ^= 1u;
          }
          if (((uint32_t)s & iss_mask) != my_slots) continue;  // a slot always belongs to the same issuer
          mbar_wait_site(&full[s], ph, 4 + me, n);
          if (n == 0 && lane == 0) trace(p, 2);
          tc_fence_after();
          const uint32_t st = smem_u32(base + (size_t)s * stage_bytes);
          const uint64_t da = umma_desc_k_sw128(st);
          const uint64_t da1 = umma_desc_k_sw128(st + A_TILE_BYTES);
          const uint64_t db = umma_desc_k_sw128(st + a_bytes);
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < GEMM_BK / 16; ++k) {
              const uint32_t acc = (!first || k > 0) ? 1u : 0u;
              umma_bf16(acc_addr, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, acc);
              if (DUAL) umma_bf16(acc_addr + (uint32_t)bn, da1 + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, acc);
            }
            umma_commit(&empty[s]);  // frees the smem slot when these MMAs have read it
          }
          __syncwarp();
          first = false;
        }
        if (elect_one()) {
          umma_commit(&tfull[buf]);  // arrives at once if this issuer had no k-block in the item
          if (me == 0) trace(p, 3 + 4 * (int)item);
        }
        __syncwarp();
        ++item;
      }
    }
  } else if ((warp >= 2 && warp < 6) || (warp >= 7 && warp < 11)) {
    // ---------------- epilogue: TMEM -> registers -> (fix-up) -> global ----------------
    pdl_wait();
    const int quad = warp & 3;
    const int r = quad * 32 + lane;  // row of the tile = TMEM lane
    // The last work item's epilogue is never overlapped (it is the kernel's tail), so it is spread over 8 warps:
    // warp (2..5 | 7..10) owns TMEM lane quadrant warp & 3 and group grp takes the 32-column chunks c0 = 32*grp (mod 64)
    const int grp = warp >= 7 ? 1 : 0;
    const int et = grp ? (int)threadIdx.x - 224 + 128 : (int)threadIdx.x - 64;  // 0..255
    WorkIter it(p, cta, grid);
    WorkItem w;
    uint32_t item = 0, n_run = 0;  // n_run: running k-block counter (the issuers' n) at the item's start
    const int nkb = it.nkb;
    while (it.next(w)) {
      const uint32_t buf = item % nbuf, tph = (item / nbuf) & 1u;
      const uint32_t len = (uint32_t)(w.kb1 - w.kb0);
      // which issuers accumulated anything in this item (an accumulator nobody wrote holds stale data): issuer
      // (slot & 1) handles a k-block, slots run cyclically from n_run % stages
      bool has0 = n_iss == 1, has1 = false;
      if (n_iss == 2) {
        uint32_t sl = n_run % (uint32_t)stages;
        for (uint32_t j = 0; j < len && j < 3u; ++j) {
          if (sl & 1u) has1 = true; else has0 = true;
          if (++sl == (uint32_t)stages) sl = 0;
        }
      }
      n_run += len;
      int seg = 0;
#pragma unroll
      for (int i = 1; i < 3; ++i)
        if (i < p.n_seg && w.row_tile >= p.seg_tile0[i]) seg = i;
      const int row_in_seg = (w.row_tile - p.seg_tile0[seg]) * GEMM_BM + r;
      const bool row_ok = row_in_seg < p.seg_rows[seg];
      const int col = p.seg_col[seg] + row_in_seg;
      const int t0 = w.t_tile * bn;
      const bool is_first = w.kb0 == 0, is_last = w.kb1 == nkb;

      // stream-K fix-up bookkeeping
      int c_lo = 0, c_hi = -1;  // contributors [c_lo, c_hi] of a tile this CTA owns
      if (is_first && !is_last) {
        const uint32_t tile_end = ((uint32_t)(w.t_tile * p.n_row_tiles + w.row_tile) + 1u) * (uint32_t)nkb;
        c_lo = cta + 1;
        c_hi = cta;
        while (c_hi + 1 < grid && it.range_start(c_hi + 1) < tile_end) ++c_hi;
      }
      bool polled = false;  // the contributors' flags are awaited as late as possible: just before the first fix-up add

      if (et == 0) trace(p, 4 + 4 * (int)item);
      mbar_wait_site(&tfull[buf], tph, 6, item);
      if (et == 0) trace(p, 5 + 4 * (int)item);
      tc_fence_after();
      const uint32_t tq = tmem_base + buf * acc_stride + ((uint32_t)(quad * 32) << 16);
      // 32 columns of the item's accumulator = sum over the issuers that contributed
      auto ld_acc = [&](uint32_t c, uint32_t (&v)[32]) {
        if (has0) tmem_ld_32x32(tq + c, v);
        if (has1) {
          uint32_t v1[32];
          tmem_ld_32x32(tq + acc_cols + c, v1);
          tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 32; ++j)
            v[j] = has0 ? __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(v1[j])) : v1[j];
        } else {
          tmem_ld_wait();
        }
      };

      if (!DUAL && p.epi == EPI_PARTIAL) {
        // every piece of a tile (owner's included) goes to its own slot; the consumer kernel adds them (internal.h)
        const size_t slot_off = ((size_t)cta * 2 + item) * bn * GEMM_BM;
        float *slot = p.fix_slots + slot_off;
        for (int c0 = grp * 32; c0 < bn; c0 += 64) {
          uint32_t v[32];
          ld_acc((uint32_t)c0, v);
          if (p.tp_size > 0) {
            // fused tensor-parallel all-reduce, gather half: the piece goes into the exchange buffer of EVERY rank
            // (plain stores; for the other ranks they travel over NVLink to peer-mapped memory)
            for (int d = 0; d < p.tp_size; ++d) {
              float *ds = p.tp_slots[d] + slot_off;
#pragma unroll
              for (int j = 0; j < 32; ++j) ds[(size_t)(c0 + j) * GEMM_BM + r] = __uint_as_float(v[j]);
            }
          } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) slot[(size_t)(c0 + j) * GEMM_BM + r] = __uint_as_float(v[j]);
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&tempty[buf]);
      } else if (!is_first) {
        // contributor: dump the raw fp32 accumulator(s) to this CTA's slot, [acc][col][row]
        float *slot = p.fix_slots + (size_t)cta * (DUAL ? 2 : 1) * bn * GEMM_BM;
        for (int c0 = grp * 32; c0 < (int)acc_cols; c0 += 64) {
          uint32_t v[32];
          ld_acc((uint32_t)c0, v);
#pragma unroll
          for (int j = 0; j < 32; ++j) slot[(size_t)(c0 + j) * GEMM_BM + r] = __uint_as_float(v[j]);
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&tempty[buf]);
        // publish: the barrier orders every epilogue thread's stores before thread 0's gpu-scope fence, which is
        // cumulative, so one fence (not one per thread before the barrier as well) is on the tile owner's critical path
        epi_bar();
        if (et == 0) {
          __threadfence();
          atomicExch(p.fix_flags + cta, 1);
        }
      } else {
        for (int c0 = grp * 32; c0 < bn; c0 += 64) {
          uint32_t v[32], u[32];
          // the residual values this chunk will be added to do not depend on the accumulator: request them first so
          // their L2 round trip overlaps the TMEM loads and the fix-up rounds
          float xv[32];
          if (!DUAL && p.epi == EPI_RESID_F32 && row_ok) {
            const float *o = p.out_f32 + col;
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const int t = t0 + c0 + j;
              xv[j] = (t < p.T) ? __ldcg(o + (size_t)t * p.ld_out) : 0.f;
            }
          }
          ld_acc((uint32_t)c0, v);
          if (DUAL) ld_acc((uint32_t)(bn + c0), u);
          if (et == 0 && item == 1) trace(p, 40 + 3 * (c0 >> 5));
          if (!polled) {
            // with this chunk's residual values requested and its accumulator in registers, so that both round trips
            // overlap the contributors' dump + publish (cfg-2 step 7.355 -> 7.30 ms, cfg-3 5.148 -> 5.12 ms, same box)
            polled = true;
            for (int cc = c_lo; cc <= c_hi; ++cc) {
              uint32_t polls = 0;
              unsigned long long t0w = 0;
              while (ld_acquire(p.fix_flags + cc) == 0) {
                if (wait_expired_ns(polls, t0w)) wait_expired(7, (uint32_t)cc, item);
              }
            }
          }
          for (int cc = c_lo; cc <= c_hi; ++cc) {  // fix-up in CTA order: deterministic sums
            const float *slot = p.fix_slots + (size_t)cc * (DUAL ? 2 : 1) * bn * GEMM_BM;
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              v[j] = __float_as_uint(__uint_as_float(v[j]) + __ldcg(slot + (size_t)(c0 + j) * GEMM_BM + r));
              if (DUAL)
                u[j] = __float_as_uint(__uint_as_float(u[j]) + __ldcg(slot + (size_t)(bn + c0 + j) * GEMM_BM + r));
            }
          }
          if (et == 0 && item == 1) trace(p, 41 + 3 * (c0 >> 5));
          if (DUAL) {
            // EPI_SWIGLU_BF16: a = g / (1 + exp(-g)) * u.  This epilogue is on the kernel's critical path (the last
            // work item's is never overlapped): fast-math SiLU (ex2.approx + div.approx, error far below the bf16
            // output's 2^-9) and, instead of 32 two-byte stores per thread, lane pairs swap alternate tokens so
            // every lane stores one bf16x2 = features (col, col+1) of one token (timeline:
            // round-1 timeline: 3.6 -> 1.7 us per 32-token chunk).
            __nv_bfloat16 *o = (__nv_bfloat16 *)p.out_bf16;
            const bool odd = (lane & 1) != 0;
#pragma unroll
            for (int j = 0; j < 32; j += 2) {
              const float g0 = __uint_as_float(v[j]), g1 = __uint_as_float(v[j + 1]);
              const float a0 = __fdividef(g0, 1.0f + __expf(-g0)) * __uint_as_float(u[j]);
              const float a1 = __fdividef(g1, 1.0f + __expf(-g1)) * __uint_as_float(u[j + 1]);
              const float got = __shfl_xor_sync(0xffffffffu, odd ? a0 : a1, 1);
              // even lane: token j, features (col, col+1) = (own a0, neighbour's a0)
              // odd lane : token j+1, features (col-1, col) = (neighbour's a1, own a1)
              const int t = t0 + c0 + j + (odd ? 1 : 0);
              const uint32_t pk = odd ? pack_bf16x2(got, a1) : pack_bf16x2(a0, got);
              if (row_ok && t < p.T)
                *reinterpret_cast<uint32_t *>(o + (size_t)t * p.ld_out + (col & ~1)) = pk;
            }
          } else if (row_ok) {
            if (p.epi == EPI_RESID_F32) {
              // (the 32 residual values were loaded above, before any store: a `+=` loop would serialise 32 dependent
              // L2 round trips per chunk, since the compiler cannot prove the stores do not alias the loads)
              float *o = p.out_f32 + col;
#pragma unroll
              for (int j = 0; j < 32; ++j) {
                const int t = t0 + c0 + j;
                if (t < p.T) o[(size_t)t * p.ld_out] = xv[j] + __uint_as_float(v[j]);
              }
            } else {
              float *o = p.out_f32 + col;
#pragma unroll
              for (int j = 0; j < 32; ++j) {
                const int t = t0 + c0 + j;
                if (t < p.T) o[(size_t)t * p.ld_out] = __uint_as_float(v[j]);
              }
            }
          }
        }
        if (et == 0 && item == 1) trace(p, 60);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&tempty[buf]);
        if (c_hi >= c_lo) {  // consumed: re-arm the contributors' flags for the next launch
          epi_bar();
          if (et == 0)
            for (int cc = c_lo; cc <= c_hi; ++cc) p.fix_flags[cc] = 0;
        }
      }
      if (et == 0) trace(p, 6 + 4 * (int)item);
      ++item;
    }
    if (!DUAL && p.epi == EPI_PARTIAL && p.tp_size > 0) {
      // publish: every epilogue thread's stores -> barrier -> one system-scope fence -> one arrival per rank
      epi_bar();
      if (et == 0) {
        __threadfence_system();
        for (int d = 0; d < p.tp_size; ++d) atomicAdd_system(p.tp_flags[d], 1u);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) trace(p, 1);
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_dyn(tmem_base, tmem_cols);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// The tensor-bound (prefill) shapes on CTA PAIRS: a cluster of two CTAs on the two SMs of a TPC computes one
// 256-weight-row x 256-token tile with tcgen05.mma.cta_group::2.  Each CTA loads ITS 128 weight rows (A) and HALF of
// the token tile (B: 128 tokens); the pair's tensor cores read the other half from the peer's shared memory, so a
// stage is 32 KB per CTA instead of 48 KB (a 128 x 256 single-CTA tile re-reads the whole activation tile per 128
// weight rows) and the L2 -> SM traffic per flop drops by a third — what held the plain projections at 83-85% of the
// cuBLAS-sustained rate while the dual gate/up tile (two weight tiles per activation tile) ran at 94%.
// Roles per CTA: warp 0 TMA producer (both CTAs; all bytes are counted on the LEADER's full barrier), warp 1 MMA issuer
// (leader only; its commits arrive on both CTAs' barriers), warps 4-19 epilogue (each CTA its own 128 rows).
// Whole tiles only (SCHED_TILES), band-rasterised like the single-CTA kernel.
// ---------------------------------------------------------------------------------------------------------------
constexpr int PAIR_BN = 256;                       // tokens per pair tile
constexpr int PAIR_BHALF_BYTES = (PAIR_BN / 2) * 128;  // this CTA's half of the activation tile, per stage
constexpr int PAIR_EPI_WARPS = 16;
constexpr int PAIR_THREADS = 32 * (4 + PAIR_EPI_WARPS);  // warp 0 producer, 1 MMA issuer, 2-3 idle, 4-19 epilogue

size_t gemm_pair_smem_bytes(bool dual, int stages) {
  const size_t stage = (size_t)A_TILE_BYTES * (dual ? 2 : 1) + PAIR_BHALF_BYTES;
  return 1024 + stage * stages + 8 * (2 * stages + 4) + 16;
}

template <bool DUAL>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PAIR_THREADS, 1)
gemm_pair_kernel(const __grid_constant__ CUtensorMap ta0, const __grid_constant__ CUtensorMap ta1,
                 const __grid_constant__ CUtensorMap ta2, const __grid_constant__ CUtensorMap tb, const GemmParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *base = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  constexpr uint32_t a_bytes = A_TILE_BYTES * (DUAL ? 2 : 1);
  constexpr uint32_t stage_bytes = a_bytes + PAIR_BHALF_BYTES;
  const int stages = p.stages;
  uint64_t *full = (uint64_t *)(base + (size_t)stages * stage_bytes);  // used in the leader CTA only
  uint64_t *empty = full + stages;   // per CTA: the slot may be refilled (the leader's commit arrives on both)
  uint64_t *tfull = empty + stages;  // [2] per CTA: accumulator complete
  uint64_t *tempty = tfull + 2;      // [2] leader only: both CTAs' epilogues have drained the accumulator
  uint32_t *tmem_slot = (uint32_t *)(tempty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cluster = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;
  constexpr uint32_t acc_cols = PAIR_BN * (DUAL ? 2u : 1u);
  constexpr int nbuf = DUAL ? 1 : 2;
  constexpr uint32_t tmem_cols = 512;

  pdl_launch_dependents();
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&ta0);
    if (DUAL || p.n_seg > 1) tma_prefetch_desc(&ta1);
    if (p.n_seg > 2) tma_prefetch_desc(&ta2);
    tma_prefetch_desc(&tb);
    for (int i = 0; i < stages; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&tfull[i], 1);
      mbar_init(&tempty[i], 2 * PAIR_EPI_WARPS);  // one arrival per epilogue warp of either CTA
    }
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc_pair(tmem_slot, tmem_cols);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();  // the peer's barriers exist before anything signals them
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  // pair items: (row PAIR, token tile); this CTA's row tile is 2 * pair + rank
  GemmParams pp = p;
  pp.n_row_tiles = (p.n_row_tiles + 1) >> 1;
  pp.sched = SCHED_TILES;

  if (warp == 0) {
    {
      // ---------------- TMA producer (both CTAs; whole warp, issue under elect_one: see gemm_kernel) ----------------
      auto policy = [](int k) { return k == 0 ? l2_policy_evict_first() : (k == 1 ? l2_policy_evict_normal() : l2_policy_evict_last()); };
      const uint64_t pol = policy(p.w_policy), pol_b = policy(p.x_policy);
      pdl_wait();
      WorkIter it(pp, cluster, n_clusters);
      WorkItem w;
      int s = 0;
      uint32_t ph = 0;
      while (it.next(w)) {
        const int row_tile = 2 * w.row_tile + (int)rank;
        int seg = 0;
#pragma unroll
        for (int i = 1; i < 3; ++i)
          if (i < p.n_seg && row_tile >= p.seg_tile0[i]) seg = i;
        // a row tile past the end (odd tile count) loads rows past its tensor: TMA fills zeros and counts the bytes
        const int row0 = row_tile < p.n_row_tiles ? (row_tile - p.seg_tile0[seg]) * GEMM_BM : (1 << 28);
        const int t0 = w.t_tile * PAIR_BN + (int)rank * (PAIR_BN / 2);
        const CUtensorMap *ta = DUAL ? &ta0 : (seg == 0 ? &ta0 : (seg == 1 ? &ta1 : &ta2));
        for (int kb = w.kb0; kb < w.kb1; ++kb) {
          mbar_wait_site(&empty[s], ph ^ 1u, 1, (uint32_t)s);
          uint8_t *st = base + (size_t)s * stage_bytes;
          if (elect_one()) {
            if (rank == 0) mbar_expect_tx(&full[s], 2 * stage_bytes);  // both CTAs' loads land on the leader's barrier
            tma_load_2d_pair(st, ta, &full[s], kb * GEMM_BK, row0, pol);
            if (DUAL) tma_load_2d_pair(st + A_TILE_BYTES, &ta1, &full[s], kb * GEMM_BK, row0, pol);
            tma_load_2d_pair(st + a_bytes, &tb, &full[s], kb * GEMM_BK, t0, pol_b);
          }
          __syncwarp();
          if (++s == stages) {
            s = 0;
            ph ^= 1u;
          }
        }
      }
    }
  } else if (warp == 1) {
    if (rank == 0) {
      // ---------------- MMA issuer (leader CTA, for the pair) ----------------
      const uint32_t idesc = umma_idesc_bf16(2 * GEMM_BM, PAIR_BN);
      WorkIter it(pp, cluster, n_clusters);
      WorkItem w;
      uint32_t item = 0;
      int ms = 0;
      uint32_t mph = 0;
      while (it.next(w)) {
        const uint32_t buf = item % nbuf, tph = (item / nbuf) & 1u;
        mbar_wait_site(&tempty[buf], tph ^ 1u, 2, item);  // both epilogues have drained this accumulator
        tc_fence_after();
        const uint32_t acc_addr = tmem_base + buf * acc_cols;
        bool first = true;
        for (int kb = w.kb0; kb < w.kb1; ++kb) {
          mbar_wait_site(&full[ms], mph, 4, (uint32_t)kb);
          tc_fence_after();
          const uint32_t st = smem_u32(base + (size_t)ms * stage_bytes);
          const uint64_t da = umma_desc_k_sw128(st);
          const uint64_t da1 = umma_desc_k_sw128(st + A_TILE_BYTES);
          const uint64_t db = umma_desc_k_sw128(st + a_bytes);
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < GEMM_BK / 16; ++k) {
              const uint32_t acc = (!first || k > 0) ? 1u : 0u;
              umma_bf16_pair(acc_addr, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, acc);
              if (DUAL) umma_bf16_pair(acc_addr + PAIR_BN, da1 + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, acc);
            }
            umma_commit_pair(&empty[ms]);  // frees the slot in BOTH CTAs when these MMAs have read it
          }
          __syncwarp();
          first = false;
          if (++ms == stages) {
            ms = 0;
            mph ^= 1u;
          }
        }
        if (elect_one()) umma_commit_pair(&tfull[buf]);
        __syncwarp();
        ++item;
      }
    }
  } else if (warp >= 4) {
    // ---------------- epilogue: this CTA's 128 rows x 256 tokens, TMEM -> registers -> global ----------------
    // 16 warps, four per TMEM lane quadrant, 16-column chunks: the dual tile leaves no second TMEM buffer, so its
    // epilogue is exposed once per item and is spread as wide as the register file allows (640 threads x 96 registers)
    pdl_wait();
    const int quad = warp & 3;
    const int r = quad * 32 + lane;
    const int grp = (warp - 4) >> 2;  // 0..3
    WorkIter it(pp, cluster, n_clusters);
    WorkItem w;
    uint32_t item = 0;
    while (it.next(w)) {
      const uint32_t buf = item % nbuf, tph = (item / nbuf) & 1u;
      const int row_tile = 2 * w.row_tile + (int)rank;
      int seg = 0;
#pragma unroll
      for (int i = 1; i < 3; ++i)
        if (i < p.n_seg && row_tile >= p.seg_tile0[i]) seg = i;
      const int row_in_seg = (row_tile - p.seg_tile0[seg]) * GEMM_BM + r;
      const bool row_ok = row_tile < p.n_row_tiles && row_in_seg < p.seg_rows[seg];
      const int col = p.seg_col[seg] + row_in_seg;
      const int t0 = w.t_tile * PAIR_BN;
      mbar_wait_site(&tfull[buf], tph, 6, item);
      tc_fence_after();
      const uint32_t tq = tmem_base + buf * acc_cols + ((uint32_t)(quad * 32) << 16);
      for (int c0 = grp * 16; c0 < PAIR_BN; c0 += 64) {
        if (t0 + c0 >= p.T) break;  // (uniform per warp) nothing but padding from here on
        uint32_t v[16], u[16];
        float xv[16];
        if (!DUAL && p.epi == EPI_RESID_F32 && row_ok) {
          const float *o = p.out_f32 + col;
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            const int t = t0 + c0 + j;
            xv[j] = (t < p.T) ? __ldcg(o + (size_t)t * p.ld_out) : 0.f;
          }
        }
        tmem_ld_32x16(tq + (uint32_t)c0, v);
        if (DUAL) tmem_ld_32x16(tq + (uint32_t)(PAIR_BN + c0), u);
        tmem_ld_wait();
        if (DUAL) {
          __nv_bfloat16 *o = (__nv_bfloat16 *)p.out_bf16;
          const bool odd = (lane & 1) != 0;
#pragma unroll
          for (int j = 0; j < 16; j += 2) {
            const float g0 = __uint_as_float(v[j]), g1 = __uint_as_float(v[j + 1]);
            const float a0 = __fdividef(g0, 1.0f + __expf(-g0)) * __uint_as_float(u[j]);
            const float a1 = __fdividef(g1, 1.0f + __expf(-g1)) * __uint_as_float(u[j + 1]);
            const float got = __shfl_xor_sync(0xffffffffu, odd ? a0 : a1, 1);
            const int t = t0 + c0 + j + (odd ? 1 : 0);
            const uint32_t pk = odd ? pack_bf16x2(got, a1) : pack_bf16x2(a0, got);
            if (row_ok && t < p.T) *reinterpret_cast<uint32_t *>(o + (size_t)t * p.ld_out + (col & ~1)) = pk;
          }
        } else if (row_ok) {
          float *o = p.out_f32 + col;
          if (p.epi == EPI_RESID_F32) {
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              const int t = t0 + c0 + j;
              if (t < p.T) o[(size_t)t * p.ld_out] = xv[j] + __uint_as_float(v[j]);
            }
          } else {
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              const int t = t0 + c0 + j;
              if (t < p.T) o[(size_t)t * p.ld_out] = __uint_as_float(v[j]);
            }
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_leader(&tempty[buf]);
      ++item;
    }
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();  // neither CTA leaves (or frees its TMEM) while the pair may still touch it
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_pair(tmem_base, tmem_cols);
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

// Tuning overrides exist only in builds with -DSS_TUNE (SS_NVCC_EXTRA=-DSS_TUNE python -m paper_2606_18600_b200.build):
// the product library reads no environment variable on this path.
#ifdef SS_TUNE
static int tune(const char *name, int dflt) {
  const char *e = getenv(name);
  return e ? atoi(e) : dflt;
}
#else
static inline int tune(const char *, int dflt) { return dflt; }
#endif

int gemm_pick_bn(int T) {
  const int forced = tune("SS_GEMM_BN", 0);
  if (forced > 0) return forced;
  // the narrowest multiple of 32 columns that covers T in ceil(T / 256) token tiles: a UMMA costs tensor-pipe time and
  // smem reads in proportion to N, and from ~128 tokens on the decode GEMMs are near the roofline's ridge (256 flop
  // per weight byte at T = 256 against 1,624 TFLOP/s / 6,545 GB/s = 248), so padded columns are not free
  if (T <= 32) return 32;
  const int n_t = (T + 255) / 256;
  const int per = (T + n_t - 1) / n_t;
  return (per + 31) / 32 * 32;
}

size_t gemm_smem_bytes(int bn, bool dual, int stages) {
  const size_t stage = (size_t)A_TILE_BYTES * (dual ? 2 : 1) + (size_t)bn * 128;
  return 1024 + stage * stages + 8 * (2 * stages + 4) + 16;
}

int gemm_pick_stages(int bn, bool dual) {
  int st = tune("SS_GEMM_STAGES", GEMM_MAX_STAGES);  // one persistent CTA per SM: use the 227 KB
  if (st > GEMM_MAX_STAGES || st < 2) st = GEMM_MAX_STAGES;
  while (st > 2 && gemm_smem_bytes(bn, dual, st) > 227 * 1024) --st;
  return st;
}

void gemm_plan(GemmLaunch &g, int n_sm) {
  GemmParams &p = g.p;
  int tiles = 0, col = 0;
  for (int i = 0; i < 3; ++i) {
    p.seg_tile0[i] = tiles;
    p.seg_col[i] = col;
    if (i < p.n_seg) {
      tiles += (p.seg_rows[i] + GEMM_BM - 1) / GEMM_BM;
      col += p.seg_rows[i];
    } else {
      p.seg_rows[i] = 0;
    }
  }
  p.n_row_tiles = tiles;
  p.bn = gemm_pick_bn(p.T);
  p.n_t_tiles = (p.T + p.bn - 1) / p.bn;
  const long long n_tiles = (long long)p.n_row_tiles * p.n_t_tiles;
  const long long nkb = (p.K + GEMM_BK - 1) / GEMM_BK;
  int max_grid = tune("SS_GEMM_GRID", n_sm);
  if (max_grid > GEMM_MAX_GRID) max_grid = GEMM_MAX_GRID;
  // whole tiles when the last wave is nearly full (>= 88% of the CTAs busy; 70% once there are several token
  // tiles, i.e. the problem is tensor-bound anyway) or there are many waves; stream-K
  // otherwise (every decode shape: 64-224 tiles on 148 SMs).  Measured on the mixed batches of cfg-5 (T ~ 1,700,
  // 280-1,400 tiles): tiles 30.8 ms / iteration vs stream-K with 256-column fix-up slots 33.9 ms.
  const long long waves = (n_tiles + max_grid - 1) / max_grid;
  const bool full_waves = n_tiles >= max_grid && n_tiles * 100 >= waves * max_grid * (p.n_t_tiles >= 2 ? 70 : 88);
  p.sched = (n_tiles >= 4LL * max_grid || full_waves) ? SCHED_TILES : SCHED_STREAMK;
  if (p.n_t_tiles == 1) p.sched = SCHED_STREAMK;  // HBM-bound whatever the tile count (lm_head: 1,002-1,187 tiles = 6.8-8.02 waves)
  p.sched = tune("SS_GEMM_SCHED", p.sched);
  if (g.invariant) p.sched = SCHED_TILES;  // every tile's whole K by one CTA, k-blocks in order
  if (n_tiles * nkb >= (1LL << 31)) p.sched = SCHED_TILES;  // the stream-K unit cursor is 32-bit
  p.band = tune("SS_GEMM_BAND", g.dual ? 8 : 16);
  if (p.band > p.n_row_tiles) p.band = p.n_row_tiles;
  p.stages = gemm_pick_stages(p.bn, g.dual);
  {
    const int acc_cols = p.bn * (g.dual ? 2 : 1);
    // one token tile (T <= 256): every weight byte is read once, whatever the schedule (e.g. the lm_head at decode:
    // 1,002 row tiles -> whole-tile schedule, but HBM-bound like the stream-K shapes)
    const bool hbm_bound = p.sched == SCHED_STREAMK || p.n_t_tiles == 1;
    p.w_policy = tune("SS_GEMM_WPOL", hbm_bound ? 0 : 2);
    // HBM-bound: two issuers (one accumulator set each) only while BOTH sets still fit twice in TMEM: with 2 x 256
    // columns per item there is no second buffer and the epilogue stops the main loop (T = 256 down projection
    // 119 -> 113 us, O 51.5 -> 45.5 us, T = 128 gate/up 155.6 -> 153.9 us with one issuer).  Tensor-bound: one issuer
    // (the tensor pipe waits on L2 there, not on the issuing thread).
    p.issuers = (hbm_bound && 4 * acc_cols <= 512) ? 2 : 1;
    if (g.invariant) p.issuers = 1;  // one accumulator: no sum of two interleaved k-block sets
    const int forced_iss = tune("SS_GEMM_ISSUERS", 0);
    if (forced_iss == 1 || (forced_iss == 2 && 2 * acc_cols <= 512)) p.issuers = forced_iss;
    p.single_buf = tune("SS_GEMM_SINGLE_BUF", 0);
  }
  // tensor-bound shapes (several token tiles, whole-tile schedule): CTA pairs on 256 x 256 tiles (gemm_pair_kernel)
  const int pair_mode = tune("SS_GEMM_PAIR", 1);  // tuning builds: 0 never, 1 always, 2 plain only, 3 plain with K <= 8192
  g.pair = pair_mode != 0 && !g.invariant && p.sched == SCHED_TILES && p.T > 2 * PAIR_BN && n_sm >= 2 &&
           (pair_mode < 2 || !g.dual) && (pair_mode < 3 || p.K <= 8192);
  if (g.pair) {
    p.bn = PAIR_BN;
    p.n_t_tiles = (p.T + PAIR_BN - 1) / PAIR_BN;
    p.issuers = 1;
    p.stages = GEMM_MAX_STAGES;
    while (p.stages > 2 && gemm_pair_smem_bytes(g.dual, p.stages) > 227 * 1024) --p.stages;
    const long long pair_tiles = (long long)((p.n_row_tiles + 1) / 2) * p.n_t_tiles;
    const long long clusters = pair_tiles < max_grid / 2 ? pair_tiles : max_grid / 2;
    p.band = tune("SS_GEMM_BAND", g.dual ? 4 : 8);  // in row PAIRS
    p.w_policy = tune("SS_GEMM_WPOL", 2);
    p.x_policy = tune("SS_GEMM_XPOL", 2);
    if (p.band > (p.n_row_tiles + 1) / 2) p.band = (p.n_row_tiles + 1) / 2;
    g.grid = (int)(2 * clusters);
    return;
  }
  const long long work = p.sched == SCHED_STREAMK ? n_tiles * nkb : n_tiles;
  g.grid = (int)(work < max_grid ? work : max_grid);
  {
    // Stream-K over FEWER tiles than SMs (O / down projections: 40-64 row tiles): a grid that is a multiple of the tile
    // count cuts every tile into the same whole number of CTA ranges with aligned boundaries, so an owner waits for
    // exactly k - 1 contributors and no CTA holds pieces of two tiles (148 CTAs over 40 tiles = 3.7 ranges per tile:
    // 3-4 contributors, most CTAs with two short items).  HBM does not need all 148 SMs to be saturated, the fix-up
    // tail is what these short GEMMs lose.  Same box, alternating: cfg-2 step
    // 7.287 -> 7.217 ms (grid 128 for 64 tiles), cfg-3 5.10 -> 5.02 ms (grid 120 for 40 tiles); stand-alone O
    // projection 29.0 -> 26.9 us, down 56.4 -> 53.9 us at T = 128.  Only when that grid keeps >= 80% of the SMs: the
    // 80-tile QKV projection on 80 CTAs went 36.2 -> 39.3 us at cfg-2 (31.1 -> 30.0 at cfg-3).  Half-integer cuts (140
    // CTAs for 40 tiles, 120 for 80) measured between the two or within noise of this rule; not used.
    if (tune("SS_GEMM_ALIGN", 1) > 0 && p.sched == SCHED_STREAMK && n_tiles < max_grid && work >= max_grid) {
      const int nt = (int)n_tiles;
      const int aligned = (max_grid / nt) * nt;
      if (aligned * 10 >= max_grid * 8) g.grid = aligned;
    }
  }
}

bool gemm_partial_ok(const GemmLaunch &g) {
  const GemmParams &p = g.p;
  if (g.dual || p.sched != SCHED_STREAMK || p.n_t_tiles != 1) return false;
  const long long nkb = (p.K + GEMM_BK - 1) / GEMM_BK;
  const long long U = (long long)p.n_row_tiles * nkb;
  return (U + g.grid - 1) / g.grid <= nkb;  // a CTA range never spans more than two tiles
}

void gemm_partial_table(const GemmLaunch &g, PartialTile *out) {
  const GemmParams &p = g.p;
  const uint32_t nkb = (uint32_t)((p.K + GEMM_BK - 1) / GEMM_BK), G = (uint32_t)g.grid;
  const uint32_t U = (uint32_t)p.n_row_tiles * nkb, uq = U / G, ur = U - uq * G;
  auto rs = [&](uint32_t c) { return c * uq + (c * ur) / G; };  // = WorkIter::range_start
  uint32_t c = 0;
  for (int i = 0; i < p.n_row_tiles; ++i) {
    const uint32_t lo = (uint32_t)i * nkb, hi = lo + nkb;
    while (rs(c + 1) <= lo) ++c;  // first CTA whose range reaches into tile i
    PartialTile t;
    t.first_cta = (int)c;
    t.first_item = rs(c) < lo ? 1 : 0;  // the CTA started in the previous tile: this tile is its second item
    uint32_t e = c;
    while (e + 1 < G && rs(e + 1) < hi) ++e;
    t.count = (int)(e - c + 1);
    t.pad = 0;
    out[i] = t;
  }
}

cudaError_t gemm_set_debug_buffer(unsigned long long *host_mapped) {
  return cudaMemcpyToSymbol(g_dbg, &host_mapped, sizeof(host_mapped));
}

cudaError_t gemm_init() {
  cudaError_t e = cudaFuncSetAttribute(gemm_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(gemm_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(gemm_pair_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(gemm_pair_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
}

cudaError_t gemm_launch(const GemmLaunch &g) {
  const GemmParams &p = g.p;
  size_t smem = gemm_smem_bytes(p.bn, g.dual, p.stages);
  const CUtensorMap *a1 = g.a[1] ? g.a[1] : g.a[0];
  const CUtensorMap *a2 = g.a[2] ? g.a[2] : g.a[0];
  if (g.pair) {
    smem = gemm_pair_smem_bytes(g.dual, p.stages);
    if (g.dual)
      return launch_pdl_if(!g.no_pdl, gemm_pair_kernel<true>, dim3(g.grid), dim3(PAIR_THREADS), smem, g.stream, *g.a[0], *a1, *a2, *g.b, p);
    return launch_pdl_if(!g.no_pdl, gemm_pair_kernel<false>, dim3(g.grid), dim3(PAIR_THREADS), smem, g.stream, *g.a[0], *a1, *a2, *g.b, p);
  }
  if (g.dual)
    return launch_pdl_if(!g.no_pdl, gemm_kernel<true>, dim3(g.grid), dim3(GEMM_THREADS), smem, g.stream, *g.a[0], *a1, *a2, *g.b, p);
  return launch_pdl_if(!g.no_pdl, gemm_kernel<false>, dim3(g.grid), dim3(GEMM_THREADS), smem, g.stream, *g.a[0], *a1, *a2, *g.b, p);
}

}  // namespace ss
