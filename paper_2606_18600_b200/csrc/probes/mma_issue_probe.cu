// mma_issue_probe.cu — stand-alone probe (not part of libshuntstage.so): cycles an issuing thread spends per
// tcgen05.mma (M in {64,128}, N in 16..256, K=16, bf16, both operands in smem) and per tcgen05.commit, with 1 or 2
// issuing threads, on 1 or 148 CTAs.  Its output is profiles/r01_mma_issue_microbench.md; it motivated the two MMA
// issuers and the division-free issue loop of gemm_tcgen05.cu.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o mma_issue_probe mma_issue_probe.cu
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
#include "../common.cuh"
using namespace ss;

struct P { int N; int groups; int mma_per_group; int commit_every; int issuers; int M; int same_acc; };

__global__ void __launch_bounds__(128, 1) k(P p, long long *out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *base = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ uint64_t bars[8];
  __shared__ uint64_t fin[2];
  __shared__ uint32_t slot;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int i = threadIdx.x; i < (64 + 64) * 1024 / 4; i += blockDim.x) ((uint32_t *)base)[i] = 0x3c003c00u + i;
  if (threadIdx.x == 0) { for (int i = 0; i < 8; ++i) mbar_init(&bars[i], 1); mbar_init(&fin[0], 1); mbar_init(&fin[1], 1); mbar_fence_init(); }
  if (warp == 0) tmem_alloc_dyn(&slot, 512);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before(); __syncthreads(); tc_fence_after();
  const uint32_t tm = slot;
  if (lane == 0 && warp < p.issuers) {
    const uint32_t idesc = umma_idesc_bf16(p.M, p.N);
    const uint32_t acc = tm + (p.same_acc ? 0 : warp * 256);
    long long t0 = clock64();
    for (int g = 0; g < p.groups; ++g) {
      const uint32_t sa = smem_u32(base + (g & 3) * 16384);
      const uint32_t sb = smem_u32(base + 65536 + (g & 1) * 32768);
      const uint64_t da = umma_desc_k_sw128(sa), db = umma_desc_k_sw128(sb);
      for (int k = 0; k < p.mma_per_group; ++k)
        umma_bf16(acc, da + (uint64_t)((k & 3) * 2), db + (uint64_t)((k & 3) * 2), idesc, (g | k) ? 1u : 0u);
      if (p.commit_every && (g % p.commit_every) == p.commit_every - 1) umma_commit(&bars[(g + warp) & 7]);
    }
    long long t1 = clock64();
    umma_commit(&fin[warp]);
    mbar_wait(&fin[warp], 0);
    long long t2 = clock64();
    if (blockIdx.x == 0) { out[warp * 2] = t1 - t0; out[warp * 2 + 1] = t2 - t0; }
  }
  tc_fence_before(); __syncthreads();
  if (warp == 0) { tc_fence_after(); tmem_dealloc_dyn(tm, 512); }
}

int main() {
  long long *d; cudaMalloc(&d, 64); long long h[4];
  cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  int Ns[] = {16, 32, 64, 128, 256};
  printf("M N mma/grp commit_every issuers grid | issue clk/mma | total clk/mma\n");
  for (int M : {128, 64}) for (int grid : {1, 148}) for (int issuers : {1, 2}) for (int ce : {0, 1, 2}) for (int N : Ns) {
    if (M == 64 && (grid == 1 || issuers == 2)) continue;
    P p{N, 2000, 4, ce, issuers, M, 0};
    k<<<grid, 128, 200 * 1024>>>(p, d);
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { printf("err %s\n", cudaGetErrorString(e)); return 1; }
    cudaMemcpy(h, d, 32, cudaMemcpyDeviceToHost);
    double n = 2000.0 * 4;
    printf("%3d %3d %d %d %d %3d | %7.1f | %7.1f\n", M, N, 4, ce, issuers, grid, h[0] / n, h[1] / n);
  }
  printf("two issuers, N=256, separate vs same accumulator, 8 MMAs per group (per issuer clk/MMA; pipe floor 128 per MMA => 256 when two issuers share the pipe)\n");
  for (int same : {0, 1}) for (int ce : {0, 1}) for (int mpg : {4, 8}) {
    P p{256, 2000, mpg, ce, 2, 128, same};
    k<<<148, 128, 200 * 1024>>>(p, d);
    if (cudaDeviceSynchronize() != cudaSuccess) { printf("err\n"); return 1; }
    cudaMemcpy(h, d, 32, cudaMemcpyDeviceToHost);
    double n = 2000.0 * mpg;
    printf("same_acc=%d commit_every=%d mma/grp=%d | issuer0 %7.1f issuer1 %7.1f (total/MMA)\n", same, ce, mpg, h[1] / n, h[3] / n);
  }
  return 0;
}
