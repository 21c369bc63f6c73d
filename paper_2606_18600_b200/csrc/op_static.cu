// op_static.cu — ss_op_gemm_bf16_static: the op-level tcgen05 GEMM for callers that may not allocate device memory
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same kernel and same launch
// plan as ss_op_gemm_bf16 (stage.cu: op_gemm); the only difference is where the stream-K fix-up scratch lives: in a
// file-scope __device__ array of a fixed, stated size instead of a buffer the caller allocates.
//
// The array costs SS_OP_GEMM_STATIC_SCRATCH_BYTES (16 MiB + 1 KiB) of device memory on every GPU that loads the
// library, from load until exit.  It is sized for T <= SS_OP_GEMM_STATIC_MAX_T = 128 tokens (the decode batches of
// BASELINE.json's configs): one fix-up slot of bn x 128 fp32 (bn <= 128) per persistent CTA, at most GEMM_MAX_GRID = 256
// CTAs, behind 1 KiB of flags.  Larger T is refused (SS_ERR_CAPACITY), never clipped.
//
// Every call shares the one array, and the array keeps what the last call left in it:
//   * the flags must be zero when the kernel starts; the kernel leaves them zero, but a call that was aborted would
//     not, so each call clears them with a 1 KiB memset node on the caller's stream, ahead of the kernel;
//   * the slots need no clearing: a slot is written in full by its contributor CTA before the flag that publishes it;
//   * two calls that overlap on the GPU (different streams, several host threads, a captured graph launched while
//     another call is in flight) RACE on the flags and slots.  Serialise them on one stream or with events.
//
// In host code the array's NAME is a host-side stand-in, not a device address: passing it to a kernel faults (or, where
// the GPU can reach host memory, silently uses the wrong memory).  The device address is taken once per device, with
// that device current, by cudaGetSymbolAddress, and it is that pointer that goes into the kernel's parameters.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <cstring>
#include <mutex>

#include "../../include/shuntstage.h"
#include "internal.h"

namespace ss {

static_assert(SS_OP_GEMM_STATIC_MAX_T == 128, "the scratch array is sized for bn <= 128");
constexpr size_t STATIC_SLOT_BYTES = (size_t)SS_OP_GEMM_STATIC_MAX_T * GEMM_BM * sizeof(float);  // 64 KiB per CTA
constexpr size_t STATIC_SCRATCH_BYTES = GEMM_FIX_FLAG_BYTES + (size_t)GEMM_MAX_GRID * STATIC_SLOT_BYTES;
static_assert(STATIC_SCRATCH_BYTES == SS_OP_GEMM_STATIC_SCRATCH_BYTES, "include/shuntstage.h states this size");

// [flags: GEMM_MAX_GRID ints | slots: GEMM_MAX_GRID x (bn x 128 fp32)]; zero-initialised when the module is loaded
static __device__ __align__(256) unsigned char g_gemm_static_scratch[STATIC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
static std::mutex g_setup_mutex;
static void *g_scratch_dev[MAX_DEVICES];  // device address of the array on device i; nullptr = not set up yet

// Set-up, once per device, with that device current: the array's device address.  No allocation: the array came with
// the module.  Returns cudaSuccess and *out, or the error of cudaGetDevice / cudaGetSymbolAddress.
static cudaError_t static_scratch(void **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_dev[dev]) {
    void *ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_gemm_static_scratch);
    if (e != cudaSuccess) return e;
    if (!ptr || ((uintptr_t)ptr & 255)) return cudaErrorInvalidSymbol;
    g_scratch_dev[dev] = ptr;
  }
  *out = g_scratch_dev[dev];
  return cudaSuccess;
}

}  // namespace ss

using namespace ss;

extern "C" int ss_op_gemm_bf16_static(const void *x_dev, const void *w_dev, float *c_dev, int T, int N, int K,
                                      void *cuda_stream) {
  if (!x_dev || !w_dev || !c_dev || T <= 0 || N <= 0 || K <= 0) return SS_ERR_INVALID_ARG;
  if (K % 8 != 0 || ((uintptr_t)x_dev & 15) || ((uintptr_t)w_dev & 15)) return SS_ERR_UNSUPPORTED;
  if (T > SS_OP_GEMM_STATIC_MAX_T)
    return note_error(SS_ERR_CAPACITY, "ss_op_gemm_bf16_static: T exceeds SS_OP_GEMM_STATIC_MAX_T (128); "
                                       "use ss_op_gemm_bf16 with caller-owned scratch");
  cudaError_t e = gemm_init();  // function attributes only
  if (e != cudaSuccess) return note_cuda_error(e, "gemm_init");
  int dev = 0, n_sm = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return note_cuda_error(e, "cudaGetDevice");
  if ((e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
    return note_cuda_error(e, "cudaDeviceGetAttribute");
  void *scratch = nullptr;
  if ((e = static_scratch(&scratch)) != cudaSuccess) return note_cuda_error(e, "cudaGetSymbolAddress(g_gemm_static_scratch)");

  CUtensorMap ta, tb;
  GemmLaunch g;
  memset(&g, 0, sizeof(g));
  GemmParams &p = g.p;
  p.n_seg = 1;
  p.seg_rows[0] = N;
  p.T = T;
  p.K = K;
  p.epi = EPI_F32;
  p.ld_out = N;
  p.out_f32 = c_dev;
  p.fix_flags = (int *)scratch;
  p.fix_slots = (float *)((uint8_t *)scratch + GEMM_FIX_FLAG_BYTES);
  g.dual = false;
  g.no_pdl = true;  // as op_gemm: the caller's operands may come straight out of a preceding kernel
  g.stream = (cudaStream_t)cuda_stream;
  gemm_plan(g, n_sm);
  // the plan must fit the array: one slot of bn x 128 fp32 per CTA (T <= 128 gives bn <= 128, one token tile, no pairs)
  if (g.pair || g.grid > GEMM_MAX_GRID || (size_t)p.bn * GEMM_BM * sizeof(float) > STATIC_SLOT_BYTES)
    return note_error(SS_ERR_CAPACITY, "ss_op_gemm_bf16_static: the launch plan does not fit the static scratch");
  if (make_tmap_bf16_2d(&ta, w_dev, (uint64_t)N, (uint64_t)K, GEMM_BM, true) != 0 ||
      make_tmap_bf16_2d(&tb, x_dev, (uint64_t)T, (uint64_t)K, (uint32_t)p.bn, false) != 0)
    return note_error(SS_ERR_CUDA, "cuTensorMapEncodeTiled failed");
  g.a[0] = &ta;
  g.b = &tb;
  // the flags must start at zero whatever the previous call left (a memset node: nothing is allocated)
  if ((e = cudaMemsetAsync(scratch, 0, GEMM_FIX_FLAG_BYTES, g.stream)) != cudaSuccess)
    return note_cuda_error(e, "cudaMemsetAsync(flags)");
  if ((e = gemm_launch(g)) != cudaSuccess) return note_cuda_error(e, "gemm_launch");
  return SS_OK;
}
