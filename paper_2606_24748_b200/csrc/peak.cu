// peak.cu -- measured fp64 FMA peak of the device: the ALU roof beside the HBM roof of the PtAP kernels
// ("report the fp64-pipe fraction beside the HBM fraction, from a measured FMA peak").
//
// Register-resident chains: every thread runs 16 independent fp64 FMA chains for `iters` rounds, enough warps per SM
// to fill the fp64 pipe; nothing touches memory until the final store.  Timed with CUDA events on the caller's stream
// after one warm-up launch; best of 5.  COLD (synchronises).  A second probe does the same with mma.sync m8n8k4 (the
// fp64 tensor-core path the dense GEMM of vcycle_refresh runs on).
#include "internal.h"

namespace bsramg {

__global__ void __launch_bounds__(256)
fp64_fma_chain_kernel(int iters, double seed, double* __restrict__ out) {
  double a[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) a[k] = seed + 1e-3 * (threadIdx.x + k);
  const double m = 1.0 - 1e-9, c = 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = fma(a[k], m, c);
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += a[k];
  if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chains alive
}

// the same for the fp64 tensor-core path: 8 independent m8n8k4 accumulator chains per warp (512 flops per MMA)
__global__ void __launch_bounds__(256)
fp64_mma_chain_kernel(int iters, double seed, double* __restrict__ out) {
  double c[8][2];
#pragma unroll
  for (int t = 0; t < 8; ++t) c[t][0] = c[t][1] = 0.0;
  const double a = seed + threadIdx.x * 1e-6, b = seed - threadIdx.x * 1e-6;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int t = 0; t < 8; ++t)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(c[t][0]), "+d"(c[t][1]) : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int t = 0; t < 8; ++t) s += c[t][0] + c[t][1];
  if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chains alive
}

}  // namespace bsramg

using namespace bsramg;

static int measure_peak(bool mma, double* tflops, void* stream) {
  if (!tflops) return fail(BSR_ERR_NULL, "bsr_measure_fp64_peak: null output");
  *tflops = 0.0;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int grid = sms * 8, block = 256, iters = 4096;
  // flops per thread and round: 16 FMAs, or 8 MMAs of 512 flops shared by the 32 lanes of a warp
  const double flops_per_thread_round = mma ? 8.0 * 512.0 / 32.0 : 2.0 * 16.0;
  double* scratch = nullptr;
  BSR_TRY(dev_alloc_t(&scratch, (size_t)grid * block));
  cudaEvent_t e0, e1;
  CUDA_TRY(cudaEventCreate(&e0));
  CUDA_TRY(cudaEventCreate(&e1));
  double best = 0.0;
  int rc = BSR_OK;
  for (int rep = 0; rep < 6 && rc == BSR_OK; ++rep) {
    cudaEventRecord(e0, st);
    if (mma) fp64_mma_chain_kernel<<<grid, block, 0, st>>>(iters, 1.0, scratch);
    else fp64_fma_chain_kernel<<<grid, block, 0, st>>>(iters, 0.5, scratch);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) {
      rc = fail(BSR_ERR_CUDA, "fp64 peak kernel failed");
      break;
    }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double tf = flops_per_thread_round * iters * (double)grid * block / (ms * 1e-3) / 1e12;
    if (rep > 0 && tf > best) best = tf;   // rep 0 is the warm-up
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  dev_free(scratch);
  *tflops = best;
  return rc;
}

extern "C" int bsr_measure_fp64_peak(double* tflops, void* stream) { return measure_peak(false, tflops, stream); }

extern "C" int bsr_measure_fp64_mma_peak(double* tflops, void* stream) { return measure_peak(true, tflops, stream); }
