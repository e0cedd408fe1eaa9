// FP64 FMA microbenchmark: the roofline denominator "measured by an FMA microbenchmark in
// the same run" (BASELINE.json north_star).  Register-resident, 8 independent DFMA chains
// per thread, 1024 threads x 2 CTAs per SM, no memory traffic inside the timed loop.
#include "xt_internal.h"

namespace xt {
namespace {

constexpr int kChains = 8;
constexpr int kInner = 64;  // DFMAs per chain per outer iteration (unrolled)

__global__ void __launch_bounds__(512) fma_peak_kernel(double *out, int outer, double a, double b) {
  double acc[kChains];
#pragma unroll
  for (int k = 0; k < kChains; ++k) acc[k] = static_cast<double>(threadIdx.x + k) * 1e-9;
  for (int it = 0; it < outer; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j) {
#pragma unroll
      for (int k = 0; k < kChains; ++k) acc[k] = fma(acc[k], a, b);
    }
  }
  double sum = 0.0;
#pragma unroll
  for (int k = 0; k < kChains; ++k) sum += acc[k];
  if (sum == 12345.6789) out[0] = sum;  // keeps the chains live; practically never true
}

}  // namespace

int run_fma_peak(double *flops_per_s, double *ms_out, cudaStream_t st) {
  int dev = 0, n_sm = 0;
  XT_CUDA(cudaGetDevice(&dev));
  XT_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  double *d_out = nullptr;
  XT_CUDA(cudaMalloc(&d_out, 8));
  cudaEvent_t e0, e1;
  XT_CUDA(cudaEventCreate(&e0));
  XT_CUDA(cudaEventCreate(&e1));
  const int block = 512, grid = n_sm * 4, outer = 2000;
  // a*x+b with |a|<1 converges to a fixed point: no overflow, no denormals
  fma_peak_kernel<<<grid, block, 0, st>>>(d_out, 50, 0.999, 1e-3);  // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, st);
    fma_peak_kernel<<<grid, block, 0, st>>>(d_out, outer, 0.999, 1e-3);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) {
      cudaFree(d_out);
      return cuda_fail(e, "fma_peak_kernel");
    }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  count_launch(4);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d_out);
  const double n_fma = static_cast<double>(grid) * block * static_cast<double>(outer) * kInner * kChains;
  if (flops_per_s) *flops_per_s = 2.0 * n_fma / (static_cast<double>(best) * 1e-3);
  if (ms_out) *ms_out = best;
  return XT_OK;
}

}  // namespace xt
