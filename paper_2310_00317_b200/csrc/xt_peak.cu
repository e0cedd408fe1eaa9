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

// Operand-pattern probes: the same DFMA count with the operand shapes
// of the tracking arithmetic.  pattern 1: acc = fma(acc, x_i, y_i), three distinct registers
// per instruction; pattern 2: the complex Horner recurrence for 4 particles per thread with
// the coefficients broadcast from shared memory (no lattice, no dispatch).
__global__ void __launch_bounds__(512) fma_distinct_kernel(double *out, int outer, double a, double b) {
  double acc[kChains], x[kChains], y[kChains];
#pragma unroll
  for (int k = 0; k < kChains; ++k) {
    acc[k] = static_cast<double>(threadIdx.x + k) * 1e-9;
    x[k] = a + 1e-6 * k + 1e-9 * threadIdx.x;
    y[k] = b + 1e-7 * k + 1e-10 * threadIdx.x;
  }
  for (int it = 0; it < outer; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j) {
#pragma unroll
      for (int k = 0; k < kChains; ++k) acc[k] = fma(acc[k], x[k], y[k]);
    }
  }
  double sum = 0.0;
#pragma unroll
  for (int k = 0; k < kChains; ++k) sum += acc[k] + x[k] + y[k];
  if (sum == 12345.6789) out[0] = sum;
}

__global__ void __launch_bounds__(512) horner_probe_kernel(double *out, int outer, double a, double b) {
  constexpr int P = 4, kCoef = 64;
  __shared__ double2 cs[kCoef];
  if (threadIdx.x < kCoef) cs[threadIdx.x] = make_double2(1e-9 * threadIdx.x, -1e-9 * threadIdx.x);
  __syncthreads();
  double re[P], im[P], x[P], y[P];
#pragma unroll
  for (int j = 0; j < P; ++j) {
    re[j] = 1e-3 * j;
    im[j] = 2e-3 * j;
    x[j] = a * 1e-3 + 1e-9 * threadIdx.x + 1e-6 * j;
    y[j] = b + 1e-9 * threadIdx.x - 1e-6 * j;
  }
  for (int it = 0; it < outer; ++it) {
#pragma unroll 4
    for (int k = 0; k < kCoef; ++k) {
      const double2 c = cs[k];
#pragma unroll
      for (int j = 0; j < P; ++j) {
        const double nre = fma(re[j], x[j], fma(-im[j], y[j], c.x));
        const double nim = fma(re[j], y[j], fma(im[j], x[j], c.y));
        re[j] = nre;
        im[j] = nim;
      }
    }
  }
  double sum = 0.0;
#pragma unroll
  for (int j = 0; j < P; ++j) sum += re[j] + im[j];
  if (sum == 12345.6789) out[0] = sum;
}

}  // namespace

int run_fma_peak(double *flops_per_s, double *ms_out, int pattern, cudaStream_t st) {
  if (pattern < 0 || pattern > 2) {
    set_error("xt_fp64_fma_probe: pattern must be 0 (shared operands), 1 (distinct operands) or 2 (Horner)");
    return XT_ERR_INVALID_ARG;
  }
  int dev = 0, n_sm = 0;
  XT_CUDA(cudaGetDevice(&dev));
  XT_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  double *d_out = nullptr;
  XT_CUDA(cudaMalloc(&d_out, 8));
  cudaEvent_t e0, e1;
  XT_CUDA(cudaEventCreate(&e0));
  XT_CUDA(cudaEventCreate(&e1));
  const int block = 512, grid = n_sm * 4;
  const int outer = pattern == 2 ? 1000 : 2000;
  auto launch = [&](int n_outer) {
    // a*x+b with |a|<1 converges to a fixed point: no overflow, no denormals
    if (pattern == 0) fma_peak_kernel<<<grid, block, 0, st>>>(d_out, n_outer, 0.999, 1e-3);
    if (pattern == 1) fma_distinct_kernel<<<grid, block, 0, st>>>(d_out, n_outer, 0.999, 1e-3);
    if (pattern == 2) horner_probe_kernel<<<grid, block, 0, st>>>(d_out, n_outer, 0.999, 1e-3);
  };
  launch(50);  // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, st);
    launch(outer);
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
  const double per_thread = pattern == 2 ? 64.0 * 16.0 : static_cast<double>(kInner) * kChains;
  const double n_fma = static_cast<double>(grid) * block * static_cast<double>(outer) * per_thread;
  if (flops_per_s) *flops_per_s = 2.0 * n_fma / (static_cast<double>(best) * 1e-3);
  if (ms_out) *ms_out = best;
  return XT_OK;
}

}  // namespace xt
