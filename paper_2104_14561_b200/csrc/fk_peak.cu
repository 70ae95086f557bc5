// fk_peak.cu -- measurement only: the fp64 fused-multiply-add rate of the device, the roof the
// row contraction is held against when it, not HBM, bounds a kernel
// (include/fk.h fk_peak_fp64; bench.py prints the derivation).
#include "fk_internal.h"

namespace {

// 8 independent dependent-chains per thread: enough to cover the DFMA latency (8 cycles) at
// 16 warps per SM sub-partition; a and b are runtime values so nothing folds away
__global__ void __launch_bounds__(512)
fk_dfma_peak(double* __restrict__ out, int iters, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5,
         x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

}  // namespace

cudaError_t fk_launch_dfma_peak(double* out, int blocks, int threads, int iters, cudaStream_t s) {
  fk_dfma_peak<<<blocks, threads, 0, s>>>(out, iters, 1.0000001, 1e-9);
  return cudaGetLastError();
}
