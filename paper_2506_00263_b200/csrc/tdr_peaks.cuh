// tdr_peaks.cuh — two micro-benchmarks behind tdr_measure_peak: the denominators SURVEY 8(d) asks for beside the HBM
// copy peak of MEASURED_PEAKS.json.  The transport path is bound by instruction issue, the fp64 pipe and L2, not by HBM,
// so bench.py quotes its rates against these measured ceilings as well.
#pragma once
#include "tdr_device.cuh"

// fp64: 8 independent DFMA chains per thread, nothing else in the loop
__global__ void __launch_bounds__(256) k_peak_dfma(double *out, int iters, double b, double c) {
  double a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
#pragma unroll 4
  for (int i = 0; i < iters; i++) {
    a0 = __fma_rn(a0, b, c); a1 = __fma_rn(a1, b, c); a2 = __fma_rn(a2, b, c); a3 = __fma_rn(a3, b, c);
    a4 = __fma_rn(a4, b, c); a5 = __fma_rn(a5, b, c); a6 = __fma_rn(a6, b, c); a7 = __fma_rn(a7, b, c);
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

// L2: copy a buffer that fits the 126 MB L2 several times over (read + write bytes counted)
__global__ void __launch_bounds__(256) k_peak_copy(const double2 *__restrict__ src, double2 *__restrict__ dst, size_t n, int reps) {
  for (int r = 0; r < reps; r++)
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}
