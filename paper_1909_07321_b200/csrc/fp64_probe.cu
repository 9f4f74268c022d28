// fp64_probe.cu -- register-resident FP64 throughput probes (include/pstgf_rmat.h, "measurement").
//
// MEASURED_PEAKS.json carries no FP64 entry, so the roofline denominator of the DMMA SYRK kernel
// is measured with these: kind 0 issues DMMA.8x8x4 (mma.sync m8n8k4 f64) on 16 independent
// accumulator tiles per warp, kind 1 issues DFMA on 8 independent chains per thread, kind 2
// interleaves both.  No memory traffic inside the loop; operands depend on the lane so nothing
// folds away, and the accumulators are written to `sink` at the end.
#include <cuda_runtime.h>

#include "../../include/pstgf_rmat.h"

namespace {

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

template <int KIND>
__global__ void __launch_bounds__(1024) probe_kernel(int iters, double *sink) {
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
  double c[16][2];
  double f[8];
#pragma unroll
  for (int t = 0; t < 16; ++t) c[t][0] = c[t][1] = 0.0;
#pragma unroll
  for (int t = 0; t < 8; ++t) f[t] = 1e-3 * t;
  for (int it = 0; it < iters; ++it) {
    if (KIND == 0 || KIND == 2) {
#pragma unroll
      for (int t = 0; t < 16; ++t) dmma(c[t][0], c[t][1], a, b);
    }
    if (KIND == 1 || KIND == 2) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int t = 0; t < 8; ++t) f[t] = fma(f[t], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int t = 0; t < 16; ++t) s += c[t][0] + c[t][1];
#pragma unroll
  for (int t = 0; t < 8; ++t) s += f[t];
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

extern "C" pstgf_status_t pstgf_fp64_probe(int kind, int iters, int blocks, int threads, double *sink,
                                           double *flop_out, void *stream) {
  if (kind < 0 || kind > 2 || iters < 0 || blocks <= 0 || threads <= 0 || threads > 1024 || threads % 32 != 0 || !sink)
    return PSTGF_ERR_INVALID_VALUE;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (kind == 0) probe_kernel<0><<<blocks, threads, 0, s>>>(iters, sink);
  else if (kind == 1) probe_kernel<1><<<blocks, threads, 0, s>>>(iters, sink);
  else probe_kernel<2><<<blocks, threads, 0, s>>>(iters, sink);
  if (cudaGetLastError() != cudaSuccess) return PSTGF_ERR_CUDA;
  if (flop_out) {
    const double warps = (double)blocks * (threads / 32);
    double flop = 0.0;
    if (kind == 0 || kind == 2) flop += warps * iters * 16.0 * 512.0;          // DMMA.8x8x4 = 256 FMA
    if (kind == 1 || kind == 2) flop += warps * 32.0 * iters * 32.0 * 2.0;     // 32 DFMA per thread per iteration
    *flop_out = flop;
  }
  return PSTGF_OK;
}
