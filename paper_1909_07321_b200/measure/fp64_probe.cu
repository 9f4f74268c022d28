// fp64_probe.cu -- register-resident FP64 throughput probes: libpstgf_probe.so, a MEASUREMENT utility that
// bench.py loads beside the product library (it is not part of libpstgf_rmat.so and shares no code with it).
//
// MEASURED_PEAKS.json carries no FP64 entry, so the roofline denominator of the DMMA SYRK kernel
// is measured with these: kind 0 issues DMMA.8x8x4 (mma.sync m8n8k4 f64) in the register-tile
// pattern of the SYRK kernel (8 A x 4 B fragments, 32 accumulator tiles per warp), kind 1 issues
// DFMA on 8 independent chains per thread, kind 2 runs DMMA on even and DFMA on odd warps.  No memory traffic inside the loop; operands depend on the lane so nothing
// folds away, and the accumulators are written to `sink` at the end.
#include <cuda_runtime.h>


namespace {

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// kind 3: ONE accumulator per warp, every DMMA depends on the one before it: elapsed time / (32 iters) is the
// dependent-issue latency of DMMA.8x8x4, which says how many independent accumulators a sub-partition needs in
// flight to fill the pipe (latency / 16 clk).
__global__ void __launch_bounds__(256) probe_chain_kernel(int iters, double *sink) {
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
  double c0 = 0.0, c1 = 0.0;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 32; ++r) dmma(c0, c1, a, b);
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = c0 + c1;
}

template <int KIND>
__global__ void __launch_bounds__(256) probe_kernel(int iters, double *sink) {
  // kind 0: the register tile of the SYRK kernel's OFF path (8 A fragments x 4 B fragments, 32
  // accumulator tiles); kind 1: 8 DFMA chains; kind 2: odd warps DFMA, even warps DMMA.
  const double a0 = 1.0 + 1e-9 * threadIdx.x, b0 = 1.0 - 1e-9 * threadIdx.x;
  const bool tensor = KIND == 0 || (KIND == 2 && ((threadIdx.x >> 5) & 1) == 0);
  double s = 0.0;
  if (tensor) {
    double a[8], b[4], c[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = a0 + i;
#pragma unroll
    for (int j = 0; j < 4; ++j) b[j] = b0 + j;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) c[i][j][0] = c[i][j][1] = 0.0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int i = 0; i < 8; ++i) dmma(c[i][j][0], c[i][j][1], a[i], b[j]);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) s += c[i][j][0] + c[i][j][1];
  } else {
    double f[8];
#pragma unroll
    for (int t = 0; t < 8; ++t) f[t] = 1e-3 * t;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int r = 0; r < 16; ++r)
#pragma unroll
        for (int t = 0; t < 8; ++t) f[t] = fma(f[t], a0, b0);
    }
#pragma unroll
    for (int t = 0; t < 8; ++t) s += f[t];
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

// kind 0 = DMMA.8x8x4 (the instruction the SYRK kernel issues, in its register-tile pattern), 1 = DFMA, 2 = DMMA on
// even warps and DFMA on odd warps, 3 = one dependent DMMA chain per warp (32 DMMAs per iteration: a latency probe).  Launches `blocks` CTAs of `threads` threads (multiple of 32, <= 256) that each
// run `iters` iterations; DEVICE `sink` receives blocks*threads doubles.  HOST `flop_out` (may be NULL) receives
// the FLOPs the launch performs (2 per FMA).  Asynchronous on `stream` (a cudaStream_t): time it with events.
// Returns 0, 1 on bad arguments, 5 when the launch fails.
extern "C" int pstgf_fp64_probe(int kind, int iters, int blocks, int threads, double *sink, double *flop_out,
                                void *stream) {
  if (kind < 0 || kind > 3 || iters < 0 || blocks <= 0 || threads <= 0 || threads > 256 || threads % 32 != 0 || !sink)
    return 1;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (kind == 0) probe_kernel<0><<<blocks, threads, 0, s>>>(iters, sink);
  else if (kind == 1) probe_kernel<1><<<blocks, threads, 0, s>>>(iters, sink);
  else if (kind == 2) probe_kernel<2><<<blocks, threads, 0, s>>>(iters, sink);
  else probe_chain_kernel<<<blocks, threads, 0, s>>>(iters, sink);
  if (cudaGetLastError() != cudaSuccess) return 5;
  if (flop_out) {
    const double warps = (double)blocks * (threads / 32);
    const double per_dmma_warp = (double)iters * 32.0 * 512.0;        // 32 DMMA.8x8x4 (256 FMA each) per iteration
    const double per_dfma_warp = (double)iters * 128.0 * 32.0 * 2.0;  // 128 DFMA per thread per iteration
    const double even = (double)blocks * ((threads / 32 + 1) / 2), odd = warps - even;
    *flop_out = kind == 0 || kind == 3 ? warps * per_dmma_warp : kind == 1 ? warps * per_dfma_warp : even * per_dmma_warp + odd * per_dfma_warp;
  }
  return 0;
}
