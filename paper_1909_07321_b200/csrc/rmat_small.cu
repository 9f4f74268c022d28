// rmat_small.cu -- eq. 4 for a TINY partial wave in one launch with no scratch and no ring.
//
// A wave with at most SMALL_MAX_CHAN channels and little work in all (BASELINE.json configs[0]: 8 channels, 160 poles,
// 1000 energies: 10 MFLOP, 0.3 us of the FP64 pipe) is bound by latencies, not by throughput: the persistent kernel's
// two launches (scratch builder + GEMM items), its mbarrier ring and its 128-energy items cost 27 us for it.  This
// kernel evaluates the SAME pair form, term for term and in the same order,
//     R[e][(n,m)] = (1/2a) sum_k P[(n,m)][k] * D[e][k],   P = rn(w_nk w_mk),   D = rn(1 / (E_k - E_e)),
// with one CTA per block of 8 energies: the CTA's warps first build D for the block's 8 energies in shared memory
// (every division done once, all of them independent) beside a copy of W, then each warp takes a few blocks of 8
// pairs and runs their DMMA chains, forming the products P in registers from the rows of W.  The operands of every
// DMMA, their lane positions and the order of the k-steps are those of a pair item of the persistent kernel
// (rmat_kernel.cuh consume_pair), so the result is bitwise the same and the choice between the two is one of speed
// alone.
#include "rmat_launch.h"
#include "rmat_common.h"

namespace pstgf {

namespace {

constexpr int SMALL_KC = 160;              // poles per chunk held in shared memory
constexpr int SMALL_PITCH = SMALL_KC + 4;  // == 4 (mod 16) doubles: conflict-free LDS.64 fragment loads

__device__ __forceinline__ void dmma884_small(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// NPBW: blocks of 8 pairs per MMA warp.  blockDim.x = 2 * 32 * ceil(pair blocks / NPBW): the first half of the CTA's
// warps run the DMMA chains, all of them stage W and build D (a launch this short is bound by instruction latencies:
// twice the warps halve each thread's loads and divisions and give the schedulers something to switch to).
// gridDim.x = ceil(n_E / 8).
template <int NPBW>
__global__ void __launch_bounds__(64 * SMALL_MAX_WARPS)
rmat_small_kernel(const __grid_constant__ DevWave w) {
  __shared__ double sW[SMALL_MAX_CHAN * SMALL_PITCH];
  __shared__ double sD[8 * SMALL_PITCH];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, q = lane & 3;
  const int C = w.n_chan, K = w.n_poles, N = w.n_E;
  const int n_pairs = C * (C + 1) / 2;
  const int e0 = blockIdx.x * 8;
  const long long sn = w.tr ? 1 : w.ldw, sk = w.tr ? w.ldw : 1;   // element (n, k) of W at W[n * sn + k * sk]
  const int hs = blockDim.x >> 1;                                  // threads per half
  const int hh = threadIdx.x >= hs ? 1 : 0, tt = threadIdx.x - hh * hs;
  const bool mma_warp = hh == 0;

  int offn[NPBW], offm[NPBW], pn[NPBW], pm[NPBW];
  double acc[NPBW][2];
#pragma unroll
  for (int b = 0; b < NPBW; ++b) acc[b][0] = acc[b][1] = 0.0;

  for (int k0 = 0; k0 < K; k0 += SMALL_KC) {
    const int kc = min(SMALL_KC, K - k0), kc4 = (kc + 3) & ~3;
    if (k0 > 0) __syncthreads();                       // the previous chunk has been consumed
    // Every global load of the chunk is issued before the first one is used, and nothing is computed ahead of them:
    // thread (hh, tt) takes the poles k = tt, tt + hs, ... and of each the channels n = hh, hh + 2, ... and the
    // energies 4 hh .. 4 hh + 3 (no index divisions; with 160 poles and 8 channels: 4 + 1 + 4 loads per thread).
    double en[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) en[j] = e0 + 4 * hh + j < N ? __ldg(w.energies + e0 + 4 * hh + j) : 0.0;
    for (int k = tt; k < kc4; k += hs) {
      const bool kin = k < kc;
      const double ek = kin ? __ldg(w.E_k + k0 + k) : 0.0;
      double v[SMALL_MAX_CHAN / 2];
#pragma unroll
      for (int j = 0; j < SMALL_MAX_CHAN / 2; ++j) {
        const int n = hh + 2 * j;
        v[j] = (kin && n < C) ? __ldg(w.W + (size_t)n * sn + (size_t)(k0 + k) * sk) : 0.0;
      }
#pragma unroll
      for (int j = 0; j < SMALL_MAX_CHAN / 2; ++j)
        if (hh + 2 * j < C) sW[(hh + 2 * j) * SMALL_PITCH + k] = v[j];      // zero beyond n_poles
      // D[e][k] = 1 / (E_k - E_e) (IEEE division), zero beyond n_poles and beyond n_E
#pragma unroll
      for (int j = 0; j < 4; ++j)
        sD[(4 * hh + j) * SMALL_PITCH + k] = (kin && e0 + 4 * hh + j < N) ? 1.0 / (ek - en[j]) : 0.0;
    }
    if (k0 == 0 && mma_warp) {
      // (while the loads are in flight) the pairs of this lane's rows: row 8 (warp NPBW + b) + g of P, in the pair
      // order of the persistent kernel
#pragma unroll
      for (int b = 0; b < NPBW; ++b) {
        const int r = (warp * NPBW + b) * 8 + g;
        int n = 0, m = 0;
        if (r < n_pairs) pair_row_channels(r, C, n, m);
        pn[b] = r < n_pairs ? n : -1;
        pm[b] = m;
        offn[b] = n * SMALL_PITCH + q;
        offm[b] = m * SMALL_PITCH + q;
      }
    }
    __syncthreads();
    if (mma_warp) {
      const double *bp = sD + g * SMALL_PITCH + q;
#pragma unroll 4
      for (int ks = 0; ks < kc4 / 4; ++ks) {
        const double bfrag = bp[ks * 4];
#pragma unroll
        for (int b = 0; b < NPBW; ++b) {
          const double a = __dmul_rn(sW[offn[b] + ks * 4], sW[offm[b] + ks * 4]);   // P[(n,m)][k] = w_nk w_mk
          dmma884_small(acc[b][0], acc[b][1], a, bfrag);
        }
      }
    }
  }
  if (!mma_warp) return;
  // epilogue: this lane holds pair rows 8 (warp NPBW + b) + g at energies e0 + 2 q + {0, 1}
  const size_t cc = (size_t)C * C;
#pragma unroll
  for (int b = 0; b < NPBW; ++b) {
    const int n = pn[b], m = pm[b];
    if (n < 0) continue;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int e = e0 + 2 * q + h;
      if (e >= N) continue;
      double v = acc[b][h] * w.inv2a;
      if (n == m && w.diag_add) v += __ldg(w.diag_add + (size_t)e * C + n);
      double *R = w.R_out + (size_t)e * cc;
      __stcs(R + (size_t)n * C + m, v);
      if (n != m) __stcs(R + (size_t)m * C + n, v);
    }
  }
}

}  // namespace

cudaError_t small_launch(const DevWave &w, cudaStream_t s) {
  const int n_pb = (w.n_chan * (w.n_chan + 1) / 2 + 7) / 8;           // blocks of 8 pairs: at most 17
  const int npbw = (n_pb + SMALL_MAX_WARPS - 1) / SMALL_MAX_WARPS;    // 1, 2 or 3
  const int warps = (n_pb + npbw - 1) / npbw;
  const dim3 grid((unsigned)((w.n_E + 7) / 8)), block((unsigned)(64 * warps));
  switch (npbw) {
    case 1: rmat_small_kernel<1><<<grid, block, 0, s>>>(w); break;
    case 2: rmat_small_kernel<2><<<grid, block, 0, s>>>(w); break;
    default: rmat_small_kernel<3><<<grid, block, 0, s>>>(w); break;
  }
  return cudaGetLastError();
}

}  // namespace pstgf
