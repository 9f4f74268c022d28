// rmat_aux.cuh -- the small kernels beside the persistent one: the pair form's scratch builder and the term-by-term
// verification kernel.  Included by pstgf_rmat.cu only.
#pragma once
#include "rmat_common.h"

namespace pstgf {

// ---- pair form: scratch builder ---------------------------------------------------------------
// P[(n,m)][k] = w_nk * w_mk for the pairs n <= m (no energy in it: once per wave; rows in the order of
// pair_row_channels, which is also recorded in pair_nm) and D[e][k] = 1/(E_k - E_e) (no channel in it), both
// [rows][pair_ld] with k contiguous, which is how the GEMM items' TMA boxes want them.
// Grid (blocks, waves); block b takes the chunks b, b + gridDim.x, ... of PAIR_BUILD_ROWS consecutive rows of the wave's
// n_E + n_pairs rows.  Thread t owns the poles t, t + 256, ...: it loads E_k once per chunk and runs down the chunk's
// rows (independent divisions, coalesced stores along k) -- one row per block and pass left the divisions' latency
// exposed and wrote at a third of the HBM rate (config 7: 600 MB of P and D per step).
constexpr int PAIR_BUILD_ROWS = 16;
template <bool BATCH>
__global__ void __launch_bounds__(256)
pair_build_kernel(const __grid_constant__ DevWave single, const DevWave *__restrict__ waves, int n_waves) {
  __shared__ int s_n[PAIR_BUILD_ROWS], s_m[PAIR_BUILD_ROWS];
  __shared__ double s_E[PAIR_BUILD_ROWS];
  for (int p = blockIdx.y; p < n_waves; p += gridDim.y) {
    const DevWave &w = BATCH ? waves[p] : single;
    if (w.n_pairs <= 0) continue;
    const int K = w.n_poles, C = w.n_chan, N = w.n_E, rows = N + (w.pair_keep_P ? 0 : w.n_pairs);   // D rows, then (unless kept) P rows
    const long long sn = w.tr ? 1 : w.ldw, sk = w.tr ? w.ldw : 1;       // element (n, k) of W at W[n * sn + k * sk]
    for (int r0 = blockIdx.x * PAIR_BUILD_ROWS; r0 < rows; r0 += gridDim.x * PAIR_BUILD_ROWS) {
      const int nr = min(PAIR_BUILD_ROWS, rows - r0);
      __syncthreads();                                           // the previous chunk's tables have been read
      if ((int)threadIdx.x < nr) {
        const int row = r0 + threadIdx.x;
        if (row < N) {
          s_E[threadIdx.x] = __ldg(w.energies + row);
        } else {
          int n, m;
          pair_row_channels(row - N, C, n, m);                   // O(n_chan) integer steps, once per row
          s_n[threadIdx.x] = n;
          s_m[threadIdx.x] = m;
          const_cast<unsigned int *>(w.pair_nm)[row - N] = (unsigned int)n | ((unsigned int)m << 16);
        }
      }
      __syncthreads();
      const int n_d = max(0, min(nr, N - r0));                   // rows [0, n_d) of the chunk are rows of D, the rest rows of P
      for (int k = threadIdx.x; k < K; k += blockDim.x) {
        if (n_d > 0) {
          const double ek = __ldg(w.E_k + k);
          double *d = w.pair_D + (size_t)r0 * w.pair_ld + k;
#pragma unroll 4
          for (int i = 0; i < n_d; ++i) d[(size_t)i * w.pair_ld] = 1.0 / (ek - s_E[i]);
        }
        for (int i = n_d; i < nr; ++i) {
          const double *wn = w.W + (size_t)s_n[i] * sn, *wm = w.W + (size_t)s_m[i] * sn;
          w.pair_P[(size_t)(r0 + i - N) * w.pair_ld + k] = __dmul_rn(wn[(size_t)k * sk], wm[(size_t)k * sk]);
        }
      }
    }
  }
}

// ---- verification kernel: eq. 4 term by term, one thread per R element ----------------------
__global__ void rmat_naive_kernel(const double *__restrict__ W, long long stride_n, long long stride_k,
                                  const double *__restrict__ E_k, const double *__restrict__ energies, int n_chan,
                                  int n_poles, long long n_elems, double a, const double *__restrict__ diag_add,
                                  double *__restrict__ R_out) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_elems) return;
  const long long cc = (long long)n_chan * n_chan;
  const long long e = idx / cc;
  const int rem = (int)(idx - e * cc);
  const int n = rem / n_chan, m = rem - n * n_chan;
  const double E = energies[e];
  const double *wn = W + (size_t)n * stride_n, *wm = W + (size_t)m * stride_n;
  double s = 0.0, c = 0.0;
  for (int k = 0; k < n_poles; ++k) {
    const double t = __ddiv_rn(__dmul_rn(wn[(size_t)k * stride_k], wm[(size_t)k * stride_k]), __dsub_rn(E_k[k], E));
    const double u = __dadd_rn(s, t);
    c = __dadd_rn(c, fabs(s) >= fabs(t) ? __dadd_rn(__dsub_rn(s, u), t) : __dadd_rn(__dsub_rn(t, u), s));
    s = u;
  }
  double r = __ddiv_rn(__dadd_rn(s, c), __dmul_rn(2.0, a));
  if (diag_add != nullptr && n == m) r = __dadd_rn(r, diag_add[e * n_chan + n]);
  R_out[idx] = r;
}

}  // namespace pstgf
