// rmat_sliced.cu -- pstgf_rmat_form_sliced: eq. 4 evaluated on the INT8 tensor pipe of sm_100a
// (tcgen05.mma kind::i8, INT32 accumulators in tensor memory) by slicing both operands into signed 7-bit digits
// ("FP64-accurate emulation on the INT8 tcgen05 pipes").  A VARIANT beside the DMMA path, never the
// default: its results are not IEEE FP64 sums (they agree with them to ~1e-12 of max|R| with 7 slices, 1e-14 with 8).
//
//   R_nm(E) = 1/(2a) sum_k a_nk b_mk,   a_nk = w_nk,   b_mk = w_mk / (E_k - E)            (eq. 4)
//   a_nk = sA_n sum_i dA_i[n][k] 2^(-6-7i),   b_mk = sB_m sum_j dB_j[m][k] 2^(-6-7j)       (digits in [-64, 64],
//                                                                  sA, sB powers of two: the row maxima rounded up)
//   sum_k a_nk b_mk ~= sA_n sB_m sum_{t < S} 2^(-12-7t) ACC_t[n][m],   ACC_t = sum_{i+j=t} dA_i dB_j^T   (exact in INT32
//                                                                  for n_poles (t + 1) < 2^19: |digit product| <= 2^12)
// Three kernels per call: slice_kernel over W (once), slice_kernel over W diag(1/(E_k - E_e)) for a chunk of energies,
// and sliced_gemm_kernel, in which one thread streams the digit tiles in by TMA (64-byte swizzle), one thread issues
// the S (S + 1) / 2 integer MMAs per k-step into S accumulators of 128 x 64 in TMEM, and four warps read the accumulators
// back (tcgen05.ld), fold them in FP64 (Horner in 2^-7), scale and store the upper triangle and its mirror.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <cfloat>
#include <cmath>
#include <mutex>

#include "../../include/pstgf_rmat.h"
#include "rmat_launch.h"

namespace {

constexpr int SL_MAX = 8;            // slices per operand, at most
constexpr int TILE_M = 128;          // rows of an output tile (channels n, digits of A = W)
constexpr int TILE_N = 64;           // columns of an output tile (channels m, digits of B = W diag(d_e))
constexpr int KB = 64;               // poles (bytes) per k-block: one 64-byte swizzle row
constexpr int UMMA_K = 32;           // poles per tcgen05.mma kind::i8
constexpr int STAGES = 2;
constexpr int GEMM_THREADS = 192;    // warp 0 TMA, warp 1 MMA, warps 2..5 epilogue (TMEM lane quadrants 2, 3, 0, 1)

__host__ __device__ inline long long round_up(long long x, long long m) { return (x + m - 1) / m * m; }

// ---- slicing -----------------------------------------------------------------------------------
// One block per (row, energy).  x_k = W[row][k] * d_k with d_k = 1 / (E_k - E) (B operand) or 1 (A operand, E_k null).
// Pass 1: the row maximum -> scale s = 2^(floor(log2 max) + 1), so that |x / s| < 1.  Pass 2: S digits per element,
// r = x / s * 64, d_0 = rint(r), r = (r - d_0) * 128, ... (every step exact in FP64), four poles per thread so that a
// slice row is written in 32-bit words.  Rows beyond n_chan and poles beyond n_poles are zero digits.
// CACHE: the row's x_k are kept in (dynamic) shared memory between the passes, so that every division is done once.
template <bool CACHE>
__global__ void __launch_bounds__(256) slice_kernel(const double *__restrict__ W, long long ldw, const double *__restrict__ E_k,
                                                    const double *__restrict__ energies, int n_chan, int n_poles, int S,
                                                    long long Cp, long long Kp, int8_t *__restrict__ digits, double *__restrict__ scales) {
  extern __shared__ double xrow[];
  const int row = blockIdx.x, e = blockIdx.y;
  __shared__ double red[256];
  const bool in_row = row < n_chan;
  const double E = E_k ? energies[e] : 0.0;
  const double *w = W + (size_t)row * ldw;
  double m = 0.0;
  if (in_row)
    for (int k = threadIdx.x; k < n_poles; k += blockDim.x) {
      const double x = E_k ? w[k] * (1.0 / (E_k[k] - E)) : w[k];
      if (CACHE) xrow[k] = x;
      m = fabs(x) <= DBL_MAX ? fmax(m, fabs(x)) : INFINITY;       // inf or NaN (an energy on a pole): fmax alone would drop a NaN
    }
  red[threadIdx.x] = m;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) red[threadIdx.x] = fmax(red[threadIdx.x], red[threadIdx.x + s]);
    __syncthreads();
  }
  m = red[0];
  // a row with a non-finite element has no digits: they are written as zeros and the row's scale as NaN, which the
  // epilogue multiplies into every R element the row enters (IEEE inf/NaN there, as the header promises)
  const bool bad = !(m <= DBL_MAX);
  int ex = 0;
  if (m > 0.0 && !bad) (void)frexp(m, &ex);                 // m = f 2^ex, f in [0.5, 1): |x| < 2^ex
  const double scale = bad ? __longlong_as_double(0x7ff8000000000000LL) : ldexp(1.0, ex), inv = ldexp(1.0, -ex);
  if (threadIdx.x == 0) scales[(size_t)e * Cp + row] = scale;
  for (long long k4 = (long long)threadIdx.x * 4; k4 < Kp; k4 += (long long)blockDim.x * 4) {
    uint32_t word[SL_MAX];
#pragma unroll
    for (int i = 0; i < SL_MAX; ++i) word[i] = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const long long k = k4 + j;
      double r = 0.0;
      if (in_row && k < n_poles) {
        const double x = CACHE ? xrow[k] : (E_k ? w[k] * (1.0 / (E_k[k] - E)) : w[k]);
        r = bad ? 0.0 : x * inv * 64.0;
      }
#pragma unroll
      for (int i = 0; i < SL_MAX; ++i) {
        if (i < S) {
          const double d = rint(r);
          word[i] |= ((uint32_t)(uint8_t)(int8_t)(int)d) << (8 * j);
          r = (r - d) * 128.0;
        }
      }
    }
    for (int i = 0; i < S; ++i)
      *reinterpret_cast<uint32_t *>(digits + (((size_t)e * S + i) * Cp + row) * Kp + k4) = word[i];
  }
}

// ---- the integer GEMM on tcgen05 -----------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "SL_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra SL_DONE;\n"
      "bra SL_WAIT;\n"
      "SL_DONE:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_2d(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
               "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(bar)
               : "memory");
}
// K-major tile of rows x 64 bytes, SWIZZLE_64B: 8-row groups of 512 bytes one after another (what the TMA box writes).
// SM100 matrix descriptor: start address >> 4 in [0, 14), leading byte offset >> 4 in [16, 30) (unused here: 1), stride
// byte offset >> 4 in [32, 46) (512 bytes between 8-row groups), version 1 in [46, 48), layout type 4 (64-byte swizzle)
// in [61, 64).
__device__ __forceinline__ uint64_t make_desc(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3ffffu) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(512 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)4 << 61;
  return d;
}
// kind::i8 instruction descriptor: c_format S32 (2) in [4, 6), a / b format signed 8 bit (1) in [7, 10) / [10, 13), both
// K-major, N >> 3 in [17, 23), M >> 4 in [24, 29).
__device__ __forceinline__ uint32_t make_idesc() {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(TILE_N >> 3) << 17) | ((uint32_t)(TILE_M >> 4) << 24);
}
__device__ __forceinline__ void mma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t"
      "}\n" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

struct GemmArgs {
  const double *sA;        // [Cp]
  const double *sB;        // [ne][Cp]
  const double *diag_add;  // optional [ne][n_chan] (already offset to the chunk's first energy)
  double *R;               // R_out of the chunk's first energy
  double inv2a;
  int n_chan, S, n_kb, ne;
  int n_ti, n_tj;          // tiles down (128 rows) and across (64 columns)
  int tiles_per_e;         // tiles with an element on or above the diagonal: sum over I of (n_tj - 2 I)
  long long Cp;
};

__global__ void __launch_bounds__(GEMM_THREADS, 1)
sliced_gemm_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, const GemmArgs g) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  __shared__ __align__(8) unsigned long long bars[2 * STAGES + 2];
  __shared__ uint32_t tmem_slot;
  unsigned char *tiles = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int S = g.S;
  const uint32_t stage_bytes = (uint32_t)S * (TILE_M + TILE_N) * KB;
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[STAGES]);
  const uint32_t acc_full = smem_u32(&bars[2 * STAGES]), acc_empty = smem_u32(&bars[2 * STAGES + 1]);
  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, 1);
    }
    mbar_init(acc_full, 1);
    mbar_init(acc_empty, 4);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    __syncwarp();                                            // lane 0 comes out of the barrier set-up: .sync.aligned wants the warp converged
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_slot)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = tmem_slot;

  // work items: (energy of the chunk, tile down I, tile across J) with some element on or above the diagonal, i.e.
  // J >= 2 I (64 J + 63 >= 128 I); CTA b takes items b, b + grid, ... of the list ordered energy-major (the tiles of
  // an energy share its B digits in L2)
  const long long tiles_per_e = g.tiles_per_e, n_items = tiles_per_e * g.ne;
  auto decode = [&](long long item, int &e, int &I, int &J) {
    e = (int)(item / tiles_per_e);
    int t = (int)(item - e * tiles_per_e);
    for (I = 0;; ++I) {
      const int cnt = g.n_tj - 2 * I;
      if (t < cnt) break;
      t -= cnt;
    }
    J = 2 * I + t;
  };

  if (warp == 0 && lane == 0) {
    // ===== TMA producer =====
    uint32_t stage = 0, phase = 0;
    for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
      int e, I, J;
      decode(item, e, I, J);
      for (int kb = 0; kb < g.n_kb; ++kb) {
        mbar_wait(empty0 + 8 * stage, phase ^ 1u);
        const uint32_t base = smem_u32(tiles) + stage * stage_bytes, full = full0 + 8 * stage;
        mbar_expect_tx(full, stage_bytes);
        for (int s = 0; s < S; ++s) {
          tma_2d(base + s * (TILE_M * KB), &mapA, kb * KB, (int)(s * g.Cp + (long long)I * TILE_M), full);
          tma_2d(base + S * (TILE_M * KB) + s * (TILE_N * KB), &mapB, kb * KB, (int)(((long long)e * S + s) * g.Cp + (long long)J * TILE_N), full);
        }
        if (++stage == STAGES) { stage = 0; phase ^= 1u; }
      }
    }
  } else if (warp == 1 && lane == 0) {
    // ===== MMA issuer =====
    const uint32_t idesc = make_idesc();
    uint32_t stage = 0, phase = 0, acc_phase = 0;
    for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
      int e, I, J;
      decode(item, e, I, J);
      mbar_wait(acc_empty, acc_phase ^ 1u);                 // the epilogue has drained the accumulators of the last item
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      for (int kb = 0; kb < g.n_kb; ++kb) {
        mbar_wait(full0 + 8 * stage, phase);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t base = smem_u32(tiles) + stage * stage_bytes;
        for (int kk = 0; kk < KB / UMMA_K; ++kk)
          for (int tt = 0; tt < S; ++tt)                      // accumulator tt: the products dA_i dB_j^T with i + j = tt
            for (int i = 0; i <= tt; ++i) {
              const uint64_t da = make_desc(base + i * (TILE_M * KB) + kk * UMMA_K);
              const uint64_t db = make_desc(base + S * (TILE_M * KB) + (tt - i) * (TILE_N * KB) + kk * UMMA_K);
              mma_i8(tmem + tt * TILE_N, da, db, idesc, (kb | kk | i) != 0 ? 1u : 0u);
            }
        umma_commit(empty0 + 8 * stage);                     // the stage is free when these MMAs have read it
        if (++stage == STAGES) { stage = 0; phase ^= 1u; }
      }
      umma_commit(acc_full);                                 // ... and the accumulators are complete
      acc_phase ^= 1u;
    }
  } else if (warp >= 2) {
    // ===== epilogue: TMEM -> registers -> FP64 -> R and its mirror =====
    const int quad = warp & 3;                               // the TMEM lanes this warp may read: 32 quad .. 32 quad + 31
    uint32_t acc_phase = 0;
    const size_t cc = (size_t)g.n_chan * g.n_chan;
    for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
      int e, I, J;
      decode(item, e, I, J);
      mbar_wait(acc_full, acc_phase);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const int n = I * TILE_M + 32 * quad + lane;
      const double sn = n < g.n_chan ? g.sA[n] * g.inv2a : 0.0;
      double *R = g.R + (size_t)e * cc;
      for (int c0 = 0; c0 < TILE_N; c0 += 16) {
        double v[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) v[c] = 0.0;
        for (int tt = S - 1; tt >= 0; --tt) {                 // Horner: v = v 2^-7 + ACC_tt, smallest terms first
          uint32_t r[16];
          const uint32_t taddr = tmem + ((uint32_t)(32 * quad) << 16) + (uint32_t)(tt * TILE_N + c0);
          asm volatile(
              "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
              : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
              : "r"(taddr));
          asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
          for (int c = 0; c < 16; ++c) v[c] = v[c] * 0.0078125 + (double)(int)r[c];
        }
        if (n < g.n_chan) {
#pragma unroll
          for (int c = 0; c < 16; ++c) {
            const int m = J * TILE_N + c0 + c;
            if (m < g.n_chan && m >= n) {
              double val = v[c] * (1.0 / 4096.0) * sn * g.sB[(size_t)e * g.Cp + m];
              if (m == n && g.diag_add) val += g.diag_add[(size_t)e * g.n_chan + n];
              __stcs(R + (size_t)n * g.n_chan + m, val);
              if (m != n) __stcs(R + (size_t)m * g.n_chan + n, val);
            }
          }
        }
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncwarp();
      if (lane == 0) mbar_arrive(acc_empty);
      acc_phase ^= 1u;
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    __syncwarp();                                            // lane 0 ran the producer loop on its own
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
  }
}

// ---- host ----------------------------------------------------------------------------------------
typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                    const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
encode_tiled_fn g_encode_sliced = nullptr;
std::once_flag g_encode_sliced_once;

bool encode_bytes_map(CUtensorMap *map, const int8_t *base, long long rows, long long Kp, int box_rows) {
  cuuint64_t dims[2] = {(cuuint64_t)Kp, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)Kp};
  cuuint32_t box[2] = {(cuuint32_t)KB, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  return g_encode_sliced(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<int8_t *>(base), dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

struct SlicedLayout {
  long long Cp, Kp;
  int chunk;               // energies sliced and contracted per pass
  size_t off_sA, off_sB, off_A, off_B, bytes;
};
SlicedLayout sliced_layout(int n_chan, int n_poles, int n_E, int S) {
  SlicedLayout L;
  L.Cp = round_up(n_chan, TILE_M);
  L.Kp = round_up(std::max(n_poles, 1), KB);
  const size_t per_op = (size_t)S * (size_t)L.Cp * (size_t)L.Kp;             // digits of one operand at one energy
  const size_t budget = (size_t)1 << 30;                                     // B digits of a chunk: at most 1 GiB
  L.chunk = (int)std::max<size_t>(1, std::min<size_t>((size_t)std::max(n_E, 1), budget / std::max<size_t>(per_op, 1)));
  L.chunk = std::min(L.chunk, 65535);                                        // the slicing launch has one grid.y per energy
  auto al = [](size_t x) { return (x + 1023) & ~(size_t)1023; };
  L.off_sA = 0;
  L.off_sB = al(L.off_sA + sizeof(double) * (size_t)L.Cp);
  L.off_A = al(L.off_sB + sizeof(double) * (size_t)L.chunk * (size_t)L.Cp);
  L.off_B = al(L.off_A + per_op);
  L.bytes = al(L.off_B + per_op * (size_t)L.chunk);
  return L;
}

}  // namespace

extern "C" {

size_t pstgf_rmat_sliced_workspace_bytes(int n_chan, int n_poles, int n_E, int n_slices) {
  if (n_chan <= 0 || n_poles <= 0 || n_E <= 0 || n_slices < 2 || n_slices > SL_MAX) return 0;
  return sliced_layout(n_chan, n_poles, n_E, n_slices).bytes;
}

pstgf_status_t pstgf_rmat_form_sliced(const pstgf_wave_t *wave, int n_slices, void *workspace, size_t workspace_bytes, void *stream) {
  pstgf::set_last_call_state(0, 0);
  if (!wave) return PSTGF_ERR_INVALID_VALUE;
  const pstgf_wave_t &w = *wave;
  if (w.n_chan < 0 || w.n_poles < 0 || w.n_E < 0 || !(w.a > 0.0) || !std::isfinite(w.a)) return PSTGF_ERR_INVALID_VALUE;
  if (n_slices < 2 || n_slices > SL_MAX) return PSTGF_ERR_INVALID_VALUE;
  if (w.n_chan == 0 || w.n_E == 0) return PSTGF_OK;
  if (w.w_layout != PSTGF_W_POLE_CONTIGUOUS) return PSTGF_ERR_INVALID_VALUE;           // pole-contiguous W only
  if (w.n_poles == 0 || (long long)w.n_poles * n_slices >= (1LL << 19)) return PSTGF_ERR_INVALID_VALUE;   // INT32 accumulators
  if (!w.W || !w.E_k || !w.energies || !w.R_out || w.ldw < w.n_poles) return PSTGF_ERR_INVALID_VALUE;
  for (const void *p : {(const void *)w.W, (const void *)w.E_k, (const void *)w.energies, (const void *)w.R_out, (const void *)w.diag_add})
    if (reinterpret_cast<uintptr_t>(p) & 7u) return PSTGF_ERR_ALIGNMENT;
  const SlicedLayout L = sliced_layout(w.n_chan, w.n_poles, w.n_E, n_slices);
  if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < L.bytes) return PSTGF_ERR_WORKSPACE;
  int dev = 0, major = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
      major != 10 || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    (void)cudaGetLastError();
    return PSTGF_ERR_UNSUPPORTED_DEVICE;
  }
  std::call_once(g_encode_sliced_once, [] {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      g_encode_sliced = reinterpret_cast<encode_tiled_fn>(fn);
  });
  if (!g_encode_sliced) return PSTGF_ERR_UNSUPPORTED_DEVICE;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  unsigned char *ws = static_cast<unsigned char *>(workspace);
  double *sA = reinterpret_cast<double *>(ws + L.off_sA), *sB = reinterpret_cast<double *>(ws + L.off_sB);
  int8_t *dA = reinterpret_cast<int8_t *>(ws + L.off_A), *dB = reinterpret_cast<int8_t *>(ws + L.off_B);
  const int S = n_slices;
  const int smem = STAGES * S * (TILE_M + TILE_N) * KB + 1024;
  auto fail = [](cudaError_t e) { pstgf::set_last_call_state(0, (int)e); (void)cudaGetLastError(); return PSTGF_ERR_CUDA; };
  cudaError_t ce = cudaFuncSetAttribute(sliced_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (ce != cudaSuccess) return fail(ce);
  CUtensorMap mapA, mapB;
  if (!encode_bytes_map(&mapA, dA, (long long)S * L.Cp, L.Kp, TILE_M) ||
      !encode_bytes_map(&mapB, dB, (long long)L.chunk * S * L.Cp, L.Kp, TILE_N))
    return fail(cudaErrorInvalidValue);
  // the slicing kernel keeps a row in shared memory between its two passes when that does not cost occupancy (a row of
  // config 5 is 80 KB: two blocks per SM, measured 12.6 ms per step against 8.8 ms with the divisions done twice)
  const size_t row_bytes = sizeof(double) * (size_t)w.n_poles;
  const bool cache = row_bytes <= 16 * 1024;
  if (cache && (ce = cudaFuncSetAttribute(slice_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)row_bytes)) != cudaSuccess) return fail(ce);
  auto slice = [&](dim3 grid, const double *Ek, const double *en, int8_t *digits, double *scales) {
    if (cache) slice_kernel<true><<<grid, 256, row_bytes, s>>>(w.W, w.ldw, Ek, en, w.n_chan, w.n_poles, S, L.Cp, L.Kp, digits, scales);
    else slice_kernel<false><<<grid, 256, 0, s>>>(w.W, w.ldw, Ek, en, w.n_chan, w.n_poles, S, L.Cp, L.Kp, digits, scales);
  };
  // digits of A = W, once
  slice(dim3((unsigned)L.Cp, 1), nullptr, nullptr, dA, sA);
  int launches = 1;
  for (int e0 = 0; e0 < w.n_E; e0 += L.chunk) {
    const int ne = std::min(L.chunk, w.n_E - e0);
    // digits of B_e = W diag(1 / (E_k - E_e)) for the chunk's energies, then the contraction
    slice(dim3((unsigned)L.Cp, (unsigned)ne), w.E_k, w.energies + e0, dB, sB);
    GemmArgs g;
    g.sA = sA;
    g.sB = sB;
    g.diag_add = w.diag_add ? w.diag_add + (size_t)e0 * w.n_chan : nullptr;
    g.R = w.R_out + (size_t)e0 * w.n_chan * w.n_chan;
    g.inv2a = 1.0 / (2.0 * w.a);
    g.n_chan = w.n_chan;
    g.S = S;
    g.n_kb = (int)(L.Kp / KB);
    g.ne = ne;
    g.n_ti = (int)(L.Cp / TILE_M);
    g.n_tj = (int)(L.Cp / TILE_N);
    g.Cp = L.Cp;
    g.tiles_per_e = 0;
    for (int I = 0; I < g.n_ti; ++I) g.tiles_per_e += std::max(0, g.n_tj - 2 * I);
    const long long items = (long long)g.tiles_per_e * ne;
    sliced_gemm_kernel<<<(unsigned)std::min<long long>(sms, items), GEMM_THREADS, smem, s>>>(mapA, mapB, g);
    launches += 2;
  }
  ce = cudaGetLastError();
  if (ce != cudaSuccess) return fail(ce);
  pstgf::set_last_call_state(launches, 0);
  return PSTGF_OK;
}

}  // extern "C"
