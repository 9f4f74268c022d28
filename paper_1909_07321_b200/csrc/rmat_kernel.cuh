// rmat_kernel.cuh -- the persistent sm_100a kernel behind pstgf_rmat_form / pstgf_rmat_form_batch.
//
// One CTA per SM, 12 warps.  Warps 8..11 are the producer warpgroup: they hand most of their
// registers to the consumers (setmaxnreg).  Warp 8 takes work items (atomic counter: in the workspace
// for the batch call, in a pool slot for the single-wave call), publishes them and issues the TMA loads of the W
// panels; warps 9..11 build the pole scaling d_e[k] = 1/(E_k - E_e) of every
// stage in shared memory (S1; the denominator of eq. 4).  Warps 0..7 are consumers.  On a classic
// item each takes one energy of the item's block of 8; on a slab item (the energies that do not fill a block of
// 8, taken four, two or one at a time) the warps of one energy split the tile between them; on a pair item (a wave
// with few channels as the GEMM over channel pairs, rmat_common.h) each takes 16 of the item's 128 energies.  Classic
// and slab items contract
// acc[n][m] += W[n][k] * (W[m][k] * d_e[k]) on the FP64 tensor pipe (mma.sync m8n8k4 -> DMMA.8x8x4) over
// upper-triangle tiles only (S3) and write R and its mirror scaled by 1/(2a) (S4).
// Producer and consumers are coupled by an mbarrier full/empty ring that runs on across item boundaries, so the
// next item's first stages land while the epilogue of the current one is being stored.
#pragma once
#include "rmat_common.h"

namespace pstgf {

struct alignas(16) ItemInfo {   // handed from the load warp to the pole-scaling and consumer warps through smem
  double *R;               // R_out of the item's first energy
  const double *diag_add;  // the wave's diagonal addend at the item's first energy, or null
  unsigned int *done;      // completion counter of the item's wave, or null
  unsigned int *done_flag; // host-mapped word set to 1 when the counter reaches done_target
  const double *E_k;       // the wave's poles
  const double *energies;  // the item's first energy
  double inv2a;
  unsigned int done_target;
  int n_chan;
  int n_poles;
  int n_valid_e;           // energies of this item (1..EB; slab items: 2 or 1)
  int row0, col0;
  int nblk;                // DIAG: valid 8x8 block rows/cols; rectangular tiles: valid 8-wide column blocks; pair items: row blocks
  int n_kt;
  int n_pairs;             // pair items: rows of P (row0 = first pair of the tile, col0 = first energy of the tile)
  int pair_rb;             // pair items: rows of P in the block section (rmat_common.h)
  const unsigned int *pair_nm;   // pair items: n | m << 16 of every row of P
  short kind;              // 0 on the diagonal (DIAG / slab S(i,i)), 1 strictly above it, 2 pair item, -1 stop
  unsigned char nrb;       // classic rectangular tiles: 8-row blocks of the I panel (16 WIDE, 8 OFF, 4 fine OFF32)
  unsigned char tr;        // stage layout: 0 row-major panels, 1 pole-major panels (channel-contiguous W)
  unsigned char slab_T;    // 0: classic item (one energy per warp); else the edge of the slab tile (32, 64, 128)
  unsigned char slab_g;    // slab items: energies in the group (2 or 1)
};
static_assert(sizeof(ItemInfo) <= 128, "ItemInfo slot (SMEM_ITEM_OFFSET reserves 2 x 128)");

// ---- PTX wrappers ------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "MBAR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra MBAR_DONE;\n"
      "bra MBAR_WAIT;\n"
      "MBAR_DONE:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}
// The same with an L2 cache policy (evict_last for a W that fits half of L2: R's streaming stores then leave it alone).
__device__ __forceinline__ void tma_load_2d_hint(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar,
                                                 uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(bar), "l"(policy)
      : "memory");
}
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_normal() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// A tensor map that lives in global memory (the batch call's workspace, rewritten by every call) must be
// acquired by the CTA before its first use by the TMA unit, or a stale cached copy may be used.
__device__ __forceinline__ void tensormap_acquire(const CUtensorMap *map) {
  asm volatile("fence.proxy.tensormap::generic.acquire.gpu [%0], 128;" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}
__device__ __forceinline__ unsigned long long global_timer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}
// D(8x8) += A(8x4) * B(4x8), FP64.  Lane l holds A[l/4][l%4], B[l%4][l/4], D[l/4][2*(l%4)+{0,1}].
__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// Host-buffer call: W may still be on its way up while the launch runs.  It is uploaded in slabs, the upload
// stream bumps a counter after every slab, and the load warp waits here until what it is about to load has
// landed.  Slabs of poles (column ranges of a pole-contiguous W, rows of a channel-contiguous one) let the k loop
// of the first items run behind the upload -- good when the upload takes about as long as an item; slabs of
// channels (rows of a pole-contiguous W) let the tiles near the top of the matrix run at full speed while the
// rest is still coming -- good when the upload takes many item times (the 6.2 GB of the paper-scale wave).
// The wait is bounded: after timeout_ns without the counter reaching `need` (a failed or serialised upload) the
// warp raises the launch's abort flag and stops waiting; every other load warp sees the flag at its next wait, the
// launch drains, and the host turns the flag into PSTGF_ERR_TIMEOUT (the R of that call is then undefined).
__device__ __forceinline__ void wait_rows_uploaded(const unsigned int *rows_ready, unsigned int need, unsigned int &seen,
                                                   unsigned int *abort_flag, unsigned int *abort_flag_host,
                                                   unsigned long long timeout_ns, int lane) {
  if (seen >= need) return;
  if (lane == 0) {
    unsigned int v;
    const unsigned long long t0 = global_timer_ns();
    for (;;) {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(rows_ready) : "memory");
      if (v >= need) break;
      if (abort_flag != nullptr) {
        // the flag that is polled lives in DEVICE memory: 148 load warps polling a word of mapped host memory
        // fill the PCIe link with small reads and slow the very upload they are waiting for (measured: config 4's
        // host call 149 -> 265 ms); the host's copy is written once, by the warp whose wait timed out
        unsigned int ab;
        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(ab) : "l"(abort_flag) : "memory");
        if (ab == 0u && global_timer_ns() - t0 > timeout_ns) {
          atomicExch(abort_flag, 1u);
          if (abort_flag_host != nullptr) {
            *reinterpret_cast<volatile unsigned int *>(abort_flag_host) = 1u;
            __threadfence_system();
          }
          ab = 1u;
        }
        if (ab != 0u) {
          v = 0xffffffffu;
          break;
        }
      }
      __nanosleep(500);
    }
    seen = v;
    asm volatile("fence.proxy.async;" ::: "memory");   // the loads that follow go through the async proxy (TMA)
  }
  seen = __shfl_sync(0xffffffffu, seen, 0);
}

// Position in the shared-memory ring, with the ring's geometry (a launch parameter: RingGeo).
struct Pipe {
  const unsigned char *ring;
  uint32_t full0, empty0;
  int stage_bytes, n_stages;
  uint32_t stage = 0, phase = 0;
  __device__ __forceinline__ void advance() {
    if (++stage == (uint32_t)n_stages) { stage = 0; phase ^= 1u; }
  }
  __device__ __forceinline__ const double *stage_ptr() const {
    return reinterpret_cast<const double *>(ring + (size_t)stage * stage_bytes);
  }
  __device__ __forceinline__ uint32_t full() const { return full0 + 8 * stage; }
  __device__ __forceinline__ uint32_t empty() const { return empty0 + 8 * stage; }
};

// ---- consumers ---------------------------------------------------------------------------
// Releasing a stage.  mbarrier.arrive does not wait for the warp's LDS that are still in flight, so an arrive
// issued right after the stage's last fragment load leaves a window in which the refill (TMA, async proxy)
// can overwrite rows a delayed LDS has yet to read.  With R_out in device memory the window never opens (an
// LDS takes tens of cycles, a refill hundreds), but with the LSU backed up for microseconds -- R_out in mapped
// host memory, every store a PCIe write -- it showed as a few wrong rows per launch.  A CTA-scope fence executed
// by the whole warp before the release closes it: the warp's loads have been performed when the fence retires
// (costs 0.5 % on config 5; releasing one stage late instead was measured and is no cheaper).
__device__ __forceinline__ void release_stage(const Pipe &ps, int lane) {
  __threadfence_block();
  __syncwarp();
  if (lane == 0) mbar_arrive(ps.empty());
}

// Warps with nothing to compute in an item (an energy slot beyond n_E, a slab below the diagonal) only keep the
// ring moving.
__device__ __forceinline__ void consume_idle(int n_kt, Pipe &ps, int lane) {
  for (int kt = 0; kt < n_kt; ++kt) {
    mbar_wait(ps.full(), ps.phase);
    __syncwarp();
    if (lane == 0) mbar_arrive(ps.empty());
    ps.advance();
  }
}

// Rectangular tile strictly above the diagonal: WIDE 128 x 16 (NRB = 16, NCB <= 2), OFF 64 x 32 (NRB = 8) or
// fine OFF32 32 x 32 (NRB = 4); NRB x NCB DMMA blocks, all needed (column blocks >= nblk lie beyond n_chan and
// are skipped).  One scaled B fragment feeds NRB DMMAs: the WIDE shape halves the DMULs per DMMA of OFF.
template <int NCB, int NRB, bool TR>
__device__ __forceinline__ void consume_off(const ItemInfo &it, Pipe &ps, int warp, int lane) {
  double acc[NRB][NCB][2];
#pragma unroll
  for (int bi = 0; bi < NRB; ++bi)
#pragma unroll
    for (int bj = 0; bj < NCB; ++bj) acc[bi][bj][0] = acc[bi][bj][1] = 0.0;
  const int g = lane >> 2, q = lane & 3;
  using L = StageLayout<TR>;
  for (int kt = 0; kt < it.n_kt; ++kt) {
    mbar_wait(ps.full(), ps.phase);
    const double *st = ps.stage_ptr();
    const double *wi = st + L::W_BASE + L::off(g, q);
    const double *wj = st + L::J_CLASSIC + L::off(g, q);
    const double *dd = st + warp * KT + q;
#pragma unroll
    for (int ks = 0; ks < KT / 4; ++ks) {
      const double dv = dd[ks * 4];
      double a[NRB];
#pragma unroll
      for (int bi = 0; bi < NRB; ++bi) a[bi] = wi[L::off(bi * 8, ks * 4)];
#pragma unroll
      for (int bj = 0; bj < NCB; ++bj) {
        const double b = wj[L::off(bj * 8, ks * 4)] * dv;   // pole scaling folded into the B fragment
#pragma unroll
        for (int bi = 0; bi < NRB; ++bi) dmma884(acc[bi][bj][0], acc[bi][bj][1], a[bi], b);
      }
    }
    release_stage(ps, lane);
    ps.advance();
  }
  // epilogue: R[r][c] and the mirror R[c][r]; rows are always inside the matrix for OFF tiles
  const int C = it.n_chan;
  double *R = it.R + (size_t)warp * C * C;
  const double s = it.inv2a;
#pragma unroll
  for (int bj = 0; bj < NCB; ++bj) {
    const int c = it.col0 + bj * 8 + 2 * q;
#pragma unroll
    for (int bi = 0; bi < NRB; ++bi) {
      const int r = it.row0 + bi * 8 + g;
      const double v0 = acc[bi][bj][0] * s, v1 = acc[bi][bj][1] * s;
      // R[r][c], R[r][c+1] are neighbours: one 16-byte store when the address allows it (always, for an even n_chan
      // and a 16-byte aligned R_out); the mirror elements R[c][r], R[c+1][r] are a row apart
      double *direct = R + (size_t)r * C + c;
      if (c + 1 < C && (reinterpret_cast<uintptr_t>(direct) & 15u) == 0) {
        __stcs(reinterpret_cast<double2 *>(direct), make_double2(v0, v1));
        __stcs(R + (size_t)c * C + r, v0);
        __stcs(R + (size_t)(c + 1) * C + r, v1);
      } else {
        if (c < C) { __stcs(direct, v0); __stcs(R + (size_t)c * C + r, v0); }
        if (c + 1 < C) { __stcs(direct + 1, v1); __stcs(R + (size_t)(c + 1) * C + r, v1); }
      }
    }
  }
}

// DIAG tile: 64 x 64 block on the diagonal; only 8x8 blocks (bi <= bj) are computed, and in
// blocks on the diagonal only elements c >= r are stored (with their mirror), so that
// R[n][m] == R[m][n] bitwise.  The optional diagonal addend (pstgf_wave_t.diag_add) goes onto R[n][n] here,
// after the 1/(2a) scale.
template <int NB, bool TR>
__device__ __forceinline__ void consume_diag(const ItemInfo &it, Pipe &ps, int warp, int lane) {
  double acc[NB * (NB + 1) / 2][2];
#pragma unroll
  for (int t = 0; t < NB * (NB + 1) / 2; ++t) acc[t][0] = acc[t][1] = 0.0;
  const int g = lane >> 2, q = lane & 3;
  using L = StageLayout<TR>;
  for (int kt = 0; kt < it.n_kt; ++kt) {
    mbar_wait(ps.full(), ps.phase);
    const double *st = ps.stage_ptr();
    const double *wi = st + L::W_BASE + L::off(g, q);
    const double *dd = st + warp * KT + q;
#pragma unroll
    for (int ks = 0; ks < KT / 4; ++ks) {
      const double dv = dd[ks * 4];
      double a[NB];
#pragma unroll
      for (int bi = 0; bi < NB; ++bi) a[bi] = wi[L::off(bi * 8, ks * 4)];
#pragma unroll
      for (int bj = 0; bj < NB; ++bj) {
        const double b = a[bj] * dv;
#pragma unroll
        for (int bi = 0; bi <= bj; ++bi) dmma884(acc[bj * (bj + 1) / 2 + bi][0], acc[bj * (bj + 1) / 2 + bi][1], a[bi], b);
      }
    }
    release_stage(ps, lane);
    ps.advance();
  }
  const int C = it.n_chan;
  double *R = it.R + (size_t)warp * C * C;
  const double *da = it.diag_add ? it.diag_add + (size_t)warp * C : nullptr;
  const double s = it.inv2a;
#pragma unroll
  for (int bj = 0; bj < NB; ++bj) {
    const int c = it.row0 + bj * 8 + 2 * q;
#pragma unroll
    for (int bi = 0; bi <= bj; ++bi) {
      const int r = it.row0 + bi * 8 + g;
      double v0 = acc[bj * (bj + 1) / 2 + bi][0] * s, v1 = acc[bj * (bj + 1) / 2 + bi][1] * s;
      if (r < C) {
        if (c < C && c >= r) {
          if (bi == bj && c == r && da) v0 += __ldg(da + r);
          __stcs(R + (size_t)r * C + c, v0);
          if (c > r) __stcs(R + (size_t)c * C + r, v0);
        }
        if (c + 1 < C && c + 1 >= r) {
          if (bi == bj && c + 1 == r && da) v1 += __ldg(da + r);
          __stcs(R + (size_t)r * C + c + 1, v1);
          if (c + 1 > r) __stcs(R + (size_t)(c + 1) * C + r, v1);
        }
      }
    }
  }
}

// Slab item: a square tile S(i, j) of edge T for a group of g = 4, 2 or 1 energies.  The 8 / g warps of one energy
// form a grid of wr x wc warps over the tile (SlabShape); this warp computes row blocks [rb0, rb0 + NR) x column
// blocks [cb0, cb0 + NCW) of 8 x 8.  The DMMA loop has no predicates: a warp whose slab is cut by the diagonal or by
// the edge of the matrix computes all of its register tile and stores only what is wanted (nrc[c] row blocks of
// column c: a prefix, because rows ascend); a warp with nothing wanted only keeps the ring moving.  A = rows of
// the I panels, B = scaled rows of the J panels (the I panels on a diagonal tile): the same operands and (NCH == 1,
// what the library uses) the same k order as a classic item gives the element, hence the same bits.  NCH == 5 sums
// the five k-steps of a stage into five chains that are added at the end: a different association of the same
// terms; measured to buy nothing (a dependent DMMA issues after 26.5 clk, so two accumulators per warp already fill
// the pipe's 16-clk slots), kept as a compile-time option only.
template <int NR, int NCW, int NCH, bool TR>
__device__ __forceinline__ void consume_slab(const ItemInfo &it, Pipe &ps, int warp, int lane, int wc) {
  using L = StageLayout<TR>;
  static_assert(NCH == 1 || NCH == KT / 4, "one summation chain, or one per k-step of a stage");
  const int T = it.slab_T, gE = it.slab_g, C = it.n_chan;
  const int e_slot = warp % gE, s = warp / gE;              // which energy of the group, which slab of the tile
  const int wci = s % wc, wri = s / wc;
  const int rb0 = wri * NR, cb0 = wci * NCW;
  const bool diag = it.kind == 0;
  const int vrb = min(T / 8, (C - it.row0 + 7) / 8);        // row blocks of the tile inside the matrix
  int nrc[NCW];
  bool any = false;
#pragma unroll
  for (int c = 0; c < NCW; ++c) {
    const int cb = cb0 + c;
    const int lim = min(diag ? cb + 1 : T / 8, vrb);         // on a diagonal tile only row blocks rb <= cb
    nrc[c] = it.col0 + cb * 8 < C ? max(0, min(NR, lim - rb0)) : 0;
    any = any || nrc[c] > 0;
  }
  if (!any || e_slot >= it.n_valid_e) {                      // nothing wanted, or the empty fourth slot of a group of three
    consume_idle(it.n_kt, ps, lane);
    return;
  }
  const int g = lane >> 2, q = lane & 3;
  const int jrow = diag ? 0 : T;                             // B fragments: rows of the J panels (behind the I panels)
  const int aoff = L::W_BASE + L::off(rb0 * 8, 0) + L::off(g, q);
  const int boff = L::W_BASE + L::off(jrow + cb0 * 8, 0) + L::off(g, q);
  const int doff = e_slot * KT + q;
  double acc[NCH][NR][NCW][2];
#pragma unroll
  for (int h = 0; h < NCH; ++h)
#pragma unroll
    for (int bi = 0; bi < NR; ++bi)
#pragma unroll
      for (int c = 0; c < NCW; ++c) acc[h][bi][c][0] = acc[h][bi][c][1] = 0.0;
  for (int kt = 0; kt < it.n_kt; ++kt) {
    mbar_wait(ps.full(), ps.phase);
    const double *st = ps.stage_ptr();
    const double *wa = st + aoff;
    const double *wb = st + boff;
    const double *dd = st + doff;
#pragma unroll
    for (int ks = 0; ks < KT / 4; ++ks) {
      const int h = NCH == 1 ? 0 : ks;                       // the chain this k-step adds to
      const double dv = dd[ks * 4];
      double a[NR];
#pragma unroll
      for (int bi = 0; bi < NR; ++bi) a[bi] = wa[L::off(bi * 8, ks * 4)];
#pragma unroll
      for (int c = 0; c < NCW; ++c) {
        const double b = wb[L::off(c * 8, ks * 4)] * dv;     // pole scaling folded into the B fragment
#pragma unroll
        for (int bi = 0; bi < NR; ++bi) dmma884(acc[h][bi][c][0], acc[h][bi][c][1], a[bi], b);
      }
    }
    release_stage(ps, lane);
    ps.advance();
  }
  // epilogue
  double *R = it.R + (size_t)e_slot * C * C;
  const double *da = it.diag_add ? it.diag_add + (size_t)e_slot * C : nullptr;
  const double sc = it.inv2a;
#pragma unroll
  for (int c = 0; c < NCW; ++c) {
    const int col = it.col0 + (cb0 + c) * 8 + 2 * q;
#pragma unroll
    for (int bi = 0; bi < NR; ++bi) {
      if (bi < nrc[c]) {
        const int r = it.row0 + (rb0 + bi) * 8 + g;
        const bool dg = diag && rb0 + bi == cb0 + c;         // a block on the diagonal: keep col >= r only
        double v0 = acc[0][bi][c][0], v1 = acc[0][bi][c][1];
        if (NCH > 1) {                                       // fixed order: ((c0 + c1) + (c2 + c3)) + c4
          v0 = __dadd_rn(__dadd_rn(__dadd_rn(v0, acc[1 % NCH][bi][c][0]), __dadd_rn(acc[2 % NCH][bi][c][0], acc[3 % NCH][bi][c][0])),
                         acc[4 % NCH][bi][c][0]);
          v1 = __dadd_rn(__dadd_rn(__dadd_rn(v1, acc[1 % NCH][bi][c][1]), __dadd_rn(acc[2 % NCH][bi][c][1], acc[3 % NCH][bi][c][1])),
                         acc[4 % NCH][bi][c][1]);
        }
        v0 *= sc;
        v1 *= sc;
        if (r < C) {
          if (col < C && (!dg || col >= r)) {
            if (dg && col == r && da) v0 += __ldg(da + r);
            __stcs(R + (size_t)r * C + col, v0);
            if (col != r) __stcs(R + (size_t)col * C + r, v0);
          }
          if (col + 1 < C && (!dg || col + 1 >= r)) {
            if (dg && col + 1 == r && da) v1 += __ldg(da + r);
            __stcs(R + (size_t)r * C + col + 1, v1);
            if (col + 1 != r) __stcs(R + (size_t)(col + 1) * C + r, v1);
          }
        }
      }
    }
  }
}

// Pair item: NR row blocks of P (8 pairs each) x 128 energies; this warp's 16 energies are rows [16 warp, +16) of the
// D panels.  acc[pair][energy] += P[pair][k] * D[energy][k]: a plain GEMM, nothing is scaled inside the loop and no
// block is cut by a diagonal.  The epilogue scatters pair (n, m) of energy e to R[e][n][m] and R[e][m][n].
template <int NR>
__device__ __forceinline__ void consume_pair(const ItemInfo &it, Pipe &ps, int warp, int lane) {
  using L = StageLayout<false>;
  if (warp * 16 >= it.n_valid_e) {
    consume_idle(it.n_kt, ps, lane);
    return;
  }
  const int g = lane >> 2, q = lane & 3;
  const int aoff = L::W_BASE + L::off(g, q);
  const int boff = L::W_BASE + L::off(PT_M + warp * 16, 0) + L::off(g, q);
  double acc[NR][2][2];
#pragma unroll
  for (int bi = 0; bi < NR; ++bi) acc[bi][0][0] = acc[bi][0][1] = acc[bi][1][0] = acc[bi][1][1] = 0.0;
  for (int kt = 0; kt < it.n_kt; ++kt) {
    mbar_wait(ps.full(), ps.phase);
    const double *st = ps.stage_ptr();
    const double *wa = st + aoff;
    const double *wb = st + boff;
#pragma unroll
    for (int ks = 0; ks < KT / 4; ++ks) {
      double a[NR];
#pragma unroll
      for (int bi = 0; bi < NR; ++bi) a[bi] = wa[L::off(bi * 8, ks * 4)];
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const double b = wb[L::off(c * 8, ks * 4)];
#pragma unroll
        for (int bi = 0; bi < NR; ++bi) dmma884(acc[bi][c][0], acc[bi][c][1], a[bi], b);
      }
    }
    release_stage(ps, lane);
    ps.advance();
  }
  // epilogue: lane (g, q) holds row row0 + 8 bi + g of P at energies col0 + 16 warp + 8 c + 2 q + {0, 1}
  const int C = it.n_chan;
  const size_t cc = (size_t)C * C;
  const double sc = it.inv2a;
  const int nfb = C / 8;
#pragma unroll
  for (int grp = 0; grp < (NR + 7) / 8; ++grp) {            // groups of 64 rows: each is one 8 x 8 channel block, or loose
    const int r0 = it.row0 + grp * 64;
    if (NR >= 8 && r0 + 64 <= it.pair_rb) {
      // block section: rows 8 j + i of the group are the pairs (8 bn + j, 8 bm + i); this lane holds i = g
      int blk = r0 >> 6, bn = 0;
      while (blk >= nfb - 1 - bn) { blk -= nfb - 1 - bn; ++bn; }
      const int n0 = 8 * bn, m = 8 * (bn + 1 + blk) + g;
#pragma unroll
      for (int c = 0; c < 2; ++c) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int el = warp * 16 + c * 8 + 2 * q + h;       // energy inside the tile
          if (el < it.n_valid_e) {
            double *R = it.R + (size_t)el * cc;
            double v[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              v[j] = acc[(grp * 8 + j) % NR][c][h] * sc;
              __stcs(R + (size_t)(n0 + j) * C + m, v[j]);       // R[n][m .. m+7] across the eight lanes g: a 64-byte run
            }
            double *mir = R + (size_t)m * C + n0;               // R[m][n0 .. n0+7]: this lane's own 64-byte run
            if ((reinterpret_cast<uintptr_t>(mir) & 15u) == 0) {
#pragma unroll
              for (int j = 0; j < 8; j += 2) __stcs(reinterpret_cast<double2 *>(mir + j), make_double2(v[j], v[j + 1]));
            } else {
#pragma unroll
              for (int j = 0; j < 8; ++j) __stcs(mir + j, v[j]);
            }
          }
        }
      }
    } else {
      // loose section (diagonal blocks' triangles, ragged last block): element by element through the table
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int bi = grp * 8 + j;
        if (bi < NR) {
          const int idx = it.row0 + bi * 8 + g;
          if (idx < it.n_pairs) {
            const unsigned int nm = __ldg(it.pair_nm + idx);
            const int n = (int)(nm & 0xffffu), m = (int)(nm >> 16);
#pragma unroll
            for (int c = 0; c < 2; ++c) {
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                const int el = warp * 16 + c * 8 + 2 * q + h;
                if (el < it.n_valid_e) {
                  double v = acc[bi][c][h] * sc;
                  if (n == m && it.diag_add) v += __ldg(it.diag_add + (size_t)el * C + n);
                  double *R = it.R + (size_t)el * cc;
                  __stcs(R + (size_t)n * C + m, v);
                  if (n != m) __stcs(R + (size_t)m * C + n, v);
                }
              }
            }
          }
        }
      }
    }
  }
}

// The tile shapes are compile-time variants (no predicates inside the DMMA loop); ragged edges of
// a wave pick the variant with fewer 8-wide blocks.
template <int FAM, bool TR>
__device__ __forceinline__ void consume_item_layout(const ItemInfo &it, Pipe &ps, int warp, int lane) {
  if constexpr (FAM >= FAM_SLAB) {
    if (it.slab_T != 0) {
      const SlabShape sh = slab_shape(it.slab_T, it.slab_g);
      switch (sh.nr) {
        case 16: consume_slab<16, 2, 1, TR>(it, ps, warp, lane, sh.wc); break;
        case 8:
          if (sh.ncw == 4) consume_slab<8, 4, 1, TR>(it, ps, warp, lane, sh.wc);
          else consume_slab<8, 2, 1, TR>(it, ps, warp, lane, sh.wc);
          break;
        case 4: consume_slab<4, 2, 1, TR>(it, ps, warp, lane, sh.wc); break;
        default: consume_slab<2, 2, 1, TR>(it, ps, warp, lane, sh.wc); break;
      }
      return;
    }
  }
  if (warp >= it.n_valid_e) {
    consume_idle(it.n_kt, ps, lane);
    return;
  }
  if (it.kind == 0) {
    switch (it.nblk) {
      case 8: consume_diag<8, TR>(it, ps, warp, lane); break;
      case 7: consume_diag<7, TR>(it, ps, warp, lane); break;
      case 6: consume_diag<6, TR>(it, ps, warp, lane); break;
      case 5: consume_diag<5, TR>(it, ps, warp, lane); break;
      case 4: consume_diag<4, TR>(it, ps, warp, lane); break;
      case 3: consume_diag<3, TR>(it, ps, warp, lane); break;
      case 2: consume_diag<2, TR>(it, ps, warp, lane); break;
      default: consume_diag<1, TR>(it, ps, warp, lane); break;
    }
  } else if (it.nrb == 16) {
    if (it.nblk == 2) consume_off<2, 16, TR>(it, ps, warp, lane);
    else consume_off<1, 16, TR>(it, ps, warp, lane);
  } else if (it.nrb == 8) {
    switch (it.nblk) {
      case 4: consume_off<4, 8, TR>(it, ps, warp, lane); break;
      case 3: consume_off<3, 8, TR>(it, ps, warp, lane); break;
      case 2: consume_off<2, 8, TR>(it, ps, warp, lane); break;
      default: consume_off<1, 8, TR>(it, ps, warp, lane); break;
    }
  } else {
    switch (it.nblk) {
      case 4: consume_off<4, 4, TR>(it, ps, warp, lane); break;
      case 3: consume_off<3, 4, TR>(it, ps, warp, lane); break;
      case 2: consume_off<2, 4, TR>(it, ps, warp, lane); break;
      default: consume_off<1, 4, TR>(it, ps, warp, lane); break;
    }
  }
}

// FAM: the item families the launch can hold (rmat_common.h): a launch without pair items (without slab items)
// runs a kernel that does not contain their code -- the mere presence of the pair consumer in the kernel cost the
// classic items 1.4 % (config 5: 20.14 -> 20.42 ms, with identical SASS in the classic loops).
template <int FAM>
__device__ __forceinline__ void consume_item(const ItemInfo &it, Pipe &ps, int warp, int lane) {
  if constexpr (FAM >= FAM_PAIR) {
    if (it.kind == 2) {
      if (it.nblk == 16) consume_pair<16>(it, ps, warp, lane);
      else if (it.nblk == 8) consume_pair<8>(it, ps, warp, lane);
      else consume_pair<4>(it, ps, warp, lane);
      return;
    }
  }
  if (it.tr) consume_item_layout<FAM, true>(it, ps, warp, lane);
  else consume_item_layout<FAM, false>(it, ps, warp, lane);
}

// ---- producer ----------------------------------------------------------------------------
// Fine tile index -> OFF32 tiles first (16 DMMA per k-step), then DIAG32 (10).
__device__ __forceinline__ void decode_tile_fine(const DevWave &w, int tile, int &kind, int &row0, int &col0, int &nblk) {
  const int n = w.n_j, n_off = n * (n - 1) / 2;
  if (tile < n_off) {
    kind = 1;
    int t = tile, i = 0;
    for (;; ++i) {
      const int cnt = n - 1 - i;
      if (t < cnt) break;
      t -= cnt;
    }
    row0 = i * TN;
    col0 = (i + 1 + t) * TN;
    const int left = w.n_chan - col0;
    nblk = left >= TN ? TN / 8 : (left + 7) / 8;
  } else {
    kind = 0;
    row0 = col0 = (tile - n_off) * TN;
    const int left = w.n_chan - row0;
    nblk = left >= TN ? TN / 8 : (left + 7) / 8;
  }
}

// Coarse tile index inside a wave -> (kind, row0, col0, nblk, nrb).  DIAG tiles first (they are the most
// expensive), then the WIDE tiles pair by pair, then the OFF squares inside the pairs.
__device__ __forceinline__ void decode_tile(const DevWave &w, int tile, int &kind, int &row0, int &col0, int &nblk,
                                            int &nrb) {
  if (tile < w.n_i) {
    kind = 0;
    row0 = col0 = tile * TM;
    const int left = w.n_chan - row0;
    nblk = left >= TM ? TM / 8 : (left + 7) / 8;
    nrb = nblk;
    return;
  }
  kind = 1;
  int t = tile - w.n_i;
  for (int p = 0; TW * p + TM < w.n_chan; ++p) {
    const int cnt = wide_tiles_in_pair(w.n_chan, p);
    if (t < cnt) {
      row0 = p * TW;
      col0 = (p + 1) * TW + t * TWN;
      const int left = w.n_chan - col0;
      nblk = left >= TWN ? TWN / 8 : (left + 7) / 8;
      nrb = TW / 8;
      return;
    }
    t -= cnt;
  }
  for (int p = 0;; ++p) {
    const int cnt = off_tiles_in_pair(w.n_chan, p);
    if (t < cnt) {
      row0 = p * TW;
      col0 = p * TW + TM + t * TN;
      const int left = w.n_chan - col0;
      nblk = left >= TN ? TN / 8 : (left + 7) / 8;
      nrb = TM / 8;
      return;
    }
    t -= cnt;
  }
}

// Slab tile index -> S(i, j), j >= i, row by row over the upper triangle of slab_nt x slab_nt tiles.
__device__ __forceinline__ void decode_tile_slab(const DevWave &w, int tile, int &kind, int &row0, int &col0) {
  int t = tile, i = 0;
  for (;; ++i) {
    const int cnt = w.slab_nt - i;
    if (t < cnt) break;
    t -= cnt;
  }
  row0 = i * w.slab_T;
  col0 = (i + t) * w.slab_T;
  kind = t == 0 ? 0 : 1;
}

// Staging without TMA (W not 16-byte aligned or ldw odd): the producer warp copies the panels
// with plain loads, zero-filling rows >= n_chan and poles >= n_poles like the TMA path does.  The loads are
// L2-coherent (ld.global.cg): in the host-buffer call W may still be arriving while earlier slabs are read.
__device__ __forceinline__ void stage_panel_plain(double *dst, const DevWave &w, int row0, int rows, int k0, int lane) {
  for (int idx = lane; idx < rows * KT; idx += 32) {
    const int r = idx / KT, kk = idx - r * KT;
    const int row = row0 + r, k = k0 + kk;
    dst[idx] = (row < w.n_chan && k < w.n_poles) ? __ldcg(w.W + (size_t)row * w.ldw + k) : 0.0;
  }
}

// The same for channel-contiguous W: one pole-major panel [KT][TR_PITCH] of 32 channels.
__device__ __forceinline__ void stage_panel_plain_tr(double *dst, const DevWave &w, int row0, int k0, int lane) {
  for (int kk = 0; kk < KT; ++kk) {
    const int row = row0 + lane, k = k0 + kk;
    dst[kk * TR_PITCH + lane] = (row < w.n_chan && k < w.n_poles) ? __ldcg(w.W + (size_t)k * w.ldw + row) : 0.0;
  }
}

template <bool BATCH, int FAM>
__global__ void __launch_bounds__(NUM_THREADS, 1)
rmat_persistent_kernel(const __grid_constant__ DevWave single, const DevWave *__restrict__ waves,
                       const long long *__restrict__ item_begin, int n_waves, long long n_items,
                       unsigned long long *counter, const RingGeo geo) {
  extern __shared__ __align__(128) unsigned char smem[];   // used directly: the shared address space is kept (LDS/STS)
  const uint32_t bar0 = smem_u32(smem + SMEM_BARRIER_OFFSET);
  const uint32_t full0 = bar0, empty0 = bar0 + 8 * MAX_STAGES;
  const uint32_t item_full0 = bar0 + 16 * MAX_STAGES, item_empty0 = item_full0 + 16;
  ItemInfo *ring = reinterpret_cast<ItemInfo *>(smem + SMEM_ITEM_OFFSET);   // 2 slots of 128 B
  unsigned char *stages = smem + SMEM_RING_OFFSET;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < geo.n_stages; ++s) {
      mbar_init(full0 + 8 * s, 2);     // load warp (TMA expect_tx / plain staging done) + the pole-scaling warp whose turn it is
      mbar_init(empty0 + 8 * s, EB);   // one arrival per consumer warp
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(item_full0 + 8 * s, 1);
      mbar_init(item_empty0 + 8 * s, EB + PRODUCER_WARPS - 1);   // consumers + pole-scaling warps
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  Pipe ps;
  ps.ring = stages;
  ps.full0 = full0;
  ps.empty0 = empty0;
  ps.stage_bytes = geo.stage_bytes;
  ps.n_stages = geo.n_stages;

  if (warp >= EB) {
    // ================= producer warpgroup: give registers away =================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PRODUCER_REGS));
    if (warp == EB) {
      // ---- load warp: takes work items, publishes them, stages the W panels (S2, S5) ----
      uint32_t iq = 0, iphase = 0;
      long long next_static = blockIdx.x;
      unsigned long long next_drawn = 0;        // lane 0: the item this CTA does next (drawn ahead of time)
      if (counter != nullptr && lane == 0) next_drawn = atomicAdd(counter, 1ULL);
      int last_section = 0;
      constexpr int DRAW_AHEAD = 6;             // stages before the end of an item's loads at which the next item is drawn
      const uint64_t keep_policy = l2_policy_evict_last(), normal_policy = l2_policy_evict_normal();
      int last_wave = -1;
      for (;;) {
        // items are drawn from an atomic counter (batch call: in the workspace; single-wave call: a slot of
        // the library's counter pool), or round-robin when the single-wave call found no free slot.  The draw for
        // the NEXT item was issued a few stages before the end of the previous item's loads (below), so its
        // round trip to L2 is off the critical path of short items.
        long long item;
        if (counter != nullptr) {
          item = (long long)__shfl_sync(0xffffffffu, next_drawn, 0);
        } else {
          item = next_static;
          next_static += gridDim.x;
        }
        const bool stop = item >= n_items;
        // locate the section: [coarse items of wave 0, 1, ... | slab items of wave 0, 1, ... | fine items of wave 0, 1, ...]
        int p = 0, sec = 0;
        if (!stop) {
          if (BATCH) {
            // the counter only goes up, so the section of this CTA's next item is never before the last one's:
            // a short scan forward instead of a binary search (ten dependent loads from L2 per item)
            int lo = last_section;               // item_begin[lo] <= item < item_begin[3 n_waves]
            while (lo + 1 < 3 * n_waves && __ldg(item_begin + lo + 1) <= item) {
              lo = lo + 16 < 3 * n_waves && __ldg(item_begin + lo + 16) <= item ? lo + 16 : lo + 1;
            }
            last_section = lo;
            item -= __ldg(item_begin + lo);
            sec = lo / n_waves;
            p = lo - sec * n_waves;
          } else {
            const bool sp = single.n_pairs > 0;
            const long long n_coarse = sp ? pair_section_items(single, 0) : (long long)single.n_tiles * single.n_eb_coarse;
            const long long n_slab = sp ? pair_section_items(single, 1)
                                        : (long long)slab_tiles(single.slab_nt) * slab_groups(single.slab_g4, single.slab_g2, single.slab_g1);
            if (item >= n_coarse + n_slab) { sec = 2; item -= n_coarse + n_slab; }
            else if (item >= n_coarse) { sec = 1; item -= n_coarse; }
          }
        }
        const DevWave &w = BATCH ? waves[p] : single;
        int kind = -1, row0 = 0, col0 = 0, nblk = 0, nrb = 0, e_first = 0, n_valid = 0, n_kt = 0, slab_T = 0, slab_g = 0;
        if (!stop) {
          if (w.n_pairs > 0) {
            // pair form: section s holds (PT_M >> s)-pair tiles: 128-pair items, then the tail in 64-pair and last in
            // 32-pair items (rmat_common.h: pair_section_items)
            int mt, nt;
            pair_decode_item(w, sec, item, mt, nt);
            kind = 2;
            row0 = mt * (PT_M >> sec);
            col0 = nt * PT_N;
            const int left = w.n_pairs - row0;
            nblk = min(PT_M >> (sec + 3), left > 64 ? 16 : left > 32 ? 8 : 4);
            e_first = col0;
            n_valid = min(PT_N, w.n_E - col0);
          } else if (sec == 1) {
            // group-major: all tiles of the first group, then of the next -- the groups of four energies come first, so
            // the longest items do (largest-first list scheduling)
            const int n_st = slab_tiles(w.slab_nt);
            const int gi = (int)(item / n_st);
            const int tile = (int)(item - (long long)gi * n_st);
            decode_tile_slab(w, tile, kind, row0, col0);
            slab_T = w.slab_T;
            // groups of four energies first, then of two, then of one
            if (gi < w.slab_g4) {
              slab_g = 4;
              e_first = w.slab_e0 + 4 * gi;
            } else if (gi < w.slab_g4 + w.slab_g2) {
              slab_g = 2;
              e_first = w.slab_e0 + 4 * w.slab_g4 + 2 * (gi - w.slab_g4);
            } else {
              slab_g = 1;
              e_first = w.slab_e0 + 4 * w.slab_g4 + 2 * w.slab_g2 + (gi - w.slab_g4 - w.slab_g2);
            }
            n_valid = min(slab_g, w.n_E - e_first);             // (a group of four may hold three)
          } else {
            const bool fine = sec == 2;
            const int n_eb_sec = fine ? w.n_eb - w.n_eb_coarse : w.n_eb_coarse;
            const int tile = (int)(item / n_eb_sec);
            const int eb = (int)(item - (long long)tile * n_eb_sec) + (fine ? w.n_eb_coarse : 0);
            if (fine) {
              decode_tile_fine(w, tile, kind, row0, col0, nblk);
              nrb = kind == 0 ? nblk : TN / 8;                   // 8-row blocks of the I panel that are read
            } else {
              decode_tile(w, tile, kind, row0, col0, nblk, nrb);
            }
            e_first = eb * EB;
            n_valid = min(EB, w.n_E - e_first);
          }
          n_kt = w.n_kt;
        }
        mbar_wait(item_empty0 + 8 * iq, iphase ^ 1u);
        if (lane == 0) {
          ItemInfo &ii = ring[iq];
          ii.kind = (short)kind;
          if (!stop) {
            ii.R = w.R_out + (size_t)e_first * w.n_chan * w.n_chan;
            ii.diag_add = w.diag_add ? w.diag_add + (size_t)e_first * w.n_chan : nullptr;
            ii.done = w.done;
            ii.done_flag = w.done_flag;
            ii.done_target = w.done_target;
            ii.E_k = w.E_k;
            ii.energies = w.energies + e_first;
            ii.inv2a = w.inv2a;
            ii.n_chan = w.n_chan;
            ii.n_poles = w.n_poles;
            ii.n_valid_e = n_valid;
            ii.row0 = row0;
            ii.col0 = col0;
            ii.nrb = (unsigned char)nrb;
            ii.tr = (unsigned char)(kind == 2 ? 0 : w.tr);
            ii.n_pairs = w.n_pairs;
            ii.pair_rb = w.pair_rb;
            ii.pair_nm = w.pair_nm;
            ii.slab_T = (unsigned char)slab_T;
            ii.slab_g = (unsigned char)slab_g;
            ii.nblk = nblk;
            ii.n_kt = n_kt;
          }
          mbar_arrive(item_full0 + 8 * iq);   // release: the stores above are visible to waiters
        }
        iq ^= 1u;
        if (iq == 0) iphase ^= 1u;
        if (stop) break;

        const bool pair = kind == 2;
        const CUtensorMap *map = &w.map;
        if (BATCH && (w.use_tma || pair) && p != last_wave) {
          if (lane == 0) {
            if (pair) {
              tensormap_acquire(&w.map_P);
              tensormap_acquire(&w.map_D);
            } else {
              tensormap_acquire(map);
            }
          }
          __syncwarp();
          last_wave = p;
        }
        // panels of 32 channels to stage: I rows [row0, ...) into panels [0, i_boxes), J rows [col0, ...) into
        // panels [j_panel0, j_panel0 + j_boxes); boxes that lie wholly beyond n_chan are not loaded (nothing reads them)
        int i_boxes, j_boxes, j_panel0;
        if (pair) {
          i_boxes = (min(nblk * 8, w.n_pairs - row0) + TN - 1) / TN;      // rows of P
          j_boxes = (n_valid + TN - 1) / TN;                               // rows of D
          j_panel0 = PT_M / TN;
        } else if (slab_T != 0) {
          i_boxes = (min(slab_T, w.n_chan - row0) + TN - 1) / TN;
          j_boxes = kind != 0 ? (min(slab_T, w.n_chan - col0) + TN - 1) / TN : 0;
          j_panel0 = slab_T / TN;
        } else {
          i_boxes = (nrb + TN / 8 - 1) / (TN / 8);     // one to four boxes of 32 rows
          j_boxes = kind != 0 ? 1 : 0;
          j_panel0 = TW / TN;
        }
        const uint32_t box = (w.tr && !pair) ? TR_BOX_BYTES : BOX_BYTES;
        const uint32_t tx_bytes = (uint32_t)(i_boxes + j_boxes) * box;
        // host-buffer call: W uploaded so far.  Slabs of channels are waited for here, once per item (the rows and
        // columns of its tile); slabs of poles stage by stage below.
        const unsigned int *rows_ready = pair ? nullptr : w.rows_ready;   // (P and D are complete before the launch)
        const unsigned long long timeout_ns = (unsigned long long)(w.wait_timeout_ms ? w.wait_timeout_ms : 2000u) * 1000000ULL;
        unsigned int rows_seen = rows_ready ? 0u : 0xffffffffu;
        if (rows_ready && w.ready_counts_channels) {
          const int last = max(row0 + i_boxes * TN, kind != 0 ? col0 + j_boxes * TN : 0);
          wait_rows_uploaded(rows_ready, (unsigned int)min(last, w.n_chan), rows_seen, w.abort_flag, w.abort_flag_host, timeout_ns, lane);
          rows_seen = 0xffffffffu;
        }
        if (w.use_tma || pair) {
          // One box per lane: lane b < i_boxes + j_boxes issues box b of every stage.  Everything that does not
          // change from stage to stage is worked out here, so that a stage costs this warp a few dozen
          // instructions: items that spend only a few hundred cycles on a stage (slab tiles of edge 32) would
          // otherwise be bound by this loop.  TMA box coordinates: (pole, channel) for pole-contiguous W,
          // (channel, pole) for the H.DAT order.
          const int nb = i_boxes + j_boxes;
          const bool my_box = lane < nb;
          const int my_chan = lane < i_boxes ? row0 + lane * TN : col0 + (lane - i_boxes) * TN;
          const uint32_t my_dst = smem_u32(stages) + D_BYTES + (uint32_t)(lane < i_boxes ? lane : j_panel0 + (lane - i_boxes)) * box;
          const bool trl = w.tr && !pair;
          int c0 = trl ? my_chan : 0, c1 = trl ? 0 : my_chan;
          const int s0 = trl ? 0 : KT, s1 = trl ? KT : 0;
          if (pair) map = lane < i_boxes ? &w.map_P : &w.map_D;
          const uint64_t policy = w.l2_keep ? keep_policy : normal_policy;
          const int n_poles = w.n_poles;
          unsigned int *const abort_flag = w.abort_flag, *const abort_flag_host = w.abort_flag_host;
          const int draw_at = max(0, n_kt - DRAW_AHEAD);
          for (int kt = 0; kt < n_kt; ++kt) {
            if (kt == draw_at && counter != nullptr && lane == 0) next_drawn = atomicAdd(counter, 1ULL);
            if (rows_ready != nullptr)
              wait_rows_uploaded(rows_ready, (unsigned int)min(kt * KT + KT, n_poles), rows_seen, abort_flag, abort_flag_host, timeout_ns, lane);
            mbar_wait(ps.empty(), ps.phase ^ 1u);
            const uint32_t full = ps.full();
            if (lane == 0) mbar_arrive_expect_tx(full, tx_bytes);
            if (my_box) tma_load_2d_hint(my_dst + ps.stage * (uint32_t)ps.stage_bytes, map, c0, c1, full, policy);
            c0 += s0;
            c1 += s1;
            ps.advance();
          }
        } else {
          if (counter != nullptr && lane == 0) next_drawn = atomicAdd(counter, 1ULL);
          for (int kt = 0; kt < n_kt; ++kt) {
            const int k0 = kt * KT;
            wait_rows_uploaded(rows_ready, (unsigned int)min(k0 + KT, w.n_poles), rows_seen, w.abort_flag, w.abort_flag_host, timeout_ns, lane);
            mbar_wait(ps.empty(), ps.phase ^ 1u);
            double *sd = reinterpret_cast<double *>(stages + (size_t)ps.stage * ps.stage_bytes) + D_DOUBLES;
            if (w.tr) {
              for (int b = 0; b < i_boxes; ++b) stage_panel_plain_tr(sd + b * TR_BOX_DOUBLES, w, row0 + b * TN, k0, lane);
              for (int b = 0; b < j_boxes; ++b) stage_panel_plain_tr(sd + (j_panel0 + b) * TR_BOX_DOUBLES, w, col0 + b * TN, k0, lane);
            } else {
              stage_panel_plain(sd, w, row0, i_boxes * TN, k0, lane);
              if (j_boxes) stage_panel_plain(sd + j_panel0 * TN * KT, w, col0, j_boxes * TN, k0, lane);
            }
            __threadfence_block();   // all lanes' stores performed before lane 0 publishes the stage
            __syncwarp();
            if (lane == 0) mbar_arrive(ps.full());
            ps.advance();
          }
        }
      }
      // single-wave call with a pool counter: the last CTA to run dry hands the slot back zeroed
      if (!BATCH && counter != nullptr && lane == 0) {
        if (atomicAdd(counter + 1, 1ULL) == (unsigned long long)gridDim.x - 1) {
          counter[0] = 0ULL;
          counter[1] = 0ULL;
        }
      }
    } else {
      // ---- pole-scaling warps (S1): d_e[k] = 1/(E_k - E_e) of every stage, built in shared memory.
      // The three warps take the stages of an item in turn (warp j the k-tiles j, j + 3, ...), lane = pole of the
      // tile, a loop over the item's energies.  An FP64 division is a dependent chain of some 300 cycles; a warp
      // computes the divisions of its NEXT stage right after it has handed the current one over, so that chain runs
      // while the warp waits for its next empty slot, and with three warps in turn a stage can be handed over
      // every ~100 cycles -- slab items of edge 32 consume one every ~300 (classic items every 5000).
      constexpr int DW = PRODUCER_WARPS - 1;                 // 3 warps
      const int sw = warp - EB - 1;
      const bool pole_lane = lane < KT;
      uint32_t iq = 0, iphase = 0;
      for (;;) {
        mbar_wait(item_full0 + 8 * iq, iphase);
        const ItemInfo it = ring[iq];
        __threadfence_block();       // the copy above has been read before the slot is handed back
        __syncwarp();
        if (lane == 0) mbar_arrive(item_empty0 + 8 * iq);
        iq ^= 1u;
        if (iq == 0) iphase ^= 1u;
        if (it.kind < 0) break;
        if (it.kind == 2) {
          // pair item: D comes from scratch, there is nothing to scale -- this warp only signs its stages off
          int turn = sw;
          for (int kt = 0; kt < it.n_kt; ++kt) {
            if (turn == 0) {
              mbar_wait(ps.empty(), ps.phase ^ 1u);
              __syncwarp();
              if (lane == 0) mbar_arrive(ps.full());
              turn = DW;
            }
            --turn;
            ps.advance();
          }
          continue;
        }
        const int nv = it.n_valid_e;
        double en[EB], dv[EB];
#pragma unroll
        for (int e = 0; e < EB; ++e) en[e] = (pole_lane && e < nv) ? __ldg(it.energies + e) : 0.0;
        auto load_pole = [&](int kt) -> double {
          const int k = kt * KT + lane;
          return (pole_lane && kt < it.n_kt && k < it.n_poles) ? __ldg(it.E_k + k) : 0.0;
        };
        auto scale = [&](int kt, double ek) {
          // 0 beyond n_poles so that zero-filled W columns stay zero; energy slots beyond the item's are never read
          const bool ok = pole_lane && kt * KT + lane < it.n_poles;
#pragma unroll
          for (int e = 0; e < EB; ++e)
            if (e < nv) dv[e] = ok ? 1.0 / (ek - en[e]) : 0.0;
        };
        scale(sw, load_pole(sw));
        double ek_next = load_pole(sw + DW);                 // poles are fetched two turns ahead (an L2 round trip)
        int turn = sw;                                       // k-tiles until this warp's next stage
        for (int kt = 0; kt < it.n_kt; ++kt) {
          if (turn == 0) {
            const double ek_after = load_pole(kt + 2 * DW);
            mbar_wait(ps.empty(), ps.phase ^ 1u);
            double *dsm = reinterpret_cast<double *>(stages + (size_t)ps.stage * ps.stage_bytes);   // d is first in a stage
            if (pole_lane) {
#pragma unroll
              for (int e = 0; e < EB; ++e)
                if (e < nv) dsm[e * KT + lane] = dv[e];
            }
            __threadfence_block();     // every lane's d has been written before lane 0 arrives
            __syncwarp();
            if (lane == 0) mbar_arrive(ps.full());
            scale(kt + DW, ek_next);
            ek_next = ek_after;
            turn = DW;
          }
          --turn;
          ps.advance();
        }
      }
    }
  } else {
    // ================= consumer warps =================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CONSUMER_REGS));
    uint32_t iq = 0, iphase = 0;
    for (;;) {
      mbar_wait(item_full0 + 8 * iq, iphase);
      const ItemInfo it = ring[iq];
      if (it.kind < 0) break;
      consume_item<FAM>(it, ps, warp, lane);
      if (it.done != nullptr) {
        // host-buffer call: the host copies a wave's R back as soon as its last item has been stored.  Every warp
        // makes its stores visible device-wide and counts itself in; the arrival that completes the wave raises
        // the wave's flag in host-mapped memory, which the calling thread polls.
        __threadfence();
        __syncwarp();
        if (lane == 0 && atomicAdd(it.done, 1u) + 1u == it.done_target) {
          __threadfence_system();
          *reinterpret_cast<volatile unsigned int *>(it.done_flag) = 1u;
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(item_empty0 + 8 * iq);
      iq ^= 1u;
      if (iq == 0) iphase ^= 1u;
    }
  }
}

}  // namespace pstgf
