// rmat_common.h -- tile constants and the device-visible tables shared by the host planner
// and the sm_100a kernel of libpstgf_rmat.so.  (Not shared with oracle/: that is a separate
// C translation unit with no includes from here.)
//
// Work decomposition of eq. 4 for one partial wave with C = n_chan,
// K = n_poles, N = n_E:
//   coarse tiles DIAG(i)    rows/cols [64 i, 64 i + 64): upper triangle of 8x8 DMMA blocks
//                WIDE(p, c) rows [128 p, 128 p + 128) x cols [128 (p + 1) + 16 c, + 16): everything to the
//                           right of the p-th pair of DIAG tiles; one scaled B fragment feeds 16 DMMAs
//                OFF(p, t)  rows [128 p, 128 p + 64) x cols [128 p + 64 + 32 t, + 32), t = 0, 1: the square
//                           between the two DIAG tiles of a pair
//   fine tiles   OFF32(i,j) rows [32 i, 32 i + 32) x cols [32 j, 32 j + 32), j > i
//                DIAG32(i)  rows/cols [32 i, 32 i + 32)
//   energy block EB = 8 consecutive energies, one per consumer warp
//   item         (wave, tile, energy block).  The first n_eb_coarse energy blocks of a wave are cut
//                into coarse tiles, the remaining ones (the "tail", sized by the planner to about one
//                round of the grid) into fine tiles of 16/36 and 10/36 of a coarse item's cost, and all
//                fine items are handed out after all coarse ones: largest-first list scheduling ends
//                on small items, so the CTAs finish together.  Inside a section the item index is
//                tile * n_eb_section + eb (energy-fastest: CTAs running side by side share one W tile
//                in L2).  An R element has the same operands and k order in both tilings (bitwise
//                the same result).
// Only tiles on or above the diagonal exist ("half of the symmetric R-matrix"),
// the mirror is written by the epilogue ("symmetrised").
#pragma once
#include <cuda.h>
#include <stdint.h>

namespace pstgf {

constexpr int TM = 64;      // DIAG / OFF tile rows
constexpr int TN = 32;      // OFF tile columns: J panel; also the TMA box height
constexpr int TW = 128;     // WIDE tile rows (the I panel region of a stage holds this many rows)
constexpr int TWN = 16;     // WIDE tile columns
constexpr int KT = 20;      // poles per pipeline stage; row pitch 20 doubles == 4 (mod 16) -> conflict-free LDS.64
constexpr int EB = 8;       // energies per item == consumer warps per CTA
constexpr int STAGES = 7;   // smem ring depth
constexpr int PRODUCER_WARPS = 4;                    // one warpgroup: 1 load warp + 3 pole-scaling warps
constexpr int NUM_THREADS = (EB + PRODUCER_WARPS) * 32;   // 8 consumer warps + the producer warpgroup
constexpr int PRODUCER_REGS = 56;                    // setmaxnreg targets: 8*224 + 4*56 = 12*168, the launch allocation
constexpr int CONSUMER_REGS = 224;
constexpr int BOX_BYTES = TN * KT * 8;               // one TMA box: 32 rows x 20 poles
constexpr int WI_BYTES = TW * KT * 8;                // I panel region: four boxes
constexpr int WJ_BYTES = TN * KT * 8;
constexpr int D_BYTES = EB * KT * 8;                 // d_e[k] = 1/(E_k - E_e) for the stage
// Channel-contiguous W (the H.DAT record order) is staged pole-major: five panels
// [KT poles][TR_PITCH channels] (I rows 0..31, 32..63, 64..95, 96..127, J), each one TMA box of 36 channels x 20 poles
// (32 used + 4 spare: the row pitch 36 == 4 (mod 16) doubles keeps the LDS.64 fragment loads conflict-free).
constexpr int TR_PITCH = TN + 4;
constexpr int TR_BOX_BYTES = KT * TR_PITCH * 8;      // 5760
constexpr int STAGE_BYTES_ROWMAJOR = WI_BYTES + WJ_BYTES + D_BYTES;   // 26880
constexpr int STAGE_BYTES_TR = 5 * TR_BOX_BYTES + D_BYTES;            // 30080
constexpr int STAGE_BYTES = STAGE_BYTES_TR > STAGE_BYTES_ROWMAJOR ? STAGE_BYTES_TR : STAGE_BYTES_ROWMAJOR;

// Offsets (in doubles) inside a stage, per layout.  i_off / j_off are additive in (row, k): the offset of
// element (8 bi + g, 4 ks + q) is off(g, q) + off(8 bi, 4 ks).
template <bool TR>
struct StageLayout {
  static constexpr int J_BASE = TR ? 4 * KT * TR_PITCH : TW * KT;
  static constexpr int D_BASE = TR ? 5 * KT * TR_PITCH : (TW + TN) * KT;
  __host__ __device__ static constexpr int i_off(int r, int k) {
    return TR ? (r >> 5) * KT * TR_PITCH + k * TR_PITCH + (r & 31) : r * KT + k;
  }
  __host__ __device__ static constexpr int j_off(int c, int k) { return TR ? k * TR_PITCH + c : c * KT + k; }
};
constexpr int SMEM_BARRIER_OFFSET = STAGES * STAGE_BYTES;
constexpr int SMEM_ITEM_OFFSET = SMEM_BARRIER_OFFSET + (2 * STAGES + 4) * 8;
constexpr int SMEM_BYTES = SMEM_ITEM_OFFSET + 2 * 96 + 128;  // two ItemInfo slots + alignment slack

// One partial wave as the kernel sees it.  Built on the host, lives in kernel parameter
// space (single-wave call) or in the caller's workspace (batch call).
struct alignas(128) DevWave {
  CUtensorMap map;         // W viewed as [n_chan][n_poles] (row stride ldw*8), box [TN][KT], no swizzle (tr: see below)
  const double *W;
  const double *E_k;
  const double *energies;
  double *R_out;
  unsigned int *done;      // optional completion counter of this wave (host-buffer call): += 1 per consumer warp and item
  unsigned int *done_flag; // ... and the (host-mapped) word that is set to 1 by the arrival that makes it done_target
  const unsigned int *rows_ready;   // optional (host-buffer call): how much of W has been uploaded so far, see the load warp
  long long ldw;
  double inv2a;            // 1/(2a), PAPER.md:108 prefactor
  int n_chan, n_poles, n_E;
  int n_kt;                // ceil(n_poles / KT)
  int n_i;                 // ceil(n_chan / TM): DIAG tiles
  int n_j;                 // ceil(n_chan / TN)
  int n_eb;                // ceil(n_E / EB)
  int n_tiles;             // coarse tiles: n_i DIAG + WIDE + OFF
  int use_tma;             // W 16-byte aligned and ldw even
  int n_eb_coarse;         // energy blocks [0, n_eb_coarse) use coarse tiles, [n_eb_coarse, n_eb) fine tiles
  unsigned int done_target;
  int ready_counts_channels;   // what rows_ready counts: 0 poles uploaded, 1 channels (rows of a pole-contiguous W)
  int tr;                  // 1: W is channel-contiguous [n_poles][ldw] (H.DAT record order), map box [KT][TR_PITCH]
};
static_assert(sizeof(DevWave) == 256, "DevWave layout");

// Host-side tile arithmetic (also used by the kernel's decoder).
// WIDE tiles of row pair p: columns from 128 (p + 1) to the end, 16 at a time.
__host__ __device__ inline int wide_tiles_in_pair(int n_chan, int p) {
  const int left = n_chan - TW * (p + 1);
  return left > 0 ? (left + TWN - 1) / TWN : 0;
}
// OFF tiles of row pair p: the (up to) 64 columns [128 p + 64, 128 p + 128), 32 at a time.
__host__ __device__ inline int off_tiles_in_pair(int n_chan, int p) {
  int left = n_chan - (TW * p + TM);
  left = left > TM ? TM : left;
  return left > 0 ? (left + TN - 1) / TN : 0;
}
__host__ __device__ inline int coarse_tiles(int n_chan) {
  int n = (n_chan + TM - 1) / TM;
  for (int p = 0; TW * p + TM < n_chan; ++p) n += wide_tiles_in_pair(n_chan, p) + off_tiles_in_pair(n_chan, p);
  return n;
}
// Fine tiling: n_j row/column panels of 32; OFF32 tiles first (n_j (n_j - 1) / 2), then DIAG32 (n_j).
__host__ __device__ inline int fine_tiles(int n_j) { return n_j * (n_j - 1) / 2 + n_j; }

// Relative cost of one item in DMMA.8x8x4 per k-step of 4 and energy: coarse DIAG 36, coarse OFF 32,
// fine OFF 16, fine DIAG 10 (full-size tiles; ragged edge tiles are cheaper).
constexpr int COST_DIAG = 36, COST_OFF = 32, COST_WIDE = 32, COST_OFF32 = 16, COST_DIAG32 = 10;

}  // namespace pstgf
