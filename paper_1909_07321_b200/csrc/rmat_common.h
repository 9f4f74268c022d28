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
//   slab tiles   the energies that do not fill a block of 8 (n_E mod 8, and every energy of a call with
//                n_E < 8: PSTGF calls RINIT once per (wave, energy)) are taken in groups
//                of g = 4, 2 or 1 energies, and the eight consumer warps split the TILE instead of the energy
//                block: square tiles S(i, j), j >= i, of edge T = 128, 64 or 32 chosen by the planner so that
//                there are enough items for the grid; the 8 / g warps of one energy each take a slab of the
//                tile (SlabShape below).  Same operands, same k order: same bits as inside a block of 8.
//   pair items   waves with FEW channels (n_chan <= PAIR_MAX_CHAN) and enough energies are not done in the SYRK form
//                above at all: an n_chan x n_chan tile there computes whole 8x8 blocks across the diagonal (36
//                blocks for 32 counted at n_chan = 64, 1 for 1/2 at n_chan = 8) and pays a scaling multiply
//                for every few DMMAs.  Eq. 4 is also the plain GEMM over channel PAIRS
//                    R[e][(n,m)] = (1/2a) sum_k P[(n,m)][k] * D[e][k],   P = w_nk w_mk,  D = 1/(E_k - E_e),
//                with the n_chan (n_chan + 1) / 2 pairs n <= m as rows and the energies as columns: no block is
//                cut by a diagonal and nothing is scaled inside the k loop.  P (once per wave) and D (once per
//                energy) are written to scratch by a small kernel first; an item is (128, 64 or 32 pairs) x 128
//                energies, each of the eight warps taking 16 energies (the WIDE register tile, 16 x 2 blocks, or 8 x 2,
//                4 x 2): 128-pair items first, then a tail of 64-pair and last of 32-pair items.
// Only tiles on or above the diagonal exist ("half of the symmetric R-matrix"),
// the mirror is written by the epilogue ("symmetrised").
#pragma once
#include <cuda.h>
#include <stdint.h>

namespace pstgf {

constexpr int TM = 64;      // DIAG / OFF tile rows
constexpr int TN = 32;      // OFF tile columns: J panel; also the TMA box height
constexpr int TW = 128;     // WIDE tile rows (the I panel region of a classic stage holds this many rows)
constexpr int TWN = 16;     // WIDE tile columns
constexpr int KT = 20;      // poles per pipeline stage; row pitch 20 doubles == 4 (mod 16) -> conflict-free LDS.64
constexpr int EB = 8;       // energies per item == consumer warps per CTA
constexpr int MAX_STAGES = 16;  // smem ring depth: as many stages as fit (7 classic, 5 with 128-row slab tiles, 16 with 32-row ones)
constexpr int PRODUCER_WARPS = 4;                    // one warpgroup: 1 load warp + 3 pole-scaling warps
constexpr int NUM_THREADS = (EB + PRODUCER_WARPS) * 32;   // 8 consumer warps + the producer warpgroup
constexpr int PRODUCER_REGS = 56;                    // setmaxnreg targets: 8*224 + 4*56 = 12*168, the launch allocation
constexpr int CONSUMER_REGS = 224;
constexpr int BOX_BYTES = TN * KT * 8;               // one TMA box: 32 rows x 20 poles
constexpr int D_DOUBLES = EB * KT;                   // d_e[k] = 1/(E_k - E_e) for the stage: first thing in a stage
constexpr int D_BYTES = D_DOUBLES * 8;               // 1280 = 10 x 128: the panels behind it keep their bank pattern
// Channel-contiguous W (the H.DAT record order) is staged pole-major: panels
// [KT poles][TR_PITCH channels], each one TMA box of 36 channels x 20 poles
// (32 used + 4 spare: the row pitch 36 == 4 (mod 16) doubles keeps the LDS.64 fragment loads conflict-free).
constexpr int TR_PITCH = TN + 4;
constexpr int TR_BOX_BYTES = KT * TR_PITCH * 8;      // 5760
constexpr int TR_BOX_DOUBLES = KT * TR_PITCH;

// A stage is [d 8 x 20 | panels of 32 channels x 20 poles].  Classic items use panels 0..3 for the I rows and
// panel 4 for the J rows; slab items of edge T use panels [0, T/32) for the I rows and [T/32, 2 T/32) for J.
// Offsets (in doubles) of element (row r, pole k) of the panel region; additive in (r, k) for 8-aligned r:
// off(8 b + g, 4 s + q) = off(g, q) + off(8 b, 4 s).
template <bool TR>
struct StageLayout {
  static constexpr int PANEL = TR ? TR_BOX_DOUBLES : TN * KT;       // doubles per panel of 32 channels
  static constexpr int PANEL_BYTES = PANEL * 8;
  static constexpr int W_BASE = D_DOUBLES;                          // panels start behind d
  static constexpr int J_CLASSIC = W_BASE + (TW / TN) * PANEL;      // classic items: J panel behind four I panels
  __host__ __device__ static constexpr int off(int r, int k) {
    return TR ? (r >> 5) * TR_BOX_DOUBLES + k * TR_PITCH + (r & 31) : r * KT + k;
  }
};
constexpr int stage_bytes_for(bool tr, int panels) { return D_BYTES + panels * (tr ? TR_BOX_BYTES : BOX_BYTES); }
constexpr int CLASSIC_PANELS = TW / TN + 1;          // 5
constexpr int slab_panels(int T) { return 2 * (T / TN); }   // 8, 4, 2 for slab tiles of edge 128, 64, 32
// Pair form (see above): pair tiles of 128 (coarse) or 64 (fine tail) rows of P, energy tiles of 128 rows of D.
constexpr int PAIR_MAX_CHAN = 96;        // 4656 pairs; P is 71 MB at n_poles = 20 n_chan
constexpr int PAIR_MIN_E = 64;           // fewer energies than this do not fill an energy tile's eight warps
constexpr int PT_M = 128, PT_MF = 64, PT_MFF = 32, PT_N = 128;   // pair tile rows of section s: PT_M >> s
constexpr int PAIR_PANELS = (PT_M + PT_N) / TN;             // 8
// Tiny waves (pair form, at most SMALL_MAX_CHAN channels, little work in all) are done by a kernel of their own
// (rmat_small.cu): one CTA per block of 8 energies, at most SMALL_MAX_WARPS warps that split the blocks of 8 pairs.
constexpr int SMALL_MAX_CHAN = 16;       // 136 pairs: 17 blocks of 8
constexpr int SMALL_MAX_WARPS = 6;
// Item families a launch can hold; the persistent kernel is compiled once per value (a template parameter), so that a
// launch of classic items only does not carry the code of the others.
constexpr int FAM_CLASSIC = 0, FAM_SLAB = 1, FAM_PAIR = 2;

// Shared memory of a CTA: [mbarriers | two ItemInfo slots | ring of n_stages stages]; the ring geometry is a launch
// parameter (RingGeo) because slab tiles of edge 128 need 8 panels per stage instead of 5.
constexpr int SMEM_BARRIER_OFFSET = 0;               // (2 MAX_STAGES + 4) x 8 B = 288
constexpr int SMEM_ITEM_OFFSET = 384;                // 2 x 128 B
constexpr int SMEM_RING_OFFSET = 640;
constexpr int SMEM_ALIGN_SLACK = 128;
constexpr int SMEM_MAX_OPTIN = 232448;               // 227 KB
struct RingGeo {
  int stage_bytes;
  int n_stages;
};
constexpr int smem_bytes_for(RingGeo g) { return SMEM_RING_OFFSET + g.n_stages * g.stage_bytes + SMEM_ALIGN_SLACK; }

// How the 8 / g consumer warps of one energy share a slab tile of edge T: a grid of wr x wc warps, each
// computing NR row blocks x NCW column blocks of 8 x 8 (predicated on the diagonal and at the matrix edge).
struct SlabShape {
  int wc;    // warps across the columns
  int nr;    // row blocks per warp: 16, 8, 4 or 2
  int ncw;   // column blocks per warp: 2 or 1
};
__host__ __device__ inline SlabShape slab_shape(int T, int g) {
  if (T == 128) return SlabShape{8, 16, 2};                 // g = 1 only: 8 warps x (16 x 2 blocks), the WIDE register tile
  if (T == 64) return g == 1 ? SlabShape{4, 4, 2} : g == 2 ? SlabShape{4, 8, 2} : SlabShape{2, 8, 4};
  // T == 32: 2 x 2 warps of 2 x 2 blocks for one or two energies.  With one energy that leaves four of the eight warps
  // idle, on purpose: 8 warps of 2 x 1 blocks issue 4 LDS.64 per 2 DMMA each, which is all of the SM's shared-memory
  // bandwidth (ncu: 48 % of its peak at 52 % DMMA utilisation); 2 x 2 blocks need 5 per 4.  Four energies: two warps
  // of 4 x 2 blocks each.
  return g == 4 ? SlabShape{2, 4, 2} : SlabShape{2, 2, 2};
}
// slab groups of a wave: all of them, and the number of energies in front of group gi
__host__ __device__ inline int slab_groups(int g4, int g2, int g1) { return g4 + g2 + g1; }

// One partial wave as the kernel sees it.  Built on the host, lives in kernel parameter
// space (single-wave call) or in the caller's workspace (batch call).
struct alignas(128) DevWave {
  CUtensorMap map;         // W viewed as [n_chan][n_poles] (row stride ldw*8), box [TN][KT], no swizzle (tr: see below)
  CUtensorMap map_P;       // pair form: P viewed as [n_pairs][n_poles] (row stride pair_ld*8), box [TN][KT]
  CUtensorMap map_D;       // pair form: D viewed as [n_E][n_poles] (row stride pair_ld*8), box [TN][KT]
  const double *W;
  const double *E_k;
  const double *energies;
  double *R_out;
  const double *diag_add;  // optional [n_E][n_chan]: added to R_nn after the 1/(2a) scale (Buttle-type correction)
  unsigned int *done;      // optional completion counter of this wave (host-buffer call): += 1 per consumer warp and item
  unsigned int *done_flag; // ... and the (host-mapped) word that is set to 1 by the arrival that makes it done_target
  const unsigned int *rows_ready;   // optional (host-buffer call): how much of W has been uploaded so far, see the load warp
  unsigned int *abort_flag;         // host-buffer call: DEVICE word set to 1 by a load warp whose wait for an upload timed out
  unsigned int *abort_flag_host;    // ... and the host-mapped word that warp sets as well (written once, never polled by the device)
  long long ldw;
  double inv2a;            // 1/(2a), PAPER.md:108 prefactor
  int n_chan, n_poles, n_E;
  int n_kt;                // ceil(n_poles / KT)
  int n_i;                 // ceil(n_chan / TM): DIAG tiles
  int n_j;                 // ceil(n_chan / TN)
  int n_eb;                // energy blocks of 8 handled by classic items (n_E / 8, or ceil when the remainder is not slabbed)
  int n_tiles;             // coarse tiles: n_i DIAG + WIDE + OFF
  int use_tma;             // W 16-byte aligned and ldw even
  int n_eb_coarse;         // energy blocks [0, n_eb_coarse) use coarse tiles, [n_eb_coarse, n_eb) fine tiles
  unsigned int done_target;
  int ready_counts_channels;   // what rows_ready counts: 0 poles uploaded, 1 channels (rows of a pole-contiguous W)
  int tr;                  // 1: W is channel-contiguous [n_poles][ldw] (H.DAT record order), map box [KT][TR_PITCH]
  int slab_e0;             // first energy handled by slab items (8 n_eb, or n_E when there are none)
  int slab_g4, slab_g2, slab_g1;   // groups of four energies (the last of them may hold three), then of two, then of one
  int slab_T;              // tile edge of the slab items: 128, 64 or 32
  int slab_nt;             // ceil(n_chan / slab_T): slab tiles = slab_nt (slab_nt + 1) / 2
  int l2_keep;             // W fits half of L2: load it with the evict_last policy so that R's stores do not push it out
  unsigned int wait_timeout_ms;   // bound on a load warp's wait for an upload slab (0 = 2000)
  // pair form (n_pairs > 0: this wave has pair items and no others)
  double *pair_P;          // scratch [n_pairs][pair_ld]: P[(n,m)][k] = w_nk w_mk, pairs row by row over the upper triangle
  double *pair_D;          // scratch [n_E][pair_ld]:     D[e][k] = 1/(E_k - E_e)
  long long pair_ld;       // even, >= n_poles
  int n_pairs;             // n_chan (n_chan + 1) / 2, or 0 when the wave is done in the SYRK form
  int pair_nt;             // energy tiles of PT_N
  int pair_nt_coarse;      // energy tiles [0, pair_nt_coarse) are cut into pair tiles of PT_M rows (section 0), ...
  int pair_nt_mid;         // ... [pair_nt_coarse, pair_nt_mid) of PT_MF rows (section 1), the rest of PT_MFF rows (section 2)
  int pair_mt, pair_mtf, pair_mtff;   // pair tiles of PT_M / PT_MF / PT_MFF rows
  int pair_x0;             // the first pair_x0 128-pair tiles of energy tile pair_nt_coarse are section-0 items too (< pair_mt; 0 unless pair_nt_coarse < pair_nt_mid)
  int pair_x1;             // the first pair_x1 64-pair tiles of energy tile pair_nt_mid are section-1 items too (< pair_mtf; 0 unless pair_nt_mid < pair_nt)
  int pair_nfb;            // n_chan / 8: channel blocks that are full
  int pair_rb;             // rows of P in the block section: 64 pair_nfb (pair_nfb - 1) / 2, see pair_row_channels
  int pair_keep_P;         // 1: P and pair_nm are there already (built once for the wave, shared by its energy ranges): the scratch builder writes D only
  const unsigned int *pair_nm;   // scratch [n_pairs]: n | m << 16 of every row of P (written by the scratch builder)
};
static_assert(sizeof(DevWave) == 768, "DevWave layout (alignas 128; the batch workspace holds an array of these)");

// Pair form: the items of a wave, section by section.  Section s holds (PT_M >> s)-pair tiles: section 0 the energy
// tiles [0, pair_nt_coarse) and the first pair_x0 tiles of energy tile pair_nt_coarse; section 1 the rest of that energy
// tile (its 64-pair tiles from 2 pair_x0 on), the energy tiles up to pair_nt_mid and the first pair_x1 tiles of energy
// tile pair_nt_mid; section 2 the rest.  The ragged boundaries let the planner end each section after any number of
// items, not only after whole energy tiles: with 3.7 rounds of 128-pair items on the grid (config 2) that is worth 5 %.
__host__ __device__ inline long long pair_section_items(const DevWave &w, int sec) {
  if (sec == 0) return (long long)w.pair_mt * w.pair_nt_coarse + w.pair_x0;
  const int x = sec == 1 ? w.pair_x0 : w.pair_x1, tiles = sec == 1 ? w.pair_mtf : w.pair_mtff;
  const int first = sec == 1 ? w.pair_nt_coarse : w.pair_nt_mid, end = sec == 1 ? w.pair_nt_mid : w.pair_nt;
  return (x > 0 ? tiles - 2 * x : 0) + (long long)tiles * (end - first - (x > 0 ? 1 : 0)) + (sec == 1 ? w.pair_x1 : 0);
}
// item of section sec -> (pair tile mt in units of PT_M >> sec rows, energy tile nt)
__host__ __device__ inline void pair_decode_item(const DevWave &w, int sec, long long item, int &mt, int &nt) {
  if (sec == 0) {
    const long long reg = (long long)w.pair_mt * w.pair_nt_coarse;
    if (item < reg) {                      // energy tile fastest: CTAs side by side share a P panel
      mt = (int)(item / w.pair_nt_coarse);
      nt = (int)(item - (long long)mt * w.pair_nt_coarse);
    } else {
      mt = (int)(item - reg);
      nt = w.pair_nt_coarse;
    }
    return;
  }
  const int x = sec == 1 ? w.pair_x0 : w.pair_x1, tiles = sec == 1 ? w.pair_mtf : w.pair_mtff;
  const int first = sec == 1 ? w.pair_nt_coarse : w.pair_nt_mid, end = sec == 1 ? w.pair_nt_mid : w.pair_nt;
  const int first_cnt = x > 0 ? tiles - 2 * x : 0;
  if (item < first_cnt) {
    nt = first;
    mt = 2 * x + (int)item;
    return;
  }
  item -= first_cnt;
  const int r0 = first + (x > 0 ? 1 : 0), n_reg = end - r0;
  const long long reg = (long long)tiles * n_reg;
  if (item < reg) {
    mt = (int)(item / n_reg);
    nt = r0 + (int)(item - (long long)mt * n_reg);
  } else {
    mt = (int)(item - reg);
    nt = end;
  }
}

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
// Order of the pairs (n, m), n <= m, as rows of P.  First the BLOCK section: the off-diagonal 8 x 8 blocks of
// channels (bn < bm < nfb = C / 8) one after the other, (0,1), (0,2), ..., (1,2), ..., 64 rows each, row 8 j + i of
// a block being the pair (8 bn + j, 8 bm + i).  A warp's 8 x 8 accumulator blocks of such a group then hold an
// 8 x 8 patch of R: R[n][m .. m+7] lies across eight lanes (a 64-byte run) and the mirror R[m][n .. n+7] in ONE lane's
// eight accumulators (a 64-byte run again, vector stores) -- both triangles are written in full sectors.  Then the
// LOOSE section: what is left (the triangles of the diagonal blocks and the strip of a ragged last block), row by
// row of the upper triangle; those rows go through a table (DevWave::pair_nm) and are stored element by element.
__host__ __device__ inline int pair_block_rows(int C) { const int nfb = C / 8; return 64 * (nfb * (nfb - 1) / 2); }
// loose pairs of channel row n: m from n to the end of n's own 8-block, plus the ragged strip m >= 8 nfb
__host__ __device__ inline int pair_loose_in_row(int n, int C) {
  const int nfb = C / 8, own_end = (n / 8 + 1) * 8 < C ? (n / 8 + 1) * 8 : C;
  return (own_end - n) + (n / 8 < nfb && 8 * nfb < C && own_end <= 8 * nfb ? C - 8 * nfb : 0);
}
// row r of P -> (n, m); O(C) for loose rows (used by the scratch builder, which records the answer in pair_nm)
__host__ __device__ inline void pair_row_channels(int r, int C, int &n, int &m) {
  const int nfb = C / 8, rb = pair_block_rows(C);
  if (r < rb) {
    int blk = r >> 6, bn = 0;
    while (blk >= nfb - 1 - bn) { blk -= nfb - 1 - bn; ++bn; }
    n = 8 * bn + ((r >> 3) & 7);
    m = 8 * (bn + 1 + blk) + (r & 7);
    return;
  }
  int l = r - rb;
  for (n = 0; n < C - 1; ++n) {
    const int cnt = pair_loose_in_row(n, C);
    if (l < cnt) break;
    l -= cnt;
  }
  const int own_end = (n / 8 + 1) * 8 < C ? (n / 8 + 1) * 8 : C;
  m = l < own_end - n ? n + l : 8 * nfb + (l - (own_end - n));
}
// Slab tiling: nt row/column panels of T; tiles row by row over the upper triangle, (0,0), (0,1), ..., (1,1), ...
__host__ __device__ inline int slab_tiles(int nt) { return nt * (nt + 1) / 2; }

// Relative cost of one item in DMMA.8x8x4 per k-step of 4 and energy: coarse DIAG 36, coarse OFF 32,
// fine OFF 16, fine DIAG 10 (full-size tiles; ragged edge tiles are cheaper).
constexpr int COST_DIAG = 36, COST_OFF = 32, COST_WIDE = 32, COST_OFF32 = 16, COST_DIAG32 = 10;

}  // namespace pstgf
