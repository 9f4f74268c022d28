// pstgf_rmat.cu -- C ABI of libpstgf_rmat.so (include/pstgf_rmat.h): argument checks, the host
// planner (tile / item tables, TMA descriptors) and the launches of the sm_100a kernel in
// rmat_kernel.cuh.  Eq. 4 of arxiv 1909.07321.
#include <cuda_runtime.h>
#include <cuda.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <map>
#include <queue>
#include <tuple>
#include <mutex>
#include <numeric>
#include <thread>
#include <vector>
#include <chrono>

#include "../../include/pstgf_rmat.h"
#include "rmat_aux.cuh"
#include "rmat_launch.h"

namespace {

using pstgf::DevWave;

thread_local int tl_cuda_error = 0;
thread_local int tl_launches = 0;

pstgf_status_t cuda_fail(cudaError_t e) {
  tl_cuda_error = (int)e;
  (void)cudaGetLastError();
  return PSTGF_ERR_CUDA;
}
#define PSTGF_CUDA(expr)                                  \
  do {                                                    \
    cudaError_t e_ = (expr);                              \
    if (e_ != cudaSuccess) return cuda_fail(e_);          \
  } while (0)

}  // namespace
void pstgf::set_last_call_state(int launches, int cuda_error) {
  tl_launches = launches;
  tl_cuda_error = cuda_error;
}
namespace {

// ---- device / driver state -----------------------------------------------------------------
typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct DeviceState {
  int device = -1;
  int sm_count = 0;
  int l2_bytes = 0;
  bool ok = false;
};

encode_tiled_fn g_encode = nullptr;
std::once_flag g_encode_once;
std::mutex g_attr_mutex;
bool g_attr_set[64] = {false};

pstgf_status_t device_state(DeviceState &ds) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    tl_cuda_error = (int)e;
    (void)cudaGetLastError();
    return PSTGF_ERR_UNSUPPORTED_DEVICE;
  }
  int major = 0, sms = 0;
  PSTGF_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  PSTGF_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (major != 10) return PSTGF_ERR_UNSUPPORTED_DEVICE;
  int l2 = 0;
  PSTGF_CUDA(cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev));
  ds.l2_bytes = l2;
  std::call_once(g_encode_once, [] {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      g_encode = reinterpret_cast<encode_tiled_fn>(fn);
  });
  if (!g_encode) return PSTGF_ERR_UNSUPPORTED_DEVICE;
  {
    std::lock_guard<std::mutex> lock(g_attr_mutex);
    if (dev < 64 && !g_attr_set[dev]) {
      PSTGF_CUDA(pstgf::persistent_prepare_all());
      g_attr_set[dev] = true;
    }
  }
  ds.device = dev;
  ds.sm_count = sms;
  ds.ok = true;
  return PSTGF_OK;
}

// ---- argument checks -----------------------------------------------------------------------
bool aligned8(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 7u) == 0; }

pstgf_status_t check_wave(const pstgf_wave_t &w) {
  if (w.n_chan < 0 || w.n_poles < 0 || w.n_E < 0) return PSTGF_ERR_INVALID_VALUE;
  if (!(w.a > 0.0) || !std::isfinite(w.a)) return PSTGF_ERR_INVALID_VALUE;
  if (w.n_chan == 0 || w.n_E == 0) return PSTGF_OK;       // nothing to read or write
  if (!w.energies || !w.R_out) return PSTGF_ERR_INVALID_VALUE;
  if (w.w_layout != PSTGF_W_POLE_CONTIGUOUS && w.w_layout != PSTGF_W_CHANNEL_CONTIGUOUS) return PSTGF_ERR_INVALID_VALUE;
  const long long ld_min = w.w_layout == PSTGF_W_CHANNEL_CONTIGUOUS ? w.n_chan : w.n_poles;
  if (w.n_poles > 0 && (!w.W || !w.E_k || w.ldw < ld_min)) return PSTGF_ERR_INVALID_VALUE;
  if (!aligned8(w.W) || !aligned8(w.E_k) || !aligned8(w.energies) || !aligned8(w.R_out) || !aligned8(w.diag_add))
    return PSTGF_ERR_ALIGNMENT;
  return PSTGF_OK;
}

// ---- planner -------------------------------------------------------------------------------
// Knobs for tests and measurements (pstgf_debug_*): thread-local, they affect the calling thread's calls only.
thread_local int tl_tail_policy = PSTGF_TAIL_AUTO;
thread_local int tl_slab_policy = PSTGF_SLAB_AUTO;
thread_local int tl_pair_policy = PSTGF_PAIRS_AUTO;
thread_local int tl_small_policy = PSTGF_SMALL_AUTO;
thread_local int tl_host_pipeline = PSTGF_HOST_PIPELINE_AUTO;
thread_local unsigned int tl_upload_timeout_ms = 0;   // 0 = the kernel's default (2 s)
thread_local int tl_stall_upload = 0;

// Fills everything of DevWave except the tensor map, the slab section and the tail; every energy block starts out
// coarse and a remainder of n_E mod 8 energies starts out as a partial classic block.
void plan_wave(const pstgf_wave_t &w, DevWave &d, int l2_bytes) {
  std::memset(&d, 0, sizeof(d));
  d.W = w.W;
  d.E_k = w.E_k;
  d.energies = w.energies;
  d.R_out = w.R_out;
  d.diag_add = w.diag_add;
  d.ldw = w.ldw;
  d.inv2a = 1.0 / (2.0 * w.a);
  d.n_chan = w.n_chan;
  d.n_poles = w.n_poles;
  d.n_E = w.n_E;
  d.n_kt = (w.n_poles + pstgf::KT - 1) / pstgf::KT;
  d.n_i = (w.n_chan + pstgf::TM - 1) / pstgf::TM;
  d.n_j = (w.n_chan + pstgf::TN - 1) / pstgf::TN;
  d.n_eb = (w.n_E + pstgf::EB - 1) / pstgf::EB;
  d.n_tiles = pstgf::coarse_tiles(w.n_chan);
  d.n_eb_coarse = d.n_eb;
  d.slab_e0 = w.n_E;
  d.slab_T = 64;
  d.slab_nt = (w.n_chan + 63) / 64;
  d.tr = w.w_layout == PSTGF_W_CHANNEL_CONTIGUOUS ? 1 : 0;
  d.use_tma = ((reinterpret_cast<uintptr_t>(w.W) & 15u) == 0 && (w.ldw % 2) == 0 && w.ldw * 8 < (1LL << 40)) ? 1 : 0;
  // a W of at most half the L2 is loaded with the evict_last policy: R's streaming stores then do not push it out
  const double w_bytes = 8.0 * (double)w.ldw * (double)(d.tr ? w.n_poles : w.n_chan);
  d.l2_keep = (l2_bytes > 0 && w_bytes <= 0.5 * (double)l2_bytes) ? 1 : 0;
}

// A wave in the pair form has its 128-pair items in section 0, its 64-pair items in section 1 (where the slab items
// of the symmetric form are) and its 32-pair items in section 2.
long long coarse_items(const DevWave &d) {
  return d.n_pairs > 0 ? pstgf::pair_section_items(d, 0) : (long long)d.n_tiles * d.n_eb_coarse;
}
long long slab_items(const DevWave &d) {
  return d.n_pairs > 0 ? pstgf::pair_section_items(d, 1)
                       : (long long)pstgf::slab_tiles(d.slab_nt) * pstgf::slab_groups(d.slab_g4, d.slab_g2, d.slab_g1);
}
long long fine_items(const DevWave &d) {
  return d.n_pairs > 0 ? pstgf::pair_section_items(d, 2)
                       : (long long)pstgf::fine_tiles(d.n_j) * (d.n_eb - d.n_eb_coarse);
}
long long wave_items(const DevWave &d) { return coarse_items(d) + slab_items(d) + fine_items(d); }

// Relative cost of a wave's items, for the largest-first order of the batch.
double wave_item_cost(const pstgf_wave_t &w) { return (double)std::min(w.n_chan, pstgf::TM) * w.n_poles; }

double simulate_makespan(const std::vector<std::pair<double, int>> &runs, int grid);

// ---- pair form: which waves, how much scratch -----------------------------------------------------
// A wave is done as the GEMM over channel pairs (rmat_common.h) when it has few channels and enough energies to
// fill an energy tile's warps.  The choice depends on the wave's own shape only (and the thread's debug knob), so
// that a wave gives the same bits alone, in any batch and through the host call.
bool wants_pair_form(int n_chan, int n_poles, int n_E) {
  if (tl_pair_policy == PSTGF_PAIRS_NONE) return false;
  if (n_chan <= 0 || n_poles <= 0 || n_chan > pstgf::PAIR_MAX_CHAN) return false;
  if (tl_pair_policy == PSTGF_PAIRS_ALWAYS) return n_E > 0;
  return n_E >= pstgf::PAIR_MIN_E;
}
// A pair-form wave that is tiny -- few channels and little work in all -- goes to the one-launch kernel of
// rmat_small.cu (single-wave calls only).  It computes the pair form term for term, so this is a choice of speed, not
// of bits: the persistent kernel needs a scratch-builder launch, a ring and 128-energy items, which cost such a wave
// tens of microseconds.
constexpr double SMALL_MAX_FLOP = 536870912.0;       // n_chan^2 n_poles n_E = 2^29, about 15 us of the FP64 pipe: measured crossover 6e8 - 1e9
bool wants_small_kernel(int n_chan, int n_poles, int n_E) {
  if (tl_small_policy == PSTGF_SMALL_NONE || n_chan > pstgf::SMALL_MAX_CHAN) return false;
  return tl_small_policy == PSTGF_SMALL_ALWAYS || (double)n_chan * n_chan * (double)n_poles * (double)n_E <= SMALL_MAX_FLOP;
}
long long pair_count(int n_chan) { return (long long)n_chan * (n_chan + 1) / 2; }
long long pair_ld(int n_poles) { return ((long long)n_poles + 1) & ~1LL; }
size_t pair_D_bytes(int n_poles, int n_E) { return (((size_t)n_E * (size_t)pair_ld(n_poles) * 8) + 255) & ~(size_t)255; }
size_t pair_scratch_bytes(int n_chan, int n_poles, int n_E) {        // P, D, the (n, m) table: each 256-byte aligned
  const size_t ld = (size_t)pair_ld(n_poles);
  const size_t p = (((size_t)pair_count(n_chan) * ld * 8) + 255) & ~(size_t)255;
  const size_t t = (((size_t)pair_count(n_chan) * 4) + 255) & ~(size_t)255;
  return p + pair_D_bytes(n_poles, n_E) + t;
}
// Cuts a wave into pair items; `scratch` is where its P and D go.  Every energy tile starts out coarse (128-pair
// items); plan_pair_tails then cuts the tail of the launch into 64-pair items.
// With kept_P / kept_nm (P and the pair table of this wave, built earlier from all of W -- they hold no energy) the
// scratch takes D alone (pair_D_bytes) and the builder is told to leave P be.
void plan_pairs(DevWave &d, unsigned char *scratch, double *kept_P = nullptr, const unsigned int *kept_nm = nullptr) {
  d.n_pairs = (int)pair_count(d.n_chan);
  d.pair_ld = pair_ld(d.n_poles);
  if (kept_P) {
    d.pair_P = kept_P;
    d.pair_nm = kept_nm;
    d.pair_D = reinterpret_cast<double *>(scratch);
    d.pair_keep_P = 1;
  } else {
    d.pair_P = reinterpret_cast<double *>(scratch);
    const size_t p_bytes = (((size_t)d.n_pairs * (size_t)d.pair_ld * 8) + 255) & ~(size_t)255;
    const size_t d_bytes = (((size_t)d.n_E * (size_t)d.pair_ld * 8) + 255) & ~(size_t)255;
    d.pair_D = reinterpret_cast<double *>(scratch + p_bytes);
    d.pair_nm = reinterpret_cast<const unsigned int *>(scratch + p_bytes + d_bytes);
  }
  d.pair_nfb = d.n_chan / 8;
  d.pair_rb = pstgf::pair_block_rows(d.n_chan);
  d.pair_mt = (d.n_pairs + pstgf::PT_M - 1) / pstgf::PT_M;
  d.pair_mtf = (d.n_pairs + pstgf::PT_MF - 1) / pstgf::PT_MF;
  d.pair_mtff = (d.n_pairs + pstgf::PT_MFF - 1) / pstgf::PT_MFF;
  d.pair_nt = (d.n_E + pstgf::PT_N - 1) / pstgf::PT_N;
  d.pair_nt_coarse = d.pair_nt_mid = d.pair_nt;
  // no classic or slab items
  d.n_eb = d.n_eb_coarse = 0;
  d.slab_g4 = d.slab_g2 = d.slab_g1 = 0;
  d.slab_e0 = d.n_E;
}

// Relative cost of a wave's pair items in row blocks of 8 pairs per item: 16 / 8 / 4 for the three tile heights
// (fewer in a wave's last pair tile), times a factor for the shorter register tiles' inner loops.
// Measured item times on config 2 (per-CTA timestamps, 64 k-tiles per item): 172.6 us for 16 row blocks, 97.8 us for 8,
// 49.6 - 61.5 us for 4, i.e. 9.35 us per row block plus 23 us per item -- the short items reload the same 128 energies
// of D for fewer pairs and run into the L2 -> SM bandwidth (3.5 TB/s chip-wide for 64-pair items).
constexpr double PAIR_Q[3] = {1.0, 1.0, 1.0};
constexpr double PAIR_ITEM_FIXED = 2.5;              // per item, in row blocks
double pair_last_tile_blocks(const DevWave &d, int sec) {
  const int rows = pstgf::PT_M >> sec;
  const int left = d.n_pairs - ((d.n_pairs + rows - 1) / rows - 1) * rows;
  return std::min<double>(rows / 8, left > 64 ? 16.0 : left > 32 ? 8.0 : 4.0);
}
int pair_tiles(const DevWave &d, int sec) { return sec == 0 ? d.pair_mt : sec == 1 ? d.pair_mtf : d.pair_mtff; }
// Sets the section boundaries of a pair-form wave from item counts: the first n0 items of the 128-pair tiling are
// section 0, then about n1 64-pair items (rounded up so that no energy tile is split three ways), the rest 32-pair.
void pair_set_sections(DevWave &d, long long n0, long long n1) {
  const int nt = d.pair_nt;
  n0 = std::min<long long>(n0, (long long)d.pair_mt * nt);
  d.pair_nt_coarse = (int)(n0 / d.pair_mt);
  d.pair_x0 = (int)(n0 % d.pair_mt);
  d.pair_x1 = 0;
  if (d.pair_nt_coarse >= nt) {            // everything coarse
    d.pair_nt_coarse = d.pair_nt_mid = nt;
    d.pair_x0 = 0;
    return;
  }
  const long long first = d.pair_x0 > 0 ? d.pair_mtf - 2 * d.pair_x0 : 0;    // the split energy tile's 64-pair items
  const long long rest = std::max<long long>(0, n1 - first);
  const int full = (int)std::min<long long>(rest / d.pair_mtf, nt - d.pair_nt_coarse - (d.pair_x0 > 0 ? 1 : 0));
  d.pair_nt_mid = d.pair_nt_coarse + (d.pair_x0 > 0 ? 1 : 0) + full;
  if (d.pair_nt_mid < nt) d.pair_x1 = (int)std::min<long long>(rest - (long long)full * d.pair_mtf, d.pair_mtf - 1);
}

// Item costs of a pair-form wave, item by item in the order the counter hands them out.
void pair_item_costs(const DevWave &d, std::vector<std::pair<double, int>> &runs) {
  runs.clear();
  for (int sec = 0; sec < 3; ++sec) {
    const long long n = pstgf::pair_section_items(d, sec);
    const int rows = pstgf::PT_M >> sec, last_mt = pair_tiles(d, sec) - 1;
    const double c_full = PAIR_Q[sec] * (rows / 8) + PAIR_ITEM_FIXED, c_last = PAIR_Q[sec] * pair_last_tile_blocks(d, sec) + PAIR_ITEM_FIXED;
    for (long long i = 0; i < n; ++i) {
      int mt, nt;
      pstgf::pair_decode_item(d, sec, i, mt, nt);
      const double c = mt == last_mt ? c_last : c_full;
      if (!runs.empty() && runs.back().first == c) ++runs.back().second;
      else runs.emplace_back(c, 1);
    }
  }
}

// The tail of the launch's pair items -- about one round of the grid -- in 64-pair and, at the very end, 32-pair items,
// so that the CTAs run dry together, like the fine tiles of the symmetric form.  One wave: the section sizes (in
// items: the boundaries may cut through an energy tile) with the smallest simulated makespan among those that end the
// 128-pair section near a whole number of rounds of the grid; several waves: whole energy tiles from the end of the
// list until a quarter of a round's worth of work has been cut into 32-pair items and a round's worth into 64-pair items.
void plan_pair_tails(std::vector<DevWave> &ds, int grid) {
  if (tl_tail_policy == PSTGF_TAIL_NONE) return;
  std::vector<DevWave *> pw;
  for (DevWave &d : ds)
    if (d.n_pairs > 0) pw.push_back(&d);
  if (pw.empty()) return;
  if (tl_tail_policy == PSTGF_TAIL_ALL) {
    for (DevWave *d : pw) {               // a bit of everything, with both boundaries inside an energy tile where there is room
      const long long all = (long long)d->pair_mt * d->pair_nt;
      pair_set_sections(*d, all / 3 + (d->pair_mt > 1 ? 1 : 0), (long long)d->pair_mtf * d->pair_nt / 3 + (d->pair_mtf > 1 ? 1 : 0));
    }
    return;
  }
  if (pw.size() == 1 && ds.size() == 1) {
    DevWave &d = *pw[0];
    // cached per shape: the simulation costs a millisecond or two of host time for a few thousand items
    static std::mutex cache_mutex;
    static std::map<std::tuple<int, int, int>, std::pair<long long, long long>> cache;   // (n_pairs, energy tiles, grid) -> (n0, n1)
    const auto key = std::make_tuple(d.n_pairs, d.pair_nt, grid);
    {
      std::lock_guard<std::mutex> lock(cache_mutex);
      auto it = cache.find(key);
      if (it != cache.end()) {
        pair_set_sections(d, it->second.first, it->second.second);
        return;
      }
    }
    const long long all = (long long)d.pair_mt * d.pair_nt;
    std::vector<long long> c0, c1;
    if (all > 64LL * grid) {              // many rounds: the last round and a half in 64-pair items, the last half round finer
      c0.push_back(std::max<long long>(0, all - grid - grid / 2));
      c1.push_back(2LL * grid);
    } else {
      // 128-pair sections that end up to a round short of the total, in steps of an eighth of a round; 64-pair
      // sections of up to two rounds of the grid (two 64-pair items are one 128-pair item)
      for (int i = 0; i <= 16; ++i) c0.push_back(std::max<long long>(0, all - (long long)i * grid / 8));
      for (int i = 0; i <= 8; ++i) c1.push_back((long long)i * grid / 4);
    }
    std::vector<std::pair<double, int>> runs;
    long long best_n0 = all, best_n1 = 0;
    double best = -1.0;
    for (long long n0 : c0)
      for (long long n1 : c1) {
        pair_set_sections(d, n0, n1);
        pair_item_costs(d, runs);
        const double m = simulate_makespan(runs, grid);
        if (best < 0.0 || m < best * (1.0 - 1e-9)) {
          best = m;
          best_n0 = n0;
          best_n1 = n1;
        }
      }
    pair_set_sections(d, best_n0, best_n1);
    std::lock_guard<std::mutex> lock(cache_mutex);
    cache[key] = std::make_pair(best_n0, best_n1);
    return;
  }
  double budget_fine = 4.0 * grid, budget_mid = 16.0 * grid;          // in row blocks
  for (size_t q = pw.size(); q-- > 0 && budget_mid > 0.0;) {
    DevWave &d = *pw[q];
    const double per_tile = 16.0 * (d.pair_mt - 1) + pair_last_tile_blocks(d, 0);   // one energy tile of this wave
    const int t2 = budget_fine > 0.0 ? (int)std::min<double>((double)d.pair_nt, std::floor(budget_fine / per_tile + 0.5)) : 0;
    budget_fine -= std::max(1, t2) * per_tile;                        // (a wave too big for it ends the 32-pair tail)
    const int t1 = (int)std::min<double>((double)(d.pair_nt - t2), std::floor(budget_mid / per_tile + 0.5));
    d.pair_nt_mid = d.pair_nt - t2;
    d.pair_nt_coarse = d.pair_nt_mid - t1;
    budget_mid -= (t1 + t2) * per_tile;
    if (t1 + t2 == 0) break;
  }
}

// Cost model in DMMA.8x8x4 per energy (full-size tiles; good enough to size the tail).
double largest_item_cost(const DevWave &d) {
  const int nb = std::min((d.n_chan + 7) / 8, pstgf::TM / 8);
  return (double)d.n_kt * (nb * (nb + 1) / 2);
}
double cost_per_energy_block(const DevWave &d) {
  return (double)d.n_kt * ((double)d.n_i * pstgf::COST_DIAG + (double)(d.n_tiles - d.n_i) * pstgf::COST_OFF);
}

// Makespan of greedy list scheduling (what the atomic counter does) of runs of equal items on `grid` CTAs.
double simulate_makespan(const std::vector<std::pair<double, int>> &runs, int grid) {
  std::priority_queue<double, std::vector<double>, std::greater<double>> free_at;
  for (int b = 0; b < grid; ++b) free_at.push(0.0);
  double last = 0.0;
  for (const auto &r : runs)
    for (int n = 0; n < r.second; ++n) {
      const double f = free_at.top() + r.first;
      free_at.pop();
      free_at.push(f);
      last = std::max(last, f);
    }
  return last;
}

// ---- slab section: the energies that do not fill a block of 8 ------------------------------------
// Time of a slab item per k-tile, in SM clocks: the slower of
//  - its busiest SM sub-partition's DMMAs: blocks per warp (SlabShape: nr x ncw) x warps per sub-partition x 5 k-steps
//    x 16 clk, times a factor for the quality of the warp's inner loop (fewer DMMAs per fragment load and per scaling
//    multiply in the small shapes; fitted to the B200 sweeps of bench.py --n-E), and
//  - the rate at which a slab item is SEEN to take its panels in: 15 B/clk per SM, 4.2 TB/s chip-wide (measured: one
//    energy at 512 x 10240 on tiles of edge 32 runs at 634 clk per k-tile for 10 KB of panels).  This is a fitted item
//    rate, NOT the L2 -> SM fabric: the probe of measure/l2_probe.cu delivers 28-31 B/clk per SM (8-9 TB/s) on this
//    chip (profiles/r03_l2_probe.md), and issuing the boxes of four stages in one TMA instruction -- the pattern
//    that takes the probe from 2.6 to 8 TB/s -- left these items where they were (0.170 -> 0.169 ms):
//    a k-tile of an edge-32 tile is 320 clk of DMMA issue on a sub-partition that holds ONE computing warp, and that
//    warp's wait / fragment loads / scaling / dependent DMMAs / release run one after the other,
// plus a fixed cost per item (epilogue, ring refill) of three k-tiles.
constexpr double SLAB_PANEL_BYTES_PER_CLK = 15.0;
double slab_item_cost(int T, int g, int n_kt) {
  const pstgf::SlabShape sh = pstgf::slab_shape(T, g);
  const int blocks = sh.nr * sh.ncw;
  const double quality = blocks >= 32 ? 1.0 : blocks >= 16 ? 1.04 : blocks >= 8 ? 1.10 : 1.15;
  const double warps_per_smsp = (T == 32 && g == 1) ? 1.0 : 2.0;          // (edge 32 with one energy keeps four warps idle)
  const double compute = blocks * warps_per_smsp * 80.0 * quality;
  const double l2 = pstgf::slab_panels(T) * (double)pstgf::BOX_BYTES / SLAB_PANEL_BYTES_PER_CLK;
  return std::max(compute, l2) * ((double)n_kt + 3.0);
}

struct SlabPlan {
  int T, g4, g2, g1;
};
std::mutex g_slab_mutex;
std::map<std::tuple<int, int, int, int, int>, SlabPlan> g_slab_cache;   // (n_chan, remainder, n_kt bucket, grid, forced edge) -> plan

// Tile edge and energy groups of a wave's slab items: the candidate with the smallest simulated makespan of the slab
// items alone.  Large tiles have the better inner loop and the smaller L2 traffic, small tiles give the grid enough
// items; groups of four or two energies share the tile's panels (tiles of edge 128 take one energy at a time), and a
// group of four may hold three.
SlabPlan best_slab_plan(int n_chan, int r, int n_kt, int grid, int forced_T) {
  const auto key = std::make_tuple(n_chan, r, std::min(n_kt, 64), grid, forced_T);
  {
    std::lock_guard<std::mutex> lock(g_slab_mutex);
    auto it = g_slab_cache.find(key);
    if (it != g_slab_cache.end()) return it->second;
  }
  SlabPlan best_plan{32, 0, 0, r};
  double best = -1.0;
  std::vector<std::pair<double, int>> runs;
  for (int T : {128, 64, 32}) {
    if (forced_T != 0 && T != forced_T) continue;
    const int nt = (n_chan + T - 1) / T;
    const long long tiles = pstgf::slab_tiles(nt);
    for (int g4 = 0; g4 <= (T == 128 ? 0 : (r + 3) / 4); ++g4) {
      const int rem = std::max(0, r - 4 * g4);
      if (g4 > 0 && 4 * g4 - r > 1) continue;                            // a group of four holds four or three energies
      const int g2 = T == 128 ? 0 : rem / 2, g1 = T == 128 ? rem : rem % 2;
      const double c4 = g4 ? slab_item_cost(T, 4, n_kt) : 0.0, c2 = g2 ? slab_item_cost(T, 2, n_kt) : 0.0,
                   c1 = g1 ? slab_item_cost(T, 1, n_kt) : 0.0;
      double m;
      if (tiles * (g4 + g2 + g1) > 16LL * grid) {
        // plenty of items: the makespan is the work divided by the grid, no need to simulate
        m = (double)tiles * (g4 * c4 + g2 * c2 + g1 * c1) / grid;
      } else {
        runs.clear();
        // group-major order, groups of four first; all tiles cost the same in this model (edge tiles are cheaper in fact)
        if (g4) runs.emplace_back(c4, (int)(tiles * g4));
        if (g2) runs.emplace_back(c2, (int)(tiles * g2));
        if (g1) runs.emplace_back(c1, (int)(tiles * g1));
        m = simulate_makespan(runs, grid);
      }
      if (best < 0.0 || m < best * (1.0 - 1e-9)) {
        best = m;
        best_plan = SlabPlan{T, g4, g2, g1};
      }
    }
  }
  std::lock_guard<std::mutex> lock(g_slab_mutex);
  g_slab_cache[key] = best_plan;
  return best_plan;
}

void plan_slabs(std::vector<DevWave> &ds, int grid) {
  const int policy = tl_slab_policy;
  if (policy == PSTGF_SLAB_NONE) return;
  for (DevWave &d : ds) {
    const int r = d.n_E % pstgf::EB;
    if (r == 0 || d.n_pairs > 0) continue;
    const int forced = policy == PSTGF_SLAB_T32 ? 32 : policy == PSTGF_SLAB_T64 ? 64 : policy == PSTGF_SLAB_T128 ? 128 : 0;
    const SlabPlan sp = best_slab_plan(d.n_chan, r, d.n_kt, grid, forced);
    d.n_eb = d.n_E / pstgf::EB;
    d.n_eb_coarse = d.n_eb;
    d.slab_e0 = d.n_eb * pstgf::EB;
    d.slab_T = sp.T;
    d.slab_nt = (d.n_chan + sp.T - 1) / sp.T;
    d.slab_g4 = sp.g4;
    d.slab_g2 = sp.g2;
    d.slab_g1 = sp.g1;
  }
}

// Item families of a launch (rmat_common.h): the kernel instantiation that holds no more code than the items need.
int launch_family(const std::vector<DevWave> &ds) {
  int fam = pstgf::FAM_CLASSIC;
  for (const DevWave &d : ds) {
    if (d.n_pairs > 0) return pstgf::FAM_PAIR;
    if (slab_items(d) > 0) fam = pstgf::FAM_SLAB;
  }
  return fam;
}

// Ring geometry of a launch: a stage holds the most panels any of its items needs (5 for classic items, 8 / 4 / 2
// for slab tiles of edge 128 / 64 / 32); as many stages as fit, at most MAX_STAGES.  Small stages make a deep ring:
// items that spend a few hundred cycles on a stage need many stages in flight to cover the load latency.
pstgf::RingGeo ring_geometry(const std::vector<DevWave> &ds) {
  int bytes = 0;
  for (const DevWave &d : ds) {
    int panels = 0;
    if (d.n_pairs > 0) panels = pstgf::PAIR_PANELS;
    else if (coarse_items(d) + fine_items(d) > 0) panels = pstgf::CLASSIC_PANELS;
    if (d.n_pairs == 0 && slab_items(d) > 0) panels = std::max(panels, pstgf::slab_panels(d.slab_T));
    bytes = std::max(bytes, pstgf::stage_bytes_for(d.tr != 0 && d.n_pairs == 0, panels));
  }
  pstgf::RingGeo g;
  g.stage_bytes = bytes;
  g.n_stages = std::min(pstgf::MAX_STAGES, (pstgf::SMEM_MAX_OPTIN - pstgf::SMEM_RING_OFFSET - pstgf::SMEM_ALIGN_SLACK) / bytes);
  return g;
}

// ---- tail size of a single wave by simulation ------------------------------------------------------
// Relative cost of one 8x8 block per k-step in the four tile kinds, fitted to sweeps of the tail size on the
// B200 (configs 2 and 5; the fit reproduces the measured step times to 0.2 %): coarse OFF 1, coarse DIAG 1.04
// (8 DMUL per 36 DMMA), fine OFF32 1.03, fine DIAG32 1.2 (4 DMUL per 10 DMMA and a stage consumed in a
// quarter of the time).
constexpr double BLK_OFF = 1.0, BLK_WIDE = 0.985, BLK_DIAG = 1.04, BLK_OFF32 = 1.03, BLK_DIAG32 = 1.2;

// Item costs of one wave in the order the counter hands them out, with `t` energy blocks in the fine tail.
void item_costs(const DevWave &d, int t, std::vector<std::pair<double, int>> &runs) {
  runs.clear();
  const int C = d.n_chan, n_c = d.n_eb - t;
  auto blocks8 = [&](int first, int cap) { return std::min(cap, (C - first + 7) / 8); };
  if (n_c > 0) {
    for (int i = 0; i < d.n_i; ++i) {
      const int nb = blocks8(pstgf::TM * i, pstgf::TM / 8);
      runs.emplace_back(BLK_DIAG * nb * (nb + 1) / 2, n_c);
    }
    for (int p = 0; pstgf::TW * p + pstgf::TM < C; ++p)
      for (int c = 0; c < pstgf::wide_tiles_in_pair(C, p); ++c)
        runs.emplace_back(BLK_WIDE * 16 * blocks8(pstgf::TW * (p + 1) + pstgf::TWN * c, pstgf::TWN / 8), n_c);
    for (int p = 0; pstgf::TW * p + pstgf::TM < C; ++p)
      for (int t2 = 0; t2 < pstgf::off_tiles_in_pair(C, p); ++t2)
        runs.emplace_back(BLK_OFF * 8 * blocks8(pstgf::TW * p + pstgf::TM + pstgf::TN * t2, pstgf::TN / 8), n_c);
  }
  if (t > 0) {
    for (int i = 0; i < d.n_j; ++i)
      for (int j = i + 1; j < d.n_j; ++j) runs.emplace_back(BLK_OFF32 * 4 * blocks8(pstgf::TN * j, pstgf::TN / 8), t);
    for (int i = 0; i < d.n_j; ++i) {
      const int nb = blocks8(pstgf::TN * i, pstgf::TN / 8);
      runs.emplace_back(BLK_DIAG32 * nb * (nb + 1) / 2, t);
    }
  }
}

std::mutex g_tail_mutex;
std::map<std::tuple<int, int, int>, int> g_tail_cache;   // (n_chan, n_eb, grid) -> energy blocks in the fine tail

// Tail size of a single wave: the candidate with the smallest simulated makespan among up to 17 sizes between
// 0 and twice the heuristic budget.  Cached per shape (the cost does not depend on n_poles: every item of a wave
// has the same number of k-steps).  Returns -1 when the wave has too many items for a simulation to be worth its
// host time (then the tail matters little anyway).
int best_tail_single_wave(const DevWave &d, int grid, double budget) {
  const long long items = (long long)d.n_tiles * d.n_eb;
  if (items > 8192) return -1;
  const auto key = std::make_tuple(d.n_chan, d.n_eb, grid);
  {
    std::lock_guard<std::mutex> lock(g_tail_mutex);
    auto it = g_tail_cache.find(key);
    if (it != g_tail_cache.end()) return it->second;
  }
  const double per_eb = cost_per_energy_block(d) / std::max(1, d.n_kt);
  const int t_max = (int)std::min<double>((double)d.n_eb, std::ceil(2.0 * budget / std::max(1, d.n_kt) / per_eb) + 1.0);
  const int stride = std::max(1, t_max / 16);
  std::vector<std::pair<double, int>> runs;
  int best_t = 0;
  double best = 0.0;
  for (int t = 0; t <= t_max; t += stride) {
    item_costs(d, t, runs);
    const double m = simulate_makespan(runs, grid);
    if (t == 0 || m < best * (1.0 - 1e-9)) {
      best = m;
      best_t = t;
    }
  }
  std::lock_guard<std::mutex> lock(g_tail_mutex);
  g_tail_cache[key] = best_t;
  return best_t;
}

// Tail of the schedule (see rmat_common.h): about one round of the grid's worth of work, taken from the
// END of the largest-first order, is cut into fine tiles so that list scheduling finishes on small items.
void plan_tails(std::vector<DevWave> &ds, int grid) {
  const int policy = tl_tail_policy;
  if (policy == PSTGF_TAIL_NONE) return;
  if (policy == PSTGF_TAIL_ALL) {
    for (DevWave &d : ds) d.n_eb_coarse = 0;
    return;
  }
  double c_max = 0.0;
  for (const DevWave &d : ds)
    if (d.n_eb > 0 && d.n_pairs == 0) c_max = std::max(c_max, largest_item_cost(d));
  double budget = c_max * grid;
  if (ds.size() == 1) {
    if (ds[0].n_eb == 0 || ds[0].n_pairs > 0) return;
    const int t = best_tail_single_wave(ds[0], grid, c_max * grid);
    if (t >= 0) {
      ds[0].n_eb_coarse = ds[0].n_eb - t;
      return;
    }
  }
  for (size_t q = ds.size(); q-- > 0 && budget > 0.0;) {
    DevWave &d = ds[q];
    if (d.n_eb == 0 || d.n_pairs > 0) continue;
    const double per_eb = cost_per_energy_block(d);
    if (largest_item_cost(d) <= 0.45 * c_max) {   // a small wave at the end of the list: its coarse items are fine enough
      budget -= d.n_eb * per_eb;
      continue;
    }
    // whole energy blocks, rounded to the nearest: a wave whose single energy block already outweighs the
    // budget (many tiles, few energies: the paper-scale wave) keeps its coarse tiles -- its items are small
    // against the whole job, and fine tiles run 5 % slower
    const int t = (int)std::min<double>((double)d.n_eb, std::floor(budget / per_eb + 0.5));
    if (t == 0) break;
    d.n_eb_coarse = d.n_eb - t;
    budget -= t * per_eb;
  }
}

pstgf_status_t encode_map(DevWave &d) {
  if (!d.use_tma) return PSTGF_OK;
  // pole-contiguous W: dims (pole, channel), box 20 poles x 32 channels; channel-contiguous W (H.DAT order):
  // dims (channel, pole), box 36 channels x 20 poles.  Out-of-range elements are zero-filled either way.
  cuuint64_t dims[2] = {(cuuint64_t)d.n_poles, (cuuint64_t)d.n_chan};
  cuuint32_t box[2] = {(cuuint32_t)pstgf::KT, (cuuint32_t)pstgf::TN};
  if (d.tr) {
    std::swap(dims[0], dims[1]);
    box[0] = (cuuint32_t)pstgf::TR_PITCH;
    box[1] = (cuuint32_t)pstgf::KT;
  }
  cuuint64_t strides[1] = {(cuuint64_t)d.ldw * 8};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = g_encode(&d.map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double *>(d.W), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    d.use_tma = 0;   // shapes the encoder refuses fall back to the plain staging path
  }
  return PSTGF_OK;
}

// Tensor maps of the pair form's scratch: P [n_pairs][pair_ld] and D [n_E][pair_ld], boxes of 32 rows x 20 poles.
pstgf_status_t encode_pair_maps(DevWave &d) {
  if (d.n_pairs <= 0) return PSTGF_OK;
  for (int which = 0; which < 2; ++which) {
    cuuint64_t dims[2] = {(cuuint64_t)d.n_poles, (cuuint64_t)(which ? d.n_E : d.n_pairs)};
    cuuint32_t box[2] = {(cuuint32_t)pstgf::KT, (cuuint32_t)pstgf::TN};
    cuuint64_t strides[1] = {(cuuint64_t)d.pair_ld * 8};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = g_encode(which ? &d.map_D : &d.map_P, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, which ? d.pair_D : d.pair_P, dims,
                          strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                          CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
      tl_cuda_error = (int)cudaErrorInvalidValue;
      return PSTGF_ERR_CUDA;
    }
  }
  return PSTGF_OK;
}

// A wave with work for the contraction kernel (n_poles == 0 is a zero-fill instead).
bool wave_has_items(const pstgf_wave_t &w) { return w.n_chan > 0 && w.n_E > 0 && w.n_poles > 0; }

// n_poles == 0: the sum of eq. 4 is empty, R is the diagonal addend alone (zero without one).
__global__ void diag_only_kernel(const double *__restrict__ diag_add, int n_chan, long long n, double *__restrict__ R_out) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;      // over [n_E][n_chan]
  if (idx >= n) return;
  const long long e = idx / n_chan;
  const int c = (int)(idx - e * n_chan);
  R_out[(size_t)e * n_chan * n_chan + (size_t)c * n_chan + c] = diag_add[idx];
}

pstgf_status_t zero_fill(const pstgf_wave_t &w, cudaStream_t s) {
  if (w.n_chan > 0 && w.n_E > 0 && w.n_poles == 0) {
    PSTGF_CUDA(cudaMemsetAsync(w.R_out, 0, sizeof(double) * (size_t)w.n_E * w.n_chan * w.n_chan, s));
    ++tl_launches;
    if (w.diag_add) {
      const long long n = (long long)w.n_E * w.n_chan;
      diag_only_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(w.diag_add, w.n_chan, n, w.R_out);
      PSTGF_CUDA(cudaGetLastError());
      ++tl_launches;
    }
  }
  return PSTGF_OK;
}

// Device memory of the host call, and the single-wave call's pair-form scratch, come from a pool the library owns (one per device, release threshold =
// never, freed by pstgf_rmat_finalize): the default pool hands its memory back at every synchronise, and
// re-growing it costs tens of milliseconds per call.
// The single-wave call's pair-form scratch has a pool of its own that keeps at most SCRATCH_POOL_KEEP bytes across a
// synchronise (what a run of RINIT calls on one wave reuses) and hands the rest back to the device, so that a caller's
// own allocator can have it.
std::mutex g_pool_mutex;
cudaMemPool_t g_pool[64] = {nullptr};
cudaMemPool_t g_scratch_pool[64] = {nullptr};
constexpr unsigned long long SCRATCH_POOL_KEEP = 256ULL << 20;

cudaError_t library_pool(int dev, cudaMemPool_t *out, bool scratch = false) {
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  cudaMemPool_t *pools = scratch ? g_scratch_pool : g_pool;
  if (!pools[dev]) {
    cudaMemPoolProps props;
    std::memset(&props, 0, sizeof(props));
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t pool;
    cudaError_t e = cudaMemPoolCreate(&pool, &props);
    if (e != cudaSuccess) return e;
    unsigned long long keep = scratch ? SCRATCH_POOL_KEEP : ~0ULL;
    e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    if (e != cudaSuccess) { cudaMemPoolDestroy(pool); return e; }
    pools[dev] = pool;
  }
  *out = pools[dev];
  return cudaSuccess;
}

// workspace layout of the batch call
constexpr size_t WS_COUNTER_BYTES = 256;
size_t ws_item_begin_bytes(int n_waves) { return ((3 * (size_t)n_waves + 2) * sizeof(long long) + 255) & ~(size_t)255; }   // two launches: two tables
size_t ws_tables_bytes(int n_waves) {
  return (WS_COUNTER_BYTES + ws_item_begin_bytes(n_waves) + (size_t)n_waves * sizeof(DevWave) + 255) & ~(size_t)255;
}
// tables, then the scratch (P, D) of every wave that is done in the pair form; force_pair, if given, overrides the
// per-wave choice (the host call cuts waves into energy ranges and wants every range to go the way of the whole wave)
size_t ws_bytes(const pstgf_wave_t *waves, int n_waves, const unsigned char *force_pair = nullptr, double *const *kept_P = nullptr) {
  size_t b = ws_tables_bytes(n_waves);
  if (waves)
    for (int p = 0; p < n_waves; ++p) {
      const pstgf_wave_t &w = waves[p];
      if (w.n_chan <= 0 || w.n_E <= 0 || w.n_poles <= 0) continue;
      const bool pair = force_pair ? force_pair[p] != 0 : wants_pair_form(w.n_chan, w.n_poles, w.n_E);
      if (pair) b += (kept_P && kept_P[p]) ? pair_D_bytes(w.n_poles, w.n_E) : pair_scratch_bytes(w.n_chan, w.n_poles, w.n_E);
    }
  return b;
}

// ---- work counters of the single-wave call ---------------------------------------------------
// pstgf_rmat_form has no workspace argument, so its atomic work counter comes from a small pool the library
// keeps per device (COUNTER_SLOTS x 128 B, allocated at first use, freed by pstgf_rmat_finalize).  A slot is
// handed to one launch at a time: an event recorded behind the launch tells when it is free again (the kernel's
// last CTA zeroes it).  With no free slot, or under stream capture, the launch falls back to round-robin item
// assignment.
constexpr int COUNTER_SLOTS = 64;
struct CounterPool {
  unsigned long long *base = nullptr;
  cudaEvent_t ev[COUNTER_SLOTS] = {nullptr};
  bool armed[COUNTER_SLOTS] = {false};
  int next = 0;
};
std::mutex g_counter_mutex;
CounterPool g_counters[64];

bool stream_is_capturing(cudaStream_t s) {
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(s, &cap) != cudaSuccess) {
    (void)cudaGetLastError();
    return true;      // cannot tell: treat as capturing (the safe side)
  }
  return cap != cudaStreamCaptureStatusNone;
}

// Called with g_counter_mutex held.  Returns the slot or -1.
int acquire_counter(int dev, cudaStream_t s, unsigned long long **out) {
  if (dev < 0 || dev >= 64) return -1;
  if (stream_is_capturing(s)) return -1;
  CounterPool &cp = g_counters[dev];
  if (!cp.base) {
    void *p = nullptr;
    if (cudaMalloc(&p, COUNTER_SLOTS * 128) != cudaSuccess || cudaMemset(p, 0, COUNTER_SLOTS * 128) != cudaSuccess) {
      (void)cudaGetLastError();
      if (p) cudaFree(p);
      return -1;
    }
    for (int i = 0; i < COUNTER_SLOTS; ++i) {
      if (cudaEventCreateWithFlags(&cp.ev[i], cudaEventDisableTiming) != cudaSuccess) {
        (void)cudaGetLastError();
        for (int k = 0; k < i; ++k) cudaEventDestroy(cp.ev[k]);
        cudaFree(p);
        return -1;
      }
    }
    cp.base = static_cast<unsigned long long *>(p);
  }
  for (int t = 0; t < COUNTER_SLOTS; ++t) {
    const int slot = (cp.next + t) % COUNTER_SLOTS;
    if (cp.armed[slot]) {
      if (cudaEventQuery(cp.ev[slot]) != cudaSuccess) {
        (void)cudaGetLastError();
        continue;                                   // that launch has not finished yet
      }
      cp.armed[slot] = false;
    }
    cp.next = (slot + 1) % COUNTER_SLOTS;
    *out = cp.base + (size_t)slot * 16;
    return slot;
  }
  return -1;
}

// ---- library-resident scratch of pstgf_rmat_form_static ------------------------------------------
// pstgf_rmat_form_static (include/pstgf_rmat.h) is the single-wave call for callers that must not allocate device
// memory.  What pstgf_rmat_form takes from cudaMalloc (the work-counter pool) and from cudaMallocFromPoolAsync (P, D and
// the pair table of a pair-form wave) lives here instead: one array of PSTGF_STATIC_SCRATCH_BYTES that is part of the
// module's image, so every device that loads libpstgf_rmat.so carries it from module load to process exit, used or not.
//   [0, 256)                               the launch's work counter (two words used)
//   [256, PSTGF_STATIC_SCRATCH_BYTES)      pair-form scratch, laid out by plan_pairs as in the other calls
// In host code `g_static_scratch` is only a handle for the runtime (a host-side shadow symbol), never a device
// address: the device address is asked for once per device with cudaGetSymbolAddress and that is what kernels get.
}  // namespace
static __device__ __align__(256) unsigned char g_static_scratch[PSTGF_STATIC_SCRATCH_BYTES];
namespace {
constexpr size_t STATIC_COUNTER_BYTES = 256;
std::mutex g_static_mutex;
unsigned char *g_static_addr[64] = {nullptr};

// Device address of g_static_scratch on device `dev`, which must be the CURRENT device (cudaGetSymbolAddress answers
// for the current device's copy of the module).  Looked up at the first call per device, remembered afterwards.
pstgf_status_t static_scratch_address(int dev, unsigned char **out) {
  if (dev < 0 || dev >= 64) return PSTGF_ERR_UNSUPPORTED_DEVICE;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_addr[dev]) {
    void *p = nullptr;
    PSTGF_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255u) != 0) return PSTGF_ERR_CUDA;
    g_static_addr[dev] = static_cast<unsigned char *>(p);
  }
  *out = g_static_addr[dev];
  return PSTGF_OK;
}

}  // namespace

extern "C" {

pstgf_status_t pstgf_debug_set_tail_policy(int policy) {
  if (policy != PSTGF_TAIL_AUTO && policy != PSTGF_TAIL_NONE && policy != PSTGF_TAIL_ALL) return PSTGF_ERR_INVALID_VALUE;
  tl_tail_policy = policy;
  return PSTGF_OK;
}

pstgf_status_t pstgf_debug_set_pair_policy(int policy) {
  if (policy < PSTGF_PAIRS_AUTO || policy > PSTGF_PAIRS_ALWAYS) return PSTGF_ERR_INVALID_VALUE;
  tl_pair_policy = policy;
  return PSTGF_OK;
}

pstgf_status_t pstgf_debug_set_small_policy(int policy) {
  if (policy < PSTGF_SMALL_AUTO || policy > PSTGF_SMALL_ALWAYS) return PSTGF_ERR_INVALID_VALUE;
  tl_small_policy = policy;
  return PSTGF_OK;
}

pstgf_status_t pstgf_debug_set_slab_policy(int policy) {
  if (policy < PSTGF_SLAB_AUTO || policy > PSTGF_SLAB_T128) return PSTGF_ERR_INVALID_VALUE;
  tl_slab_policy = policy;
  return PSTGF_OK;
}

// One persistent launch of a single-wave plan on `s`, with a work counter from the pool when there are more items
// than CTAs.
static pstgf_status_t launch_single(std::vector<DevWave> &d, const DeviceState &ds, cudaStream_t s) {
  const long long n_items = wave_items(d[0]);
  const int grid = (int)std::min<long long>(ds.sm_count, n_items);
  const pstgf::RingGeo geo = ring_geometry(d);
  std::lock_guard<std::mutex> lock(g_counter_mutex);
  unsigned long long *counter = nullptr;
  // no more items than CTAs: item b goes to CTA b, no counter needed (one L2 round trip less for the tiny calls)
  const int slot = n_items <= grid ? -1 : acquire_counter(ds.device, s, &counter);
  pstgf::PersistentArgs pa{&d[0], nullptr, nullptr, 1, n_items, counter, geo, grid};
  PSTGF_CUDA(pstgf::persistent_launch_family(launch_family(d), false, pa, s));
  if (slot >= 0) {
    CounterPool &cp = g_counters[ds.device];
    PSTGF_CUDA(cudaEventRecord(cp.ev[slot], s));
    cp.armed[slot] = true;
  }
  return PSTGF_OK;
}

// The pair form of the single-wave call.  Scratch is stream-ordered memory from the library's scratch pool, allocated
// here and freed behind the last launch: P and the pair table once, D for at most PAIR_D_RANGE_BYTES worth of energies
// at a time -- a long mesh goes out as several (builder, GEMM) launch pairs over energy ranges that start on energy-tile
// boundaries, all reading the one P, so the scratch does not grow with n_E (a 64 x 1280 wave with 10^6 energies would
// otherwise want 10 GB of D).  Every R element is still one thread's sum in the fixed k order: same bits as one launch.
// *no_memory is set, and nothing has been enqueued, when the scratch cannot be had; the caller then takes the
// symmetric form, which needs none.
constexpr size_t PAIR_D_RANGE_BYTES = (size_t)128 << 20;
static pstgf_status_t form_single_pairs(const pstgf_wave_t &w, const DeviceState &ds, cudaStream_t s, bool *no_memory) {
  *no_memory = false;
  const size_t row_bytes = (size_t)pair_ld(w.n_poles) * 8;
  int range = w.n_E;
  if (pair_D_bytes(w.n_poles, w.n_E) > PAIR_D_RANGE_BYTES)
    range = std::max<long long>(pstgf::PT_N, (long long)(PAIR_D_RANGE_BYTES / row_bytes) / pstgf::PT_N * pstgf::PT_N);
  range = std::min(range, w.n_E);
  cudaMemPool_t pool;
  PSTGF_CUDA(library_pool(ds.device, &pool, true));
  void *scratch = nullptr;
  const cudaError_t ae = cudaMallocFromPoolAsync(&scratch, pair_scratch_bytes(w.n_chan, w.n_poles, range), pool, s);
  if (ae != cudaSuccess) {
    (void)cudaGetLastError();
    if (ae != cudaErrorMemoryAllocation) return cuda_fail(ae);
    *no_memory = true;
    return PSTGF_OK;
  }
  pstgf_status_t st = PSTGF_OK;
  int launches = 0;
  double *kept_P = nullptr;
  const unsigned int *kept_nm = nullptr;
  for (int e0 = 0; e0 < w.n_E && st == PSTGF_OK; e0 += range) {
    pstgf_wave_t part = w;
    part.n_E = std::min(range, w.n_E - e0);
    part.energies = w.energies + e0;
    part.R_out = w.R_out + (size_t)e0 * w.n_chan * w.n_chan;
    if (w.diag_add) part.diag_add = w.diag_add + (size_t)e0 * w.n_chan;
    std::vector<DevWave> d(1);
    plan_wave(part, d[0], ds.l2_bytes);
    if (e0 == 0) {
      plan_pairs(d[0], static_cast<unsigned char *>(scratch));     // the first range is a full one: P | D[range] | table
      kept_P = d[0].pair_P;
      kept_nm = d[0].pair_nm;
    } else {                                                       // later ranges: the same P and table, D in the same place
      plan_pairs(d[0], reinterpret_cast<unsigned char *>(kept_P) + ((((size_t)pair_count(w.n_chan) * row_bytes) + 255) & ~(size_t)255),
                 kept_P, kept_nm);
    }
    plan_pair_tails(d, ds.sm_count);
    st = encode_pair_maps(d[0]);
    if (st != PSTGF_OK) break;
    const int rows = d[0].n_E + (d[0].pair_keep_P ? 0 : d[0].n_pairs);
    const int chunks = (rows + pstgf::PAIR_BUILD_ROWS - 1) / pstgf::PAIR_BUILD_ROWS;
    pstgf::pair_build_kernel<false><<<dim3((unsigned)std::min(chunks, 8 * ds.sm_count), 1), 256, 0, s>>>(d[0], nullptr, 1);
    const cudaError_t le = cudaGetLastError();
    if (le != cudaSuccess) { st = cuda_fail(le); break; }
    st = launch_single(d, ds, s);
    launches += 2;
  }
  cudaFreeAsync(scratch, s);
  if (st == PSTGF_OK) tl_launches = launches;
  return st;
}

static pstgf_status_t form_single(const pstgf_wave_t &w, void *stream) {
  const int n_chan = w.n_chan, n_poles = w.n_poles, n_E = w.n_E;
  tl_launches = 0;
  pstgf_status_t st = check_wave(w);
  if (st != PSTGF_OK) return st;
  if (n_chan == 0 || n_E == 0) return PSTGF_OK;
  DeviceState ds;
  st = device_state(ds);
  if (st != PSTGF_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (n_poles == 0) return zero_fill(w, s);
  std::vector<DevWave> d(1);
  plan_wave(w, d[0], ds.l2_bytes);
  if (wants_pair_form(n_chan, n_poles, n_E) && wants_small_kernel(n_chan, n_poles, n_E)) {
    PSTGF_CUDA(pstgf::small_launch(d[0], s));
    tl_launches = 1;
    return PSTGF_OK;
  }
  if (wants_pair_form(n_chan, n_poles, n_E)) {
    bool no_memory = false;
    st = form_single_pairs(w, ds, s, &no_memory);
    if (!no_memory) return st;
    // no device memory for P and D: the symmetric form below needs none (a few ulp apart, see the header)
  }
  plan_slabs(d, ds.sm_count);
  plan_tails(d, ds.sm_count);
  st = encode_map(d[0]);
  if (st != PSTGF_OK) return st;
  st = launch_single(d, ds, s);
  if (st != PSTGF_OK) return st;
  tl_launches = 1;
  return PSTGF_OK;
}

pstgf_status_t pstgf_rmat_form(const double *W, long long ldw, const double *E_k, const double *energies, int n_chan,
                               int n_poles, int n_E, double a, double *R_out, void *stream) {
  pstgf_wave_t w{n_chan, n_poles, n_E, PSTGF_W_POLE_CONTIGUOUS, ldw, a, W, E_k, energies, R_out, nullptr};
  return form_single(w, stream);
}

pstgf_status_t pstgf_rmat_form_hdat(const double *Wt, long long ldw, const double *E_k, const double *energies,
                                    int n_chan, int n_poles, int n_E, double a, double *R_out, void *stream) {
  pstgf_wave_t w{n_chan, n_poles, n_E, PSTGF_W_CHANNEL_CONTIGUOUS, ldw, a, Wt, E_k, energies, R_out, nullptr};
  return form_single(w, stream);
}

// pstgf_rmat_form without any device allocation: the same plan, the same kernels and therefore the same bits, with
// the scratch and the work counter in g_static_scratch.  No cudaMalloc*, cudaFree*, memory pool or event is touched.
pstgf_status_t pstgf_rmat_form_static(const double *W, long long ldw, const double *E_k, const double *energies,
                                      int n_chan, int n_poles, int n_E, double a, double *R_out, void *stream) {
  const pstgf_wave_t w{n_chan, n_poles, n_E, PSTGF_W_POLE_CONTIGUOUS, ldw, a, W, E_k, energies, R_out, nullptr};
  tl_launches = 0;
  pstgf_status_t st = check_wave(w);
  if (st != PSTGF_OK) return st;
  if (n_chan == 0 || n_E == 0) return PSTGF_OK;
  const bool pair = wants_pair_form(n_chan, n_poles, n_E);
  const bool small = pair && wants_small_kernel(n_chan, n_poles, n_E);      // one launch, no scratch at all
  // the size check needs no device: too large a wave is refused before any CUDA call
  if (pair && !small && pair_scratch_bytes(n_chan, n_poles, n_E) > (size_t)PSTGF_STATIC_SCRATCH_BYTES - STATIC_COUNTER_BYTES)
    return PSTGF_ERR_STATIC_LIMIT;
  DeviceState ds;
  st = device_state(ds);
  if (st != PSTGF_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (n_poles == 0) return zero_fill(w, s);
  std::vector<DevWave> d(1);
  plan_wave(w, d[0], ds.l2_bytes);
  if (small) {
    PSTGF_CUDA(pstgf::small_launch(d[0], s));
    tl_launches = 1;
    return PSTGF_OK;
  }
  unsigned char *base = nullptr;
  st = static_scratch_address(ds.device, &base);       // the first call on this device looks the address up
  if (st != PSTGF_OK) return st;
  int launches = 0;
  if (pair) {
    // P, D and the pair table are written in full by the builder before the GEMM items read them, so what the last
    // call left in the array does not matter
    plan_pairs(d[0], base + STATIC_COUNTER_BYTES);
    plan_pair_tails(d, ds.sm_count);
    st = encode_pair_maps(d[0]);
    if (st != PSTGF_OK) return st;
    const int rows = d[0].n_E + d[0].n_pairs;
    const int chunks = (rows + pstgf::PAIR_BUILD_ROWS - 1) / pstgf::PAIR_BUILD_ROWS;
    pstgf::pair_build_kernel<false><<<dim3((unsigned)std::min(chunks, 8 * ds.sm_count), 1), 256, 0, s>>>(d[0], nullptr, 1);
    PSTGF_CUDA(cudaGetLastError());
    ++launches;
  } else {
    plan_slabs(d, ds.sm_count);
    plan_tails(d, ds.sm_count);
    st = encode_map(d[0]);
    if (st != PSTGF_OK) return st;
  }
  const long long n_items = wave_items(d[0]);
  const int grid = (int)std::min<long long>(ds.sm_count, n_items);
  const pstgf::RingGeo geo = ring_geometry(d);
  unsigned long long *counter = nullptr;
  if (n_items > grid) {
    // the work counter must start at zero: cleared on the stream ahead of every launch (a launch that ran to its end
    // leaves it zeroed, one that was cut short does not)
    counter = reinterpret_cast<unsigned long long *>(base);
    PSTGF_CUDA(cudaMemsetAsync(counter, 0, 2 * sizeof(unsigned long long), s));
    ++launches;
  }
  pstgf::PersistentArgs pa{&d[0], nullptr, nullptr, 1, n_items, counter, geo, grid};
  PSTGF_CUDA(pstgf::persistent_launch_family(launch_family(d), false, pa, s));
  tl_launches = launches + 1;
  return PSTGF_OK;
}

size_t pstgf_rmat_batch_workspace_bytes(const pstgf_wave_t *waves, int n_waves) {
  return n_waves > 0 ? ws_bytes(waves, n_waves) : 0;
}

// What the host-buffer call needs to know about a batch launch to copy the waves back as they finish.
struct BatchCompletion {
  unsigned int *const *done = nullptr;   // in: per input wave, a zeroed device counter or null
  unsigned int *const *flag = nullptr;   // in: per input wave, a zeroed host-mapped word (device-visible address)
  const unsigned int *const *rows_ready = nullptr;   // in, optional: per input wave, the upload counter of its W
  const int *ready_counts_channels = nullptr;        // ... and what it counts (DevWave::ready_counts_channels)
  unsigned int *abort_flag = nullptr;                // in: zeroed DEVICE word the load warps poll and set when an upload wait times out
  unsigned int *abort_flag_host = nullptr;           // in: host-mapped word the warp that timed out sets as well
  const unsigned char *force_pair = nullptr;         // in, optional: per input wave, 1 = pair form, 0 = SYRK form
  double *const *kept_P = nullptr;                   // in, optional: per input wave, its P built earlier (null = build it here) ...
  const unsigned int *const *kept_nm = nullptr;      // ... and the pair table that goes with it
  std::vector<int> order;                // out: input wave indices in the order the launch completes them
  std::vector<long long> items;          // out: items of each input wave (arrivals = items * EB)
};

static pstgf_status_t form_batch_impl(const pstgf_wave_t *waves, int n_waves, void *workspace, size_t workspace_bytes,
                                      void *stream, BatchCompletion *completion) {
  tl_launches = 0;
  if (n_waves < 0) return PSTGF_ERR_INVALID_VALUE;
  if (n_waves == 0) return PSTGF_OK;
  if (!waves) return PSTGF_ERR_INVALID_VALUE;
  for (int p = 0; p < n_waves; ++p) {
    pstgf_status_t st = check_wave(waves[p]);
    if (st != PSTGF_OK) return st;
  }
  const unsigned char *force_pair = completion ? completion->force_pair : nullptr;
  double *const *kept_P = completion ? completion->kept_P : nullptr;
  if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) != 0 || workspace_bytes < ws_bytes(waves, n_waves, force_pair, kept_P))
    return PSTGF_ERR_WORKSPACE;
  DeviceState dstate;
  pstgf_status_t st = device_state(dstate);
  if (st != PSTGF_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  // the tables go to the workspace by a copy from this call's own host memory: a captured graph would replay a
  // copy from memory that is long gone, so the batch call refuses to be captured
  if (stream_is_capturing(s)) return PSTGF_ERR_CAPTURE;
  int launches = 0;
  // waves with work, most expensive items first (largest-first list scheduling)
  std::vector<int> order;
  for (int p = 0; p < n_waves; ++p) {
    if (wave_has_items(waves[p])) order.push_back(p);
    else {
      st = zero_fill(waves[p], s);
      if (st != PSTGF_OK) return st;
    }
  }
  launches = tl_launches;
  if (order.empty()) return PSTGF_OK;
  std::stable_sort(order.begin(), order.end(),
                   [&](int x, int y) { return wave_item_cost(waves[x]) > wave_item_cost(waves[y]); });
  const int nw = (int)order.size();
  if (nw == 1 && !completion) {
    // one tiny wave: the one-launch kernel, as in the single-wave call (same bits: rmat_small.cu)
    const pstgf_wave_t &w = waves[order[0]];
    if (wants_pair_form(w.n_chan, w.n_poles, w.n_E) && wants_small_kernel(w.n_chan, w.n_poles, w.n_E)) {
      DevWave d;
      plan_wave(w, d, dstate.l2_bytes);
      PSTGF_CUDA(pstgf::small_launch(d, s));
      tl_launches = launches + 1;
      return PSTGF_OK;
    }
  }
  // A batch that mixes pair-form waves with others goes out as TWO launches, the pair-form waves first (they are the
  // small ones): each launch then runs the kernel instantiation that holds only its own item families, with the ring
  // geometry that suits them -- in one launch the pair consumer's code costs the classic items 1.4 % and the pair
  // items' 8-panel stages cut the ring from 7 stages to 5 (config 4: 137.2 ms in one launch).
  auto is_pair = [&](int p) {
    const pstgf_wave_t &w = waves[p];
    return force_pair ? force_pair[p] != 0 : wants_pair_form(w.n_chan, w.n_poles, w.n_E);
  };
  const int n_pair_waves = (int)std::count_if(order.begin(), order.end(), is_pair);
  if (n_pair_waves > 0 && n_pair_waves < nw) std::stable_partition(order.begin(), order.end(), is_pair);
  const int n_groups = (n_pair_waves > 0 && n_pair_waves < nw) ? 2 : 1;
  const int group_begin[3] = {0, n_groups == 2 ? n_pair_waves : nw, nw};
  // host image of the workspace: [counters | item_begin tables, 3 n + 1 entries per launch | DevWave[nw]]; the item
  // sections of a launch are the coarse items of every wave (largest first), then the slab items of every wave, then
  // the fine items of every wave
  const size_t off_begin = WS_COUNTER_BYTES, off_waves = WS_COUNTER_BYTES + ws_item_begin_bytes(n_waves);
  std::vector<unsigned char> img(off_waves + (size_t)nw * sizeof(DevWave), 0);
  long long *item_begin = reinterpret_cast<long long *>(img.data() + off_begin);
  std::vector<DevWave> ds((size_t)nw);
  unsigned char *ws = static_cast<unsigned char *>(workspace);
  size_t scratch_off = ws_tables_bytes(n_waves);
  int max_build_rows = 0;
  for (int q = 0; q < nw; ++q) {
    const pstgf_wave_t &w = waves[order[q]];
    plan_wave(w, ds[q], dstate.l2_bytes);
    if (is_pair(order[q])) {
      if (kept_P && kept_P[order[q]]) {                  // the host call built this wave's P once for all its energy ranges
        plan_pairs(ds[q], ws + scratch_off, kept_P[order[q]], completion->kept_nm[order[q]]);
        scratch_off += pair_D_bytes(w.n_poles, w.n_E);
      } else {
        plan_pairs(ds[q], ws + scratch_off);
        scratch_off += pair_scratch_bytes(w.n_chan, w.n_poles, w.n_E);
      }
      max_build_rows = std::max(max_build_rows, ds[q].n_E + (ds[q].pair_keep_P ? 0 : ds[q].n_pairs));
      st = encode_pair_maps(ds[q]);
      if (st != PSTGF_OK) return st;
    }
  }
  // every launch is planned on its own: its slab tiles, its tails
  std::vector<std::vector<DevWave>> parts((size_t)n_groups);
  for (int g = 0; g < n_groups; ++g) {
    parts[(size_t)g].assign(ds.begin() + group_begin[g], ds.begin() + group_begin[g + 1]);
    plan_slabs(parts[(size_t)g], dstate.sm_count);
    plan_tails(parts[(size_t)g], dstate.sm_count);
    plan_pair_tails(parts[(size_t)g], dstate.sm_count);
    std::copy(parts[(size_t)g].begin(), parts[(size_t)g].end(), ds.begin() + group_begin[g]);
  }
  if (completion && completion->done)
    for (int q = 0; q < nw; ++q) {
      ds[q].done = completion->done[order[q]];
      ds[q].done_flag = completion->flag[order[q]];
      ds[q].done_target = (unsigned int)(wave_items(ds[q]) * pstgf::EB);   // one arrival per consumer warp and item
      if (completion->rows_ready) {
        ds[q].rows_ready = completion->rows_ready[order[q]];
        ds[q].ready_counts_channels = completion->ready_counts_channels[order[q]];
        ds[q].abort_flag = completion->abort_flag;
        ds[q].abort_flag_host = completion->abort_flag_host;
        ds[q].wait_timeout_ms = tl_upload_timeout_ms;
      }
    }
  if (completion) {
    // launch by launch; inside a launch coarse items, then slab items, then fine items: a wave is complete when its
    // last section is
    completion->items.assign((size_t)n_waves, 0);
    completion->order.clear();
    for (int g = 0; g < n_groups; ++g)
      for (int pass = 0; pass < 3; ++pass)
        for (int q = group_begin[g]; q < group_begin[g + 1]; ++q) {
          const int last = fine_items(ds[q]) > 0 ? 2 : slab_items(ds[q]) > 0 ? 1 : 0;
          if (last == pass) completion->order.push_back(order[q]);
        }
    for (int q = 0; q < nw; ++q) completion->items[(size_t)order[q]] = wave_items(ds[q]);
  }
  long long totals[2] = {0, 0};
  size_t table_off[2] = {0, 0};
  for (int g = 0; g < n_groups; ++g) {
    const int q0 = group_begin[g], n = group_begin[g + 1] - q0;
    table_off[g] = g == 0 ? 0 : (size_t)(3 * group_begin[1] + 1);
    long long *tb = item_begin + table_off[g];
    long long total = 0;
    for (int i = 0; i < n; ++i) {
      if (ds[q0 + i].n_pairs == 0) {
        st = encode_map(ds[q0 + i]);
        if (st != PSTGF_OK) return st;
      }
      std::memcpy(img.data() + off_waves + (size_t)(q0 + i) * sizeof(DevWave), &ds[q0 + i], sizeof(DevWave));
      tb[i] = total;
      total += coarse_items(ds[q0 + i]);
    }
    for (int i = 0; i < n; ++i) {
      tb[n + i] = total;
      total += slab_items(ds[q0 + i]);
    }
    for (int i = 0; i < n; ++i) {
      tb[2 * n + i] = total;
      total += fine_items(ds[q0 + i]);
    }
    tb[3 * n] = total;
    totals[g] = total;
  }
  PSTGF_CUDA(cudaMemcpyAsync(ws, img.data(), img.size(), cudaMemcpyHostToDevice, s));
  if (n_pair_waves > 0) {
    // P and D of every pair-form wave in one launch (grid.y = the waves; the others return at once)
    DevWave none;
    std::memset(&none, 0, sizeof(none));
    const int bx = std::max(1, std::min((max_build_rows + pstgf::PAIR_BUILD_ROWS - 1) / pstgf::PAIR_BUILD_ROWS, std::max(2, 8 * dstate.sm_count / nw)));
    pstgf::pair_build_kernel<true><<<dim3((unsigned)bx, (unsigned)std::min(nw, 65535)), 256, 0, s>>>(none, reinterpret_cast<const DevWave *>(ws + off_waves), nw);
    PSTGF_CUDA(cudaGetLastError());
    ++launches;
  }
  for (int g = 0; g < n_groups; ++g) {
    const int q0 = group_begin[g], n = group_begin[g + 1] - q0;
    const std::vector<DevWave> part(ds.begin() + q0, ds.begin() + q0 + n);
    const int grid = (int)std::min<long long>(dstate.sm_count, totals[g]);
    const pstgf::RingGeo geo = ring_geometry(part);
    pstgf::PersistentArgs pa{nullptr, reinterpret_cast<const DevWave *>(ws + off_waves) + q0,
                             reinterpret_cast<const long long *>(ws + off_begin) + table_off[g], n, totals[g],
                             reinterpret_cast<unsigned long long *>(ws + 128 * g), geo, grid};   // a work counter per launch
    PSTGF_CUDA(pstgf::persistent_launch_family(launch_family(part), true, pa, s));
    ++launches;
  }
  tl_launches = launches;
  return PSTGF_OK;
}

pstgf_status_t pstgf_rmat_form_batch(const pstgf_wave_t *waves, int n_waves, void *workspace, size_t workspace_bytes,
                                     void *stream) {
  return form_batch_impl(waves, n_waves, workspace, workspace_bytes, stream, nullptr);
}

pstgf_status_t pstgf_rmat_form_naive(const pstgf_wave_t *wave, void *stream) {
  tl_launches = 0;
  if (!wave) return PSTGF_ERR_INVALID_VALUE;
  const pstgf_wave_t &w = *wave;
  pstgf_status_t st = check_wave(w);
  if (st != PSTGF_OK) return st;
  if (w.n_chan == 0 || w.n_E == 0) return PSTGF_OK;
  DeviceState ds;
  st = device_state(ds);
  if (st != PSTGF_OK) return st;
  const long long n_elems = (long long)w.n_E * w.n_chan * w.n_chan;
  const int threads = 128;
  const long long blocks = (n_elems + threads - 1) / threads;
  if (blocks > 0x7fffffffLL) return PSTGF_ERR_INVALID_VALUE;
  const bool tr = w.w_layout == PSTGF_W_CHANNEL_CONTIGUOUS;
  pstgf::rmat_naive_kernel<<<(unsigned)blocks, threads, 0, static_cast<cudaStream_t>(stream)>>>(
      w.W, tr ? 1LL : w.ldw, tr ? w.ldw : 1LL, w.E_k, w.energies, w.n_chan, w.n_poles, n_elems, w.a, w.diag_add, w.R_out);
  PSTGF_CUDA(cudaGetLastError());
  tl_launches = 1;
  return PSTGF_OK;
}

/* the mesh of the namelists is in z-scaled Rydberg, E/z^2; eq. 4 wants E on the scale of the poles. */
pstgf_status_t pstgf_mesh_from_zscaled(const double *e_scaled, long long n, double z, double *e_out) {
  if (n < 0 || !std::isfinite(z) || !(z > 0.0)) return PSTGF_ERR_INVALID_VALUE;
  if (n == 0) return PSTGF_OK;
  if (!e_scaled || !e_out) return PSTGF_ERR_INVALID_VALUE;
  const double z2 = z * z;
  for (long long i = 0; i < n; ++i) e_out[i] = e_scaled[i] * z2;
  return PSTGF_OK;
}

// ---- end-to-end call over HOST buffers ---------------------------------------------------------
namespace {
constexpr int HOST_RING = 3;          // R staging buffers in flight
constexpr int HOST_COMPUTE_STREAMS = 2;

constexpr size_t MAX_CHUNK_SEGMENTS = 4096;

// Completion state of the signalled pipeline, per device and host thread, allocated at the thread's first host
// call: 2 x MAX_CHUNK_SEGMENTS device counters and as many flag words in mapped pinned host memory, plus one
// abort word.  The blocks are owned by a registry so that pstgf_rmat_finalize can free them whatever thread made
// them; a thread notices through the generation number that its cached block is gone.
constexpr size_t MAX_UPLOAD_WAVES = 1024, MAX_UPLOAD_SLABS = 16;
struct HostFlags {
  unsigned int *counters = nullptr;            // device
  volatile unsigned int *flags_host = nullptr; // host view
  unsigned int *flags_dev = nullptr;           // device view of the same words; word [2 MAX_CHUNK_SEGMENTS] is the abort flag
  unsigned int *upload_counters = nullptr;     // device: rows of each wave's W uploaded so far
  unsigned int *upload_values = nullptr;       // pinned host: the values the upload stream copies into them
  int device = -1;
};
std::mutex g_flags_mutex;
std::vector<HostFlags *> g_flags_registry;
std::atomic<unsigned long long> g_flags_generation{1};

void free_host_flags(HostFlags *f) {
  if (f->counters) cudaFree(f->counters);
  if (f->flags_host) cudaFreeHost(const_cast<unsigned int *>(f->flags_host));
  if (f->upload_counters) cudaFree(f->upload_counters);
  if (f->upload_values) cudaFreeHost(f->upload_values);
  delete f;
}

cudaError_t host_call_flags(int dev, HostFlags *out) {
  static thread_local HostFlags *cache[64] = {nullptr};
  static thread_local unsigned long long cache_generation = 0;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  const unsigned long long gen = g_flags_generation.load();
  if (cache_generation != gen) {
    for (HostFlags *&c : cache) c = nullptr;      // freed by pstgf_rmat_finalize
    cache_generation = gen;
  }
  if (!cache[dev]) {
    HostFlags *f = new HostFlags;
    f->device = dev;
    void *c = nullptr, *h = nullptr, *d = nullptr, *uc = nullptr, *uv = nullptr;
    const size_t bytes = (2 * MAX_CHUNK_SEGMENTS + 1) * sizeof(unsigned int);
    cudaError_t e = cudaMalloc(&c, bytes);
    if (e == cudaSuccess) e = cudaHostAlloc(&h, bytes, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&d, h, 0);
    if (e == cudaSuccess) e = cudaMalloc(&uc, MAX_UPLOAD_WAVES * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaHostAlloc(&uv, MAX_UPLOAD_WAVES * (MAX_UPLOAD_SLABS + 1) * sizeof(unsigned int), cudaHostAllocDefault);
    f->counters = static_cast<unsigned int *>(c);
    f->flags_host = static_cast<volatile unsigned int *>(h);
    f->flags_dev = static_cast<unsigned int *>(d);
    f->upload_counters = static_cast<unsigned int *>(uc);
    f->upload_values = static_cast<unsigned int *>(uv);
    if (e != cudaSuccess) {
      free_host_flags(f);
      return e;
    }
    std::lock_guard<std::mutex> lock(g_flags_mutex);
    g_flags_registry.push_back(f);
    cache[dev] = f;
  }
  *out = *cache[dev];
  return cudaSuccess;
}

struct HostCallResources {
  cudaStream_t s = nullptr, copy = nullptr, compute[HOST_COMPUTE_STREAMS] = {nullptr, nullptr};
  cudaEvent_t inputs = nullptr, computed[HOST_RING] = {nullptr}, copied[HOST_RING] = {nullptr};
  std::vector<void *> allocs;
  ~HostCallResources() {
    for (cudaStream_t c : compute) if (c) cudaStreamSynchronize(c);
    if (copy) cudaStreamSynchronize(copy);
    cudaStreamSynchronize(s);
    for (void *p : allocs) cudaFreeAsync(p, s);
    cudaStreamSynchronize(s);
    if (inputs) cudaEventDestroy(inputs);
    for (int b = 0; b < HOST_RING; ++b) {
      if (computed[b]) cudaEventDestroy(computed[b]);
      if (copied[b]) cudaEventDestroy(copied[b]);
    }
    for (cudaStream_t c : compute) if (c) cudaStreamDestroy(c);
    if (copy) cudaStreamDestroy(copy);
  }
};
struct Segment { int wave, e0, ne; size_t off; };
}  // namespace

pstgf_status_t pstgf_rmat_form_batch_host(const pstgf_wave_t *waves, int n_waves, size_t max_chunk_bytes, void *stream) {
  tl_launches = 0;
  if (n_waves < 0) return PSTGF_ERR_INVALID_VALUE;
  if (n_waves == 0) return PSTGF_OK;
  if (!waves) return PSTGF_ERR_INVALID_VALUE;
  size_t total_r = 0;
  for (int p = 0; p < n_waves; ++p) {
    pstgf_status_t st = check_wave(waves[p]);
    if (st != PSTGF_OK) return st;
    if (wave_has_items(waves[p])) total_r += sizeof(double) * (size_t)waves[p].n_E * waves[p].n_chan * waves[p].n_chan;
  }
  DeviceState ds;
  pstgf_status_t st = device_state(ds);
  if (st != PSTGF_OK) return st;
  if (stream_is_capturing(static_cast<cudaStream_t>(stream))) return PSTGF_ERR_CAPTURE;   // the call synchronises
  // Pipeline choice: the signalled single launch, unless the knob asks for one launch per piece or the whole
  // job is a matter of a millisecond or two (then the naps of the flag polling cost more than launches do).
  double est_flop = 0.0;
  for (int p = 0; p < n_waves; ++p)
    if (wave_has_items(waves[p])) est_flop += (double)waves[p].n_E * waves[p].n_chan * (double)waves[p].n_chan * waves[p].n_poles;
  const bool signalled = tl_host_pipeline == PSTGF_HOST_PIPELINE_AUTO && est_flop / 33e12 >= 2e-3;
  // copy-back granularity (a piece): 1/32 of R in [8, 64] MiB when pieces are free (signalled), 1/8 of R in
  // [16, 256] MiB when each piece is a launch
  size_t cap = max_chunk_bytes;
  if (!cap)
    cap = signalled ? std::min<size_t>((size_t)64 << 20, std::max<size_t>((size_t)8 << 20, total_r / 32))
                    : std::min<size_t>((size_t)256 << 20, std::max<size_t>((size_t)16 << 20, total_r / 8));
  HostCallResources res;
  res.s = static_cast<cudaStream_t>(stream);
  cudaMemPool_t pool;
  PSTGF_CUDA(library_pool(ds.device, &pool));
  PSTGF_CUDA(cudaStreamCreateWithFlags(&res.copy, cudaStreamNonBlocking));
  for (cudaStream_t &c : res.compute) PSTGF_CUDA(cudaStreamCreateWithFlags(&c, cudaStreamNonBlocking));
  PSTGF_CUDA(cudaEventCreateWithFlags(&res.inputs, cudaEventDisableTiming));
  for (int b = 0; b < HOST_RING; ++b) {
    PSTGF_CUDA(cudaEventCreateWithFlags(&res.computed[b], cudaEventDisableTiming));
    PSTGF_CUDA(cudaEventCreateWithFlags(&res.copied[b], cudaEventDisableTiming));
  }
  auto dev_alloc = [&](size_t bytes, void **out) -> cudaError_t {
    cudaError_t e = cudaMallocFromPoolAsync(out, bytes ? bytes : 8, pool, res.s);
    if (e == cudaSuccess) res.allocs.push_back(*out);
    return e;
  };
  // inputs, first part: allocations and the small arrays (poles, energies, diagonal addends).  W follows further
  // down: in the signalled pipeline it is uploaded in slabs of poles WHILE the launch runs, each slab followed by an
  // update of the wave's upload counter that the kernel's load warp waits on stage by stage.
  HostFlags flags;
  if (signalled) PSTGF_CUDA(host_call_flags(ds.device, &flags));
  const bool overlap_upload = signalled && (size_t)n_waves <= MAX_UPLOAD_WAVES;
  volatile unsigned int *abort_host = signalled ? flags.flags_host + 2 * MAX_CHUNK_SEGMENTS : nullptr;
  if (signalled) {
    *abort_host = 0u;
    PSTGF_CUDA(cudaMemsetAsync(flags.counters + 2 * MAX_CHUNK_SEGMENTS, 0, sizeof(unsigned int), res.s));   // the device's copy
  }
  if (overlap_upload) PSTGF_CUDA(cudaMemsetAsync(flags.upload_counters, 0, sizeof(unsigned int) * (size_t)n_waves, res.s));
  std::vector<pstgf_wave_t> dev(waves, waves + n_waves);
  // poles [k0, k1) of all channels, or (by_channels, pole-contiguous W only) channels [k0, k1) with all their poles
  auto upload_W = [&](int p, long long k0, long long k1, bool by_channels) -> cudaError_t {
    const pstgf_wave_t &w = waves[p];
    double *dst = const_cast<double *>(dev[p].W);
    const bool tr = w.w_layout == PSTGF_W_CHANNEL_CONTIGUOUS;
    if (tr || by_channels)                              // whole rows of the array
      return cudaMemcpy2DAsync(dst + k0 * dev[p].ldw, (size_t)dev[p].ldw * 8, w.W + k0 * w.ldw, (size_t)w.ldw * 8,
                               (size_t)(tr ? w.n_chan : w.n_poles) * 8, (size_t)(k1 - k0), cudaMemcpyHostToDevice, res.s);
    return cudaMemcpy2DAsync(dst + k0, (size_t)dev[p].ldw * 8, w.W + k0, (size_t)w.ldw * 8, (size_t)(k1 - k0) * 8,
                             (size_t)w.n_chan, cudaMemcpyHostToDevice, res.s);   // a column range of every channel
  };
  std::vector<int> by_channels((size_t)n_waves, 0);
  // waves done in the pair form: decided on the WHOLE wave (every energy range of it then goes the same way, so the
  // host call gives the bits of the device calls), and their W is uploaded before the launches (P is built from all of it)
  std::vector<unsigned char> pair_wave((size_t)n_waves, 0);
  std::vector<double *> kept_P((size_t)n_waves, nullptr);
  std::vector<const unsigned int *> kept_nm((size_t)n_waves, nullptr);
  int p_launches = 0;
  for (int p = 0; p < n_waves; ++p) pair_wave[(size_t)p] = wants_pair_form(waves[p].n_chan, waves[p].n_poles, waves[p].n_E) ? 1 : 0;
  for (int p = 0; p < n_waves; ++p) {
    const pstgf_wave_t &w = waves[p];
    if (w.n_chan == 0 || w.n_E == 0) continue;
    if (w.n_poles == 0) {
      const size_t cc = (size_t)w.n_chan * w.n_chan;
      std::memset(w.R_out, 0, sizeof(double) * (size_t)w.n_E * cc);
      if (w.diag_add)
        for (int e = 0; e < w.n_E; ++e)
          for (int n = 0; n < w.n_chan; ++n) w.R_out[(size_t)e * cc + (size_t)n * w.n_chan + n] = w.diag_add[(size_t)e * w.n_chan + n];
      continue;
    }
    const bool tr = w.w_layout == PSTGF_W_CHANNEL_CONTIGUOUS;
    const long long w_rows = tr ? w.n_poles : w.n_chan, w_cols = tr ? w.n_chan : w.n_poles;
    const long long pitch = (w_cols + 1) & ~1LL;     // even leading dimension: the TMA staging path applies
    void *dW, *dEk, *dEn;
    PSTGF_CUDA(dev_alloc(sizeof(double) * (size_t)pitch * w_rows, &dW));
    PSTGF_CUDA(dev_alloc(sizeof(double) * (size_t)w.n_poles, &dEk));
    PSTGF_CUDA(dev_alloc(sizeof(double) * (size_t)w.n_E, &dEn));
    PSTGF_CUDA(cudaMemcpyAsync(dEk, w.E_k, sizeof(double) * (size_t)w.n_poles, cudaMemcpyHostToDevice, res.s));
    PSTGF_CUDA(cudaMemcpyAsync(dEn, w.energies, sizeof(double) * (size_t)w.n_E, cudaMemcpyHostToDevice, res.s));
    if (w.diag_add) {
      void *dDa;
      PSTGF_CUDA(dev_alloc(sizeof(double) * (size_t)w.n_E * w.n_chan, &dDa));
      PSTGF_CUDA(cudaMemcpyAsync(dDa, w.diag_add, sizeof(double) * (size_t)w.n_E * w.n_chan, cudaMemcpyHostToDevice, res.s));
      dev[p].diag_add = static_cast<double *>(dDa);
    }
    dev[p].W = static_cast<double *>(dW);
    dev[p].ldw = pitch;
    dev[p].E_k = static_cast<double *>(dEk);
    dev[p].energies = static_cast<double *>(dEn);
    if (!overlap_upload || pair_wave[(size_t)p]) PSTGF_CUDA(upload_W(p, 0, w.n_poles, false));
    if (pair_wave[(size_t)p]) {
      // P = w_n w_m and the pair table hold no energy: built ONCE per wave here, behind its W on `stream`, and shared
      // by every energy range (segment) of the wave in every chunk; the segments' own scratch is D alone
      void *dP;
      PSTGF_CUDA(dev_alloc(pair_scratch_bytes(w.n_chan, w.n_poles, 0), &dP));
      DevWave d;
      plan_wave(dev[p], d, ds.l2_bytes);
      d.n_E = 0;                                         // rows of P only
      plan_pairs(d, static_cast<unsigned char *>(dP));
      kept_P[(size_t)p] = d.pair_P;
      kept_nm[(size_t)p] = d.pair_nm;
      const int chunks_p = (d.n_pairs + pstgf::PAIR_BUILD_ROWS - 1) / pstgf::PAIR_BUILD_ROWS;
      pstgf::pair_build_kernel<false><<<dim3((unsigned)std::min(chunks_p, 8 * ds.sm_count), 1), 256, 0, res.s>>>(d, nullptr, 1);
      PSTGF_CUDA(cudaGetLastError());
      ++p_launches;
    }
  }
  // Two ways to overlap the copy-back with the formation (pstgf_debug_set_host_pipeline):
  //  signalled  ONE launch forms a whole chunk (as much of R as the device budget allows); its segments (a wave's
  //             energy range of at most `cap` bytes) are the waves of that launch, each with a completion
  //             counter; the warp whose arrival completes a segment raises a flag in mapped host memory, and
  //             this thread, which polls the flags in completion order, enqueues the segment's copy-back at
  //             once.  No launch boundaries, no per-chunk tails.  (Stream wait-value on the counters was tried
  //             first: its polling made the copy stream erratic, 7-20 ms against 3 ms on config 2.)
  //  chunked    one launch per chunk of at most `cap` bytes, copy-back ordered by events.
  size_t chunk_cap = cap;
  if (signalled) {
    // device budget of a chunk: a quarter of the device's memory, at most 16 GiB (two chunks may be in flight),
    // halved below when the allocation fails (another allocator holding the memory); the total is queried once
    // per device -- cudaMemGetInfo on every call showed up as occasional stalls of tens of ms
    static std::atomic<size_t> budget[64];
    size_t bud = ds.device < 64 ? budget[ds.device].load() : 0;
    if (!bud) {
      size_t free_b = 0, total_b = 0;
      PSTGF_CUDA(cudaMemGetInfo(&free_b, &total_b));
      bud = std::min<size_t>((size_t)16 << 30, total_b / 4);
      if (ds.device < 64) budget[ds.device].store(bud);
    }
    chunk_cap = std::max<size_t>(cap, bud);
  }
  // chunks of (wave, energy range) segments: a segment holds at most `cap` bytes of R (at least one energy
  // block), a chunk at most `chunk_cap` bytes and MAX_CHUNK_SEGMENTS segments
  std::vector<std::vector<Segment>> chunks;
  size_t max_chunk = 0, max_segs = 1;
  auto plan_chunks = [&]() {
    chunks.clear();
    max_chunk = 0;
    max_segs = 1;
    size_t cur = 0;
    chunks.emplace_back();
    for (int p = 0; p < n_waves; ++p) {
      const pstgf_wave_t &w = waves[p];
      if (!wave_has_items(w)) continue;
      const size_t per_e = sizeof(double) * (size_t)w.n_chan * w.n_chan;
      int e0 = 0;
      while (e0 < w.n_E) {
        size_t room = chunk_cap > cur ? chunk_cap - cur : 0;
        if (signalled) room = std::min(room, cap);
        int ne = (int)std::min<size_t>((size_t)(w.n_E - e0), room / per_e);
        if (ne < w.n_E - e0) ne -= ne % pstgf::EB;      // split only at energy-block boundaries
        if (signalled && ne <= 0 && chunk_cap > cur && chunk_cap - cur >= per_e * (size_t)pstgf::EB) ne = std::min(pstgf::EB, w.n_E - e0);
        if (ne <= 0 || chunks.back().size() >= MAX_CHUNK_SEGMENTS) {
          if (cur > 0) {                               // close the chunk and retry in an empty one
            chunks.emplace_back();
            cur = 0;
            continue;
          }
          ne = std::min(pstgf::EB, w.n_E - e0);          // one block does not fit the cap: take it anyway
        }
        chunks.back().push_back(Segment{p, e0, ne, cur});
        cur += per_e * (size_t)ne;
        max_chunk = std::max(max_chunk, cur);
        max_segs = std::max(max_segs, chunks.back().size());
        e0 += ne;
      }
    }
    if (chunks.back().empty()) chunks.pop_back();
  };
  plan_chunks();
  if (chunks.empty()) {
    PSTGF_CUDA(cudaStreamSynchronize(res.s));
    return PSTGF_OK;
  }
  int ring = 0;
  void *rbuf[HOST_RING] = {nullptr}, *wsbuf[HOST_RING] = {nullptr};
  size_t wsb = 0;
  for (int attempt = 0;; ++attempt) {
    ring = (int)std::min<size_t>(signalled ? 2 : HOST_RING, chunks.size());
    wsb = 0;     // tables plus the pair-form scratch of the chunk that needs the most
    for (const auto &ch : chunks) {
      size_t b = ws_tables_bytes((int)max_segs);
      for (const Segment &g : ch)
        if (pair_wave[(size_t)g.wave]) b += pair_D_bytes(waves[g.wave].n_poles, g.ne);
      wsb = std::max(wsb, b);
    }
    cudaError_t e = cudaSuccess;
    int got = 0;
    for (; got < ring && e == cudaSuccess; ++got) {
      e = dev_alloc(max_chunk, &rbuf[got]);
      if (e == cudaSuccess) e = dev_alloc(wsb, &wsbuf[got]);
    }
    if (e == cudaSuccess) break;
    (void)cudaGetLastError();
    // out of device memory: give back what this attempt took and retry with chunks of half the size
    // (down to one energy block per chunk)
    if (e != cudaErrorMemoryAllocation || attempt >= 8 || max_chunk <= cap) return cuda_fail(e);
    for (int b = 0; b < got; ++b)
      for (void *ptr : {rbuf[b], wsbuf[b]})
        if (ptr) {
          cudaFreeAsync(ptr, res.s);
          res.allocs.erase(std::remove(res.allocs.begin(), res.allocs.end(), ptr), res.allocs.end());
        }
    for (int b = 0; b < HOST_RING; ++b) rbuf[b] = wsbuf[b] = nullptr;
    chunk_cap = std::max<size_t>(cap, max_chunk / 2);
    plan_chunks();
  }
  // the formation kernels run on two streams of the library's own, so that the first CTAs of chunk c+1 start on
  // the SMs the tail of chunk c has left; both wait for the inputs (and the allocations) enqueued on `stream`
  PSTGF_CUDA(cudaEventRecord(res.inputs, res.s));
  for (cudaStream_t c : res.compute) PSTGF_CUDA(cudaStreamWaitEvent(c, res.inputs, 0));
  // inputs, second part: W in slabs of poles on `stream`, behind the event the launches wait for, so that the
  // k loops of the first items run on the first slabs while the others are still on their way
  if (overlap_upload) {
    for (int p = 0; p < n_waves; ++p) {
      const pstgf_wave_t &w = waves[p];
      if (!wave_has_items(w) || pair_wave[(size_t)p]) continue;
      const size_t bytes = sizeof(double) * (size_t)w.n_chan * (size_t)w.n_poles;
      // Slabs of poles when the upload takes no more than about two item times (~1.4 us per k-tile of 20 poles,
      // ~50 GB/s): the first items' k loops then hide it.  Otherwise slabs of channels, if W's rows are channels.
      const double t_upload = (double)bytes / 50e9, t_item = 1.4e-6 * ((w.n_poles + pstgf::KT - 1) / pstgf::KT);
      by_channels[(size_t)p] = (w.w_layout == PSTGF_W_POLE_CONTIGUOUS && t_upload > 2.0 * t_item) ? 1 : 0;
      const long long extent = by_channels[(size_t)p] ? w.n_chan : w.n_poles;
      // slabs of at least 4 MiB, and at least 512 bytes per row segment when a slab is a column range
      const long long n_slabs = std::max<long long>(1, std::min<long long>({(long long)MAX_UPLOAD_SLABS, by_channels[(size_t)p] ? extent : extent / 64,
                                                                            (long long)(bytes >> 22)}));
      unsigned int *vals = flags.upload_values + (size_t)p * (MAX_UPLOAD_SLABS + 1);
      for (long long sl = 0; sl < n_slabs; ++sl) {
        const long long k0 = extent * sl / n_slabs, k1 = extent * (sl + 1) / n_slabs;
        PSTGF_CUDA(upload_W(p, k0, k1, by_channels[(size_t)p] != 0));
        vals[sl] = (unsigned int)k1;
        if (!tl_stall_upload)     // (pstgf_debug_stall_upload: the signal is withheld and the launch must time out)
          PSTGF_CUDA(cudaMemcpyAsync(flags.upload_counters + p, vals + sl, sizeof(unsigned int), cudaMemcpyHostToDevice, res.s));
      }
    }
  }
  int launches = p_launches;
  std::vector<double *> sub_P;
  std::vector<const unsigned int *> sub_nm;
  std::vector<pstgf_wave_t> sub;
  std::vector<unsigned int *> done, flag;
  std::vector<const unsigned int *> rows_ready;
  std::vector<int> ready_kind;
  std::vector<unsigned char> force;
  BatchCompletion completion;
  for (size_t c = 0; c < chunks.size(); ++c) {
    const int b = (int)(c % ring);
    cudaStream_t cs = res.compute[c % HOST_COMPUTE_STREAMS];
    if (c >= (size_t)ring) PSTGF_CUDA(cudaStreamWaitEvent(cs, res.copied[b], 0));
    sub.clear();
    done.clear();
    flag.clear();
    rows_ready.clear();
    ready_kind.clear();
    force.clear();
    sub_P.clear();
    sub_nm.clear();
    const size_t f0 = (size_t)b * MAX_CHUNK_SEGMENTS;
    for (const Segment &g : chunks[c]) {
      pstgf_wave_t w = dev[g.wave];
      w.energies = dev[g.wave].energies + g.e0;
      if (w.diag_add) w.diag_add = dev[g.wave].diag_add + (size_t)g.e0 * w.n_chan;
      w.n_E = g.ne;
      w.R_out = reinterpret_cast<double *>(static_cast<unsigned char *>(rbuf[b]) + g.off);
      sub.push_back(w);
      force.push_back(pair_wave[(size_t)g.wave]);
      sub_P.push_back(kept_P[(size_t)g.wave]);
      sub_nm.push_back(kept_nm[(size_t)g.wave]);
      if (signalled) {
        done.push_back(flags.counters + f0 + (sub.size() - 1));
        flag.push_back(flags.flags_dev + f0 + (sub.size() - 1));
        rows_ready.push_back(overlap_upload && !pair_wave[(size_t)g.wave] ? flags.upload_counters + g.wave : nullptr);
        ready_kind.push_back(by_channels[(size_t)g.wave]);
      }
    }
    auto copy_back = [&](const Segment &g) -> cudaError_t {
      const pstgf_wave_t &w = waves[g.wave];
      const size_t per_e = sizeof(double) * (size_t)w.n_chan * w.n_chan;
      return cudaMemcpyAsync(w.R_out + (size_t)g.e0 * w.n_chan * w.n_chan, static_cast<unsigned char *>(rbuf[b]) + g.off,
                             per_e * (size_t)g.ne, cudaMemcpyDeviceToHost, res.copy);
    };
    if (signalled) {
      if (c >= (size_t)ring) PSTGF_CUDA(cudaEventSynchronize(res.copied[b]));   // this slot's flags are being reused
      for (size_t q = 0; q < sub.size(); ++q) flags.flags_host[f0 + q] = 0u;
      PSTGF_CUDA(cudaMemsetAsync(flags.counters + f0, 0, sizeof(unsigned int) * sub.size(), cs));
      completion.done = done.data();
      completion.flag = flag.data();
      completion.rows_ready = rows_ready.data();
      completion.ready_counts_channels = ready_kind.data();
      completion.abort_flag = flags.counters + 2 * MAX_CHUNK_SEGMENTS;
      completion.abort_flag_host = flags.flags_dev + 2 * MAX_CHUNK_SEGMENTS;
      completion.force_pair = force.data();
      completion.kept_P = sub_P.data();
      completion.kept_nm = sub_nm.data();
      st = form_batch_impl(sub.data(), (int)sub.size(), wsbuf[b], wsb, cs, &completion);
      if (st != PSTGF_OK) return st;
      launches += tl_launches;
      // poll the flags in completion order: a short spin, then naps of 20 us (a thread that spins for the whole
      // launch can run into the CPU quota of a container and be parked for tens of milliseconds)
      for (int q : completion.order) {
        unsigned long long polls = 0;
        while (flags.flags_host[f0 + (size_t)q] == 0u) {
          if (++polls < 2000) continue;
          std::this_thread::sleep_for(std::chrono::microseconds(20));
          if ((polls & 0xffULL) == 0) {                 // every ~250 naps: has the launch, or the upload, died?
            cudaError_t e = cudaStreamQuery(cs);
            if (e != cudaSuccess && e != cudaErrorNotReady) return cuda_fail(e);
            if (e == cudaSuccess && flags.flags_host[f0 + (size_t)q] == 0u) return cuda_fail(cudaErrorUnknown);
            e = cudaStreamQuery(res.s);
            if (e != cudaSuccess && e != cudaErrorNotReady) return cuda_fail(e);
          }
        }
        if (*abort_host != 0u) break;                    // the launch is draining: its R is not worth copying
        PSTGF_CUDA(copy_back(chunks[c][(size_t)q]));
      }
      if (*abort_host != 0u) {
        PSTGF_CUDA(cudaStreamSynchronize(cs));
        return PSTGF_ERR_TIMEOUT;
      }
    } else {
      BatchCompletion plain;
      plain.force_pair = force.data();
      plain.kept_P = sub_P.data();
      plain.kept_nm = sub_nm.data();
      st = form_batch_impl(sub.data(), (int)sub.size(), wsbuf[b], wsb, cs, &plain);
      if (st != PSTGF_OK) return st;
      launches += tl_launches;
      PSTGF_CUDA(cudaEventRecord(res.computed[b], cs));
      PSTGF_CUDA(cudaStreamWaitEvent(res.copy, res.computed[b], 0));
      for (const Segment &g : chunks[c]) PSTGF_CUDA(copy_back(g));
    }
    PSTGF_CUDA(cudaEventRecord(res.copied[b], res.copy));
  }
  PSTGF_CUDA(cudaStreamSynchronize(res.copy));
  for (cudaStream_t c : res.compute) PSTGF_CUDA(cudaStreamSynchronize(c));
  PSTGF_CUDA(cudaStreamSynchronize(res.s));
  if (signalled && *abort_host != 0u) return PSTGF_ERR_TIMEOUT;
  tl_launches = launches;
  return PSTGF_OK;
}

pstgf_status_t pstgf_debug_set_host_pipeline(int mode) {
  if (mode != PSTGF_HOST_PIPELINE_AUTO && mode != PSTGF_HOST_PIPELINE_CHUNKED) return PSTGF_ERR_INVALID_VALUE;
  tl_host_pipeline = mode;
  return PSTGF_OK;
}

pstgf_status_t pstgf_debug_set_upload_timeout_ms(unsigned int ms) {
  tl_upload_timeout_ms = ms;
  return PSTGF_OK;
}

pstgf_status_t pstgf_debug_stall_upload(int on) {
  tl_stall_upload = on ? 1 : 0;
  return PSTGF_OK;
}

// Frees what the library keeps between calls: the counter pools of pstgf_rmat_form, the memory pools and the
// completion blocks of pstgf_rmat_form_batch_host, the planner caches.  Waits for each device to go idle first.
pstgf_status_t pstgf_rmat_finalize(void) {
  int prev = 0;
  const bool have_dev = cudaGetDevice(&prev) == cudaSuccess;
  if (!have_dev) (void)cudaGetLastError();
  pstgf_status_t result = PSTGF_OK;
  auto on_device = [&](int dev) -> bool {
    if (cudaSetDevice(dev) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) {
      tl_cuda_error = (int)cudaGetLastError();
      result = PSTGF_ERR_CUDA;
      return false;
    }
    return true;
  };
  {
    std::lock_guard<std::mutex> lock(g_counter_mutex);
    for (int dev = 0; dev < 64; ++dev) {
      CounterPool &cp = g_counters[dev];
      if (!cp.base || !on_device(dev)) continue;
      for (int i = 0; i < COUNTER_SLOTS; ++i) cudaEventDestroy(cp.ev[i]);
      cudaFree(cp.base);
      cp = CounterPool();
    }
  }
  {
    std::lock_guard<std::mutex> lock(g_flags_mutex);
    for (HostFlags *f : g_flags_registry)
      if (on_device(f->device)) free_host_flags(f);
    g_flags_registry.clear();
    g_flags_generation.fetch_add(1);
  }
  {
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    for (int dev = 0; dev < 64; ++dev) {
      if ((!g_pool[dev] && !g_scratch_pool[dev]) || !on_device(dev)) continue;
      for (cudaMemPool_t *pools : {g_pool, g_scratch_pool})
        if (pools[dev]) {
          cudaMemPoolDestroy(pools[dev]);
          pools[dev] = nullptr;
        }
    }
  }
  {
    std::lock_guard<std::mutex> lock(g_tail_mutex);
    g_tail_cache.clear();
  }
  {
    std::lock_guard<std::mutex> lock(g_slab_mutex);
    g_slab_cache.clear();
  }
  if (have_dev) cudaSetDevice(prev);
  return result;
}

int pstgf_last_launch_count(void) { return tl_launches; }

const char *pstgf_status_string(pstgf_status_t status) {
  switch (status) {
    case PSTGF_OK: return "PSTGF_OK";
    case PSTGF_ERR_INVALID_VALUE: return "PSTGF_ERR_INVALID_VALUE: null pointer, negative size, ldw < n_poles, or a not finite and > 0";
    case PSTGF_ERR_ALIGNMENT: return "PSTGF_ERR_ALIGNMENT: a pointer is not 8-byte aligned";
    case PSTGF_ERR_WORKSPACE: return "PSTGF_ERR_WORKSPACE: workspace null, not 256-byte aligned, or too small";
    case PSTGF_ERR_UNSUPPORTED_DEVICE: return "PSTGF_ERR_UNSUPPORTED_DEVICE: needs a CUDA device of compute capability 10.x";
    case PSTGF_ERR_CUDA: return "PSTGF_ERR_CUDA: a CUDA call failed, see pstgf_last_cuda_error()";
    case PSTGF_ERR_TIMEOUT: return "PSTGF_ERR_TIMEOUT: the launch gave up waiting for an upload of W; R_out is undefined";
    case PSTGF_ERR_CAPTURE: return "PSTGF_ERR_CAPTURE: this call cannot be captured into a CUDA graph";
    case PSTGF_ERR_STATIC_LIMIT: return "PSTGF_ERR_STATIC_LIMIT: pstgf_rmat_form_static: the wave's pair-form scratch exceeds PSTGF_STATIC_SCRATCH_BYTES";
  }
  return "unknown pstgf_status_t";
}

int pstgf_last_cuda_error(void) { return tl_cuda_error; }

int pstgf_version(void) { return PSTGF_RMAT_VERSION; }

}  // extern "C"
