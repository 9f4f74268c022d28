/*
 * pstgf_rmat.h -- C ABI of libpstgf_rmat.so: R-matrix formation on one B200 (sm_100a).
 *
 * The operation is eq. 4 of arxiv 1909.07321 (section 3):
 *
 *     R_nm(E) = 1/(2 r0) * sum_{k=1..M} w_nk w_mk / (E_k - E)
 *
 * evaluated for every energy E of a mesh and every partial wave, i.e. the
 * batched energy-scaled symmetric contraction
 * R(E) = (1/2a) W diag(1/(E_k - E)) W^T (PSTGF's subroutine RINIT,
 * PAPER.md:168).  a == r0 is the R-matrix radius (record RA),
 * W the surface amplitudes w_nk (record WMAT), E_k the R-matrix
 * poles (record VALUE), one (W, E_k) pair per partial wave with
 * its own NCHAN and MNP2.
 *
 * All arithmetic is IEEE FP64.  There is no CPU fallback and no other device
 * path: every call either enqueues sm_100a kernels or returns an error.
 *
 * Conventions for every call
 *  - Pointers named in "DEVICE" lists are device pointers owned by the caller
 *    (allocate them with any CUDA allocator, e.g. PyTorch).  Any pointer the
 *    device can dereference works, mapped pinned host memory included (R_out
 *    there makes every store a PCIe write: about six times slower than device
 *    memory plus a copy; pstgf_rmat_form_batch_host is the fast host path).
 *  - Device memory owned by the library.  The DEVICE-pointer calls allocate
 *    none, but for the 8 KiB counter pool of pstgf_rmat_form (once per
 *    device) and that call's stream-ordered scratch for few-channel waves
 *    (P plus at most 128 MiB of D whatever n_E is, freed behind the last
 *    launch; the pool it comes from keeps at most 256 MiB across a
 *    synchronise and returns the rest to the device; if the scratch cannot
 *    be had the wave is done in the symmetric form, which needs none);
 *    pstgf_rmat_form_static allocates nothing at all; the batch call keeps
 *    its tables and scratch in the caller's workspace.
 *    pstgf_rmat_form_batch_host stages through a memory pool of its own (one
 *    per device) and keeps 33 KiB of completion words per calling thread.
 *    pstgf_rmat_finalize() frees all of it.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default
 *    stream).  DEVICE-pointer calls enqueue work and return without
 *    synchronising; buffers must stay alive until the stream reaches the end
 *    of the enqueued work.  Host structs (pstgf_wave_t arrays) are consumed
 *    before the call returns.  pstgf_rmat_form / _form_hdat may be captured
 *    into a CUDA graph; the batch calls may not (PSTGF_ERR_CAPTURE: their
 *    tables travel by a copy from the call's own host memory).
 *  - Layout: W is row-major [n_chan][ldw], element (n,k) at W[n*ldw + k],
 *    ldw >= n_poles (k contiguous), unless the wave says
 *    PSTGF_W_CHANNEL_CONTIGUOUS (the H.DAT record order).  R_out is dense row-major
 *    [n_E][n_chan][n_chan]; BOTH triangles are written and R_out[e][n][m] ==
 *    R_out[e][m][n] bitwise.  R_out must not overlap any input or another
 *    wave's R_out.  Inputs may be shared between waves.
 *  - Sizes: n_E == 0, n_chan == 0 or n_waves == 0 -> PSTGF_OK, nothing
 *    written.  n_poles == 0 -> the sum is empty: R_out is zero-filled (plus
 *    diag_add on the diagonal, if given).
 *  - An energy equal to a pole is not detected (data lives on the device):
 *    IEEE semantics apply (inf/NaN in that energy's R).  The paper is silent;
 *    callers keep a clearance (the synthetic workloads use 1e-3 Ryd).
 *  - Alignment: every pointer must be 8-byte aligned (else
 *    PSTGF_ERR_ALIGNMENT).  W 16-byte aligned with even ldw selects the TMA
 *    staging path (for an H.DAT record with an odd NCHAN: copy it with an even
 *    pitch, or accept the slower path); otherwise a slower load path inside the same kernel is
 *    used.  Any n_chan (odd included) is supported.
 *  - Results are deterministic: each R element is produced by exactly one
 *    thread with a fixed k order, whatever CTA picked the work item up, and
 *    however the energies of a call are tiled and grouped.  (A wave with
 *    n_chan <= 96 switches to the pair form at 64 energies, which rounds each
 *    term differently: a few ulp, see pstgf_debug_set_pair_policy.)
 *  - Errors are returned as pstgf_status_t; nothing is thrown or printed.
 *    Argument errors are detected before anything is enqueued.
 */
#ifndef PSTGF_RMAT_H
#define PSTGF_RMAT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PSTGF_RMAT_VERSION 201 /* major*100 + minor; 2.x: pstgf_wave_t grew diag_add (72 bytes); 2.01: pstgf_rmat_form_static */

typedef enum {
  PSTGF_OK = 0,
  PSTGF_ERR_INVALID_VALUE = 1,      /* NULL where data is required, negative size, ldw too small, unknown w_layout, a not finite or <= 0 */
  PSTGF_ERR_ALIGNMENT = 2,          /* a pointer is not 8-byte aligned */
  PSTGF_ERR_WORKSPACE = 3,          /* workspace NULL, not 256-byte aligned, or smaller than the query says */
  PSTGF_ERR_UNSUPPORTED_DEVICE = 4, /* no CUDA device, or the current device is not compute capability 10.x */
  PSTGF_ERR_CUDA = 5,               /* a CUDA runtime/driver call failed; see pstgf_last_cuda_error() */
  PSTGF_ERR_TIMEOUT = 6,            /* pstgf_rmat_form_batch_host: the launch gave up waiting for an upload of W; R_out undefined */
  PSTGF_ERR_CAPTURE = 7,            /* the stream is being captured and this call cannot be (see above) */
  PSTGF_ERR_STATIC_LIMIT = 8        /* pstgf_rmat_form_static: the wave needs more scratch than PSTGF_STATIC_SCRATCH_BYTES */
} pstgf_status_t;

/*
 * One partial wave of a ragged batch: a HOST struct holding DEVICE pointers
 * (or HOST pointers for pstgf_rmat_form_batch_host).  Field meanings as in
 * pstgf_rmat_form.
 */
typedef struct {
  int n_chan;             /* NCHAN */
  int n_poles;            /* MNP2, */
  int n_E;                /* energies of this wave's mesh */
  int w_layout;           /* PSTGF_W_POLE_CONTIGUOUS (0) or PSTGF_W_CHANNEL_CONTIGUOUS (1), see below */
  long long ldw;          /* leading dimension of W in elements, >= n_poles */
  double a;               /* RA, a.u., > 0 */
  const double *W;        /* [n_chan][ldw] */
  const double *E_k;      /* [n_poles] */
  const double *energies; /* [n_E] */
  double *R_out;          /* [n_E][n_chan][n_chan] */
  const double *diag_add; /* optional (NULL = none) [n_E][n_chan]: R_out[e][n][n] = eq. 4 + diag_add[e][n], see below */
} pstgf_wave_t;

/*
 * diag_add: a per-(energy, channel) addend for the diagonal of R, applied by
 * the same epilogue that scales by 1/(2a) and writes R (no second pass over
 * R): R_out[e][n][n] = (1/2a) sum_k w_nk^2 / (E_k - E_e) + diag_add[e][n];
 * off-diagonal elements are untouched (bitwise).  This is where a Buttle
 * correction goes.  PAPER.md lists the DATA of that correction -- records
 * NBUTD / EBUTD / CBUTD per target angular momentum ("the
 * coefficients of the Buttle correction", :544; file DBUT for old inner-region
 * codes, :581-583) -- but NOT its formula (that is in the paper's refs [3],
 * [17]): the formula is not in PAPER.md, so the caller evaluates it and
 * supplies the diagonal.
 */

/*
 * Memory order of W.
 *   PSTGF_W_POLE_CONTIGUOUS     W[n_chan][ldw], element (n,k) at W[n*ldw + k], ldw >= n_poles
 *                               (north_star's W[n_chan x n_poles]).
 *   PSTGF_W_CHANNEL_CONTIGUOUS  W[n_poles][ldw], element (n,k) at W[k*ldw + n], ldw >= n_chan:
 *                               the order of the H.DAT record "((WMAT(I,K) K=1-NCHAN), I=1-MNP2)"
 *                               (channels run fastest, one pole after the other), so a
 *                               record read from H.DATXXX can be handed over as it is, with no
 *                               transposition pass.  The panels are then staged pole-major in shared
 *                               memory by TMA boxes of 36 channels x 20 poles.
 * Both orders give bitwise the same R.
 */
#define PSTGF_W_POLE_CONTIGUOUS 0
#define PSTGF_W_CHANNEL_CONTIGUOUS 1

/*
 * Eq. 4 for one partial wave at n_E energies.
 * DEVICE: W, E_k, energies, R_out.
 *   W        [n_chan][ldw]   surface amplitudes w_nk
 *   E_k      [n_poles]       poles, Ryd, any order
 *   energies [n_E]           energies, same units and origin as E_k
 *   a                        R-matrix radius r0 in a.u., finite and > 0
 *   R_out    [n_E][n_chan][n_chan]
 * One persistent kernel launch (a memset when n_poles == 0; a small scratch-
 * builder launch ahead of it for a wave in the pair form, see
 * pstgf_rmat_form_batch; ONE small launch in all for a tiny pair-form wave of
 * at most 16 channels); work
 * items (energy block, upper-triangle tile) are drawn by the CTAs from an
 * atomic counter.  PSTGF forms R once per (partial wave, energy) (loop over
 * E -> RINIT; one energy per processor at :694): a call
 * with few energies (and the n_E mod 8 energies of any call) is cut into
 * items in which the CTA's eight compute warps share FOUR, TWO or ONE energies
 * and split the tile instead, so n_E = 1 is a first-class
 * shape.  The counter lives in a pool of 64 slots (8 KiB of device
 * memory per device, allocated by the library at the first call -- beside the
 * pair form's stream-ordered scratch the only device allocation of the
 * DEVICE-pointer calls); when 64 launches are in
 * flight at once, or `stream` is being captured into a CUDA graph, items are
 * assigned round-robin instead.  Results do not depend on the assignment.
 */
pstgf_status_t pstgf_rmat_form(const double *W, long long ldw, const double *E_k,
                               const double *energies, int n_chan, int n_poles, int n_E,
                               double a, double *R_out, void *stream);

/*
 * pstgf_rmat_form for W in the H.DAT record order (PSTGF_W_CHANNEL_CONTIGUOUS):
 * DEVICE Wt [n_poles][ldw], element (n,k) at Wt[k*ldw + n], ldw >= n_chan.
 * Everything else as pstgf_rmat_form.
 */
pstgf_status_t pstgf_rmat_form_hdat(const double *Wt, long long ldw, const double *E_k,
                                    const double *energies, int n_chan, int n_poles, int n_E,
                                    double a, double *R_out, void *stream);

/*
 * pstgf_rmat_form for callers that cannot allocate device memory.
 *
 * Who that is: code running where a cudaMalloc / cudaFree is forbidden or harmful.  A process whose device memory
 * is handed out in full at start-up to one arena (a framework's caching allocator, a job that several MPI ranks
 * share one GPU for -- PSTGF's own set-up, Fig. 2 -- each with a fixed slice) has nothing left for a
 * library to take, and a failed allocation deep inside a formation is an error the caller cannot plan for.  A
 * latency-bound loop of one RINIT call per energy cannot afford cudaMalloc / cudaFree either:
 * both may synchronise the whole device.  And a host thread that already holds its framework's allocator lock, or
 * runs as a stream callback, must not enter the CUDA allocator at all.  pstgf_rmat_form does allocate: its work
 * counters come from cudaMalloc at the first call, the pair form's P and D from a memory pool at every call.
 *
 * This call allocates nothing, frees nothing and creates no pool or event.  Its scratch is a fixed array of
 * PSTGF_STATIC_SCRATCH_BYTES (16 MiB) compiled into the library's device image: EVERY GPU on which a process uses
 * libpstgf_rmat.so gives up that much memory from the moment the library's module is loaded until the process
 * exits, whether this call is ever made or not.  That is the price, and the reason the array is modest.
 *
 * Arguments, layout, alignment rules, planning and kernels are those of pstgf_rmat_form; so are the bits of
 * R_out (the tests compare the two calls bitwise).  DEVICE: W, E_k, energies, R_out -- all the caller's.
 *
 * Limit.  A wave that goes the pair form (n_chan <= 96 and n_E >= 64, unless it is tiny enough for the
 * one-launch kernel) needs 8 * ld * (n_chan (n_chan + 1) / 2 + n_E) bytes, ld = n_poles rounded up to even, plus
 * 4 bytes per channel pair, each of the three parts rounded up to 256 bytes; that must fit in
 * PSTGF_STATIC_SCRATCH_BYTES - 256.  E.g. 24 x 480 with 2000 energies (8.8 MB) fits, BASELINE.json's 64 x 1280 x 4096
 * (63 MB) does not.  A larger wave is refused with PSTGF_ERR_STATIC_LIMIT before anything is enqueued and R_out
 * is untouched; nothing is cut down silently.  (pstgf_debug_set_pair_policy(PSTGF_PAIRS_NONE) sends such a wave
 * through the symmetric form, which needs no scratch; a few ulp apart, see there.)  Waves in the symmetric form
 * use only the 16-byte work counter and are accepted at any size.
 *
 * First call on a device.  It asks the runtime once for the array's device address (cudaGetSymbolAddress, with the
 * caller's current device current; the result is remembered per device) and, like every call of this library,
 * raises the kernels' shared-memory limit once.  Make that first call on each device ahead of time, outside any
 * stream capture; later calls only enqueue: one 16-byte memset of the work counter when the launch has more items
 * than CTAs, the scratch builder for a pair-form wave, the persistent kernel.  pstgf_last_launch_count() counts
 * the memset as one.
 *
 * Sharing.  There is ONE array per device and every call of pstgf_rmat_form_static on that device uses it, from
 * any thread and on any stream.  Two calls whose kernels can run on the GPU at the same time (different streams
 * without an event between them, or two host threads) overwrite each other's P, D and counter: wrong R, no error.
 * Keep such calls on one stream, or order them with events.  The array keeps the previous call's contents; the
 * call clears the counter and rewrites every scratch element it later reads, so nothing carries over into R.
 * pstgf_rmat_finalize neither frees nor resets the array (there is nothing to free).
 */
#define PSTGF_STATIC_SCRATCH_BYTES 16777216
pstgf_status_t pstgf_rmat_form_static(const double *W, long long ldw, const double *E_k,
                                      const double *energies, int n_chan, int n_poles, int n_E,
                                      double a, double *R_out, void *stream);

/*
 * Bytes of device workspace pstgf_rmat_form_batch needs for these waves: the
 * tables (about 800 bytes per wave) plus, for every wave that is done in
 * the pair form (n_chan <= 96 with at least 64 energies, see
 * pstgf_rmat_form_batch), 8 * n_poles * (n_chan (n_chan + 1) / 2 + n_E) bytes
 * of scratch.  `waves` is the HOST array that will be passed to the batch call
 * (only the sizes are read; NULL gives the size of the tables alone, which is
 * enough only if no wave takes the pair form).  Returns 0 for n_waves <= 0.
 */
size_t pstgf_rmat_batch_workspace_bytes(const pstgf_wave_t *waves, int n_waves);

/*
 * Eq. 4 for every wave of a ragged batch in ONE persistent kernel launch (two,
 * the pair-form waves first, for a batch that mixes pair-form waves with
 * others; plus their scratch builder).
 * `waves` is a HOST array of n_waves structs with DEVICE pointers.
 * `workspace` is DEVICE memory, 256-byte aligned, at least
 * pstgf_rmat_batch_workspace_bytes() long; it holds the wave table (with one
 * TMA descriptor per wave), the item-range table and the work counter, and
 * may be reused by the next call on the same stream.  Work items (wave,
 * energy block, tile), waves ordered by decreasing cost, are handed to CTAs
 * through an atomic counter: the counterpart of the paper's energy-permuting
 * distribution over MPI ranks (Fig. 1).
 * Waves with few channels (n_chan <= 96) and at least 64 energies are
 * evaluated as the plain GEMM over channel pairs, R[e][(n,m)] = (1/2a) sum_k
 * (w_nk w_mk) * (1/(E_k - E_e)) -- the same eq. 4, term for term, with the
 * products w_nk w_mk and the reciprocals written to scratch first (a second
 * small launch): tiles of an n_chan x n_chan matrix that small are mostly
 * diagonal blocks, which the symmetric form computes in full.  pstgf_rmat_form
 * does the same with stream-ordered scratch of its own (cudaMallocAsync on
 * `stream`, freed behind the last launch): P once, the reciprocals for at most
 * 128 MiB worth of energies at a time -- a longer mesh goes out as several
 * (builder, GEMM) launch pairs over energy ranges.  The host-buffer call
 * builds P once per wave and shares it between the wave's pieces.  The choice
 * depends on the wave's shape only, so a wave gives the same bits through
 * every call (the one exception: pstgf_rmat_form falls back to the symmetric
 * form, a few ulp apart, when the device has no memory left for the scratch).
 */
pstgf_status_t pstgf_rmat_form_batch(const pstgf_wave_t *waves, int n_waves, void *workspace,
                                     size_t workspace_bytes, void *stream);

/*
 * The same result as the calls above for ONE wave (HOST struct, DEVICE
 * pointers) from a one-thread-per-element kernel that follows eq. 4 term by
 * term ((w_n*w_m)/(E_k-E), k ascending, compensated sum, then diag_add).
 * Slow; provided so that callers and tests can check every energy of a large
 * run against an independent device evaluation.
 */
pstgf_status_t pstgf_rmat_form_naive(const pstgf_wave_t *wave, void *stream);

/*
 * VARIANT, never chosen by the calls above: eq. 4 for ONE wave (HOST struct, DEVICE pointers, pole-contiguous W)
 * evaluated on the INT8 tensor pipe (tcgen05.mma kind::i8, INT32 accumulators in tensor memory) instead of the FP64
 * tensor pipe, by slicing W and W diag(1/(E_k - E_e)) into n_slices signed 7-bit digits per element with one
 * power-of-two scale per row and summing the n_slices (n_slices + 1) / 2 leading digit products exactly (SURVEY.md
 * 8f-4).  The result is NOT an IEEE FP64 sum of the terms of eq. 4: it agrees with one to about
 * 1e-12 of max|R| per energy with 7 slices and 1e-14 with 8 (6 miss north_star's 1e-11); both triangles are written
 * and bitwise equal, diag_add is honoured.  n_slices in [2, 8]; n_poles * n_slices < 2^19 (INT32 accumulators).
 * `workspace` is DEVICE memory, 256-byte aligned, of pstgf_rmat_sliced_workspace_bytes() (the digit arrays: n_slices
 * bytes per element of W, once for W and once per energy of a chunk of at most 1 GiB).  Asynchronous on `stream`;
 * measured slower than pstgf_rmat_form on this chip, provided for comparison.
 */
size_t pstgf_rmat_sliced_workspace_bytes(int n_chan, int n_poles, int n_E, int n_slices);
pstgf_status_t pstgf_rmat_form_sliced(const pstgf_wave_t *wave, int n_slices, void *workspace, size_t workspace_bytes,
                                      void *stream);

/*
 * End-to-end convenience over HOST buffers: `waves` holds HOST pointers
 * (pinned memory recommended; pageable memory works but copies synchronously).
 * Inputs are copied to the device on `stream`, R is formed on streams of the
 * library's own in pieces of whole energy blocks and copied back into the host
 * R_out on another stream while the next pieces are being formed.  Device
 * staging for R is bounded per chunk by a quarter of the device's memory, at
 * most 16 GiB, and halved (down to one piece) when that allocation fails
 * because another allocator holds the memory.  Device memory comes from a
 * stream-ordered pool the library owns (one per device, kept until
 * pstgf_rmat_finalize so that repeated calls do not re-grow it).
 * SYNCHRONISES before returning.
 * `max_chunk_bytes` bounds a piece (0 = default: 1/32 of all R in [8, 64] MiB
 * for the signalled pipeline, 1/8 in [16, 256] MiB for the chunked one); a
 * piece always holds at least one energy block.
 * W is uploaded in slabs behind the launch, which waits for the slab it needs
 * next; that wait is bounded (2 s): if an upload never arrives the launch
 * drains and the call returns PSTGF_ERR_TIMEOUT with R_out undefined.
 */
pstgf_status_t pstgf_rmat_form_batch_host(const pstgf_wave_t *waves, int n_waves,
                                          size_t max_chunk_bytes, void *stream);

/*
 * Energy mesh in the units of eq. 4 from the mesh of the namelists: PSTGF's
 * input meshes are "z-scaled energies in Rydberg, E/z^2" (E0, EINCR:
 * PAPER.md:431-435; EMESH: PAPER.md:503), while eq. 4 needs E
 * on the scale of the poles E_k.  HOST arrays: e_out[i] = z*z * e_scaled[i]
 * for i in [0, n) (one rounding of z*z, one per product); e_out may alias
 * e_scaled.  z is the scaling charge, finite and > 0 (the paper does not say
 * what scale a neutral target uses: the caller passes the one its mesh was
 * written in, e.g. 1).  The origin is not moved: meshes given relative to a
 * threshold are the caller's to shift.
 */
pstgf_status_t pstgf_mesh_from_zscaled(const double *e_scaled, long long n, double z, double *e_out);

/*
 * Frees everything the library keeps between calls (counter pools, the host
 * call's memory pools and completion words, planner caches) after waiting for
 * the devices it used to go idle.  No call of this library may be in flight in
 * another thread.  The library may be used again afterwards.
 */
pstgf_status_t pstgf_rmat_finalize(void);

/* ---- knobs for tests and measurements ------------------------------------------------------------
 * THREAD-LOCAL: each affects only the calls the calling thread makes afterwards.  None but the pair
 * policy changes a single bit of any result. */

/*
 * Work items are handed to the persistent CTAs largest first; the END of that list
 * -- about one round of the grid's worth of work -- is cut into finer tiles
 * (32-row instead of 64-row) so that the CTAs run dry together, the device-
 * side counterpart of the paper's concern that no processor be left waiting
 * (Fig. 1).  PSTGF_TAIL_AUTO (default) sizes that tail
 * itself, PSTGF_TAIL_NONE uses coarse tiles only, PSTGF_TAIL_ALL fine tiles
 * only.
 */
#define PSTGF_TAIL_AUTO 0
#define PSTGF_TAIL_NONE 1
#define PSTGF_TAIL_ALL 2
pstgf_status_t pstgf_debug_set_tail_policy(int policy);

/*
 * The n_E mod 8 energies that do not fill a block of 8 are taken four, two or
 * one at a time by "slab" items whose eight warps split a square tile.
 * PSTGF_SLAB_AUTO (default) picks the tile edge (128, 64 or 32) that gives
 * the grid enough items; PSTGF_SLAB_NONE leaves the remainder to a partly
 * idle block of 8 (the round-1 behaviour); _T32/_T64/_T128 force an edge.
 */
#define PSTGF_SLAB_AUTO 0
#define PSTGF_SLAB_NONE 1
#define PSTGF_SLAB_T32 2
#define PSTGF_SLAB_T64 3
#define PSTGF_SLAB_T128 4
pstgf_status_t pstgf_debug_set_slab_policy(int policy);

/*
 * Which waves are evaluated as the GEMM over channel pairs (see
 * pstgf_rmat_form_batch): PSTGF_PAIRS_AUTO (default: n_chan <= 96 and
 * n_E >= 64), PSTGF_PAIRS_NONE (none: the symmetric form for everything, the
 * round-1 behaviour), PSTGF_PAIRS_ALWAYS (every wave with n_chan <= 96).  The
 * two forms round differently (a few ulp apart, both far inside 1e-11).
 */
#define PSTGF_PAIRS_AUTO 0
#define PSTGF_PAIRS_NONE 1
#define PSTGF_PAIRS_ALWAYS 2
pstgf_status_t pstgf_debug_set_pair_policy(int policy);

/*
 * A pair-form wave with at most 16 channels and little work in all (n_chan^2 n_poles n_E <= 2^29, e.g. BASELINE.json
 * configs[0]) is done by a one-launch kernel without scratch when it is the only wave of a call
 * (PSTGF_SMALL_AUTO); PSTGF_SMALL_NONE sends it through the persistent kernel like any pair-form wave,
 * PSTGF_SMALL_ALWAYS drops the bound on the work.  Same bits either way.
 */
#define PSTGF_SMALL_AUTO 0
#define PSTGF_SMALL_NONE 1
#define PSTGF_SMALL_ALWAYS 2
pstgf_status_t pstgf_debug_set_small_policy(int policy);

/*
 * How pstgf_rmat_form_batch_host overlaps formation and copy-back.
 * PSTGF_HOST_PIPELINE_AUTO (default): one launch per device-sized chunk of R; every piece of at
 * most max_chunk_bytes has a completion counter the kernel bumps, the arrival that completes a piece raises a
 * flag in mapped host memory, and the calling thread, which polls the flags, enqueues the piece's copy-back
 * while the same launch goes on forming the next ones; W is uploaded in slabs (ranges of poles or of channels)
 * behind the launch, whose load warp waits on a per-wave upload counter (jobs of under about 2 ms of formation
 * take the CHUNKED route anyway).  PSTGF_HOST_PIPELINE_CHUNKED: one launch per piece, copy-back ordered by events.
 */
#define PSTGF_HOST_PIPELINE_AUTO 0
#define PSTGF_HOST_PIPELINE_CHUNKED 1
pstgf_status_t pstgf_debug_set_host_pipeline(int mode);

/* Bound, in ms, on the kernel's wait for an upload slab of W (0 = the default, 2000). */
pstgf_status_t pstgf_debug_set_upload_timeout_ms(unsigned int ms);
/* on != 0: the host call uploads W but withholds the "slab uploaded" signals, so the launch must take its
 * time-out path (a test of PSTGF_ERR_TIMEOUT). */
pstgf_status_t pstgf_debug_stall_upload(int on);

/* Kernel launches enqueued by this thread's last successful call (for accounting). */
int pstgf_last_launch_count(void);

/* Static description of a status code (never NULL). */
const char *pstgf_status_string(pstgf_status_t status);

/* cudaError_t (as int) behind this thread's last PSTGF_ERR_CUDA, else 0. */
int pstgf_last_cuda_error(void);

/* PSTGF_RMAT_VERSION of the loaded library. */
int pstgf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PSTGF_RMAT_H */
