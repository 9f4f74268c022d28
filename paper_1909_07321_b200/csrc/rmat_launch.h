// rmat_launch.h -- host-side entry points of the persistent kernel (rmat_kernel.cuh).  The kernel is compiled once per
// item family set (rmat_common.h: FAM_CLASSIC, FAM_SLAB, FAM_PAIR), each in a translation unit of its own
// (rmat_launch.cu with -DPSTGF_FAM=0|1|2, built in parallel by build.py); pstgf_rmat.cu picks the smallest set that
// holds the launch's items.
#pragma once
#include <cuda_runtime.h>

#include "rmat_common.h"

namespace pstgf {

struct PersistentArgs {
  const DevWave *single;          // single-wave call: the wave (copied into kernel parameter space); batch call: ignored
  const DevWave *waves;           // batch call: DEVICE array of waves (in the workspace), else null
  const long long *item_begin;    // batch call: DEVICE item-range table, else null
  int n_waves;
  long long n_items;
  unsigned long long *counter;    // DEVICE work counter, or null for round-robin assignment
  RingGeo geo;
  int grid;
};

// persistent_prepare_f<k>: raises the dynamic shared-memory limit of both instantiations (batch / single) of family
// set k on the current device.  persistent_launch_f<k>: enqueues the kernel on `s`; returns the launch error, if any.
cudaError_t persistent_prepare_f0();
cudaError_t persistent_prepare_f1();
cudaError_t persistent_prepare_f2();
cudaError_t persistent_launch_f0(bool batch, const PersistentArgs &a, cudaStream_t s);
cudaError_t persistent_launch_f1(bool batch, const PersistentArgs &a, cudaStream_t s);
cudaError_t persistent_launch_f2(bool batch, const PersistentArgs &a, cudaStream_t s);

// rmat_small.cu: eq. 4 for a tiny wave (pair form, n_chan <= SMALL_MAX_CHAN) in one launch; uses W, E_k, energies,
// R_out, diag_add, ldw, inv2a, n_chan, n_poles, n_E and tr of `w`.
cudaError_t small_launch(const DevWave &w, cudaStream_t s);

// pstgf_rmat.cu: the calling thread's "launches of the last call" / "cudaError_t of the last failure" (what
// pstgf_last_launch_count and pstgf_last_cuda_error report), for entry points that live in other units.
void set_last_call_state(int launches, int cuda_error);

inline cudaError_t persistent_prepare_all() {
  cudaError_t e = persistent_prepare_f0();
  if (e == cudaSuccess) e = persistent_prepare_f1();
  if (e == cudaSuccess) e = persistent_prepare_f2();
  return e;
}
inline cudaError_t persistent_launch_family(int fam, bool batch, const PersistentArgs &a, cudaStream_t s) {
  if (fam >= FAM_PAIR) return persistent_launch_f2(batch, a, s);
  if (fam >= FAM_SLAB) return persistent_launch_f1(batch, a, s);
  return persistent_launch_f0(batch, a, s);
}

}  // namespace pstgf
