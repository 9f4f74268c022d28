// rmat_launch.cu -- one instantiation of the persistent kernel (rmat_kernel.cuh) per item family set; compiled three
// times, with -DPSTGF_FAM=0, 1 and 2 (see rmat_launch.h).
#include "rmat_launch.h"
#include "rmat_kernel.cuh"

#ifndef PSTGF_FAM
#error "compile with -DPSTGF_FAM=0|1|2"
#endif

#define PSTGF_CAT2(a, b) a##b
#define PSTGF_CAT(a, b) PSTGF_CAT2(a, b)

namespace pstgf {

cudaError_t PSTGF_CAT(persistent_prepare_f, PSTGF_FAM)() {
  cudaError_t e = cudaFuncSetAttribute(rmat_persistent_kernel<false, PSTGF_FAM>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_MAX_OPTIN);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(rmat_persistent_kernel<true, PSTGF_FAM>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_MAX_OPTIN);
  return e;
}

cudaError_t PSTGF_CAT(persistent_launch_f, PSTGF_FAM)(bool batch, const PersistentArgs &a, cudaStream_t s) {
  if (batch) {
    DevWave none;
    memset(&none, 0, sizeof(none));
    rmat_persistent_kernel<true, PSTGF_FAM><<<a.grid, NUM_THREADS, smem_bytes_for(a.geo), s>>>(none, a.waves, a.item_begin, a.n_waves, a.n_items,
                                                                                             a.counter, a.geo);
  } else {
    rmat_persistent_kernel<false, PSTGF_FAM><<<a.grid, NUM_THREADS, smem_bytes_for(a.geo), s>>>(*a.single, nullptr, nullptr, 1, a.n_items, a.counter,
                                                                                              a.geo);
  }
  return cudaGetLastError();
}

}  // namespace pstgf
