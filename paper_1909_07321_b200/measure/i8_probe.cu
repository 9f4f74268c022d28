// i8_probe.cu -- measurement utility (bench side, NOT part of libpstgf_rmat.so): issue rate of the INT8 tensor pipe of
// sm_100a, tcgen05.mma.cta_group::1.kind::i8 (SASS UTCIMMA) with both operands resident in shared memory and the
// INT32 accumulators in tensor memory.  It exists to put a MEASURED number under DESIGN.md 11.6, the bound on an
// FP64-accurate evaluation of eq. 4 by INT8 slicing: the product path does not use it.
//
// One CTA per SM, 128 threads.  Warp 0 allocates all 512 TMEM columns; one thread issues `iters` rounds of
// 2 (accumulators) x 4 (k-steps of 32 inside a 128-byte row) MMAs of 128 x 256 x 32 on a fixed pair of shared-memory
// tiles (their contents do not matter to the pipe; the descriptors are the canonical K-major, 128-byte-swizzle ones),
// commits them to an mbarrier and waits.  Operations counted: 2 * 128 * 256 * 32 per MMA.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

// K-major operand tile of `rows` rows x 128 bytes, SWIZZLE_128B: 8-row groups of 1024 bytes one after another.
// Descriptor fields (SM100 matrix descriptor): start address >> 4 in bits [0, 14), leading byte offset >> 4 in
// [16, 30) (unused for swizzled K-major layouts: 1), stride byte offset >> 4 in [32, 46) (1024 bytes between 8-row
// groups), version 1 in [46, 48), layout type 2 (128-byte swizzle) in [61, 64).
__device__ __forceinline__ uint64_t make_desc(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3ffffu) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(1024 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}

// Instruction descriptor of kind::i8: c_format S32 (2) in bits [4, 6), a/b format signed 8 bit (1) in [7, 10) and
// [10, 13), both K-major (0), N >> 3 in [17, 23), M >> 4 in [24, 29).
__device__ __forceinline__ uint32_t make_idesc(int M, int N) {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
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

constexpr int M = 128, N = 256, KSTEP = 32;

__global__ void __launch_bounds__(128, 1) i8_probe_kernel(int iters, unsigned int *sink) {
  extern __shared__ __align__(1024) unsigned char smem[];      // [A 128 x 128 B | B 256 x 128 B], 1024-byte aligned
  __shared__ __align__(8) unsigned long long bar;
  __shared__ uint32_t tmem_base;
  const int warp = threadIdx.x >> 5;
  unsigned char *tiles = smem + ((1024u - (smem_u32(smem) & 1023u)) & 1023u);    // swizzle-128B tiles want 1024-byte alignment
  for (int i = threadIdx.x; i < (M + N) * 128 / 4; i += blockDim.x) reinterpret_cast<uint32_t *>(tiles)[i] = 0x01010101u * (i & 3);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&bar)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the tiles were written through the generic proxy
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = tmem_base;
  if (threadIdx.x == 0) {
    const uint32_t a0 = smem_u32(tiles), b0 = a0 + M * 128;
    const uint32_t idesc = make_idesc(M, N);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int acc = 0; acc < 2; ++acc)
#pragma unroll
        for (int k = 0; k < 128 / KSTEP; ++k)
          mma_i8(tmem + acc * N, make_desc(a0 + k * KSTEP), make_desc(b0 + k * KSTEP), idesc, (it | k) != 0 ? 1u : 0u);
    }
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&bar)) : "memory");
  }
  // everybody waits for the MMAs to drain (phase 0 of the barrier)
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "I8_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n"
      "@p bra I8_DONE;\n"
      "bra I8_WAIT;\n"
      "I8_DONE:\n"
      "}\n" ::"r"(smem_u32(&bar))
      : "memory");
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  // read one accumulator word per thread back so that the work is observable
  uint32_t v;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(tmem + ((uint32_t)(warp * 32) << 16)));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
  if (sink != nullptr && v == 0xdeadbeefu) sink[blockIdx.x] = v;
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
}

}  // namespace

extern "C" {

// Enqueues the probe on `stream` (grid CTAs, one per SM) and returns the INT8 operations (multiply and add counted
// separately) it performs, or -1 on a launch error.
double pstgf_i8_probe(int iters, int grid, unsigned int *sink, void *stream) {
  const int smem = (M + N) * 128 + 1024;
  if (cudaFuncSetAttribute(i8_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return -1.0;
  i8_probe_kernel<<<grid, 128, smem, static_cast<cudaStream_t>(stream)>>>(iters, sink);
  if (cudaGetLastError() != cudaSuccess) return -1.0;
  return 2.0 * M * N * KSTEP * 8.0 * (double)iters * (double)grid;
}

}  // extern "C"
