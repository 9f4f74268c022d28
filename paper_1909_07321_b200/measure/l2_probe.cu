// l2_probe.cu -- how fast can one SM pull an L2-resident array into shared memory, and what does it depend on?
//
// Three of the library's item families (single-energy slab items, short pair items, the INT8 variant) are bound by
// the arrival of W panels from L2, and the planner carries that rate as a constant.  This probe measures it with
// nothing else going on: persistent CTAs (one per SM) stream boxes of an array that fits L2 into a shared-memory ring
// and do nothing with them.  One warp per CTA issues and waits; the knobs are the things the load pattern of a kernel
// can choose:
//   mode 0   cp.async.bulk.tensor.2d (TMA) boxes of `inner_bytes` x `box_rows` out of a row-major array with a long
//            pitch (80 KB, a row of config 5's W) -- the library's pattern is 160 B x 32 rows
//   mode 1   1-D cp.async.bulk of `inner_bytes * box_rows` contiguous bytes
//   lanes    how many lanes of the warp issue (each issues boxes_per_stage / lanes boxes of a stage)
//   stages   ring depth; bytes in flight per CTA = stages * boxes_per_stage * box bytes
//   cluster  1, 2 or 4 (mode 0 only): every CTA of a cluster issues 1/cluster of each stage's boxes with
//            .multicast::cluster to all of them, so that each box crosses the L2 -> SM fabric once per cluster;
//            a stage is handed back through an `empty` barrier in every CTA that all CTAs of the cluster arrive on
// The launch returns the bytes DELIVERED into shared memory (per CTA: iters * stage bytes, whatever the cluster size);
// the caller times it with CUDA events.  Every wait is bounded: a barrier that does not complete within ~1 s of
// polling sets *status and the CTA leaves (no hang).  Bench-side only: part of libpstgf_probe.so, not of the product.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

namespace {

constexpr int MAX_STAGES = 16;

struct L2ProbeArgs {
  const unsigned char *src;     // mode 1
  unsigned long long src_bytes;
  int mode, inner_bytes, box_rows, boxes_per_stage, lanes, stages, cluster, iters;
  int n_col_tiles, n_row_tiles; // mode 0: tiles of the tensor
  unsigned int *status;         // set to 1 by a CTA whose wait timed out
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

__device__ __forceinline__ bool mbar_wait_bounded(uint32_t bar, uint32_t parity) {
  for (long long spin = 0; spin < (1LL << 22); ++spin) {
    uint32_t done;
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.b32 %0, 1, 0, p;\n}\n"
        : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    if (done) return true;
  }
  return false;
}

__global__ void __launch_bounds__(32) l2_probe_kernel(const __grid_constant__ CUtensorMap map, const L2ProbeArgs a) {
  extern __shared__ __align__(1024) unsigned char ring[];
  __shared__ __align__(8) unsigned long long full[MAX_STAGES], empty[MAX_STAGES];
  const int lane = threadIdx.x;
  const uint32_t box_bytes = (uint32_t)a.inner_bytes * (uint32_t)a.box_rows;
  const uint32_t stage_bytes = box_bytes * (uint32_t)a.boxes_per_stage;
  uint32_t rank = 0;
  if (a.cluster > 1) asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
  if (lane == 0) {
    for (int s = 0; s < a.stages; ++s) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(&full[s])), "r"(1u) : "memory");
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(&empty[s])), "r"((uint32_t)a.cluster) : "memory");
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
  if (a.cluster > 1) {                         // every CTA's barriers exist before anyone multicasts into them
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
  }
  // the boxes of a stage that this CTA issues: [b0, b1) of boxes_per_stage (all of them without a cluster)
  const int per_cta = a.boxes_per_stage / a.cluster;
  const int b0 = (int)rank * per_cta, b1 = b0 + per_cta;
  const unsigned long long cluster_id = blockIdx.x / a.cluster;
  const uint16_t mask = (uint16_t)((1u << a.cluster) - 1u);
  bool ok = true;
  // issue stage `it`'s boxes (this CTA's part); box index -> a tile of the array, different for every cluster and step
  auto issue = [&](int it) {
    const int s = it % a.stages;
    const uint32_t bar = smem_u32(&full[s]);
    if (lane == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(stage_bytes) : "memory");
    __syncwarp();
    for (int b = b0 + lane; b < b1; b += a.lanes) {
      if (lane >= a.lanes) break;
      const unsigned long long idx = (cluster_id * 7919ULL + (unsigned long long)it * 104729ULL) * (unsigned long long)a.boxes_per_stage + b;
      const uint32_t dst = smem_u32(ring + (size_t)s * stage_bytes + (size_t)b * box_bytes);
      if (a.mode == 0) {
        const int c0 = (int)(idx % a.n_col_tiles) * (a.inner_bytes / 8), c1 = (int)((idx / a.n_col_tiles) % a.n_row_tiles) * a.box_rows;
        if (a.cluster > 1)
          asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%2, %3}], [%4], %5;"
                       ::"r"(dst), "l"(&map), "r"(c0), "r"(c1), "r"(bar), "h"(mask) : "memory");
        else
          asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                       ::"r"(dst), "l"(&map), "r"(c0), "r"(c1), "r"(bar) : "memory");
      } else {
        const unsigned long long off = (idx * (unsigned long long)box_bytes) % (a.src_bytes - box_bytes) & ~15ULL;
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(dst), "l"(a.src + off), "r"(box_bytes), "r"(bar) : "memory");
      }
    }
  };
  const int prologue = min(a.stages, a.iters);
  for (int it = 0; it < prologue; ++it) issue(it);
  for (int it = 0; it < a.iters && ok; ++it) {
    const int s = it % a.stages;
    const uint32_t ph = (uint32_t)(it / a.stages) & 1u;
    ok = mbar_wait_bounded(smem_u32(&full[s]), ph);          // the stage has landed (all CTAs' parts of it)
    if (!ok) break;
    const int next = it + a.stages;
    if (next < a.iters) {
      if (a.cluster > 1) {
        // hand the stage back to every CTA of the cluster, then wait until every CTA has handed back ours
        __syncwarp();
        if (lane < a.cluster) {
          uint32_t remote;
          asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(&empty[s])), "r"((uint32_t)lane));
          asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(remote) : "memory");
        }
        ok = mbar_wait_bounded(smem_u32(&empty[s]), ph);
        if (!ok) break;
      }
      issue(next);
    }
  }
  if (!ok && lane == 0) atomicExch(a.status, 1u);
  __syncwarp();
  if (a.cluster > 1) {                         // nobody leaves while a peer may still write into its shared memory
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
  }
}

typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                    const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
encode_tiled_fn g_encode_probe = nullptr;
std::once_flag g_encode_probe_once;

}  // namespace

// src: DEVICE array of src_bytes (a multiple of the 80 KB pitch; at most ~40 MB so that it stays in L2), status: DEVICE
// word (zeroed by the caller).  Returns the bytes delivered into shared memory by the launch, or a negative number for
// bad arguments / a failed launch.  Asynchronous on `stream`.
extern "C" double pstgf_l2_probe(int mode, int inner_bytes, int box_rows, int boxes_per_stage, int lanes, int stages, int cluster,
                                 int iters, int n_ctas, const void *src, unsigned long long src_bytes, unsigned int *status,
                                 void *stream) {
  constexpr unsigned long long PITCH = 81920;                          // bytes: a row of config 5's W
  if (mode < 0 || mode > 1 || inner_bytes < 16 || inner_bytes % 16 || box_rows < 1 || box_rows > 256 || boxes_per_stage < 1 ||
      lanes < 1 || lanes > 32 || stages < 1 || stages > MAX_STAGES || iters < 1 || n_ctas < 1 || !src || !status)
    return -1.0;
  if (cluster != 1 && cluster != 2 && cluster != 4) return -1.0;
  if (cluster > 1 && (mode != 0 || boxes_per_stage % cluster || n_ctas % cluster)) return -1.0;
  if (mode == 0 && (inner_bytes > 2048 || PITCH % inner_bytes)) return -1.0;
  const size_t box_bytes = (size_t)inner_bytes * box_rows, smem = box_bytes * boxes_per_stage * (size_t)stages;
  if (smem > 200 * 1024 || src_bytes < 4 * PITCH * (unsigned long long)box_rows || src_bytes % PITCH) return -1.0;
  std::call_once(g_encode_probe_once, [] {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      g_encode_probe = reinterpret_cast<encode_tiled_fn>(fn);
  });
  if (!g_encode_probe) return -2.0;
  L2ProbeArgs a;
  a.src = static_cast<const unsigned char *>(src);
  a.src_bytes = src_bytes;
  a.mode = mode;
  a.inner_bytes = inner_bytes;
  a.box_rows = box_rows;
  a.boxes_per_stage = boxes_per_stage;
  a.lanes = lanes;
  a.stages = stages;
  a.cluster = cluster;
  a.iters = iters;
  const unsigned long long rows = src_bytes / PITCH;
  a.n_col_tiles = (int)(PITCH / inner_bytes);
  a.n_row_tiles = (int)(rows / box_rows);
  a.status = status;
  CUtensorMap map;
  cuuint64_t dims[2] = {PITCH / 8, rows};
  cuuint64_t strides[1] = {PITCH};
  cuuint32_t box[2] = {(cuuint32_t)(mode == 0 ? inner_bytes / 8 : 2), (cuuint32_t)(mode == 0 ? box_rows : 1)};   // mode 1 does not use the map
  cuuint32_t estr[2] = {1, 1};
  const CUresult er = g_encode_probe(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(src), dims, strides, box, estr,
                                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (er != CUDA_SUCCESS) return -1000.0 - (double)er;
  if (cudaFuncSetAttribute(l2_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -4.0;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)n_ctas);
  cfg.blockDim = dim3(32);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = static_cast<cudaStream_t>(stream);
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cluster;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, l2_probe_kernel, map, a) != cudaSuccess) {
    (void)cudaGetLastError();
    return -5.0;
  }
  return (double)n_ctas * (double)iters * (double)box_bytes * (double)boxes_per_stage;
}
