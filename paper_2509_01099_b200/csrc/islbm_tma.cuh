// islbm_tma.cuh — sm_100a PTX wrappers shared by the TMA-staged step kernels
// (mbarrier pipeline, cp.async.bulk.tensor loads with an L2 eviction policy,
// policy-hinted global stores) and the host-side tensor-map encoder.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <utility>

namespace islbmk {

// ------------------------------ device side -------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// arrive and learn whether this arrival completed the barrier's phase (i.e. every consumer warp has released the slot)
__device__ __forceinline__ bool mbar_arrive_is_last(uint64_t *bar) {
  uint32_t done;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      ".reg .b64 t;\n"
      "mbarrier.arrive.shared::cta.b64 t, [%1];\n"
      "mbarrier.test_wait.shared::cta.b64 p, [%1], t;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(done)
      : "r"(smem_u32(bar))
      : "memory");
  return done != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

// Programmatic dependent launch (PDL): a step kernel lets the next step's CTAs become resident as soon as its own
// have all started, so their prologue (barrier init, weight staging, descriptor prefetch) and this grid's tail
// overlap; the dependent touches the population buffers only after pdl_wait(), which returns when the
// preceding grid has completed and its stores are visible.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// L2 eviction policy: 0 normal, 1 evict_first, 2 evict_last
__device__ __forceinline__ uint64_t make_policy(int kind) {
  uint64_t p;
  if (kind == 1)
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  else if (kind == 2)
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  else
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}

__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%3, %4, %5}], [%2], %6;" ::"r"(smem_u32(dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2, int c3,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%3, %4, %5, %6}], [%2], %7;" ::"r"(smem_u32(dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%3, %4}], [%2], %5;" ::"r"(smem_u32(dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap *map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

__device__ __forceinline__ void st_hint(double *p, double v, uint64_t policy) {
  asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(policy) : "memory");
}
__device__ __forceinline__ void st_hint(float *p, float v, uint64_t policy) {
  asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(policy) : "memory");
}

// ------------------------------ host side ---------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

inline CUtensorMapL2promotion promo_of(int k) {
  switch (k) {
    case 0: return CU_TENSOR_MAP_L2_PROMOTION_NONE;
    case 1: return CU_TENSOR_MAP_L2_PROMOTION_L2_64B;
    case 2: return CU_TENSOR_MAP_L2_PROMOTION_L2_128B;
    default: return CU_TENSOR_MAP_L2_PROMOTION_L2_256B;
  }
}

// Tensor view of one population buffer for TMA: dims[0] = nx is x (fastest) with a row pitch of row_pitch >= nx
// elements (the padding columns lie outside the tensor, so they read as zero like every out-of-mesh element);
// the other dimensions are dense; the last one is the storage plane.  elem_bytes 8 (fp64) or 4 (fp32 storage).
inline bool make_map(CUtensorMap *m, void *base, int elem_bytes, int rank, const long long *dims, const int *box, int promo,
                     long long row_pitch) {
  EncodeTiledFn enc = get_encode_fn();
  if (!enc || rank < 2 || rank > 5) return false;
  const CUtensorMapDataType dt = elem_bytes == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
  cuuint64_t gd[5], gs[4];
  cuuint32_t bx[5], es[5];
  unsigned long long pitch = (unsigned long long)elem_bytes;
  for (int i = 0; i < rank; ++i) {
    gd[i] = (cuuint64_t)dims[i];
    bx[i] = (cuuint32_t)box[i];
    es[i] = 1;
    pitch *= (unsigned long long)(i == 0 ? row_pitch : dims[i]);
    if (i < rank - 1) gs[i] = (cuuint64_t)pitch;
  }
  return enc(m, dt, (cuuint32_t)rank, base, gd, gs, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
             promo_of(promo), CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// launch with or without the programmatic-stream-serialization attribute
template <typename... KArgs, typename... Args>
inline cudaError_t launch_step(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, bool pdl,
                               Args &&...args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(std::forward<Args>(args))...);
}

constexpr int pad128(int bytes) { return (bytes + 127) / 128 * 128; }

// number of SMs of the current device (148 on a B200), queried once
inline int sm_count() {
  static int sms = 0;
  if (sms <= 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
      cudaGetLastError();
      return 148;   // no device (host-only calls such as islbm_workspace_bytes): sizing only
    }
  }
  return sms;
}

// run-time knobs of the tiled kernels (islbm_set_tuning); defaults chosen from measurements (profiles/)
struct Tuning {
  int chunk = 0;        // marching-chunk length (slices / rows); 0 = automatic
  int l2promo = 0;      // tensor-map L2 promotion: 0 none, 1 64 B, 2 128 B, 3 256 B (none measured fastest)
  int load_policy = 0;  // L2 eviction policy of the TMA loads: 0 normal, 1 evict_first, 2 evict_last
  int store_policy = 0; // ... of the population stores
  int tx2d = 0;         // 2-D strip width: 128 or 224; 0 = automatic
  int shape3d = 0;      // 3-D tile shape (x by y nodes per CTA): 0 automatic, 1 64x4, 2 128x2, 3 32x6, 4 32x4, 5 32x8
  int pdl = 1;          // programmatic dependent launch of consecutive step kernels
  int serpentine = 0;   // 2-D: reverse the CTA -> chunk map on odd steps (L2 reuse of the freshly written rows)
  int fill = 0;         // first ring fill: 1 before the weight rows and the CTA barrier, 2 after them; 0 = automatic
  int ring2d = 0;       // 2-D fp64 ring: 3 stages x 4 CTAs per SM, or 4 stages x 3 CTAs; 0 = automatic
  int rows2d = 0;       // 2-D chunk rule: longest chunk of a multi-wave launch (0 = automatic)
  int rows2d1 = 0;      // 2-D chunk rule: longest chunk for which a single wave is taken (0 = automatic)
  int graph = 0;        // islbm_step(n >= 32): replay a captured CUDA graph of 32 step kernels; 0 = meshes up to 2^20 nodes, 1 always, 2 never
  int slab_wait_ms = 10000;  // fused slab exchange: longest wait for a neighbour's step flag in milliseconds (0 = for ever)
  int walls = 0;        // 3-D: 0 wall rules inside the step kernel; 1 a separate boundary kernel over the shell (A/B variant)
  int cluster = 0;      // islbm_step(n >= 2) on a tiny 2-D fp64 mesh: all n steps in one launch of a thread-block cluster
                        // with the state in distributed shared memory (islbm_cluster2.cuh); 0 automatic, 2 never
};

}  // namespace islbmk
