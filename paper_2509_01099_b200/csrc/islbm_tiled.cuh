// islbm_tiled.cuh — the fused, shared-memory-staged ISLBM step for sm_100a.
//
// 3-D (D3Q19 + D3Q7), "z-marching" design:
//   * a CTA owns a TX x TY column of nodes (one thread per (x,y)) and marches
//     through a chunk of z-slices;
//   * one elected thread streams, per z-slice, haloed (TX+4)x(TY+2) boxes of the
//     20 population planes that have an in-plane stencil and halo-free TX x TY
//     boxes of the 6 that do not, with TMA (cp.async.bulk.tensor.3d) into a
//     ring of shared-memory stages guarded by full/empty mbarriers;
//   * consumer threads interpolate in-plane (x, then y) from shared memory;
//     the z-direction of the separable interpolation is a
//     3-slice combination kept in REGISTERS: for the 12 populations with
//     e_z != 0 each thread carries the in-plane-interpolated values of the two
//     previous slices, so every post-collision value is read from HBM once
//     and never re-staged;
//   * the node then collides once (islbm_lattice.cuh) and stores its 26
//     post-collision values with coalesced 8-byte stores.
// Bounce-back / anti-bounce-back values (Eq. 21-23) are the node's own
// opposite populations and are fetched straight from global memory by the few
// threads that sit on a wall.
//
// Summation order is the same as the oracle's: x, then y, then z.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <string>

#include "islbm_kernels.cuh"

namespace islbmk {

// ------------------------------ PTX wrappers ------------------------------
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
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap *map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// ------------------------------ geometry ----------------------------------
struct Tile3 {
  static constexpr int TX = 32, TY = 8;
  // haloed box: TMA needs a 16-byte aligned box origin, i.e. an even x coordinate for 8-byte elements (measured:
  // an odd origin raises an illegal-instruction fault), so the x-halo is 2 nodes wide on each side
  static constexpr int XH = 2;
  static constexpr int HX = TX + 2 * XH, HY = TY + 2;
  static constexpr int HALO_PLANES = 20, CORE_PLANES = 6;
  static constexpr int HALO_STRIDE = 368;                // doubles; 36*10 = 360 padded to a multiple of 128 B
  static constexpr int CORE_STRIDE = TX * TY;            // 256 doubles = 2048 B
  static constexpr int STAGE_DOUBLES = HALO_PLANES * HALO_STRIDE + CORE_PLANES * CORE_STRIDE;   // 8896 doubles = 71168 B
  static constexpr int STAGES = 3;
  static constexpr int CONSUMER_WARPS = TX * TY / 32;
  static constexpr int THREADS = TX * TY;                // thread 0 doubles as the TMA producer
  static constexpr uint32_t HALO_BYTES = HX * HY * 8, CORE_BYTES = TX * TY * 8;
  static constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_DOUBLES * 8 + 2 * STAGES * 8 + 128;
};

// shared-memory slot of each population inside a stage
//   halo slots 0..11 : e_z = 0 planes with an in-plane stencil (slice z)   f1 f2 f3 f4 f7 f8 f9 f10 g1 g2 g3 g4
//   halo slots 12..19: e_z != 0 planes with an in-plane stencil (slice m)  f11..f18
//   core slots 0..1  : rest populations f0 g0 (slice z);  2..5: pure-z populations f5 f6 g5 g6 (slice m)
__host__ __device__ constexpr int halo_slot_f(int q) { return q <= 4 ? q - 1 : (q <= 10 ? q - 3 : q + 1); }
__host__ __device__ constexpr int halo_slot_g(int q) { return 7 + q; }

struct TiledPlan {
  bool available = false;
  const char *name = "tiled_zmarch_tma";
  int launches_per_step = 1;
  int dim = 0, precision = 0;
  int n[3] = {0, 0, 0};
  int zchunk = 32;
  CUtensorMap halo_map[2];   // per ping-pong buffer: box (TX+4, TY+2, 1)
  CUtensorMap core_map[2];   // per ping-pong buffer: box (TX, TY, 1)
  void *buf[2] = {nullptr, nullptr};
  char why_not[96] = "";
};

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

// tensor view of one population buffer: (x, y, q*nz + z), fp64, zero fill outside the mesh in x and y
inline bool make_map(CUtensorMap *m, void *base, int nx, int ny, int nz, int q, int bx, int by) {
  EncodeTiledFn enc = get_encode_fn();
  if (!enc) return false;
  cuuint64_t dims[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz * q};
  cuuint64_t strides[2] = {(cuuint64_t)nx * 8, (cuuint64_t)nx * ny * 8};
  cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1};
  cuuint32_t es[3] = {1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// ------------------------------ device helpers -----------------------------
// 3-point sums in the oracle's order: ((w0*v0) + w1*v1) + w2*v2
__device__ __forceinline__ double tap3(const double *__restrict__ s, int stride, const double (&w)[3]) {
  double a = w[0] * s[0];
  a = fma(w[1], s[stride], a);
  return fma(w[2], s[2 * stride], a);
}
__device__ __forceinline__ double tap9(const double *__restrict__ s, const double (&wx)[3], const double (&wy)[3]) {
  double a = wy[0] * tap3(s, 1, wx);
  a = fma(wy[1], tap3(s + Tile3::HX, 1, wx), a);
  return fma(wy[2], tap3(s + 2 * Tile3::HX, 1, wx), a);
}
__device__ __forceinline__ double comb3(const double (&w)[3], double a, double b, double c) {
  return fma(w[2], c, fma(w[1], b, w[0] * a));
}

struct WallFlags {
  bool lo[3], hi[3];
};

// Eq. 21: a flow population whose departure point lies beyond a wall takes the node's own
// opposite post-collision value.
template <int Q>
__device__ __forceinline__ void bb_fix_f(double &v, const WallFlags &wf, const double *__restrict__ src, long long nn,
                                         long long c) {
  constexpr int EX = evel<3>(Q, 0), EY = evel<3>(Q, 1), EZ = evel<3>(Q, 2);
  bool cross = false;
  if (EX == 1) cross |= wf.lo[0];
  if (EX == -1) cross |= wf.hi[0];
  if (EY == 1) cross |= wf.lo[1];
  if (EY == -1) cross |= wf.hi[1];
  if (EZ == 1) cross |= wf.lo[2];
  if (EZ == -1) cross |= wf.hi[2];
  if (cross) v = __ldg(src + (long long)opposite<3>(Q) * nn + c);
}
// Eq. 22 (isothermal x-walls) and Eq. 23 (adiabatic walls)
template <int Q>
__device__ __forceinline__ void bb_fix_g(double &v, const WallFlags &wf, const double *__restrict__ srcg, long long nn,
                                         long long c, const DevMesh &m) {
  constexpr int EX = evel<3>(Q, 0), EY = evel<3>(Q, 1), EZ = evel<3>(Q, 2);
  constexpr int A = EX != 0 ? 0 : (EY != 0 ? 1 : 2);
  constexpr int S = EX + EY + EZ;
  const bool cross = S == 1 ? wf.lo[A] : wf.hi[A];
  if (cross) {
    const double gb = __ldg(srcg + (long long)opposite<3>(Q) * nn + c);
    v = A == 0 ? -gb + m.omega_bc * (wf.lo[0] ? m.T_hot : m.T_cold) : gb;
  }
}
template <int... Qs>
__device__ __forceinline__ void bb_fix_all_f(double *f, const WallFlags &wf, const double *src, long long nn, long long c,
                                             std::integer_sequence<int, Qs...>) {
  (bb_fix_f<Qs + 1>(f[Qs + 1], wf, src, nn, c), ...);
}
template <int... Qs>
__device__ __forceinline__ void bb_fix_all_g(double *g, const WallFlags &wf, const double *srcg, long long nn, long long c,
                                             const DevMesh &m, std::integer_sequence<int, Qs...>) {
  (bb_fix_g<Qs + 1>(g[Qs + 1], wf, srcg, nn, c, m), ...);
}

__device__ __forceinline__ int zbase(int z, int nz) { return min(max(z - 1, 0), nz - 3); }

// One pipeline stage = the TMA boxes one z-iteration needs (see k_step_zmarch).  Issued by one thread.
__device__ __forceinline__ void issue_stage(int s, int z0, int nz, int x0, int y0, double *stage0, uint64_t *full,
                                            uint64_t *empty, const CUtensorMap *halo_map, const CUtensorMap *core_map) {
  using T = Tile3;
  const int st = s % T::STAGES;
  const uint32_t ph = (uint32_t)(s / T::STAGES) & 1u;
  if (s >= T::STAGES) mbar_wait(&empty[st], ph ^ 1u);   // every consumer warp has released the slot
  int mslice = -1, zslice = -1;
  if (s < 2) {
    mslice = zbase(z0, nz) + s;
  } else {
    zslice = z0 + (s - 2);
    if (s == 2 || zbase(zslice, nz) != zbase(zslice - 1, nz)) mslice = zbase(zslice, nz) + 2;
  }
  const uint32_t bytes = (mslice >= 0 ? 8u * T::HALO_BYTES + 4u * T::CORE_BYTES : 0u) +
                         (zslice >= 0 ? 12u * T::HALO_BYTES + 2u * T::CORE_BYTES : 0u);
  mbar_expect_tx(&full[st], bytes);
  double *sb = stage0 + (size_t)st * T::STAGE_DOUBLES;
  double *core = sb + T::HALO_PLANES * T::HALO_STRIDE;
  if (zslice >= 0) {
#pragma unroll
    for (int q = 1; q <= 10; ++q) {
      if (q == 5 || q == 6) continue;
      tma_load_3d(sb + halo_slot_f(q) * T::HALO_STRIDE, halo_map, &full[st], x0 - T::XH, y0 - 1, q * nz + zslice);
    }
#pragma unroll
    for (int q = 1; q <= 4; ++q)
      tma_load_3d(sb + halo_slot_g(q) * T::HALO_STRIDE, halo_map, &full[st], x0 - T::XH, y0 - 1, (19 + q) * nz + zslice);
    tma_load_3d(core + 0 * T::CORE_STRIDE, core_map, &full[st], x0, y0, 0 * nz + zslice);
    tma_load_3d(core + 1 * T::CORE_STRIDE, core_map, &full[st], x0, y0, 19 * nz + zslice);
  }
  if (mslice >= 0) {
#pragma unroll
    for (int q = 11; q <= 18; ++q)
      tma_load_3d(sb + halo_slot_f(q) * T::HALO_STRIDE, halo_map, &full[st], x0 - T::XH, y0 - 1, q * nz + mslice);
    tma_load_3d(core + 2 * T::CORE_STRIDE, core_map, &full[st], x0, y0, 5 * nz + mslice);
    tma_load_3d(core + 3 * T::CORE_STRIDE, core_map, &full[st], x0, y0, 6 * nz + mslice);
    tma_load_3d(core + 4 * T::CORE_STRIDE, core_map, &full[st], x0, y0, (19 + 5) * nz + mslice);
    tma_load_3d(core + 5 * T::CORE_STRIDE, core_map, &full[st], x0, y0, (19 + 6) * nz + mslice);
  }
}

// ------------------------------ the kernel --------------------------------
__global__ void __launch_bounds__(Tile3::THREADS, 1)
k_step_zmarch(const __grid_constant__ CUtensorMap halo_map, const __grid_constant__ CUtensorMap core_map, DevMesh m,
              NodeParams np, const double *__restrict__ src, double *__restrict__ dst, int zchunk) {
  using T = Tile3;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double *stage0 = reinterpret_cast<double *>(smem_raw);
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + (size_t)T::STAGES * T::STAGE_DOUBLES * 8);
  uint64_t *empty = full + T::STAGES;

  const int x0 = blockIdx.x * T::TX, y0 = blockIdx.y * T::TY;
  const int z0 = blockIdx.z * zchunk, z1 = min(z0 + zchunk, m.nz);
  const int nstage = 2 + (z1 - z0);

  if (threadIdx.x == 0) {
    for (int s = 0; s < T::STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], T::CONSUMER_WARPS);
    }
    fence_barrier_init();
  }
  __syncthreads();

  // thread 0 is also the TMA producer: it runs STAGES-1 stages ahead of the consumers
  if (threadIdx.x == 0) {
    tma_prefetch_desc(&halo_map);
    tma_prefetch_desc(&core_map);
    for (int s = 0; s < T::STAGES - 1 && s < nstage; ++s)
      issue_stage(s, z0, m.nz, x0, y0, stage0, full, empty, &halo_map, &core_map);
  }


  // ===================== consumer threads =====================
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int x = x0 + tx, y = y0 + ty;
  const bool valid = x < m.nx && y < m.ny;
  WallFlags wf;
  wf.lo[0] = valid && x == 0;  wf.hi[0] = valid && x == m.nx - 1;
  wf.lo[1] = valid && y == 0;  wf.hi[1] = valid && y == m.ny - 1;
  const bool wall_xy = wf.lo[0] | wf.hi[0] | wf.lo[1] | wf.hi[1];
  const int sx = wf.lo[0] ? 1 : (wf.hi[0] ? -1 : 0);
  const int sy = wf.lo[1] ? 1 : (wf.hi[1] ? -1 : 0);
  // per-thread shared-memory offsets (doubles) inside a haloed plane / a core plane
  const int o_x = (ty + 1) * T::HX + (tx + T::XH - 1 + sx);      // x-stencil, taps +0,+1,+2
  const int o_y = (ty + sy) * T::HX + (tx + T::XH);              // y-stencil, taps +0,+HX,+2HX
  const int o_xy = (ty + sy) * T::HX + (tx + T::XH - 1 + sx);    // 3x3 stencil
  const int o_n = ty * T::TX + tx;                   // halo-free plane
  double wx[2][3], wy[2][3];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      wx[s][k] = valid ? __ldg(wrow(m, 0, s, k) + x) : 0.0;
      wy[s][k] = valid ? __ldg(wrow(m, 1, s, k) + y) : 0.0;
    }
  const long long plane = (long long)m.nx * m.ny;
  const long long cxy = (long long)y * m.nx + x;

  // in-plane-interpolated values of the three z-stencil slices for the 12 populations with e_z != 0:
  //   index: 0 f5, 1 f6, 2..5 f11..f14, 6..9 f15..f18, 10 g5, 11 g6
  double A[12], B[12], C[12];
#pragma unroll
  for (int i = 0; i < 12; ++i) A[i] = B[i] = C[i] = 0.0;

#pragma unroll 1
  for (int s = 0; s < nstage; ++s) {
    const int st = s % T::STAGES;
    const uint32_t ph = (uint32_t)(s / T::STAGES) & 1u;
    const int z = z0 + (s - 2);
    const bool has_emit = s >= 2;
    const bool has_mov = s <= 2 || zbase(z, m.nz) != zbase(z - 1, m.nz);
    const double *sb = stage0 + (size_t)st * T::STAGE_DOUBLES;
    const double *core = sb + T::HALO_PLANES * T::HALO_STRIDE;
    if (threadIdx.x == 0 && s + T::STAGES - 1 < nstage)
      issue_stage(s + T::STAGES - 1, z0, m.nz, x0, y0, stage0, full, empty, &halo_map, &core_map);
    __syncwarp();
    mbar_wait(&full[st], ph);

    if (has_mov) {
#pragma unroll
      for (int i = 0; i < 12; ++i) { A[i] = B[i]; B[i] = C[i]; }
      C[0] = core[2 * T::CORE_STRIDE + o_n];
      C[1] = core[3 * T::CORE_STRIDE + o_n];
      C[2] = tap3(sb + 12 * T::HALO_STRIDE + o_x, 1, wx[1]);       // f11 ( 1,0, 1)
      C[3] = tap3(sb + 13 * T::HALO_STRIDE + o_x, 1, wx[0]);       // f12 (-1,0, 1)
      C[4] = tap3(sb + 14 * T::HALO_STRIDE + o_x, 1, wx[1]);       // f13 ( 1,0,-1)
      C[5] = tap3(sb + 15 * T::HALO_STRIDE + o_x, 1, wx[0]);       // f14 (-1,0,-1)
      C[6] = tap3(sb + 16 * T::HALO_STRIDE + o_y, T::HX, wy[1]);   // f15 (0, 1, 1)
      C[7] = tap3(sb + 17 * T::HALO_STRIDE + o_y, T::HX, wy[0]);   // f16 (0,-1, 1)
      C[8] = tap3(sb + 18 * T::HALO_STRIDE + o_y, T::HX, wy[1]);   // f17 (0, 1,-1)
      C[9] = tap3(sb + 19 * T::HALO_STRIDE + o_y, T::HX, wy[0]);   // f18 (0,-1,-1)
      C[10] = core[4 * T::CORE_STRIDE + o_n];
      C[11] = core[5 * T::CORE_STRIDE + o_n];
    }

    if (has_emit) {
      double wz[2][3];
#pragma unroll
      for (int sg = 0; sg < 2; ++sg)
#pragma unroll
        for (int k = 0; k < 3; ++k) wz[sg][k] = __ldg(wrow(m, 2, sg, k) + z);
      double f[19], g[7];
      f[0] = core[0 * T::CORE_STRIDE + o_n];
      g[0] = core[1 * T::CORE_STRIDE + o_n];
      f[1] = tap3(sb + 0 * T::HALO_STRIDE + o_x, 1, wx[1]);
      f[2] = tap3(sb + 1 * T::HALO_STRIDE + o_x, 1, wx[0]);
      f[3] = tap3(sb + 2 * T::HALO_STRIDE + o_y, T::HX, wy[1]);
      f[4] = tap3(sb + 3 * T::HALO_STRIDE + o_y, T::HX, wy[0]);
      f[7] = tap9(sb + 4 * T::HALO_STRIDE + o_xy, wx[1], wy[1]);
      f[8] = tap9(sb + 5 * T::HALO_STRIDE + o_xy, wx[0], wy[1]);
      f[9] = tap9(sb + 6 * T::HALO_STRIDE + o_xy, wx[1], wy[0]);
      f[10] = tap9(sb + 7 * T::HALO_STRIDE + o_xy, wx[0], wy[0]);
      g[1] = tap3(sb + 8 * T::HALO_STRIDE + o_x, 1, wx[1]);
      g[2] = tap3(sb + 9 * T::HALO_STRIDE + o_x, 1, wx[0]);
      g[3] = tap3(sb + 10 * T::HALO_STRIDE + o_y, T::HX, wy[1]);
      g[4] = tap3(sb + 11 * T::HALO_STRIDE + o_y, T::HX, wy[0]);
      // all shared-memory reads of this stage are done: hand the slot back to the producer
      __syncwarp();
      if ((threadIdx.x & 31) == 0) mbar_arrive(&empty[st]);
      f[5] = comb3(wz[1], A[0], B[0], C[0]);
      f[6] = comb3(wz[0], A[1], B[1], C[1]);
      f[11] = comb3(wz[1], A[2], B[2], C[2]);
      f[12] = comb3(wz[1], A[3], B[3], C[3]);
      f[13] = comb3(wz[0], A[4], B[4], C[4]);
      f[14] = comb3(wz[0], A[5], B[5], C[5]);
      f[15] = comb3(wz[1], A[6], B[6], C[6]);
      f[16] = comb3(wz[1], A[7], B[7], C[7]);
      f[17] = comb3(wz[0], A[8], B[8], C[8]);
      f[18] = comb3(wz[0], A[9], B[9], C[9]);
      g[5] = comb3(wz[1], A[10], B[10], C[10]);
      g[6] = comb3(wz[0], A[11], B[11], C[11]);
      const long long c = (long long)z * plane + cxy;
      wf.lo[2] = z == 0;
      wf.hi[2] = z == m.nz - 1;
      if (valid && (wall_xy | wf.lo[2] | wf.hi[2])) {
        bb_fix_all_f(f, wf, src, m.nn, c, std::make_integer_sequence<int, 18>{});
        bb_fix_all_g(g, wf, src + 19 * m.nn, m.nn, c, m, std::make_integer_sequence<int, 6>{});
      }
      collide_node(f, g, np);
      if (valid) {
#pragma unroll
        for (int q = 0; q < 19; ++q) dst[(long long)q * m.nn + c] = f[q];
#pragma unroll
        for (int q = 0; q < 7; ++q) dst[(long long)(19 + q) * m.nn + c] = g[q];
      }
    } else {
      __syncwarp();
      if ((threadIdx.x & 31) == 0) mbar_arrive(&empty[st]);
    }
  }
}

// ------------------------------ host side ---------------------------------
inline int tiled_plan_create(TiledPlan &p, int dim, const int *n, int precision, void *buf0, void *buf1, std::string &err) {
  (void)err;
  p.available = false;
  p.dim = dim;
  p.precision = precision;
  for (int a = 0; a < 3; ++a) p.n[a] = n[a];
  p.buf[0] = buf0;
  p.buf[1] = buf1;
  auto no = [&](const char *why) { snprintf(p.why_not, sizeof p.why_not, "%s", why); return 0; };
  if (dim != 3) return no("tiled kernel: 3-D only");
  if (precision != 0) return no("tiled kernel: fp64 storage only");
  if (n[0] % 2) return no("tiled kernel: TMA needs a 16-byte row pitch (nx even)");
  if (n[1] % Tile3::TY == 1) return no("tiled kernel: last tile would hold a single row");
  if (n[0] < 3 || n[1] < 3 || n[2] < 3) return no("tiled kernel: n >= 3");
  int dev = 0, cc_major = 0, smem_optin = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return no("no device");
  cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev);
  cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (cc_major < 10 || (size_t)smem_optin < Tile3::SMEM_BYTES) return no("tiled kernel: needs sm_100 and 207 KB shared memory");
  for (int i = 0; i < 2; ++i) {
    if (!make_map(&p.halo_map[i], p.buf[i], n[0], n[1], n[2], 26, Tile3::HX, Tile3::HY)) return no("cuTensorMapEncodeTiled failed");
    if (!make_map(&p.core_map[i], p.buf[i], n[0], n[1], n[2], 26, Tile3::TX, Tile3::TY)) return no("cuTensorMapEncodeTiled failed");
  }
  if (cudaFuncSetAttribute(k_step_zmarch, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tile3::SMEM_BYTES) != cudaSuccess) {
    cudaGetLastError();
    return no("cudaFuncSetAttribute failed");
  }
  // z-chunks: enough CTAs for >= ~6 waves of 148 SMs, chunk >= 16 slices to amortise the 2-slice prologue
  const int tiles = ((n[0] + Tile3::TX - 1) / Tile3::TX) * ((n[1] + Tile3::TY - 1) / Tile3::TY);
  int chunk = n[2];
  while (chunk > 16 && (long long)tiles * ((n[2] + chunk - 1) / chunk) < 148 * 6) chunk = (chunk + 1) / 2;
  p.zchunk = chunk;
  p.available = true;
  return 0;
}

inline int tiled_step(TiledPlan &p, const DevMesh &m, const NodeParams &np, int cur, cudaStream_t stream, std::string &err) {
  dim3 grid((p.n[0] + Tile3::TX - 1) / Tile3::TX, (p.n[1] + Tile3::TY - 1) / Tile3::TY, (p.n[2] + p.zchunk - 1) / p.zchunk);
  k_step_zmarch<<<grid, Tile3::THREADS, Tile3::SMEM_BYTES, stream>>>(p.halo_map[cur], p.core_map[cur], m, np,
                                                                     (const double *)p.buf[cur], (double *)p.buf[1 - cur],
                                                                     p.zchunk);
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) {
    err = std::string("k_step_zmarch launch: ") + cudaGetErrorString(e);
    return -5;
  }
  return 0;
}

}  // namespace islbmk
