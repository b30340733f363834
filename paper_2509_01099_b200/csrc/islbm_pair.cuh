// islbm_pair.cuh — fp32-storage variants of the TMA-staged step kernels with TWO x-adjacent nodes per thread.
//
// With fp32 storage the step is bound by instruction issue, not by HBM (profiles/r1_c5_256cu_f32_v5.md: 980 warp
// instructions per 32 nodes, of which only 293 are the fp64 collision).  These kernels keep the data movement of
// islbm_tiled3.cuh / islbm_tiled2.cuh (same TMA boxes, same ring, same storage) and cut the instruction stream:
//   * a thread owns the nodes (x, x+1): every interpolated value is a float2 whose lanes are the two nodes, and the
//     separable interpolation is issued as packed fma.rn.f32x2 / mul.rn.f32x2 (sm_100: one issue
//     slot for two fused multiply-adds), lane by lane the same operations in the same order as the one-node kernels,
//     so the results are BIT-IDENTICAL to them (tests/test_gpu_parity.py compares the two);
//   * planes without an x-stencil (rest, y-, z- and yz-populations) are read with one 64-bit shared-memory load per
//     pair, and every plane is stored with one 64-bit global store per pair;
//   * loop control, barrier protocol, address arithmetic and the wall predicates are paid once per two nodes.
// The collision stays fp64, one node after the other (collide_node<DEV>, islbm_lattice.cuh).
// Needs an even nx (the BASELINE.json meshes); other meshes take the one-node kernels.
#pragma once

#include "islbm_tiled2.cuh"

namespace islbmk {

constexpr int kPairDefault3 = 6;   // default two-nodes-per-thread tile of the 3-D fp32-storage step (measured, profiles/)

__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }

// 3-point sums in the oracle's order ((w0*v0) + w1*v1) + w2*v2, per lane; sa / sb point at the first tap of node a / b
__device__ __forceinline__ float2 tap3p(const float *__restrict__ sa, const float *__restrict__ sb, int stride,
                                        const float2 (&w)[3]) {
  float2 a = mul2(w[0], make_float2(sa[0], sb[0]));
  a = fma2(w[1], make_float2(sa[stride], sb[stride]), a);
  return fma2(w[2], make_float2(sa[2 * stride], sb[2 * stride]), a);
}
// both nodes read the same rows: one 64-bit load per tap (s is 8-byte aligned)
__device__ __forceinline__ float2 tap3v(const float *__restrict__ s, int stride, const float2 (&w)[3]) {
  float2 a = mul2(w[0], *reinterpret_cast<const float2 *>(s));
  a = fma2(w[1], *reinterpret_cast<const float2 *>(s + stride), a);
  return fma2(w[2], *reinterpret_cast<const float2 *>(s + 2 * stride), a);
}
__device__ __forceinline__ float2 tap9p(const float *__restrict__ sa, const float *__restrict__ sb, int pitch,
                                        const float2 (&wx)[3], const float2 (&wy)[3]) {
  float2 a = mul2(wy[0], tap3p(sa, sb, 1, wx));
  a = fma2(wy[1], tap3p(sa + pitch, sb + pitch, 1, wx), a);
  return fma2(wy[2], tap3p(sa + 2 * pitch, sb + 2 * pitch, 1, wx), a);
}
__device__ __forceinline__ float2 comb3p(const float2 (&w)[3], float2 a, float2 b, float2 c) {
  return fma2(w[2], c, fma2(w[1], b, mul2(w[0], a)));
}
__device__ __forceinline__ float2 ld2(const float *__restrict__ s) { return *reinterpret_cast<const float2 *>(s); }

__device__ __forceinline__ void st_hint(float2 *p, float2 v, uint64_t policy) {
  asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v.x), "f"(v.y), "l"(policy) : "memory");
}

// wall fixes (Eq. 21-23) of one lane; LANE 0 = node a (.x), 1 = node b (.y)
template <int DIM, int LANE, int... Qs>
__device__ __forceinline__ void bb_fix_lane_f(float2 *f, const WallFlags &wf, const float *src, long long nn, long long c,
                                              std::integer_sequence<int, Qs...>) {
  (bb_fix_f<DIM, Qs + 1>(LANE == 0 ? f[Qs + 1].x : f[Qs + 1].y, wf, src, nn, c), ...);
}
template <int DIM, int LANE, int... Qs>
__device__ __forceinline__ void bb_fix_lane_g(float2 *g, const WallFlags &wf, const float *src, long long nn, long long c,
                                              const DevMesh &m, std::integer_sequence<int, Qs...>) {
  (bb_fix_g<DIM, Qs + 1>(LANE == 0 ? g[Qs + 1].x : g[Qs + 1].y, wf, src, nn, c, m), ...);
}

// collide the two nodes of a pair one after the other (fp64 arithmetic on the fp32 deviations, collide_node<true>)
template <int QF, int QG>
__device__ __forceinline__ void collide_pair(float2 (&f)[QF], float2 (&g)[QG], const NodeParams &np) {
  {
    float fa[QF], ga[QG];
#pragma unroll
    for (int q = 0; q < QF; ++q) fa[q] = f[q].x;
#pragma unroll
    for (int q = 0; q < QG; ++q) ga[q] = g[q].x;
    collide_node<true>(fa, ga, np);
#pragma unroll
    for (int q = 0; q < QF; ++q) f[q].x = fa[q];
#pragma unroll
    for (int q = 0; q < QG; ++q) g[q].x = ga[q];
  }
  {
    float fb[QF], gb[QG];
#pragma unroll
    for (int q = 0; q < QF; ++q) fb[q] = f[q].y;
#pragma unroll
    for (int q = 0; q < QG; ++q) gb[q] = g[q].y;
    collide_node<true>(fb, gb, np);
#pragma unroll
    for (int q = 0; q < QF; ++q) f[q].y = fb[q];
#pragma unroll
    for (int q = 0; q < QG; ++q) g[q].y = gb[q];
  }
}

// store the pair's populations plane by plane in storage order (64-bit stores; the pointer is walked by the plane pitch)
template <int DIM, int P>
__device__ __forceinline__ void store_plane2(float2 *&p, long long nn2, const float2 *f, const float2 *g, uint64_t spol) {
  constexpr int QF = Lat<DIM>::QF;
  constexpr int code = pop_of_plane<DIM>(P);
  if constexpr (code < QF) st_hint(p, f[code], spol);
  else st_hint(p, g[code - QF], spol);
  p += nn2;
  asm volatile("" : "+l"(p));
}
template <int DIM, int... Ps>
__device__ __forceinline__ void store_pair(float2 *p, long long nn2, const float2 *f, const float2 *g, uint64_t spol,
                                           std::integer_sequence<int, Ps...>) {
  (store_plane2<DIM, Ps>(p, nn2, f, g, spol), ...);
}

// fused halo exchange (islbm_kernels.cuh: peer_store_node) for the two nodes of a pair; rare path (boundary layers of a slab).
// Inlined on purpose: a call would take the address of the node arrays and force them into local memory on the hot path.
template <int DIM, int QF, int QG>
__device__ __forceinline__ void peer_store_pair(const DevMesh &m, int layer, long long inplane, const float2 (&f)[QF],
                                             const float2 (&g)[QG]) {
  float fa[QF], ga[QG];
#pragma unroll
  for (int q = 0; q < QF; ++q) fa[q] = f[q].x;
#pragma unroll
  for (int q = 0; q < QG; ++q) ga[q] = g[q].x;
  peer_store_node<DIM, float, true>(m, layer, inplane, fa, ga);
#pragma unroll
  for (int q = 0; q < QF; ++q) fa[q] = f[q].y;
#pragma unroll
  for (int q = 0; q < QG; ++q) ga[q] = g[q].y;
  peer_store_node<DIM, float, true>(m, layer, inplane + 1, fa, ga);
}

// ------------------------------ 3-D: z-marching, two nodes per thread --------------------------------------------
// in-plane-interpolated values of one z-stencil slice for the 12 populations with e_z != 0 (index map: ISLBM_LOAD_M3)
#define ISLBM_LOAD_M3P(S)                                              \
  do {                                                                 \
    S[0] = ld2(PC4(0) + o_c);                          /* f5 */        \
    S[1] = ld2(PC4(1) + o_c);                          /* f6 */        \
    S[2] = tap3p(PXM(0) + o_xa, PXM(0) + o_xb, 1, wx[1]);   /* f11 */  \
    S[3] = tap3p(PXM(1) + o_xa, PXM(1) + o_xb, 1, wx[0]);   /* f12 */  \
    S[4] = tap3p(PXM(2) + o_xa, PXM(2) + o_xb, 1, wx[1]);   /* f13 */  \
    S[5] = tap3p(PXM(3) + o_xa, PXM(3) + o_xb, 1, wx[0]);   /* f14 */  \
    S[6] = tap3v(PYM(0) + o_y, T::TX, wy[1]);          /* f15 */       \
    S[7] = tap3v(PYM(1) + o_y, T::TX, wy[0]);          /* f16 */       \
    S[8] = tap3v(PYM(2) + o_y, T::TX, wy[1]);          /* f17 */       \
    S[9] = tap3v(PYM(3) + o_y, T::TX, wy[0]);          /* f18 */       \
    S[10] = ld2(PC4(2) + o_c);                         /* g5 */        \
    S[11] = ld2(PC4(3) + o_c);                         /* g6 */        \
  } while (0)
#define ISLBM_ZCOMB3P(P0, P1, P2)                  \
  do {                                             \
    f[5] = comb3p(wz[1], P0[0], P1[0], P2[0]);     \
    f[6] = comb3p(wz[0], P0[1], P1[1], P2[1]);     \
    f[11] = comb3p(wz[1], P0[2], P1[2], P2[2]);    \
    f[12] = comb3p(wz[1], P0[3], P1[3], P2[3]);    \
    f[13] = comb3p(wz[0], P0[4], P1[4], P2[4]);    \
    f[14] = comb3p(wz[0], P0[5], P1[5], P2[5]);    \
    f[15] = comb3p(wz[1], P0[6], P1[6], P2[6]);    \
    f[16] = comb3p(wz[1], P0[7], P1[7], P2[7]);    \
    f[17] = comb3p(wz[0], P0[8], P1[8], P2[8]);    \
    f[18] = comb3p(wz[0], P0[9], P1[9], P2[9]);    \
    g[5] = comb3p(wz[1], P0[10], P1[10], P2[10]);  \
    g[6] = comb3p(wz[0], P0[11], P1[11], P2[11]);  \
  } while (0)

template <int TX, int TY, int MINB>
__global__ void __launch_bounds__(TX / 2 * TY, MINB)
k_step_zmarch_pair(const __grid_constant__ Maps3 mp, DevMesh m, NodeParams np, const float *__restrict__ src,
                   float *__restrict__ dst, int zchunk, int load_policy, int store_policy, int late_fill) {
  using T = Tile3<float, TX, TY>;
  constexpr int THREADS = TX / 2 * TY, WARPS = THREADS / 32, TXH = TX / 2;
  static_assert(THREADS % 32 == 0 && TX % 2 == 0, "whole warps of node pairs");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *stage0 = smem_raw;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + T::BAR_OFF);
  uint64_t *empty = full + T::STAGES;
  float2 *wzs = reinterpret_cast<float2 *>(smem_raw + T::W_OFF);   // marching-axis weights, both lanes equal
  int *claim = reinterpret_cast<int *>(smem_raw + T::BAR_OFF + 2 * T::STAGES * 8);
  pdl_launch_dependents();

  const int x0 = blockIdx.x * T::TX, y0 = min((int)blockIdx.y * T::TY, max(m.ny - T::TY, 0));
  const int z0 = m.em_lo + blockIdx.z * zchunk, z1 = min(z0 + zchunk, m.em_hi);
  const int nstage = 2 + (z1 - z0);
  const uint64_t lpol = make_policy(load_policy);
  const uint64_t spol = make_policy(store_policy);
  if (threadIdx.x == 0) {
    for (int s = 0; s < T::STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], WARPS);
      claim[s] = 0;
    }
    fence_barrier_init();
    tma_prefetch_desc(&mp.c2);
    tma_prefetch_desc(&mp.c4);
    tma_prefetch_desc(&mp.x);
    tma_prefetch_desc(&mp.y);
    tma_prefetch_desc(&mp.xy);
    if (!late_fill) {
      pdl_wait();
      for (int s = 0; s < T::STAGES && s < nstage; ++s) issue_stage3<T>(s, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
    }
  }
  for (int i = (int)threadIdx.x - 32; i >= 0 && i < 6 * (z1 - z0); i += THREADS - 32) {   // warps 1..: warp 0 is waiting above
    const int sk = i / (z1 - z0), zi = i - sk * (z1 - z0);
    const float w = (float)__ldg(wrow(m, 2, sk / 3, sk % 3) + z0 + zi);
    wzs[sk * kMaxChunk + zi] = make_float2(w, w);
  }
  pdl_wait();
  __syncthreads();
  if (late_fill && threadIdx.x == 0) {
    for (int s = 0; s < T::STAGES && s < nstage; ++s) issue_stage3<T>(s, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
  }

  const int tx = threadIdx.x % TXH, ty = threadIdx.x / TXH;
  const int xa = x0 + 2 * tx, y = y0 + ty;           // nodes (xa, y) and (xa + 1, y); nx is even
  const bool valid = xa < m.nx && y < m.ny;
  WallFlags wfa, wfb;
  wfa.lo[0] = valid && xa == 0;      wfa.hi[0] = false;
  wfb.lo[0] = false;                 wfb.hi[0] = valid && xa + 1 == m.nx - 1;
  wfa.lo[1] = wfb.lo[1] = valid && y == 0;
  wfa.hi[1] = wfb.hi[1] = valid && y == m.ny - 1;
  const bool wall_xy = wfa.lo[0] | wfb.hi[0] | wfa.lo[1] | wfa.hi[1];
  const int sy = wfa.lo[1] ? 1 : (wfa.hi[1] ? -1 : 0);
  // per-thread element offsets inside the four box shapes (node a / node b where the x-stencil differs)
  const int o_xa = ty * T::HX + (2 * tx + T::XH - 1 + (wfa.lo[0] ? 1 : 0));
  const int o_xb = ty * T::HX + (2 * tx + T::XH + (wfb.hi[0] ? -1 : 0));
  const int o_xya = o_xa + sy * T::HX, o_xyb = o_xb + sy * T::HX;
  const int o_y = (ty + sy) * T::TX + 2 * tx;
  const int o_c = ty * T::TX + 2 * tx;
  float2 wx[2][3], wy[2][3];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      wx[s][k] = valid ? make_float2((float)__ldg(wrow(m, 0, s, k) + xa), (float)__ldg(wrow(m, 0, s, k) + xa + 1))
                       : make_float2(0.f, 0.f);
      const float w = valid ? (float)__ldg(wrow(m, 1, s, k) + y) : 0.f;
      wy[s][k] = make_float2(w, w);
    }
  const long long plane = (long long)m.nxp * m.ny;
  const long long cxy = (long long)y * m.nxp + xa;

  float2 S0[12], S1[12], S2[12];
  int newest = 2;

#pragma unroll 1
  for (int s = 0; s < nstage; ++s) {
    const int st = s % T::STAGES;
    const uint32_t ph = (uint32_t)(s / T::STAGES) & 1u;
    const int z = z0 + (s - 2);
    const bool has_emit = s >= 2;
    const bool has_mov = s <= 2 || sbase(z, m.nz) != sbase(z - 1, m.nz);
    const unsigned char *sb = stage0 + (size_t)st * T::STAGE_BYTES;
    auto PC2 = [&](int k) { return reinterpret_cast<const float *>(sb + T::OFF_C2 + k * T::P_C); };
    auto PXZ = [&](int k) { return reinterpret_cast<const float *>(sb + T::OFF_XZ + k * T::P_X); };
    auto PYZ = [&](int k) { return reinterpret_cast<const float *>(sb + T::OFF_YZ + k * T::P_Y); };
    auto PXY = [&](int k) { return reinterpret_cast<const float *>(sb + T::OFF_XY + k * T::P_XY); };
    auto PC4 = [&](int k) { return reinterpret_cast<const float *>(sb + T::OFF_C4 + k * T::P_C); };
    auto PXM = [&](int k) { return reinterpret_cast<const float *>(sb + T::OFF_XM + k * T::P_X); };
    auto PYM = [&](int k) { return reinterpret_cast<const float *>(sb + T::OFF_YM + k * T::P_Y); };
    mbar_wait(&full[st], ph);

    if (has_mov) {
      newest = newest == 2 ? 0 : newest + 1;
      if (newest == 0) ISLBM_LOAD_M3P(S0);
      else if (newest == 1) ISLBM_LOAD_M3P(S1);
      else ISLBM_LOAD_M3P(S2);
    }

    if (has_emit) {
      float2 f[19], g[7];   // fp32 deviations, lanes = the two nodes
      f[0] = ld2(PC2(0) + o_c);
      g[0] = ld2(PC2(1) + o_c);
      f[1] = tap3p(PXZ(0) + o_xa, PXZ(0) + o_xb, 1, wx[1]);
      f[2] = tap3p(PXZ(1) + o_xa, PXZ(1) + o_xb, 1, wx[0]);
      g[1] = tap3p(PXZ(2) + o_xa, PXZ(2) + o_xb, 1, wx[1]);
      g[2] = tap3p(PXZ(3) + o_xa, PXZ(3) + o_xb, 1, wx[0]);
      f[3] = tap3v(PYZ(0) + o_y, T::TX, wy[1]);
      f[4] = tap3v(PYZ(1) + o_y, T::TX, wy[0]);
      g[3] = tap3v(PYZ(2) + o_y, T::TX, wy[1]);
      g[4] = tap3v(PYZ(3) + o_y, T::TX, wy[0]);
      f[7] = tap9p(PXY(0) + o_xya, PXY(0) + o_xyb, T::HX, wx[1], wy[1]);
      f[8] = tap9p(PXY(1) + o_xya, PXY(1) + o_xyb, T::HX, wx[0], wy[1]);
      f[9] = tap9p(PXY(2) + o_xya, PXY(2) + o_xyb, T::HX, wx[1], wy[0]);
      f[10] = tap9p(PXY(3) + o_xya, PXY(3) + o_xyb, T::HX, wx[0], wy[0]);
      // all shared-memory reads of this stage are done: hand the slot back; the warp whose release is the last one
      // refills it at once with stage s + STAGES
      __syncwarp();
      if ((threadIdx.x & 31) == 0 && mbar_arrive_is_last(&empty[st]) && s + T::STAGES < nstage &&
          atomicCAS(&claim[st], s / T::STAGES, s / T::STAGES + 1) == s / T::STAGES)
        issue_stage3<T>(s + T::STAGES, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
      float2 wz[2][3];
#pragma unroll
      for (int sg = 0; sg < 2; ++sg)
#pragma unroll
        for (int k = 0; k < 3; ++k) wz[sg][k] = wzs[(sg * 3 + k) * kMaxChunk + (s - 2)];
      if (newest == 0) ISLBM_ZCOMB3P(S1, S2, S0);
      else if (newest == 1) ISLBM_ZCOMB3P(S2, S0, S1);
      else ISLBM_ZCOMB3P(S0, S1, S2);
      const long long c = (long long)z * plane + cxy;
      const bool wlo = z == 0 && m.wall_mlo, whi = z == m.nz - 1 && m.wall_mhi;
      if (valid && (wall_xy | wlo | whi)) {
        wfa.lo[2] = wfb.lo[2] = wlo;
        wfa.hi[2] = wfb.hi[2] = whi;
        bb_fix_lane_f<3, 0>(f, wfa, src, m.nnp, c, std::make_integer_sequence<int, 18>{});
        bb_fix_lane_g<3, 0>(g, wfa, src, m.nnp, c, m, std::make_integer_sequence<int, 6>{});
        bb_fix_lane_f<3, 1>(f, wfb, src, m.nnp, c + 1, std::make_integer_sequence<int, 18>{});
        bb_fix_lane_g<3, 1>(g, wfb, src, m.nnp, c + 1, m, std::make_integer_sequence<int, 6>{});
      }
      collide_pair(f, g, np);
      if (valid) {
        store_pair<3>(reinterpret_cast<float2 *>(dst + c), m.nnp / 2, f, g, spol, std::make_integer_sequence<int, 26>{});
        if ((m.peer[0] != nullptr && z == m.em_lo) || (m.peer[1] != nullptr && z == m.em_hi - 1))
          peer_store_pair<3, 19, 7>(m, z, cxy, f, g);   // slab decomposition: boundary layer into the neighbour's ghost layer
      }
    } else {
      __syncwarp();
      if ((threadIdx.x & 31) == 0 && mbar_arrive_is_last(&empty[st]) && s + T::STAGES < nstage &&
          atomicCAS(&claim[st], s / T::STAGES, s / T::STAGES + 1) == s / T::STAGES)
        issue_stage3<T>(s + T::STAGES, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
    }
  }
}

template <int TX, int TY, int MINB>
inline bool pair3_setup(Plan3 &p, const int *n, int nxp, void *buf0, void *buf1, const Tuning &tn) {
  // same tensor maps, shared-memory layout and chunk rule as the one-node kernel of this tile
  if (!plan3_maps<float, TX, TY>(p, n, nxp, buf0, buf1, tn)) return false;
  p.available = false;
  if (n[0] % 2) { snprintf(p.why_not, sizeof p.why_not, "pair kernel: nx must be even"); return false; }
  if (cudaFuncSetAttribute(k_step_zmarch_pair<TX, TY, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)Tile3<float, TX, TY>::SMEM_BYTES) != cudaSuccess) {
    cudaGetLastError();
    snprintf(p.why_not, sizeof p.why_not, "cudaFuncSetAttribute failed");
    return false;
  }
  p.available = true;
  return true;
}

template <int TX, int TY, int MINB>
inline void launch3_pair(const Plan3 &p, const int *n, const DevMesh &m, const NodeParams &np, int cur, void *const *buf,
                         const Tuning &tn, cudaStream_t stream) {
  using T = Tile3<float, TX, TY>;
  dim3 grid((n[0] + T::TX - 1) / T::TX, (n[1] + T::TY - 1) / T::TY, (m.em_hi - m.em_lo + p.zchunk - 1) / p.zchunk);
  launch_step(k_step_zmarch_pair<TX, TY, MINB>, grid, dim3(TX / 2 * TY), T::SMEM_BYTES, stream, tn.pdl != 0, p.maps[cur], m,
              np, (const float *)buf[cur], (float *)buf[1 - cur], p.zchunk, tn.load_policy, tn.store_policy,
              tn.fill == 2 ? 1 : 0);
}

// ------------------------------ 3-D dispatch over tile shapes --------------------------------------------------
// shape3d: 1 64x4, 2 128x2, 3 32x6, 4 32x4, 5 32x8 (one node per thread); fp32 storage only, two nodes per thread:
// 6 64x4 (128 threads, two CTAs per SM), 7 64x8 (256 threads, one CTA per SM), 8 32x8 (128 threads, two CTAs per SM)
template <typename ST>
inline bool plan3_create(Plan3 &p, const int *n, int nxp, void *buf0, void *buf1, const Tuning &tn) {
  // fp64 storage: 32x8 (254 registers, one CTA per SM; DRAM-bound).  fp32 storage is bound by instruction issue: even
  // nx takes the two-nodes-per-thread kernel (profiles/r2_c5_256cu_f32.md), odd nx the one-node kernel with 32x6 CTAs
  // (two per SM, 168 registers) or 32x4 (three per SM) on short y-axes (profiles/attempts.md).
  int shape = tn.shape3d;
  if (shape == 0) shape = sizeof(ST) == 4 ? (n[0] % 2 == 0 ? kPairDefault3 : (n[1] >= 192 ? 3 : 4)) : 5;
  if (sizeof(ST) != 4 && shape >= 6) shape = 5;
  p.shape = shape;
  switch (shape) {
    case 1: return plan3_setup<ST, 64, 4>(p, n, nxp, buf0, buf1, tn);
    case 2: return plan3_setup<ST, 128, 2>(p, n, nxp, buf0, buf1, tn);
    case 3: return plan3_setup<ST, 32, 6>(p, n, nxp, buf0, buf1, tn);
    case 4: return plan3_setup<ST, 32, 4>(p, n, nxp, buf0, buf1, tn);
    case 6: return pair3_setup<64, 4, 2>(p, n, nxp, buf0, buf1, tn);
    case 7: return pair3_setup<64, 8, 1>(p, n, nxp, buf0, buf1, tn);
    case 8: return pair3_setup<32, 8, 2>(p, n, nxp, buf0, buf1, tn);
    default: p.shape = 5; return plan3_setup<ST, 32, 8>(p, n, nxp, buf0, buf1, tn);
  }
}

template <typename ST>
inline cudaError_t launch3(const Plan3 &p, const int *n, const DevMesh &m, const NodeParams &np, int cur, void *const *buf,
                           const Tuning &tn, cudaStream_t stream) {
  switch (p.shape) {
    case 1: launch3_shape<ST, 64, 4>(p, n, m, np, cur, buf, tn, stream); break;
    case 2: launch3_shape<ST, 128, 2>(p, n, m, np, cur, buf, tn, stream); break;
    case 3: launch3_shape<ST, 32, 6>(p, n, m, np, cur, buf, tn, stream); break;
    case 4: launch3_shape<ST, 32, 4>(p, n, m, np, cur, buf, tn, stream); break;
    case 6: launch3_pair<64, 4, 2>(p, n, m, np, cur, buf, tn, stream); break;
    case 7: launch3_pair<64, 8, 1>(p, n, m, np, cur, buf, tn, stream); break;
    case 8: launch3_pair<32, 8, 2>(p, n, m, np, cur, buf, tn, stream); break;
    default: launch3_shape<ST, 32, 8>(p, n, m, np, cur, buf, tn, stream);
  }
  return cudaPeekAtLastError();
}

}  // namespace islbmk
