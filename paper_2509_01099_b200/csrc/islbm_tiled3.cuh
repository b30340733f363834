// islbm_tiled3.cuh — fused, TMA-staged ISLBM step for D3Q19 + D3Q7 on sm_100a.
//
// "z-marching" design:
//   * a CTA owns a TX x TY column of nodes (one thread per (x,y)) and marches
//     through a chunk of z-slices;
//   * one elected thread streams, per z-slice, one TMA box per population plane
//     (cp.async.bulk.tensor.3d) into a ring of shared-memory stages guarded by
//     full/empty mbarriers.  The box of a plane carries a halo only along the
//     axes its velocity has a component on:
//        XY (TX+2XH)x(TY+2): f7..f10          X (TX+2XH)xTY: f1 f2 g1 g2 f11..f14
//        Y  TX x(TY+2): f3 f4 g3 g4 f15..f18   C  TX x TY: f0 g0 f5 f6 g5 g6
//   * consumer threads interpolate in-plane (x, then y) from shared memory;
//     the z-direction of the separable interpolation is a
//     3-slice combination kept in REGISTERS: for the 12 populations with
//     e_z != 0 each thread carries the in-plane-interpolated values of the two
//     previous slices, so every post-collision value is staged once;
//   * the node then collides once (islbm_lattice.cuh) and stores its 26
//     post-collision values with coalesced stores.
// Bounce-back / anti-bounce-back values (Eq. 21-23) are the node's own
// opposite populations, fetched straight from global memory by the few
// threads that sit on a wall.
//
// Summation order is the oracle's: x, then y, then z.  ST = double, or float
// holding f_q - w_q (ISLBM_F32_STORAGE); arithmetic is fp64 either way.
#pragma once

#include <cstdio>
#include <string>

#include "islbm_kernels.cuh"
#include "islbm_tma.cuh"

namespace islbmk {

constexpr int kMaxChunk = 64;   // longest marching chunk (its weights are staged in shared memory)

template <typename ST, int TX_ = 32, int TY_ = 8>
struct Tile3 {
  static constexpr int TX = TX_, TY = TY_;
  // TMA needs a 16-byte aligned box origin (measured: a misaligned origin raises an illegal-instruction
  // fault), so the x-halo is 16 bytes wide on each side: 2 nodes in fp64, 4 in fp32 storage
  static constexpr int XH = 16 / (int)sizeof(ST);
  static constexpr int HX = TX + 2 * XH, HY = TY + 2;
  static constexpr int N_XY = 4, N_X = 8, N_Y = 8, N_C = 6;
  static constexpr int B_XY = HX * HY * (int)sizeof(ST), B_X = HX * TY * (int)sizeof(ST);
  static constexpr int B_Y = TX * HY * (int)sizeof(ST), B_C = TX * TY * (int)sizeof(ST);
  static constexpr int S_XY = pad128(B_XY), S_X = pad128(B_X), S_Y = pad128(B_Y), S_C = pad128(B_C);
  static constexpr int OFF_XY = 0, OFF_X = OFF_XY + N_XY * S_XY, OFF_Y = OFF_X + N_X * S_X, OFF_C = OFF_Y + N_Y * S_Y;
  static constexpr int STAGE_BYTES = OFF_C + N_C * S_C;
  static constexpr int STAGES = 3;
  static constexpr int CONSUMER_WARPS = TX * TY / 32;
  static constexpr int THREADS = TX * TY;                // thread 0 doubles as the TMA producer
  static constexpr uint32_t Z_BYTES = 4u * B_XY + 4u * B_X + 4u * B_Y + 2u * B_C;   // planes of the emitted slice
  static constexpr uint32_t M_BYTES = 4u * B_X + 4u * B_Y + 4u * B_C;              // planes of the z-stencil slice
  static constexpr int BAR_OFF = STAGES * STAGE_BYTES;             // full[STAGES], empty[STAGES]
  static constexpr int W_OFF = BAR_OFF + 64;                        // marching-axis weights [sign][k][kMaxChunk]
  static constexpr size_t SMEM_BYTES = (size_t)W_OFF + 6 * kMaxChunk * 8 + 128;
};

struct Maps3 {
  CUtensorMap xy, x, y, c;
};

// ------------------------------ device helpers -----------------------------
// 3-point sums in the oracle's order: ((w0*v0) + w1*v1) + w2*v2
template <typename ST>
__device__ __forceinline__ double tap3(const ST *__restrict__ s, int stride, const double (&w)[3]) {
  double a = w[0] * (double)s[0];
  a = fma(w[1], (double)s[stride], a);
  return fma(w[2], (double)s[2 * stride], a);
}
template <typename ST>
__device__ __forceinline__ double tap9(const ST *__restrict__ s, int pitch, const double (&wx)[3], const double (&wy)[3]) {
  double a = wy[0] * tap3(s, 1, wx);
  a = fma(wy[1], tap3(s + pitch, 1, wx), a);
  return fma(wy[2], tap3(s + 2 * pitch, 1, wx), a);
}
__device__ __forceinline__ double comb3(const double (&w)[3], double a, double b, double c) {
  return fma(w[2], c, fma(w[1], b, w[0] * a));
}

struct WallFlags {
  bool lo[3], hi[3];
};

// Eq. 21: a flow population whose departure point lies beyond a wall takes the node's own
// opposite post-collision value (storage form: the deviation, same lattice weight as its opposite).
template <int DIM, int Q, typename ST>
__device__ __forceinline__ void bb_fix_f(double &v, const WallFlags &wf, const ST *__restrict__ src, long long nn,
                                         long long c) {
  constexpr int EX = evel<DIM>(Q, 0), EY = evel<DIM>(Q, 1), EZ = evel<DIM>(Q, 2);
  bool cross = false;
  if (EX == 1) cross |= wf.lo[0];
  if (EX == -1) cross |= wf.hi[0];
  if (EY == 1) cross |= wf.lo[1];
  if (EY == -1) cross |= wf.hi[1];
  if (DIM == 3 && EZ == 1) cross |= wf.lo[2];
  if (DIM == 3 && EZ == -1) cross |= wf.hi[2];
  if (cross) v = ldv(src + (long long)opposite<DIM>(Q) * nn + c);
}
// Eq. 22 (isothermal x-walls) and Eq. 23 (adiabatic walls)
template <int DIM, int Q, typename ST>
__device__ __forceinline__ void bb_fix_g(double &v, const WallFlags &wf, const ST *__restrict__ srcg, long long nn,
                                         long long c, const DevMesh &m) {
  constexpr int EX = evel<DIM>(Q, 0), EY = evel<DIM>(Q, 1), EZ = evel<DIM>(Q, 2);
  constexpr int A = EX != 0 ? 0 : (EY != 0 ? 1 : 2);
  constexpr int S = EX + EY + EZ;
  const bool cross = S == 1 ? wf.lo[A] : wf.hi[A];
  if (cross) {
    const double gb = ldv(srcg + (long long)opposite<DIM>(Q) * nn + c);
    v = A == 0 ? -gb + m.omega_bc * (wf.lo[0] ? m.T_hot : m.T_cold) : gb;
  }
}
template <int DIM, typename ST, int... Qs>
__device__ __forceinline__ void bb_fix_all_f(double *f, const WallFlags &wf, const ST *src, long long nn, long long c,
                                             std::integer_sequence<int, Qs...>) {
  (bb_fix_f<DIM, Qs + 1>(f[Qs + 1], wf, src, nn, c), ...);
}
template <int DIM, typename ST, int... Qs>
__device__ __forceinline__ void bb_fix_all_g(double *g, const WallFlags &wf, const ST *srcg, long long nn, long long c,
                                             const DevMesh &m, std::integer_sequence<int, Qs...>) {
  (bb_fix_g<DIM, Qs + 1>(g[Qs + 1], wf, srcg, nn, c, m), ...);
}

__device__ __forceinline__ int sbase(int j, int n) { return min(max(j - 1, 0), n - 3); }

// One pipeline stage = the TMA boxes one z-iteration needs.  Issued by one thread.
//   stage s < 2 : the first two slices of the z-stencil of the chunk's first slice;
//   stage s >= 2: the planes of emitted slice z = z0+s-2, plus the new z-stencil slice if the stencil base moves.
template <typename T>
__device__ __forceinline__ void issue_stage3(int s, int z0, int nz, int x0, int y0, unsigned char *stage0, uint64_t *full,
                                             uint64_t *empty, const Maps3 &mp, uint64_t pol) {
  const int st = s % T::STAGES;
  const uint32_t ph = (uint32_t)(s / T::STAGES) & 1u;
  if (s >= T::STAGES) mbar_wait(&empty[st], ph ^ 1u);   // every consumer warp has released the slot
  int mslice = -1, zslice = -1;
  if (s < 2) {
    mslice = sbase(z0, nz) + s;
  } else {
    zslice = z0 + (s - 2);
    if (s == 2 || sbase(zslice, nz) != sbase(zslice - 1, nz)) mslice = sbase(zslice, nz) + 2;
  }
  mbar_expect_tx(&full[st], (mslice >= 0 ? T::M_BYTES : 0u) + (zslice >= 0 ? T::Z_BYTES : 0u));
  unsigned char *sb = stage0 + (size_t)st * T::STAGE_BYTES;
  uint64_t *bar = &full[st];
  const int xh = x0 - T::XH, yh = y0 - 1;
  if (zslice >= 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k)   // f7..f10
      tma_load_3d(sb + T::OFF_XY + k * T::S_XY, &mp.xy, bar, xh, yh, (7 + k) * nz + zslice, pol);
    tma_load_3d(sb + T::OFF_X + 0 * T::S_X, &mp.x, bar, xh, y0, 1 * nz + zslice, pol);          // f1
    tma_load_3d(sb + T::OFF_X + 1 * T::S_X, &mp.x, bar, xh, y0, 2 * nz + zslice, pol);          // f2
    tma_load_3d(sb + T::OFF_X + 2 * T::S_X, &mp.x, bar, xh, y0, (19 + 1) * nz + zslice, pol);   // g1
    tma_load_3d(sb + T::OFF_X + 3 * T::S_X, &mp.x, bar, xh, y0, (19 + 2) * nz + zslice, pol);   // g2
    tma_load_3d(sb + T::OFF_Y + 0 * T::S_Y, &mp.y, bar, x0, yh, 3 * nz + zslice, pol);          // f3
    tma_load_3d(sb + T::OFF_Y + 1 * T::S_Y, &mp.y, bar, x0, yh, 4 * nz + zslice, pol);          // f4
    tma_load_3d(sb + T::OFF_Y + 2 * T::S_Y, &mp.y, bar, x0, yh, (19 + 3) * nz + zslice, pol);   // g3
    tma_load_3d(sb + T::OFF_Y + 3 * T::S_Y, &mp.y, bar, x0, yh, (19 + 4) * nz + zslice, pol);   // g4
    tma_load_3d(sb + T::OFF_C + 0 * T::S_C, &mp.c, bar, x0, y0, 0 * nz + zslice, pol);          // f0
    tma_load_3d(sb + T::OFF_C + 1 * T::S_C, &mp.c, bar, x0, y0, 19 * nz + zslice, pol);         // g0
  }
  if (mslice >= 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      tma_load_3d(sb + T::OFF_X + (4 + k) * T::S_X, &mp.x, bar, xh, y0, (11 + k) * nz + mslice, pol);   // f11..f14
      tma_load_3d(sb + T::OFF_Y + (4 + k) * T::S_Y, &mp.y, bar, x0, yh, (15 + k) * nz + mslice, pol);   // f15..f18
    }
    tma_load_3d(sb + T::OFF_C + 2 * T::S_C, &mp.c, bar, x0, y0, 5 * nz + mslice, pol);          // f5
    tma_load_3d(sb + T::OFF_C + 3 * T::S_C, &mp.c, bar, x0, y0, 6 * nz + mslice, pol);          // f6
    tma_load_3d(sb + T::OFF_C + 4 * T::S_C, &mp.c, bar, x0, y0, (19 + 5) * nz + mslice, pol);   // g5
    tma_load_3d(sb + T::OFF_C + 5 * T::S_C, &mp.c, bar, x0, y0, (19 + 6) * nz + mslice, pol);   // g6
  }
}

// ------------------------------ the kernel --------------------------------
template <typename ST, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 1)
k_step_zmarch(const __grid_constant__ Maps3 mp, DevMesh m, NodeParams np, const ST *__restrict__ src,
              ST *__restrict__ dst, int zchunk, int load_policy, int store_policy) {
  using T = Tile3<ST, TX, TY>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *stage0 = smem_raw;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + T::BAR_OFF);
  uint64_t *empty = full + T::STAGES;
  double *wzs = reinterpret_cast<double *>(smem_raw + T::W_OFF);

  const int x0 = blockIdx.x * T::TX, y0 = blockIdx.y * T::TY;
  const int z0 = blockIdx.z * zchunk, z1 = min(z0 + zchunk, m.nz);
  const int nstage = 2 + (z1 - z0);
  for (int i = threadIdx.x; i < 6 * (z1 - z0); i += T::THREADS) {
    const int sk = i / (z1 - z0), zi = i - sk * (z1 - z0);
    wzs[sk * kMaxChunk + zi] = __ldg(wrow(m, 2, sk / 3, sk % 3) + z0 + zi);
  }

  if (threadIdx.x == 0) {
    for (int s = 0; s < T::STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], T::CONSUMER_WARPS);
    }
    fence_barrier_init();
  }
  __syncthreads();

  // thread 0 is also the TMA producer: it runs STAGES-1 stages ahead of the consumers
  const uint64_t lpol = make_policy(load_policy);
  const uint64_t spol = make_policy(store_policy);
  if (threadIdx.x == 0) {
    tma_prefetch_desc(&mp.xy);
    tma_prefetch_desc(&mp.x);
    tma_prefetch_desc(&mp.y);
    tma_prefetch_desc(&mp.c);
    for (int s = 0; s < T::STAGES - 1 && s < nstage; ++s)
      issue_stage3<T>(s, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
  }

  const int tx = threadIdx.x % T::TX, ty = threadIdx.x / T::TX;
  const int x = x0 + tx, y = y0 + ty;
  const bool valid = x < m.nx && y < m.ny;
  WallFlags wf;
  wf.lo[0] = valid && x == 0;  wf.hi[0] = valid && x == m.nx - 1;
  wf.lo[1] = valid && y == 0;  wf.hi[1] = valid && y == m.ny - 1;
  const bool wall_xy = wf.lo[0] | wf.hi[0] | wf.lo[1] | wf.hi[1];
  const int sx = wf.lo[0] ? 1 : (wf.hi[0] ? -1 : 0);
  const int sy = wf.lo[1] ? 1 : (wf.hi[1] ? -1 : 0);
  // per-thread element offsets inside the four box shapes
  const int o_xy = (ty + sy) * T::HX + (tx + T::XH - 1 + sx);    // 3x3 stencil, pitch HX
  const int o_x = ty * T::HX + (tx + T::XH - 1 + sx);            // x-stencil, taps +0,+1,+2
  const int o_y = (ty + sy) * T::TX + tx;                        // y-stencil, taps +0,+TX,+2TX
  const int o_c = ty * T::TX + tx;
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
    const bool has_mov = s <= 2 || sbase(z, m.nz) != sbase(z - 1, m.nz);
    const unsigned char *sb = stage0 + (size_t)st * T::STAGE_BYTES;
    auto XY = [&](int k) { return reinterpret_cast<const ST *>(sb + T::OFF_XY + k * T::S_XY); };
    auto PX = [&](int k) { return reinterpret_cast<const ST *>(sb + T::OFF_X + k * T::S_X); };
    auto PY = [&](int k) { return reinterpret_cast<const ST *>(sb + T::OFF_Y + k * T::S_Y); };
    auto PC = [&](int k) { return reinterpret_cast<const ST *>(sb + T::OFF_C + k * T::S_C); };
    if (threadIdx.x == 0 && s + T::STAGES - 1 < nstage)
      issue_stage3<T>(s + T::STAGES - 1, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
    __syncwarp();
    mbar_wait(&full[st], ph);

    if (has_mov) {
#pragma unroll
      for (int i = 0; i < 12; ++i) { A[i] = B[i]; B[i] = C[i]; }
      C[0] = (double)PC(2)[o_c];                          // f5
      C[1] = (double)PC(3)[o_c];                          // f6
      C[2] = tap3(PX(4) + o_x, 1, wx[1]);                 // f11 ( 1,0, 1)
      C[3] = tap3(PX(5) + o_x, 1, wx[0]);                 // f12 (-1,0, 1)
      C[4] = tap3(PX(6) + o_x, 1, wx[1]);                 // f13 ( 1,0,-1)
      C[5] = tap3(PX(7) + o_x, 1, wx[0]);                 // f14 (-1,0,-1)
      C[6] = tap3(PY(4) + o_y, T::TX, wy[1]);             // f15 (0, 1, 1)
      C[7] = tap3(PY(5) + o_y, T::TX, wy[0]);             // f16 (0,-1, 1)
      C[8] = tap3(PY(6) + o_y, T::TX, wy[1]);             // f17 (0, 1,-1)
      C[9] = tap3(PY(7) + o_y, T::TX, wy[0]);             // f18 (0,-1,-1)
      C[10] = (double)PC(4)[o_c];                         // g5
      C[11] = (double)PC(5)[o_c];                         // g6
    }

    if (has_emit) {
      double wz[2][3];
#pragma unroll
      for (int sg = 0; sg < 2; ++sg)
#pragma unroll
        for (int k = 0; k < 3; ++k) wz[sg][k] = wzs[(sg * 3 + k) * kMaxChunk + (s - 2)];
      double f[19], g[7];
      f[0] = (double)PC(0)[o_c];
      g[0] = (double)PC(1)[o_c];
      f[1] = tap3(PX(0) + o_x, 1, wx[1]);
      f[2] = tap3(PX(1) + o_x, 1, wx[0]);
      g[1] = tap3(PX(2) + o_x, 1, wx[1]);
      g[2] = tap3(PX(3) + o_x, 1, wx[0]);
      f[3] = tap3(PY(0) + o_y, T::TX, wy[1]);
      f[4] = tap3(PY(1) + o_y, T::TX, wy[0]);
      g[3] = tap3(PY(2) + o_y, T::TX, wy[1]);
      g[4] = tap3(PY(3) + o_y, T::TX, wy[0]);
      f[7] = tap9(XY(0) + o_xy, T::HX, wx[1], wy[1]);
      f[8] = tap9(XY(1) + o_xy, T::HX, wx[0], wy[1]);
      f[9] = tap9(XY(2) + o_xy, T::HX, wx[1], wy[0]);
      f[10] = tap9(XY(3) + o_xy, T::HX, wx[0], wy[0]);
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
        bb_fix_all_f<3>(f, wf, src, m.nn, c, std::make_integer_sequence<int, 18>{});
        bb_fix_all_g<3>(g, wf, src + 19 * m.nn, m.nn, c, m, std::make_integer_sequence<int, 6>{});
      }
#pragma unroll
      for (int q = 0; q < 19; ++q) f[q] += Store<ST, 3>::bias(q);
      collide_node(f, g, np);
      if (valid) {
#pragma unroll
        for (int q = 0; q < 19; ++q) st_hint(dst + (long long)q * m.nn + c, (ST)(f[q] - Store<ST, 3>::bias(q)), spol);
#pragma unroll
        for (int q = 0; q < 7; ++q) st_hint(dst + (long long)(19 + q) * m.nn + c, (ST)g[q], spol);
      }
    } else {
      __syncwarp();
      if ((threadIdx.x & 31) == 0) mbar_arrive(&empty[st]);
    }
  }
}

// ------------------------------ host side ---------------------------------
struct Plan3 {
  bool available = false;
  Maps3 maps[2];            // per ping-pong buffer
  int zchunk = 32;
  int shape = 0;            // tile shape index: 0 32x8, 1 64x4, 2 128x2
  char why_not[96] = "";
};

template <typename ST, int TX, int TY>
inline bool plan3_setup(Plan3 &p, const int *n, void *buf0, void *buf1, const Tuning &tn) {
  using T = Tile3<ST, TX, TY>;
  p.available = false;
  auto no = [&](const char *why) { snprintf(p.why_not, sizeof p.why_not, "%s", why); return false; };
  if (n[0] < 3 || n[1] < 3 || n[2] < 3) return no("tiled kernel: n >= 3");
  if (n[0] % T::XH) return no("tiled kernel: TMA needs a 16-byte row pitch");
  if (n[1] % T::TY == 1) return no("tiled kernel: last tile would hold a single row");
  int dev = 0, cc_major = 0, smem_optin = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return no("no device");
  cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev);
  cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (cc_major < 10 || (size_t)smem_optin < T::SMEM_BYTES) return no("tiled kernel: needs sm_100 and its shared memory");
  void *bufs[2] = {buf0, buf1};
  const int eb = (int)sizeof(ST);
  const long long ns = 26LL * n[2];
  for (int i = 0; i < 2; ++i) {
    if (!make_map(&p.maps[i].xy, bufs[i], 3, eb, n[0], n[1], ns, T::HX, T::HY, tn.l2promo) ||
        !make_map(&p.maps[i].x, bufs[i], 3, eb, n[0], n[1], ns, T::HX, T::TY, tn.l2promo) ||
        !make_map(&p.maps[i].y, bufs[i], 3, eb, n[0], n[1], ns, T::TX, T::HY, tn.l2promo) ||
        !make_map(&p.maps[i].c, bufs[i], 3, eb, n[0], n[1], ns, T::TX, T::TY, tn.l2promo))
      return no("cuTensorMapEncodeTiled failed");
  }
  if (cudaFuncSetAttribute(k_step_zmarch<ST, TX, TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM_BYTES) != cudaSuccess) {
    cudaGetLastError();
    return no("cudaFuncSetAttribute failed");
  }
  // z-chunks: enough CTAs for >= ~12 waves of 148 SMs (measured: shorter chunks win up to there), chunk >= 16
  // slices to amortise the 2-slice prologue
  const int tiles = ((n[0] + T::TX - 1) / T::TX) * ((n[1] + T::TY - 1) / T::TY);
  int chunk = n[2];
  if (tn.chunk > 0) {
    chunk = tn.chunk < n[2] ? tn.chunk : n[2];
  } else {
    if (chunk > kMaxChunk) chunk = kMaxChunk;
    while (chunk > 16 && (long long)tiles * ((n[2] + chunk - 1) / chunk) < 148 * 12) chunk = (chunk + 1) / 2;
  }
  p.zchunk = chunk < kMaxChunk ? chunk : kMaxChunk;
  p.available = true;
  return true;
}

template <typename ST>
inline bool plan3_create(Plan3 &p, const int *n, void *buf0, void *buf1, const Tuning &tn) {
  p.shape = tn.shape3d;
  switch (tn.shape3d) {
    case 1: return plan3_setup<ST, 64, 4>(p, n, buf0, buf1, tn);
    case 2: return plan3_setup<ST, 128, 2>(p, n, buf0, buf1, tn);
    default: p.shape = 0; return plan3_setup<ST, 32, 8>(p, n, buf0, buf1, tn);
  }
}

template <typename ST, int TX, int TY>
inline void launch3_shape(const Plan3 &p, const int *n, const DevMesh &m, const NodeParams &np, int cur, void *const *buf,
                          const Tuning &tn, cudaStream_t stream) {
  using T = Tile3<ST, TX, TY>;
  dim3 grid((n[0] + T::TX - 1) / T::TX, (n[1] + T::TY - 1) / T::TY, (n[2] + p.zchunk - 1) / p.zchunk);
  k_step_zmarch<ST, TX, TY><<<grid, T::THREADS, T::SMEM_BYTES, stream>>>(
      p.maps[cur], m, np, (const ST *)buf[cur], (ST *)buf[1 - cur], p.zchunk, tn.load_policy, tn.store_policy);
}

template <typename ST>
inline cudaError_t launch3(const Plan3 &p, const int *n, const DevMesh &m, const NodeParams &np, int cur, void *const *buf,
                           const Tuning &tn, cudaStream_t stream) {
  switch (p.shape) {
    case 1: launch3_shape<ST, 64, 4>(p, n, m, np, cur, buf, tn, stream); break;
    case 2: launch3_shape<ST, 128, 2>(p, n, m, np, cur, buf, tn, stream); break;
    default: launch3_shape<ST, 32, 8>(p, n, m, np, cur, buf, tn, stream);
  }
  return cudaPeekAtLastError();
}

}  // namespace islbmk
