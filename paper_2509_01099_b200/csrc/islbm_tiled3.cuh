// islbm_tiled3.cuh — fused, TMA-staged ISLBM step for D3Q19 + D3Q7 on sm_100a.
//
// "z-marching" design:
//   * a CTA owns a TX x TY column of nodes (one thread per (x,y)) and marches
//     through a chunk of z-slices;
//   * one elected thread streams, per z-slice, SEVEN TMA boxes
//     (cp.async.bulk.tensor.4d over the view (x, y, z, plane)) into a ring of
//     shared-memory stages guarded by full/empty mbarriers.  The storage planes
//     are ordered so that each box covers the 2 or 4 consecutive planes that
//     share a halo shape (plane_f / plane_g in islbm_lattice.cuh), and a plane
//     carries a halo only along the axes its velocity has a component on:
//        C  TX x TY: f0 g0 | f5 g5 f6 g6          X (TX+2XH)xTY: f1 f2 g1 g2 | f11..f14
//        Y  TX x(TY+2): f3 f4 g3 g4 | f15..f18     XY (TX+2XH)x(TY+2): f7..f10
//   * consumer threads interpolate in-plane (x, then y) from shared memory;
//     the z-direction of the separable interpolation is a
//     3-slice combination kept in REGISTERS: for the 12 populations with
//     e_z != 0 each thread carries the in-plane-interpolated values of three
//     slices in three register sets whose roles rotate (no register shifting),
//     so every post-collision value is staged once;
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

// ring depth of the fp32-storage tiles (compile-time knob; the default is the measured optimum)
#ifndef ISLBM_Z_STAGES_F32
#define ISLBM_Z_STAGES_F32 3
#endif

#ifndef ISLBM_S_IN_SMEM
#define ISLBM_S_IN_SMEM 1
#endif
// The fp64 32x8 kernel runs a dedicated TMA producer warpgroup: 4 extra warps, of which one lane waits for each ring
// slot to be released and issues the next stage into it; `setmaxnreg` hands the group's registers to the 8 consumer
// warps (launch at 168 per thread, then 40 / 232), so no consumer warp stalls on the empty barriers or spends issue
// slots on the 7 TMA instructions per slice.  Measured +1-2 % on the sustained 256^3 step (profiles/attempts.md);
// 0 = thread 0 of consumer warp 0 is the producer (round 1).  fp32 storage keeps its last-releasing-warp refill
// (6 consumer warps per CTA are not a whole number of warpgroups).
#ifndef ISLBM_PRODUCER_WG
#define ISLBM_PRODUCER_WG 1
#endif
template <typename ST, int TX, int TY> __host__ __device__ constexpr int producer_threads() {
  return (ISLBM_PRODUCER_WG && sizeof(ST) == 8 && TX * TY == 256) ? 128 : 0;
}

// resident CTAs per SM the step kernels are compiled for (the register cap follows).  fp32 storage, 32x8 tiles: two
// CTAs per SM = 16 warps at 128 registers on a 2-stage ring (2 x (66 KB ring + 37 KB of stencil sets)): the all-fp32
// node arithmetic (ISLBM_F_FP32_3D) needs 120 registers, and the step is bound by latency, not by bytes in flight
// (256^3: 32x6 x 2 CTAs on 3 stages 741-745 us, 32x5 x 3 CTAs on 2 stages 719 us, 32x8 x 2 CTAs 711-713 us;
// profiles/attempts.md).
template <typename ST, int TX, int TY> __host__ __device__ constexpr bool f32_two_wide_ctas() {
  return sizeof(ST) == 4 && TX == 32 && TY == 8;
}
template <typename ST, int TX, int TY> __host__ __device__ constexpr int min_ctas3() {
  if (f32_two_wide_ctas<ST, TX, TY>()) return 2;
  return TX * TY <= 128 ? 3 : (TX * TY <= 192 ? 2 : 1);
}

constexpr int kMaxChunk = 64;   // longest marching chunk (its weights are staged in shared memory)

// SK = stencil kind: 0 destination-centred {j-1,j,j+1} (A2), 1 upwind {j-2,j-1,j} for c = +1 and
// {j,j+1,j+2} for c = -1 (the A2 alternative): a 2-row y-halo, and the two halves of each z-stencil group (the
// populations with e_z = +1 / -1) come from different slices (z and z+2).
template <typename ST, int TX_ = 32, int TY_ = 8, int SK_ = 0>
struct Tile3 {
  static constexpr int TX = TX_, TY = TY_, SK = SK_;
  static constexpr int YH = SK ? 2 : 1;
  // TMA needs a 16-byte aligned box origin (measured: a misaligned origin raises an illegal-instruction
  // fault), so the x-halo is 16 bytes wide on each side: 2 nodes in fp64, 4 in fp32 storage
  static constexpr int XH = 16 / (int)sizeof(ST);
  static constexpr int HX = TX + 2 * XH, HY = TY + 2 * YH;
  // bytes of one plane inside a box of each shape
  static constexpr int P_XY = HX * HY * (int)sizeof(ST), P_X = HX * TY * (int)sizeof(ST);
  static constexpr int P_Y = TX * HY * (int)sizeof(ST), P_C = TX * TY * (int)sizeof(ST);
  // groups of a stage, in storage-plane order (each starts 128-byte aligned):
  //   emitted slice z:      C2 = f0 g0, XZ = f1 f2 g1 g2, YZ = f3 f4 g3 g4, XY = f7..f10
  //   z-stencil slice (m):  C4 = f5 g5 f6 g6, XM = f11..f14, YM = f15..f18  (first half of each: e_z = +1)
  // a z-stencil group is two halves of two planes (e_z = +1, then e_z = -1); the upwind kernels load the halves with
  // separate boxes, whose shared-memory destinations must be 128-byte aligned: H_* = distance between the halves
  static constexpr int H_C = SK ? pad128(2 * P_C) : 2 * P_C, H_X = SK ? pad128(2 * P_X) : 2 * P_X;
  static constexpr int H_Y = SK ? pad128(2 * P_Y) : 2 * P_Y;
  static constexpr int OFF_C2 = 0;
  static constexpr int OFF_XZ = pad128(OFF_C2 + 2 * P_C);
  static constexpr int OFF_YZ = pad128(OFF_XZ + 4 * P_X);
  static constexpr int OFF_XY = pad128(OFF_YZ + 4 * P_Y);
  static constexpr int OFF_C4 = pad128(OFF_XY + 4 * P_XY);
  static constexpr int OFF_XM = pad128(OFF_C4 + 2 * H_C);
  static constexpr int OFF_YM = pad128(OFF_XM + 2 * H_X);
  static constexpr int STAGE_BYTES = pad128(OFF_YM + 2 * H_Y);
  // byte offset of plane k (0..3) of a z-stencil group that starts at `off`, planes of `pbytes`, halves `half` apart
  static __host__ __device__ constexpr int moff(int off, int k, int pbytes, int half) { return off + (k / 2) * half + (k % 2) * pbytes; }
  // fp64: 3 x 62.7 KB is all that fits.  fp32 storage, upwind stencil: 2 stages, so that two CTAs (2 x (58 KB ring + 27 KB
  // of stencil sets)) still share an SM; for 32x6 tiles a 2-stage ring measures the same as a 3-stage one (profiles/attempts.md)
  static constexpr int STAGES = sizeof(ST) == 4 ? ((SK || f32_two_wide_ctas<ST, TX, TY>()) ? 2 : ISLBM_Z_STAGES_F32) : 3;
  static constexpr int CONSUMER_WARPS = TX * TY / 32;
  static constexpr int THREADS = TX * TY;                // thread 0 doubles as the TMA producer
  static constexpr uint32_t Z_BYTES = 2u * P_C + 4u * P_X + 4u * P_Y + 4u * P_XY;   // planes of the emitted slice
  static constexpr uint32_t M_BYTES = 4u * P_C + 4u * P_X + 4u * P_Y;               // planes of the z-stencil slice
  static constexpr uint32_t F_BYTES = M_BYTES / 2;                                  // ... of one half (SK = 1)
  static constexpr int BAR_OFF = STAGES * STAGE_BYTES;             // full[STAGES], empty[STAGES]
  static constexpr int W_OFF = BAR_OFF + 128;                       // marching-axis weights [sign][k][kMaxChunk]
  // fp32 storage: the in-plane-interpolated values of the three z-stencil slices live in shared memory, not in
  // registers: [slot 3][pair 6][thread] float2 (each thread reads back only what it wrote: no barrier).  The kernel is
  // latency-bound, and 36 registers of carried state put loop invariants into local memory on the critical path under
  // the 168-register cap of 12 warps per SM, let alone the 128 of the 16 warps it runs at now (profiles/r2_c5_256cu_f32.md)
  static constexpr bool S_IN_SMEM = sizeof(ST) == 4 && ISLBM_S_IN_SMEM;
  static constexpr int S_OFF = W_OFF + 6 * kMaxChunk * 8 + 128;
  static constexpr size_t SMEM_BYTES = (size_t)S_OFF + (S_IN_SMEM ? 3 * 6 * THREADS * 8 : 0);
};

// tensor maps over (x, y, z, plane): one per box shape
struct Maps3 {
  CUtensorMap c2, c4, x, y, xy;
  CUtensorMap x2, y2;   // two-plane boxes of the x / y shapes (upwind stencil: half a z-stencil group)
};

// ------------------------------ device helpers -----------------------------
// Arithmetic type of the stencil interpolation, and the type the node's 26 values are held in up to the collision:
// fp64 for fp64 storage (bit-compatible with the oracle's order of operations).  For fp32 storage the stored
// deviations f_q - w_q are interpolated in fp32 (one or two more fp32 roundings of the deviation, the size of the
// storage rounding itself) and stay in fp32 registers, and the 3-D node is collided in fp32 too (ISLBM_F_FP32_3D,
// islbm_lattice.cuh): no conversion and no fp64 instruction is left in the step.  (The A/B build with the fp64 flow
// collision widens each value for the moments and again for the update f+ = fl32(fl64(f) + M^T d): 52 conversions
// per node in the SASS instead of the 116 of an fp64 interpolation; they issue at a quarter of the fp64 rate.)
template <typename ST> struct Acc { using type = double; };
template <> struct Acc<float> { using type = float; };

// A PAIR of populations of one node that share their stencil shape and differ in the sign of their velocity
// components, e.g. (f1, f2) = (+x, -x).  The separable interpolation works on such pairs: the two
// lanes take the same taps of two different planes with the weights of the two signs.  In fp32 a pair is one float2
// and a tap is ONE packed instruction (fma.rn.f32x2 / mul.rn.f32x2, sm_100), which halves the fp32 instruction
// stream of the fp32-storage kernels; in fp64 a pair is two doubles and two scalar instructions.  Either
// way each lane performs exactly the operations of the scalar form ((w0*v0) + w1*v1) + w2*v2, the oracle's order.
template <typename AT> struct Pr;
template <> struct Pr<double> { double a, b; };
template <> struct Pr<float> { float2 v; };
__device__ __forceinline__ Pr<double> mkpr(double a, double b) { return Pr<double>{a, b}; }
__device__ __forceinline__ Pr<float> mkpr(float a, float b) { Pr<float> p; p.v = make_float2(a, b); return p; }
__device__ __forceinline__ double lane_a(const Pr<double> &p) { return p.a; }
__device__ __forceinline__ double lane_b(const Pr<double> &p) { return p.b; }
__device__ __forceinline__ float lane_a(const Pr<float> &p) { return p.v.x; }
__device__ __forceinline__ float lane_b(const Pr<float> &p) { return p.v.y; }
__device__ __forceinline__ Pr<double> pmul(const Pr<double> &w, const Pr<double> &v) { return Pr<double>{w.a * v.a, w.b * v.b}; }
__device__ __forceinline__ Pr<double> pfma(const Pr<double> &w, const Pr<double> &v, const Pr<double> &c) {
  return Pr<double>{fma(w.a, v.a, c.a), fma(w.b, v.b, c.b)};
}
__device__ __forceinline__ Pr<float> pmul(const Pr<float> &w, const Pr<float> &v) { Pr<float> r; r.v = __fmul2_rn(w.v, v.v); return r; }
__device__ __forceinline__ Pr<float> pfma(const Pr<float> &w, const Pr<float> &v, const Pr<float> &c) {
  Pr<float> r;
  r.v = __ffma2_rn(w.v, v.v, c.v);
  return r;
}

// 3-point sums of a pair in the oracle's order ((w0*v0) + w1*v1) + w2*v2; pa / pb: first tap in the two planes
template <typename ST, typename AT>
__device__ __forceinline__ Pr<AT> ptap3(const ST *__restrict__ pa, const ST *__restrict__ pb, int stride, const Pr<AT> (&w)[3]) {
  Pr<AT> a = pmul(w[0], mkpr((AT)pa[0], (AT)pb[0]));
  a = pfma(w[1], mkpr((AT)pa[stride], (AT)pb[stride]), a);
  return pfma(w[2], mkpr((AT)pa[2 * stride], (AT)pb[2 * stride]), a);
}
template <typename ST, typename AT>
__device__ __forceinline__ Pr<AT> ptap9(const ST *__restrict__ pa, const ST *__restrict__ pb, int pitch, const Pr<AT> (&wx)[3],
                                        const Pr<AT> (&wy)[3]) {
  Pr<AT> a = pmul(wy[0], ptap3(pa, pb, 1, wx));
  a = pfma(wy[1], ptap3(pa + pitch, pb + pitch, 1, wx), a);
  return pfma(wy[2], ptap3(pa + 2 * pitch, pb + 2 * pitch, 1, wx), a);
}
template <typename AT>
__device__ __forceinline__ Pr<AT> pcomb3(const Pr<AT> (&w)[3], const Pr<AT> &a, const Pr<AT> &b, const Pr<AT> &c) {
  return pfma(w[2], c, pfma(w[1], b, pmul(w[0], a)));
}

struct WallFlags {
  bool lo[3], hi[3];
};

// Eq. 21: a flow population whose departure point lies beyond a wall takes the node's own opposite
// post-collision value (storage form: the deviation, same lattice weight as its opposite); Eq. 22 (isothermal x-walls)
// and Eq. 23 (adiabatic walls), for the temperature populations.  One call fixes the populations that
// cross ONE wall (AXIS, SIGN = +1: the low wall, crossed by e_AXIS = +1; -1: the high wall); a node on an edge or in a
// corner is fixed once per wall it touches, and a diagonal population that crosses two walls is loaded twice with the
// same value (A4: bounce back as soon as any component crosses).  sc = src + node index.
// The wall reads are coherent loads (ld.global.cg), not ld.global.nc: with programmatic dependent launch step t+1 is
// resident while step t still writes the buffer these loads read, so the data is not read-only for the kernel's
// lifetime (the loads themselves come after griddepcontrol.wait).
template <int DIM, int AXIS, int SIGN, int Q, typename ST, typename NT>
__device__ __forceinline__ void wall_fix_f1(NT *f, const ST *__restrict__ sc, long long nn) {
  if constexpr (evel<DIM>(Q, AXIS) == SIGN) f[Q] = (NT)ld_coherent(sc + (long long)plane_f<DIM>(opposite<DIM>(Q)) * nn);
}
template <int DIM, int AXIS, int SIGN, int Q, typename ST, typename NT>
__device__ __forceinline__ void wall_fix_g1(NT *g, const ST *__restrict__ sc, long long nn, const DevMesh &m) {
  if constexpr (evel<DIM>(Q, AXIS) == SIGN) {
    const double gb = (double)ld_coherent(sc + (long long)plane_g<DIM>(opposite<DIM>(Q)) * nn);
    g[Q] = (NT)(AXIS == 0 ? -gb + m.omega_bc * (SIGN > 0 ? m.T_hot : m.T_cold) : gb);
  }
}
template <int DIM, int AXIS, int SIGN, typename ST, typename NT, int... Qf, int... Qg>
__device__ __forceinline__ void wall_fix(NT *f, NT *g, const ST *__restrict__ sc, long long nn, const DevMesh &m,
                                         std::integer_sequence<int, Qf...>, std::integer_sequence<int, Qg...>) {
  (wall_fix_f1<DIM, AXIS, SIGN, Qf + 1>(f, sc, nn), ...);
  (wall_fix_g1<DIM, AXIS, SIGN, Qg + 1>(g, sc, nn, m), ...);
}
template <int DIM, typename ST, typename NT>
__device__ __forceinline__ void wall_fix_node(NT *f, NT *g, const WallFlags &wf, const ST *__restrict__ sc, long long nn,
                                              const DevMesh &m) {
  using QF = std::make_integer_sequence<int, Lat<DIM>::QF - 1>;
  using QG = std::make_integer_sequence<int, Lat<DIM>::QG - 1>;
  if (wf.lo[0]) wall_fix<DIM, 0, 1>(f, g, sc, nn, m, QF{}, QG{});
  if (wf.hi[0]) wall_fix<DIM, 0, -1>(f, g, sc, nn, m, QF{}, QG{});
  if (wf.lo[1]) wall_fix<DIM, 1, 1>(f, g, sc, nn, m, QF{}, QG{});
  if (wf.hi[1]) wall_fix<DIM, 1, -1>(f, g, sc, nn, m, QF{}, QG{});
  if constexpr (DIM == 3) {
    if (wf.lo[2]) wall_fix<DIM, 2, 1>(f, g, sc, nn, m, QF{}, QG{});
    if (wf.hi[2]) wall_fix<DIM, 2, -1>(f, g, sc, nn, m, QF{}, QG{});
  }
}

// store the node's populations plane by plane in storage order.  The pointer is walked by the plane pitch and made
// opaque after each step, so that ptxas keeps two integer adds per plane (a 64-bit address per plane is the floor: STG
// takes no uniform-base + 32-bit-offset form, and a 32 x 32 -> 64-bit multiply-add per plane compiles to 2.6
// instructions, measured: profiles/attempts.md)
template <int DIM, int P, bool DEV, typename ST, typename NT>
__device__ __forceinline__ void store_plane(ST *&p, long long nn, const NT *f, const NT *g, uint64_t spol) {
  constexpr int QF = Lat<DIM>::QF;
  constexpr int code = pop_of_plane<DIM>(P);
  if constexpr (code < QF) st_hint(p, to_storage_from<ST, DIM, DEV>(f[code], code), spol);
  else st_hint(p, (ST)g[code - QF], spol);
  p += nn;
  asm volatile("" : "+l"(p));
}
template <int DIM, bool DEV = false, typename ST, typename NT, int... Ps>
__device__ __forceinline__ void store_node(ST *p, long long nn, const NT *f, const NT *g, uint64_t spol,
                                           std::integer_sequence<int, Ps...>) {
  (store_plane<DIM, Ps, DEV>(p, nn, f, g, spol), ...);
}

__device__ __forceinline__ int sbase(int j, int n) { return min(max(j - 1, 0), n - 3); }
// does the stencil base move from layer j-1 to layer j?  (sbase(j) != sbase(j-1)  <=>  2 <= j <= n-2)
__device__ __forceinline__ bool sbase_moves(int j, int n) { return j >= 2 && j <= n - 2; }
// upwind stencil: base of the populations with c = +1 ({j-2,j-1,j}) and with c = -1 ({j,j+1,j+2}), clamped alike
__device__ __forceinline__ int ubase_p(int j, int n) { return min(max(j - 2, 0), n - 3); }
__device__ __forceinline__ int ubase_m(int j, int n) { return min(max(j, 0), n - 3); }
__device__ __forceinline__ bool ubase_p_moves(int j, int n) { return j >= 3; }             // ubase_p(j) != ubase_p(j-1), j < n
__device__ __forceinline__ bool ubase_m_moves(int j, int n) { return j >= 1 && j <= n - 3; }

// One pipeline stage = the TMA boxes one z-iteration needs.  Issued by one thread.
//   stage s < 2 : the first two slices of the z-stencil of the chunk's first slice;
//   stage s >= 2: the planes of emitted slice z = z0+s-2, plus the new z-stencil slice if the stencil base moves.
template <typename T>
__device__ __forceinline__ void issue_stage3(int s, int z0, int nz, int x0, int y0, unsigned char *stage0, uint64_t *full,
                                             uint64_t *empty, const Maps3 &mp, uint64_t pol) {
  const int st = s % T::STAGES;   // the caller knows the slot is free (initial fill, or it saw the last release)
  unsigned char *sb = stage0 + (size_t)st * T::STAGE_BYTES;
  uint64_t *bar = &full[st];
  const int xh = x0 - T::XH, yh = y0 - T::YH;
  int zslice = -1;
  if constexpr (T::SK == 0) {
    int mslice = -1;
    if (s < 2) {
      mslice = sbase(z0, nz) + s;
    } else {
      zslice = z0 + (s - 2);
      if (s == 2 || sbase_moves(zslice, nz)) mslice = sbase(zslice, nz) + 2;
    }
    mbar_expect_tx(bar, (mslice >= 0 ? T::M_BYTES : 0u) + (zslice >= 0 ? T::Z_BYTES : 0u));
    if (mslice >= 0) {
      tma_load_4d(sb + T::OFF_C4, &mp.c4, bar, x0, y0, mslice, 14, pol);    // f5 g5 f6 g6
      tma_load_4d(sb + T::OFF_XM, &mp.x, bar, xh, y0, mslice, 18, pol);     // f11..f14
      tma_load_4d(sb + T::OFF_YM, &mp.y, bar, x0, yh, mslice, 22, pol);     // f15..f18
    }
  } else {
    // the e_z = +1 halves (f5 g5 | f11 f12 | f15 f16) trail the emitted slice, the e_z = -1 halves lead it by two
    int pslice = -1, mslice = -1;
    if (s < 2) {
      pslice = ubase_p(z0, nz) + s;
      mslice = ubase_m(z0, nz) + s;
    } else {
      zslice = z0 + (s - 2);
      if (s == 2 || ubase_p_moves(zslice, nz)) pslice = ubase_p(zslice, nz) + 2;
      if (s == 2 || ubase_m_moves(zslice, nz)) mslice = ubase_m(zslice, nz) + 2;
    }
    mbar_expect_tx(bar, (pslice >= 0 ? T::F_BYTES : 0u) + (mslice >= 0 ? T::F_BYTES : 0u) + (zslice >= 0 ? T::Z_BYTES : 0u));
    if (pslice >= 0) {
      tma_load_4d(sb + T::OFF_C4, &mp.c2, bar, x0, y0, pslice, 14, pol);                   // f5 g5
      tma_load_4d(sb + T::OFF_XM, &mp.x2, bar, xh, y0, pslice, 18, pol);                   // f11 f12
      tma_load_4d(sb + T::OFF_YM, &mp.y2, bar, x0, yh, pslice, 22, pol);                   // f15 f16
    }
    if (mslice >= 0) {
      tma_load_4d(sb + T::OFF_C4 + T::H_C, &mp.c2, bar, x0, y0, mslice, 16, pol);          // f6 g6
      tma_load_4d(sb + T::OFF_XM + T::H_X, &mp.x2, bar, xh, y0, mslice, 20, pol);          // f13 f14
      tma_load_4d(sb + T::OFF_YM + T::H_Y, &mp.y2, bar, x0, yh, mslice, 24, pol);          // f17 f18
    }
  }
  if (zslice >= 0) {
    tma_load_4d(sb + T::OFF_C2, &mp.c2, bar, x0, y0, zslice, 0, pol);     // f0 g0
    tma_load_4d(sb + T::OFF_XZ, &mp.x, bar, xh, y0, zslice, 2, pol);      // f1 f2 g1 g2
    tma_load_4d(sb + T::OFF_YZ, &mp.y, bar, x0, yh, zslice, 6, pol);      // f3 f4 g3 g4
    tma_load_4d(sb + T::OFF_XY, &mp.xy, bar, xh, yh, zslice, 10, pol);    // f7..f10
  }
}

// marching-axis weights of one layer as pairs.  Central stencil (SK = 0): A = (weight of c=+1, weight of c=-1),
// B = the two swapped.  Upwind (SK = 1): A = (c=+1, c=+1), B = (c=-1, c=-1), because a pair then holds two
// populations of the same sign.  fp64: the chunk's weights sit in shared memory as scalars [sign][k][kMaxChunk] (a
// pair is just two registers); fp32: both forms sit there as float2 [form][k][kMaxChunk], one 64-bit load each.
template <int SK>
__device__ __forceinline__ void stage_march_weight(double *ws, int sk, int i, double w) { ws[sk * kMaxChunk + i] = w; }
template <int SK>
__device__ __forceinline__ void stage_march_weight(float *ws, int sk, int i, double w) {
  const int sign = sk / 3, k = sk - 3 * sign;   // sk = sign * 3 + k
  if constexpr (SK == 0) {
    ws[((0 * 3 + k) * kMaxChunk + i) * 2 + (sign ? 0 : 1)] = (float)w;
    ws[((1 * 3 + k) * kMaxChunk + i) * 2 + (sign ? 1 : 0)] = (float)w;
  } else {
    ws[(((sign ? 0 : 1) * 3 + k) * kMaxChunk + i) * 2 + 0] = (float)w;
    ws[(((sign ? 0 : 1) * 3 + k) * kMaxChunk + i) * 2 + 1] = (float)w;
  }
}
template <int SK>
__device__ __forceinline__ void load_march_weights(const double *ws, int i, Pr<double> (&A)[3], Pr<double> (&B)[3]) {
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const double w1 = ws[(3 + k) * kMaxChunk + i], w0 = ws[k * kMaxChunk + i];
    A[k] = SK == 0 ? mkpr(w1, w0) : mkpr(w1, w1);
    B[k] = SK == 0 ? mkpr(w0, w1) : mkpr(w0, w0);
  }
}
template <int SK>
__device__ __forceinline__ void load_march_weights(const float *ws, int i, Pr<float> (&A)[3], Pr<float> (&B)[3]) {
  const float2 *w2 = reinterpret_cast<const float2 *>(ws);
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    A[k].v = w2[k * kMaxChunk + i];
    B[k].v = w2[(3 + k) * kMaxChunk + i];
  }
}

// ------------------------------ the kernel --------------------------------
// in-plane-interpolated values of one z-stencil slice for the 12 populations with e_z != 0, as 6 pairs:
//   0 (f5, f6)  1 (g5, g6)  2 (f11, f14)  3 (f13, f12)  4 (f15, f18)  5 (f17, f16)
// (lane a has e_z = +1 in pairs 0, 1, 2, 4 and e_z = -1 in pairs 3 and 5, which take the swapped z-weights)
#define ISLBM_LOAD_M3(S)                                                                     \
  do {                                                                                       \
    S[0] = mkpr((AT)PC4(0)[0], (AT)PC4(2)[0]);              /* f5, f6 */             \
    S[1] = mkpr((AT)PC4(1)[0], (AT)PC4(3)[0]);              /* g5, g6 */             \
    S[2] = ptap3(PXM(0), PXM(3), 1, wxN);                   /* f11 (+x), f14 (-x) */ \
    S[3] = ptap3(PXM(2), PXM(1), 1, wxN);                   /* f13 (+x), f12 (-x) */ \
    S[4] = ptap3(PYM(0), PYM(3), T::TX, wyN);               /* f15 (+y), f18 (-y) */ \
    S[5] = ptap3(PYM(2), PYM(1), T::TX, wyN);               /* f17 (+y), f16 (-y) */ \
  } while (0)
// z-direction of the separable interpolation; (P0,P1,P2) = stencil slices in ascending z
#define ISLBM_ZCOMB3(P0, P1, P2)                                     \
  do {                                                               \
    const Pr<AT> q0 = pcomb3(wzN, P0[0], P1[0], P2[0]);              \
    const Pr<AT> q1 = pcomb3(wzN, P0[1], P1[1], P2[1]);              \
    const Pr<AT> q2 = pcomb3(wzN, P0[2], P1[2], P2[2]);              \
    const Pr<AT> q3 = pcomb3(wzS, P0[3], P1[3], P2[3]);              \
    const Pr<AT> q4 = pcomb3(wzN, P0[4], P1[4], P2[4]);              \
    const Pr<AT> q5 = pcomb3(wzS, P0[5], P1[5], P2[5]);              \
    f[5] = lane_a(q0);  f[6] = lane_b(q0);                           \
    g[5] = lane_a(q1);  g[6] = lane_b(q1);                           \
    f[11] = lane_a(q2); f[14] = lane_b(q2);                          \
    f[13] = lane_a(q3); f[12] = lane_b(q3);                          \
    f[15] = lane_a(q4); f[18] = lane_b(q4);                          \
    f[17] = lane_a(q5); f[16] = lane_b(q5);                          \
  } while (0)

template <typename ST, int TX, int TY>
__global__ void __launch_bounds__(TX * TY + producer_threads<ST, TX, TY>(), min_ctas3<ST, TX, TY>())
k_step_zmarch(const __grid_constant__ Maps3 mp, DevMesh m, NodeParams np, const ST *__restrict__ src,
              ST *__restrict__ dst, int zchunk, int load_policy, int store_policy, int flags) {
  using T = Tile3<ST, TX, TY>;
  constexpr bool PW = producer_threads<ST, TX, TY>() != 0;
  constexpr int ALL_THREADS = T::THREADS + producer_threads<ST, TX, TY>();
  // flags: bit 0 = first ring fill after the CTA barrier; bit 1 = leave the wall rules to k_step_shell3 (the
  // separate-boundary-kernel variant of BASELINE.json north_star, islbm_set_tuning("walls", 1); measured slower)
  const bool late_fill = flags & 1, skip_walls = flags & 2;
  using AT = typename Acc<ST>::type;
  // Ring refill policy (measured, profiles/): with fp64 storage the launch is DRAM-bound and thread 0 refilling the
  // slot released in the previous iteration (STAGES - 2 .. STAGES - 1 stages in flight) is 1.7 % faster; with fp32
  // storage the stages are half as large and the SM side dominates, and refilling each slot the moment its last
  // reader releases it (always STAGES - 1 stages in flight) is 6 % faster.
  constexpr bool EARLY = sizeof(ST) == 4;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *stage0 = smem_raw;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + T::BAR_OFF);
  uint64_t *empty = full + T::STAGES;
  AT *wzs = reinterpret_cast<AT *>(smem_raw + T::W_OFF);
  int *claim = reinterpret_cast<int *>(smem_raw + T::BAR_OFF + 2 * T::STAGES * 8);   // refill generation per slot
  pdl_launch_dependents();

  // the last y-tile is pulled back inside the mesh (it recomputes a few rows of its neighbour, bit-identically),
  // so that the shifted wall stencil of row ny-1 never leaves the box
  const int x0 = blockIdx.x * T::TX, y0 = min((int)blockIdx.y * T::TY, max(m.ny - T::TY, 0));
  const int z0 = m.em_lo + blockIdx.z * zchunk, z1 = min(z0 + zchunk, m.em_hi);
  const int nstage = 2 + (z1 - z0);
  // slab decomposition with the fused exchange: does this CTA touch the low / high boundary layer?  Then it waits for
  // that neighbour's step flag before its first load, and is counted when it is done (islbm_kernels.cuh)
  const bool b_lo = z0 == m.em_lo, b_hi = z1 == m.em_hi;
  const uint64_t lpol = make_policy(load_policy);
  const uint64_t spol = make_policy(store_policy);
  // thread 0 sets up the ring and (unless late_fill) fills it BEFORE warps 1.. load the weight rows, so the two
  // latencies overlap;
  // afterwards thread 0 (fp64 storage) or the last releasing warp (fp32) refills the slots.  griddepcontrol.wait
  // comes before the first access to a population buffer (everything else reads only tables).
  if (threadIdx.x == 0) {
    for (int s = 0; s < T::STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], T::CONSUMER_WARPS);
      claim[s] = 0;
    }
    fence_barrier_init();
    tma_prefetch_desc(&mp.c2);
    tma_prefetch_desc(&mp.c4);
    tma_prefetch_desc(&mp.x);
    tma_prefetch_desc(&mp.y);
    tma_prefetch_desc(&mp.xy);
    if (!late_fill && !PW) {
      pdl_wait();
      if (b_lo) slab_wait_neighbour(m, 0);
      if (b_hi) slab_wait_neighbour(m, 1);
      for (int s = 0; s < T::STAGES - (EARLY ? 0 : 1) && s < nstage; ++s)
        issue_stage3<T>(s, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
    }
  }
  for (int i = (int)threadIdx.x - 32; i >= 0 && i < 6 * (z1 - z0); i += ALL_THREADS - 32) {   // warps 1..: warp 0 is waiting above
    const int sk = i / (z1 - z0), zi = i - sk * (z1 - z0);
    stage_march_weight<0>(wzs, sk, zi, __ldg(wrow(m, 2, sk / 3, sk % 3) + z0 + zi));
  }
  pdl_wait();
  __syncthreads();
  if constexpr (PW) {
    if (threadIdx.x >= T::THREADS) {          // the producer warpgroup: one lane streams every stage, the rest retire
      asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
      if (threadIdx.x == T::THREADS) {
        if (b_lo) slab_wait_neighbour(m, 0);
        if (b_hi) slab_wait_neighbour(m, 1);
        for (int s = 0; s < nstage; ++s) {
          if (s >= T::STAGES) mbar_wait(&empty[s % T::STAGES], ((uint32_t)(s / T::STAGES) & 1u) ^ 1u);
          issue_stage3<T>(s, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
        }
      }
      return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
  }
  if (!PW && late_fill && threadIdx.x == 0) {
    if (b_lo) slab_wait_neighbour(m, 0);
    if (b_hi) slab_wait_neighbour(m, 1);
    for (int s = 0; s < T::STAGES - (EARLY ? 0 : 1) && s < nstage; ++s)
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
  // per-thread element offsets inside the four box shapes.  Made opaque so that they stay in registers: under
  // register pressure the compiler otherwise re-derives them from threadIdx in every iteration (~40 instructions)
  int o_xy = (ty + sy) * T::HX + (tx + T::XH - 1 + sx);    // 3x3 stencil, pitch HX
  int o_x = ty * T::HX + (tx + T::XH - 1 + sx);            // x-stencil, taps +0,+1,+2
  int o_y = (ty + sy) * T::TX + tx;                        // y-stencil, taps +0,+TX,+2TX
  int o_c = ty * T::TX + tx;
#ifdef ISLBM_OPAQUE_OFFSETS
  asm volatile("" : "+r"(o_xy), "+r"(o_x), "+r"(o_y), "+r"(o_c));
#endif
  // weights of the two signs as pairs: N = (c = +1, c = -1), S = swapped
  Pr<AT> wxN[3], wyN[3], wyS[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const AT x1 = valid ? (AT)__ldg(wrow(m, 0, 1, k) + x) : (AT)0, x0w = valid ? (AT)__ldg(wrow(m, 0, 0, k) + x) : (AT)0;
    const AT y1 = valid ? (AT)__ldg(wrow(m, 1, 1, k) + y) : (AT)0, y0w = valid ? (AT)__ldg(wrow(m, 1, 0, k) + y) : (AT)0;
    wxN[k] = mkpr(x1, x0w);
    wyN[k] = mkpr(y1, y0w);
    wyS[k] = mkpr(y0w, y1);
  }
  const long long plane = (long long)m.nxp * m.ny;
  // the node's index in plane 0 at the chunk's first slice; advanced by one slice per emitted slice
  long long c = (long long)z0 * plane + (long long)y * m.nxp + x;

  // three register sets hold the z-stencil slices; `newest` names the one written last, so the ascending-z
  // order is (newest+1, newest+2, newest) mod 3 and nothing is ever copied between sets
  Pr<AT> S0[6], S1[6], S2[6];
  int newest = 2;
  Pr<AT> *ssm = reinterpret_cast<Pr<AT> *>(smem_raw + T::S_OFF) + threadIdx.x;   // S_IN_SMEM: [slot][pair][thread]
  constexpr int SSLOT = 6 * T::THREADS;

#pragma unroll 1
  for (int s = 0; s < nstage; ++s) {
    const int st = s % T::STAGES;     // warp-uniform: these live on the uniform datapath, not in vector registers
    const uint32_t ph = (uint32_t)(s / T::STAGES) & 1u;
    const int z = z0 + (s - 2);
    const bool has_emit = s >= 2;
    const bool has_mov = s <= 2 || sbase_moves(z, m.nz);
    const ST *sb = reinterpret_cast<const ST *>(stage0 + (size_t)st * T::STAGE_BYTES);
    const ST *sbc = sb + o_c, *sbx = sb + o_x, *sby = sb + o_y, *sbxy = sb + o_xy;
    constexpr int ES = (int)sizeof(ST);
#define PC2(k) (sbc + (T::OFF_C2 + (k) * T::P_C) / ES)
#define PXZ(k) (sbx + (T::OFF_XZ + (k) * T::P_X) / ES)
#define PYZ(k) (sby + (T::OFF_YZ + (k) * T::P_Y) / ES)
#define PXY(k) (sbxy + (T::OFF_XY + (k) * T::P_XY) / ES)
#define PC4(k) (sbc + T::moff(T::OFF_C4, k, T::P_C, T::H_C) / ES)
#define PXM(k) (sbx + T::moff(T::OFF_XM, k, T::P_X, T::H_X) / ES)
#define PYM(k) (sby + T::moff(T::OFF_YM, k, T::P_Y, T::H_Y) / ES)
    if (!EARLY && !PW && threadIdx.x == 0 && s + T::STAGES - 1 < nstage) {
      const int sn = s + T::STAGES - 1;
      if (sn >= T::STAGES) mbar_wait(&empty[sn % T::STAGES], ((uint32_t)(sn / T::STAGES) & 1u) ^ 1u);
      issue_stage3<T>(sn, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
    }
    __syncwarp();
    mbar_wait(&full[st], ph);

    if (has_mov) {
      newest = newest == 2 ? 0 : newest + 1;
      if constexpr (T::S_IN_SMEM) {
        ISLBM_LOAD_M3(S2);       // S2 = the newest slice, in registers for this iteration and in its shared-memory slot
#pragma unroll
        for (int k = 0; k < 6; ++k) ssm[newest * SSLOT + k * T::THREADS] = S2[k];
      } else {
        if (newest == 0) ISLBM_LOAD_M3(S0);
        else if (newest == 1) ISLBM_LOAD_M3(S1);
        else ISLBM_LOAD_M3(S2);
      }
    }

    AT f[19], g[7];   // fp64, or fp32 deviations (fp32 storage)
    if (has_emit) {
      f[0] = PC2(0)[0];
      g[0] = PC2(1)[0];
      const Pr<AT> p1 = ptap3(PXZ(0), PXZ(1), 1, wxN);               // f1 (+x), f2 (-x)
      const Pr<AT> p2 = ptap3(PXZ(2), PXZ(3), 1, wxN);               // g1, g2
      const Pr<AT> p3 = ptap3(PYZ(0), PYZ(1), T::TX, wyN);           // f3 (+y), f4 (-y)
      const Pr<AT> p4 = ptap3(PYZ(2), PYZ(3), T::TX, wyN);           // g3, g4
      const Pr<AT> p5 = ptap9(PXY(0), PXY(3), T::HX, wxN, wyN);      // f7 (+x,+y), f10 (-x,-y)
      const Pr<AT> p6 = ptap9(PXY(2), PXY(1), T::HX, wxN, wyS);      // f9 (+x,-y), f8 (-x,+y)
      f[1] = lane_a(p1); f[2] = lane_b(p1);
      g[1] = lane_a(p2); g[2] = lane_b(p2);
      f[3] = lane_a(p3); f[4] = lane_b(p3);
      g[3] = lane_a(p4); g[4] = lane_b(p4);
      f[7] = lane_a(p5); f[10] = lane_b(p5);
      f[9] = lane_a(p6); f[8] = lane_b(p6);
    }
    // all shared-memory reads of this stage are done: hand the slot back to the producer (EARLY: the warp whose
    // release is the last one refills it at once with stage s + STAGES)
    __syncwarp();
    if ((threadIdx.x & 31) == 0) {
      if (!EARLY) mbar_arrive(&empty[st]);
      else if (mbar_arrive_is_last(&empty[st]) && s + T::STAGES < nstage &&
               atomicCAS(&claim[st], s / T::STAGES, s / T::STAGES + 1) == s / T::STAGES)
        issue_stage3<T>(s + T::STAGES, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
    }

    if (has_emit) {
      Pr<AT> wzN[3], wzS[3];
      load_march_weights<0>(wzs, s - 2, wzN, wzS);
      if constexpr (T::S_IN_SMEM) {
        // ascending z = slots (newest+1, newest+2, newest) mod 3; the newest slice is still in registers unless the
        // stencil base did not move (first / last two slices of the mesh)
        const Pr<AT> *p0 = ssm + (newest == 2 ? 0 : newest + 1) * SSLOT, *p1 = ssm + (newest == 0 ? 2 : newest - 1) * SSLOT;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
          S0[k] = p0[k * T::THREADS];
          S1[k] = p1[k * T::THREADS];
        }
        if (!has_mov) {
#pragma unroll
          for (int k = 0; k < 6; ++k) S2[k] = ssm[newest * SSLOT + k * T::THREADS];
        }
        ISLBM_ZCOMB3(S0, S1, S2);
      } else {
        if (newest == 0) ISLBM_ZCOMB3(S1, S2, S0);
        else if (newest == 1) ISLBM_ZCOMB3(S2, S0, S1);
        else ISLBM_ZCOMB3(S0, S1, S2);
      }
      wf.lo[2] = z == 0 && m.wall_mlo;
      wf.hi[2] = z == m.nz - 1 && m.wall_mhi;
      if (!skip_walls && valid && (wall_xy | wf.lo[2] | wf.hi[2])) wall_fix_node<3>(f, g, wf, src + c, m.nnp, m);
      constexpr bool DEV = Store<ST, 3>::kBiased;   // fp32 storage: collide the deviations as they are
      collide_node<DEV>(f, g, np);
      if (valid) {
        store_node<3, DEV>(dst + c, m.nnp, f, g, spol, std::make_integer_sequence<int, 26>{});
        if (m.peer[0] != nullptr || m.peer[1] != nullptr)     // slab boundary layers only: keep the 64-bit index arithmetic out of the march
          peer_store_node<3, ST, DEV>(m, z, c - (long long)z * plane, f, g);
      }
      c += plane;
    }
#undef PC2
#undef PXZ
#undef PYZ
#undef PXY
#undef PC4
#undef PXM
#undef PYM
  }
  if ((b_lo && m.flag_out[0] != nullptr) || (b_hi && m.flag_out[1] != nullptr)) {   // CTA-uniform
    if constexpr (PW) asm volatile("bar.sync 1, %0;" ::"n"(T::THREADS) : "memory");   // the consumer warps only
    else __syncthreads();
    if (threadIdx.x == 0) {
      if (b_lo) slab_publish(m, 0);
      if (b_hi) slab_publish(m, 1);
    }
  }
}

// ------------------------------ the kernel, upwind stencil -----------------------------------------------------
// Same march with the A2-alternative stencil {j-2,j-1,j} (c = +1) / {j,j+1,j+2} (c = -1) (islbm_set_stencil(h, 1);
// SURVEY.md 8(f)-3).  What changes against k_step_zmarch: the two lanes of a pair read different
// windows (lane a, the c = +1 population, starts two nodes upstream; lane b, c = -1, at the node itself), the y-halo
// is two rows, and the z-stencil state splits into two families of three pairs each:
//   family P (e_z = +1): (f5, g5) (f11, f12) (f15, f16), slices {z-2, z-1, z};
//   family M (e_z = -1): (f6, g6) (f13, f14) (f17, f18), slices {z, z+1, z+2};
// each with its own rotating register sets (fp64) or shared-memory slots (fp32 storage) and its own stencil-base
// bookkeeping at the ends of the axis.  Both lanes of a family pair take the z-weights of the same sign.
#define ISLBM_LOAD_U3(S, H)                                                                           \
  do {                                                                                                \
    S[0] = mkpr((AT)PC4(2 * H)[o_c], (AT)PC4(2 * H + 1)[o_c]);              /* f5 g5 | f6 g6 */       \
    S[1] = ptap3(PXM(2 * H) + o_xa, PXM(2 * H + 1) + o_xb, 1, wxN);         /* f11 f12 | f13 f14 */   \
    S[2] = ptap3(PYM(2 * H) + o_ya, PYM(2 * H + 1) + o_yb, T::TX, wyN);     /* f15 f16 | f17 f18 */   \
  } while (0)
#define ISLBM_ZCOMB_U3(W, P0, P1, P2, F0, G0, F1A, F1B, F2A, F2B)   \
  do {                                                              \
    const Pr<AT> q0 = pcomb3(W, P0[0], P1[0], P2[0]);               \
    const Pr<AT> q1 = pcomb3(W, P0[1], P1[1], P2[1]);               \
    const Pr<AT> q2 = pcomb3(W, P0[2], P1[2], P2[2]);               \
    f[F0] = lane_a(q0);  g[G0] = lane_b(q0);                        \
    f[F1A] = lane_a(q1); f[F1B] = lane_b(q1);                       \
    f[F2A] = lane_a(q2); f[F2B] = lane_b(q2);                       \
  } while (0)

template <typename ST, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, TX * TY <= 128 ? 3 : (TX * TY <= 192 ? 2 : 1))
k_step_zmarch_up(const __grid_constant__ Maps3 mp, DevMesh m, NodeParams np, const ST *__restrict__ src,
                 ST *__restrict__ dst, int zchunk, int load_policy, int store_policy, int late_fill) {
  using T = Tile3<ST, TX, TY, 1>;
  using AT = typename Acc<ST>::type;
  constexpr bool EARLY = sizeof(ST) == 4;   // ring refill policy: see k_step_zmarch
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *stage0 = smem_raw;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + T::BAR_OFF);
  uint64_t *empty = full + T::STAGES;
  AT *wzs = reinterpret_cast<AT *>(smem_raw + T::W_OFF);
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
      mbar_init(&empty[s], T::CONSUMER_WARPS);
      claim[s] = 0;
    }
    fence_barrier_init();
    tma_prefetch_desc(&mp.c2);
    tma_prefetch_desc(&mp.x);
    tma_prefetch_desc(&mp.y);
    tma_prefetch_desc(&mp.xy);
    tma_prefetch_desc(&mp.x2);
    tma_prefetch_desc(&mp.y2);
    if (!late_fill) {
      pdl_wait();
      for (int s = 0; s < T::STAGES - (EARLY ? 0 : 1) && s < nstage; ++s)
        issue_stage3<T>(s, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
    }
  }
  for (int i = (int)threadIdx.x - 32; i >= 0 && i < 6 * (z1 - z0); i += T::THREADS - 32) {
    const int sk = i / (z1 - z0), zi = i - sk * (z1 - z0);
    stage_march_weight<1>(wzs, sk, zi, __ldg(wrow(m, 2, sk / 3, sk % 3) + z0 + zi));
  }
  pdl_wait();
  __syncthreads();
  if (late_fill && threadIdx.x == 0) {
    for (int s = 0; s < T::STAGES - (EARLY ? 0 : 1) && s < nstage; ++s)
      issue_stage3<T>(s, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
  }

  const int tx = threadIdx.x % T::TX, ty = threadIdx.x / T::TX;
  const int x = x0 + tx, y = y0 + ty;
  const bool valid = x < m.nx && y < m.ny;
  WallFlags wf;
  wf.lo[0] = valid && x == 0;  wf.hi[0] = valid && x == m.nx - 1;
  wf.lo[1] = valid && y == 0;  wf.hi[1] = valid && y == m.ny - 1;
  const bool wall_xy = wf.lo[0] | wf.hi[0] | wf.lo[1] | wf.hi[1];
  // first stencil node of lane a (c = +1) / lane b (c = -1) inside the boxes: columns of the x-haloed shapes, rows of
  // the y-haloed ones (a thread outside the mesh reads inside the box all the same; its results are not stored)
  const int col_a = ubase_p(min(x, m.nx - 1), m.nx) - x0 + T::XH, col_b = ubase_m(min(x, m.nx - 1), m.nx) - x0 + T::XH;
  const int row_a = ubase_p(min(y, m.ny - 1), m.ny) - y0 + T::YH, row_b = ubase_m(min(y, m.ny - 1), m.ny) - y0 + T::YH;
  const int o_xa = ty * T::HX + col_a, o_xb = ty * T::HX + col_b;                 // x-stencil, taps +0,+1,+2
  const int o_ya = row_a * T::TX + tx, o_yb = row_b * T::TX + tx;                 // y-stencil, taps +0,+TX,+2TX
  const int o_aa = row_a * T::HX + col_a, o_bb = row_b * T::HX + col_b;           // 3x3 stencils, pitch HX
  const int o_ba = row_b * T::HX + col_a, o_ab = row_a * T::HX + col_b;           // (row of -y, column of +x), (+y, -x)
  const int o_c = ty * T::TX + tx;
  Pr<AT> wxN[3], wyN[3], wyS[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const AT x1 = valid ? (AT)__ldg(wrow(m, 0, 1, k) + x) : (AT)0, x0w = valid ? (AT)__ldg(wrow(m, 0, 0, k) + x) : (AT)0;
    const AT y1 = valid ? (AT)__ldg(wrow(m, 1, 1, k) + y) : (AT)0, y0w = valid ? (AT)__ldg(wrow(m, 1, 0, k) + y) : (AT)0;
    wxN[k] = mkpr(x1, x0w);
    wyN[k] = mkpr(y1, y0w);
    wyS[k] = mkpr(y0w, y1);
  }
  const long long plane = (long long)m.nxp * m.ny;
  long long c = (long long)z0 * plane + (long long)y * m.nxp + x;

  // per family three sets; `newest_*` names the one written last, ascending z = (newest+1, newest+2, newest) mod 3
  Pr<AT> P0[3], P1[3], P2[3], M0[3], M1[3], M2[3];
  int newest_p = 2, newest_m = 2;
  Pr<AT> *ssm = reinterpret_cast<Pr<AT> *>(smem_raw + T::S_OFF) + threadIdx.x;   // S_IN_SMEM: [family][slot][pair][thread]
  constexpr int SSLOT = 3 * T::THREADS;

#pragma unroll 1
  for (int s = 0; s < nstage; ++s) {
    const int st = s % T::STAGES;
    const uint32_t ph = (uint32_t)(s / T::STAGES) & 1u;
    const int z = z0 + (s - 2);
    const bool has_emit = s >= 2;
    const bool mov_p = s <= 2 || ubase_p_moves(z, m.nz), mov_m = s <= 2 || ubase_m_moves(z, m.nz);
    const ST *sb = reinterpret_cast<const ST *>(stage0 + (size_t)st * T::STAGE_BYTES);
    constexpr int ES = (int)sizeof(ST);
#define PC2(k) (sb + (T::OFF_C2 + (k) * T::P_C) / ES)
#define PXZ(k) (sb + (T::OFF_XZ + (k) * T::P_X) / ES)
#define PYZ(k) (sb + (T::OFF_YZ + (k) * T::P_Y) / ES)
#define PXY(k) (sb + (T::OFF_XY + (k) * T::P_XY) / ES)
#define PC4(k) (sb + T::moff(T::OFF_C4, k, T::P_C, T::H_C) / ES)
#define PXM(k) (sb + T::moff(T::OFF_XM, k, T::P_X, T::H_X) / ES)
#define PYM(k) (sb + T::moff(T::OFF_YM, k, T::P_Y, T::H_Y) / ES)
    if (!EARLY && threadIdx.x == 0 && s + T::STAGES - 1 < nstage) {
      const int sn = s + T::STAGES - 1;
      if (sn >= T::STAGES) mbar_wait(&empty[sn % T::STAGES], ((uint32_t)(sn / T::STAGES) & 1u) ^ 1u);
      issue_stage3<T>(sn, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
    }
    __syncwarp();
    mbar_wait(&full[st], ph);

    if (mov_p) {
      newest_p = newest_p == 2 ? 0 : newest_p + 1;
      if constexpr (T::S_IN_SMEM) {
        ISLBM_LOAD_U3(P2, 0);
#pragma unroll
        for (int k = 0; k < 3; ++k) ssm[newest_p * SSLOT + k * T::THREADS] = P2[k];
      } else {
        if (newest_p == 0) ISLBM_LOAD_U3(P0, 0);
        else if (newest_p == 1) ISLBM_LOAD_U3(P1, 0);
        else ISLBM_LOAD_U3(P2, 0);
      }
    }
    if (mov_m) {
      newest_m = newest_m == 2 ? 0 : newest_m + 1;
      if constexpr (T::S_IN_SMEM) {
        ISLBM_LOAD_U3(M2, 1);
#pragma unroll
        for (int k = 0; k < 3; ++k) ssm[(3 + newest_m) * SSLOT + k * T::THREADS] = M2[k];
      } else {
        if (newest_m == 0) ISLBM_LOAD_U3(M0, 1);
        else if (newest_m == 1) ISLBM_LOAD_U3(M1, 1);
        else ISLBM_LOAD_U3(M2, 1);
      }
    }

    AT f[19], g[7];
    if (has_emit) {
      f[0] = PC2(0)[o_c];
      g[0] = PC2(1)[o_c];
      const Pr<AT> p1 = ptap3(PXZ(0) + o_xa, PXZ(1) + o_xb, 1, wxN);                 // f1 (+x), f2 (-x)
      const Pr<AT> p2 = ptap3(PXZ(2) + o_xa, PXZ(3) + o_xb, 1, wxN);                 // g1, g2
      const Pr<AT> p3 = ptap3(PYZ(0) + o_ya, PYZ(1) + o_yb, T::TX, wyN);             // f3 (+y), f4 (-y)
      const Pr<AT> p4 = ptap3(PYZ(2) + o_ya, PYZ(3) + o_yb, T::TX, wyN);             // g3, g4
      const Pr<AT> p5 = ptap9(PXY(0) + o_aa, PXY(3) + o_bb, T::HX, wxN, wyN);        // f7 (+x,+y), f10 (-x,-y)
      const Pr<AT> p6 = ptap9(PXY(2) + o_ba, PXY(1) + o_ab, T::HX, wxN, wyS);        // f9 (+x,-y), f8 (-x,+y)
      f[1] = lane_a(p1); f[2] = lane_b(p1);
      g[1] = lane_a(p2); g[2] = lane_b(p2);
      f[3] = lane_a(p3); f[4] = lane_b(p3);
      g[3] = lane_a(p4); g[4] = lane_b(p4);
      f[7] = lane_a(p5); f[10] = lane_b(p5);
      f[9] = lane_a(p6); f[8] = lane_b(p6);
    }
    __syncwarp();
    if ((threadIdx.x & 31) == 0) {
      if (!EARLY) mbar_arrive(&empty[st]);
      else if (mbar_arrive_is_last(&empty[st]) && s + T::STAGES < nstage &&
               atomicCAS(&claim[st], s / T::STAGES, s / T::STAGES + 1) == s / T::STAGES)
        issue_stage3<T>(s + T::STAGES, z0, m.nz, x0, y0, stage0, full, empty, mp, lpol);
    }

    if (has_emit) {
      Pr<AT> wzA[3], wzB[3];    // (c=+1, c=+1) for family P, (c=-1, c=-1) for family M
      load_march_weights<1>(wzs, s - 2, wzA, wzB);
      if constexpr (T::S_IN_SMEM) {
        const Pr<AT> *pp0 = ssm + (newest_p == 2 ? 0 : newest_p + 1) * SSLOT, *pp1 = ssm + (newest_p == 0 ? 2 : newest_p - 1) * SSLOT;
        const Pr<AT> *pm0 = ssm + (3 + (newest_m == 2 ? 0 : newest_m + 1)) * SSLOT, *pm1 = ssm + (3 + (newest_m == 0 ? 2 : newest_m - 1)) * SSLOT;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          P0[k] = pp0[k * T::THREADS];
          P1[k] = pp1[k * T::THREADS];
          M0[k] = pm0[k * T::THREADS];
          M1[k] = pm1[k * T::THREADS];
        }
        if (!mov_p) {
#pragma unroll
          for (int k = 0; k < 3; ++k) P2[k] = ssm[newest_p * SSLOT + k * T::THREADS];
        }
        if (!mov_m) {
#pragma unroll
          for (int k = 0; k < 3; ++k) M2[k] = ssm[(3 + newest_m) * SSLOT + k * T::THREADS];
        }
        ISLBM_ZCOMB_U3(wzA, P0, P1, P2, 5, 5, 11, 12, 15, 16);
        ISLBM_ZCOMB_U3(wzB, M0, M1, M2, 6, 6, 13, 14, 17, 18);
      } else {
        if (newest_p == 0) ISLBM_ZCOMB_U3(wzA, P1, P2, P0, 5, 5, 11, 12, 15, 16);
        else if (newest_p == 1) ISLBM_ZCOMB_U3(wzA, P2, P0, P1, 5, 5, 11, 12, 15, 16);
        else ISLBM_ZCOMB_U3(wzA, P0, P1, P2, 5, 5, 11, 12, 15, 16);
        if (newest_m == 0) ISLBM_ZCOMB_U3(wzB, M1, M2, M0, 6, 6, 13, 14, 17, 18);
        else if (newest_m == 1) ISLBM_ZCOMB_U3(wzB, M2, M0, M1, 6, 6, 13, 14, 17, 18);
        else ISLBM_ZCOMB_U3(wzB, M0, M1, M2, 6, 6, 13, 14, 17, 18);
      }
      wf.lo[2] = z == 0 && m.wall_mlo;
      wf.hi[2] = z == m.nz - 1 && m.wall_mhi;
      if (valid && (wall_xy | wf.lo[2] | wf.hi[2])) wall_fix_node<3>(f, g, wf, src + c, m.nnp, m);
      constexpr bool DEV = Store<ST, 3>::kBiased;
      collide_node<DEV>(f, g, np);
      if (valid) store_node<3, DEV>(dst + c, m.nnp, f, g, spol, std::make_integer_sequence<int, 26>{});
      c += plane;
    }
#undef PC2
#undef PXZ
#undef PYZ
#undef PXY
#undef PC4
#undef PXM
#undef PYM
  }
}

// ------------------------------ separate boundary kernel (A/B variant) ----------------------------------------
// BASELINE.json north_star names "wall nodes handled by a separate boundary kernel".  This is that design, kept as a
// measurable alternative (islbm_set_tuning("walls", 1)): the march skips the wall rules, and this kernel then
// recomputes the shell of wall-adjacent nodes (6 faces, 2.3 % of the nodes at 256^3) from the source buffer — pull,
// Eq. 21-23, collide — and overwrites what the march stored there.  It moves more bytes (the shell is read through
// the stencil and written twice) and two of its faces are strided by a whole row; profiles/attempts.md has the A/B.
template <typename ST>
__global__ void __launch_bounds__(256)
k_step_shell3(DevMesh m, NodeParams np, const ST *__restrict__ src, ST *__restrict__ dst) {
  const int face = blockIdx.z, a = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y * blockDim.y + threadIdx.y;
  int ix, iy, iz;
  if (face < 2) { ix = face == 0 ? 0 : m.nx - 1; iy = a; iz = b; }
  else if (face < 4) { ix = a; iy = face == 2 ? 0 : m.ny - 1; iz = b; }
  else { ix = a; iy = b; iz = face == 4 ? 0 : m.nz - 1; }
  if (ix >= m.nx || iy >= m.ny || iz >= m.nz) return;
  NodeCtx<3> cx;
  make_ctx<3>(m, ix, iy, iz, cx);
  double f[19], g[7];
  pull_all_f<3>(m, src, cx, f, std::make_integer_sequence<int, 19>{});
  pull_all_g<3>(m, src, cx, g, std::make_integer_sequence<int, 7>{});
  add_bias<ST, 3>(f);
  collide_node(f, g, np);
#pragma unroll
  for (int q = 0; q < 19; ++q) dst[(long long)plane_f<3>(q) * m.nnp + cx.c] = to_storage<ST, 3>(f[q], q);
#pragma unroll
  for (int q = 0; q < 7; ++q) dst[(long long)plane_g<3>(q) * m.nnp + cx.c] = (ST)g[q];
}

// ------------------------------ host side ---------------------------------
struct Plan3 {
  bool available = false;
  Maps3 maps[2];            // per ping-pong buffer
  int zchunk = 32;
  int shape = 0;            // tile shape index (Tuning::shape3d)
  int sk = 0;               // stencil kind the plan was built for: 0 central, 1 upwind
  char why_not[96] = "";
};

template <typename ST, int TX, int TY, int SK>
inline bool plan3_setup(Plan3 &p, const int *n, int nxp, void *buf0, void *buf1, const Tuning &tn) {
  using T = Tile3<ST, TX, TY, SK>;
  p.available = false;
  auto no = [&](const char *why) { snprintf(p.why_not, sizeof p.why_not, "%s", why); return false; };
  if (n[0] < 3 || n[1] < 3 || n[2] < 3) return no("tiled kernel: n >= 3");
  if ((nxp * (int)sizeof(ST)) % 16) return no("tiled kernel: TMA needs a 16-byte row pitch");
  int dev = 0, cc_major = 0, smem_optin = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return no("no device");
  cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev);
  cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (cc_major < 10 || (size_t)smem_optin < T::SMEM_BYTES) return no("tiled kernel: needs sm_100 and its shared memory");
  void *bufs[2] = {buf0, buf1};
  const int eb = (int)sizeof(ST);
  const long long dims[4] = {n[0], n[1], n[2], 26};
  const int b_c2[4] = {T::TX, T::TY, 1, 2}, b_c4[4] = {T::TX, T::TY, 1, 4}, b_x[4] = {T::HX, T::TY, 1, 4};
  const int b_y[4] = {T::TX, T::HY, 1, 4}, b_xy[4] = {T::HX, T::HY, 1, 4};
  const int b_x2[4] = {T::HX, T::TY, 1, 2}, b_y2[4] = {T::TX, T::HY, 1, 2};
  for (int i = 0; i < 2; ++i) {
    if (!make_map(&p.maps[i].c2, bufs[i], eb, 4, dims, b_c2, tn.l2promo, nxp) ||
        !make_map(&p.maps[i].c4, bufs[i], eb, 4, dims, b_c4, tn.l2promo, nxp) ||
        !make_map(&p.maps[i].x, bufs[i], eb, 4, dims, b_x, tn.l2promo, nxp) ||
        !make_map(&p.maps[i].y, bufs[i], eb, 4, dims, b_y, tn.l2promo, nxp) ||
        !make_map(&p.maps[i].xy, bufs[i], eb, 4, dims, b_xy, tn.l2promo, nxp) ||
        !make_map(&p.maps[i].x2, bufs[i], eb, 4, dims, b_x2, tn.l2promo, nxp) ||
        !make_map(&p.maps[i].y2, bufs[i], eb, 4, dims, b_y2, tn.l2promo, nxp))
      return no("cuTensorMapEncodeTiled failed");
  }
  cudaError_t e;
  if constexpr (SK == 0) e = cudaFuncSetAttribute(k_step_zmarch<ST, TX, TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM_BYTES);
  else e = cudaFuncSetAttribute(k_step_zmarch_up<ST, TX, TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM_BYTES);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return no("cudaFuncSetAttribute failed");
  }
  // z-chunks (measured, profiles/): short chunks win — neighbouring CTAs stay in step, so the halo overlap is found in
  // L2, and the tail is fine-grained.  Meshes with at least one CTA per SM in every z-layer of tiles take 16 slices (the
  // 2-slice prologue then re-reads 12 of 26 planes twice per 16: +6 % reads through L2); smaller meshes take one full
  // wave of still shorter chunks (a CTA needs ~2 us per slice whatever the mesh).
  const int tiles = ((n[0] + T::TX - 1) / T::TX) * ((n[1] + T::TY - 1) / T::TY);
  auto ctas = [&](int c) { return (long long)tiles * ((n[2] + c - 1) / c); };
  const int sms = sm_count();
  int chunk = n[2] < kMaxChunk ? n[2] : kMaxChunk;
  if (tn.chunk > 0) {
    chunk = tn.chunk < n[2] ? tn.chunk : n[2];
  } else if (tiles >= sms) {
    chunk = n[2] < 16 ? n[2] : 16;
  } else {
    while (chunk > 4 && ctas((chunk + 1) / 2) <= sms + 16) chunk = (chunk + 1) / 2;
    while (chunk > 8 && ctas(chunk) < sms * 12) chunk = (chunk + 1) / 2;
  }
  p.zchunk = chunk < kMaxChunk ? chunk : kMaxChunk;
  p.available = true;
  return true;
}

template <typename ST, int TX, int TY, int SK>
inline void launch3_shape(const Plan3 &p, const int *n, const DevMesh &m, const NodeParams &np, int cur, void *const *buf,
                          const Tuning &tn, cudaStream_t stream) {
  using T = Tile3<ST, TX, TY, SK>;
  dim3 grid((n[0] + T::TX - 1) / T::TX, (n[1] + T::TY - 1) / T::TY, (m.em_hi - m.em_lo + p.zchunk - 1) / p.zchunk);
  DevMesh mm = m;
  mm.bctas = (int)(grid.x * grid.y);   // CTAs that touch one boundary layer of a slab
  if constexpr (SK == 0)
  {
    const bool shell = tn.walls == 1 && m.em_lo == 0 && m.em_hi == m.nz && m.peer[0] == nullptr && m.peer[1] == nullptr;
    launch_step(k_step_zmarch<ST, TX, TY>, grid, dim3(T::THREADS + producer_threads<ST, TX, TY>()), T::SMEM_BYTES, stream, tn.pdl != 0 && !shell, p.maps[cur], mm,
                np, (const ST *)buf[cur], (ST *)buf[1 - cur], p.zchunk, tn.load_policy, tn.store_policy,
                (tn.fill == 2 ? 1 : 0) | (shell ? 2 : 0));
    if (shell) {
      const int e1 = n[0] > n[1] ? n[0] : n[1], e2 = n[1] > n[2] ? n[1] : n[2];
      dim3 sg((e1 + 31) / 32, (e2 + 7) / 8, 6);
      k_step_shell3<ST><<<sg, dim3(32, 8), 0, stream>>>(m, np, (const ST *)buf[cur], (ST *)buf[1 - cur]);
    }
  }
  else
    launch_step(k_step_zmarch_up<ST, TX, TY>, grid, dim3(T::THREADS), T::SMEM_BYTES, stream, tn.pdl != 0, p.maps[cur], m, np,
                (const ST *)buf[cur], (ST *)buf[1 - cur], p.zchunk, tn.load_policy, tn.store_policy, tn.fill == 2 ? 1 : 0);
}

// sk = 0: the destination-centred stencil; 1: the upwind stencil (islbm_set_stencil)
template <typename ST>
inline bool plan3_create(Plan3 &p, const int *n, int nxp, void *buf0, void *buf1, const Tuning &tn, int sk) {
  // tile shape (x by y nodes per CTA).  fp64 storage: 32x8 (one CTA of 8 consumer warps per SM; DRAM-bound).  fp32
  // storage is bound by latency: 32x8 with two CTAs per SM (16 warps at 128 registers, 2-stage ring) for the central
  // stencil; the upwind kernels (168 registers) exist as 32x6 (two per SM) and 32x4 (three per SM, short y-axes) and
  // as 32x8 for fp64 (profiles/attempts.md).
  int shape = tn.shape3d;
  if (sk) {
    if (shape != 3 && shape != 4) shape = sizeof(ST) == 4 ? (n[1] >= 192 ? 3 : 4) : 5;
  } else if (shape == 0) {
    shape = 5;
  }
  p.shape = shape;
  p.sk = sk;
  if (sk) {
    if constexpr (sizeof(ST) == 4) {
      if (shape == 4) return plan3_setup<ST, 32, 4, 1>(p, n, nxp, buf0, buf1, tn);
      p.shape = 3;
      return plan3_setup<ST, 32, 6, 1>(p, n, nxp, buf0, buf1, tn);
    } else {
      p.shape = 5;
      return plan3_setup<ST, 32, 8, 1>(p, n, nxp, buf0, buf1, tn);
    }
  }
  switch (shape) {
    case 1: return plan3_setup<ST, 64, 4, 0>(p, n, nxp, buf0, buf1, tn);
    case 2: return plan3_setup<ST, 128, 2, 0>(p, n, nxp, buf0, buf1, tn);
    case 3: return plan3_setup<ST, 32, 6, 0>(p, n, nxp, buf0, buf1, tn);
    case 4: return plan3_setup<ST, 32, 4, 0>(p, n, nxp, buf0, buf1, tn);
    default: p.shape = 5; return plan3_setup<ST, 32, 8, 0>(p, n, nxp, buf0, buf1, tn);
  }
}

template <typename ST>
inline cudaError_t launch3(const Plan3 &p, const int *n, const DevMesh &m, const NodeParams &np, int cur, void *const *buf,
                           const Tuning &tn, cudaStream_t stream) {
  if (p.sk) {
    if constexpr (sizeof(ST) == 4) {
      if (p.shape == 4) launch3_shape<ST, 32, 4, 1>(p, n, m, np, cur, buf, tn, stream);
      else launch3_shape<ST, 32, 6, 1>(p, n, m, np, cur, buf, tn, stream);
    } else {
      launch3_shape<ST, 32, 8, 1>(p, n, m, np, cur, buf, tn, stream);
    }
    return cudaPeekAtLastError();
  }
  switch (p.shape) {
    case 1: launch3_shape<ST, 64, 4, 0>(p, n, m, np, cur, buf, tn, stream); break;
    case 2: launch3_shape<ST, 128, 2, 0>(p, n, m, np, cur, buf, tn, stream); break;
    case 3: launch3_shape<ST, 32, 6, 0>(p, n, m, np, cur, buf, tn, stream); break;
    case 4: launch3_shape<ST, 32, 4, 0>(p, n, m, np, cur, buf, tn, stream); break;
    default: launch3_shape<ST, 32, 8, 0>(p, n, m, np, cur, buf, tn, stream);
  }
  return cudaPeekAtLastError();
}

}  // namespace islbmk
