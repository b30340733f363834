// islbm_tiled2.cuh — fused, TMA-staged ISLBM step for D2Q9 + D2Q5 on sm_100a.
//
// "y-marching" design, the 2-D counterpart of islbm_tiled3.cuh:
//   * a CTA owns a strip of TX nodes in x (one thread per x) and marches
//     through a chunk of rows;
//   * one elected thread streams, per row, FOUR TMA boxes
//     (cp.async.bulk.tensor.3d over the view (x, y, plane); the storage planes
//     are ordered so that a box covers consecutive planes, plane_f / plane_g)
//     into a ring of shared-memory stages guarded by full/empty mbarriers;
//     planes with e_x != 0 (f1 f3 g1 g3 | f5..f8) carry a 16-byte x-halo on each
//     side, the others (f0 g0 | f2 g2 f4 g4) none;
//   * consumers interpolate along x from shared memory; the y-direction of the
//     separable interpolation is a 3-row combination kept
//     in REGISTERS (three rotating register sets) for the 8 populations with
//     e_y != 0, so every post-collision value is staged once and there is no
//     y-halo at all;
//   * the node collides once and stores its 14 values with coalesced stores.
// DIR = +1 marches a chunk upwards, DIR = -1 downwards ("serpentine" tuning: odd
// steps march downwards, so a step starts on the rows the previous step wrote
// last, which are the ones most likely still in L2; the 2-D states are of the
// order of the 126 MB L2).  Summation order is the oracle's either way: x, then y.
#pragma once

#include "islbm_tiled3.cuh"

namespace islbmk {

// CTAs per SM of the fp32-storage kernels (launch bounds): five = 96 registers (measured, profiles/attempts.md)
#ifndef ISLBM_F32_CTAS2D
#define ISLBM_F32_CTAS2D 5
#endif

template <typename ST, int TX_, int STAGES_, int SK_ = 0>
struct Tile2 {
  static constexpr int TX = TX_, STAGES = STAGES_, SK = SK_;   // SK: stencil kind (Tile3)
  static constexpr int XH = 16 / (int)sizeof(ST);
  static constexpr int HX = TX + 2 * XH;
  static constexpr int P_X = HX * (int)sizeof(ST), P_C = TX * (int)sizeof(ST);   // bytes of one plane row in a box
  // groups of a stage, in storage-plane order (each starts 128-byte aligned):
  //   emitted row y:      C2 = f0 g0, XR = f1 f3 g1 g3        y-stencil row (m):  C4 = f2 g2 f4 g4, XM = f5..f8
  static constexpr int OFF_C2 = 0;
  static constexpr int OFF_XR = pad128(OFF_C2 + 2 * P_C);
  // halves of a y-stencil group (e_y = +1, then e_y = -1): loaded by separate boxes with the upwind stencil, whose
  // shared-memory destinations must be 128-byte aligned (Tile3::H_*)
  static constexpr int H_C = SK ? pad128(2 * P_C) : 2 * P_C, H_X = SK ? pad128(2 * P_X) : 2 * P_X;
  static constexpr int OFF_C4 = pad128(OFF_XR + 4 * P_X);
  static constexpr int OFF_XM = pad128(OFF_C4 + 2 * H_C);
  static constexpr int STAGE_BYTES = pad128(OFF_XM + 2 * H_X);
  static __host__ __device__ constexpr int moff(int off, int k, int pbytes, int half) { return off + (k / 2) * half + (k % 2) * pbytes; }
  static constexpr int WARPS = TX / 32;
  static constexpr uint32_t Y_BYTES = 2u * P_C + 4u * P_X;   // planes of the emitted row
  static constexpr uint32_t M_BYTES = 4u * P_C + 4u * P_X;   // planes of the y-stencil row
  static constexpr uint32_t F_BYTES = M_BYTES / 2;           // ... of one half of it (upwind stencil)
  static constexpr int BAR_OFF = STAGES * STAGE_BYTES;
  static constexpr int W_OFF = BAR_OFF + 128;                // y-weights of the chunk [sign][k][kMaxChunk]
  // fp32 storage: the x-interpolated values of the three y-stencil rows live in shared memory, [slot 3][pair 4][thread]
  // float2, not in registers (Tile3::S_IN_SMEM, islbm_tiled3.cuh)
  static constexpr bool S_IN_SMEM = sizeof(ST) == 4 && ISLBM_S_IN_SMEM;
  static constexpr int S_OFF = W_OFF + 6 * kMaxChunk * 8 + 128;
  static constexpr size_t SMEM_BYTES = (size_t)S_OFF + (S_IN_SMEM ? 3 * 4 * TX * 8 : 0);
};

// tensor maps over (x, y, plane): one per box shape
struct Maps2 {
  CUtensorMap c2, c4, x;
  CUtensorMap x2;   // two-plane box of the x shape (upwind stencil: half of the group f5..f8)
};

// yf = first emitted row of the chunk (its lowest row for DIR = +1, its highest for DIR = -1).
// stage s < 2 : the first two rows (in marching order) of the y-stencil of row yf;
// stage s >= 2: the planes of emitted row y = yf + DIR*(s-2), plus the next y-stencil row if the stencil base moves.
template <typename T, int DIR>
__device__ __forceinline__ void issue_stage2(int s, int yf, int ny, int x0, unsigned char *stage0, uint64_t *full,
                                             uint64_t *empty, const Maps2 &mp, uint64_t pol) {
  const int st = s % T::STAGES;   // the caller knows the slot is free (initial fill, or it saw the last release)
  int mrow = -1, yrow = -1;
  if (s < 2) {
    mrow = DIR > 0 ? sbase(yf, ny) + s : sbase(yf, ny) + 2 - s;
  } else {
    yrow = yf + DIR * (s - 2);
    if (s == 2 || sbase(yrow, ny) != sbase(yrow - DIR, ny)) mrow = DIR > 0 ? sbase(yrow, ny) + 2 : sbase(yrow, ny);
  }
  mbar_expect_tx(&full[st], (mrow >= 0 ? T::M_BYTES : 0u) + (yrow >= 0 ? T::Y_BYTES : 0u));
  unsigned char *sb = stage0 + (size_t)st * T::STAGE_BYTES;
  uint64_t *bar = &full[st];
  const int xh = x0 - T::XH;
  if (yrow >= 0) {
    tma_load_3d(sb + T::OFF_C2, &mp.c2, bar, x0, yrow, 0, pol);    // f0 g0
    tma_load_3d(sb + T::OFF_XR, &mp.x, bar, xh, yrow, 2, pol);     // f1 f3 g1 g3
  }
  if (mrow >= 0) {
    tma_load_3d(sb + T::OFF_C4, &mp.c4, bar, x0, mrow, 6, pol);    // f2 g2 f4 g4
    tma_load_3d(sb + T::OFF_XM, &mp.x, bar, xh, mrow, 10, pol);    // f5..f8
  }
}

// x-interpolated values of one y-stencil row for the 8 populations with e_y != 0, as 4 pairs (islbm_tiled3.cuh: Pr):
//   0 (f2, f4)  1 (g2, g4)  2 (f5, f7)  3 (f8, f6)
// (lane a has e_y = +1 in pairs 0, 1, 2 and e_y = -1 in pair 3, which takes the swapped y-weights)
#define ISLBM_LOAD_M2(S)                                                            \
  do {                                                                              \
    S[0] = mkpr((AT)PC4(0)[0], (AT)PC4(2)[0]);         /* f2, f4 */                 \
    S[1] = mkpr((AT)PC4(1)[0], (AT)PC4(3)[0]);         /* g2, g4 */                 \
    S[2] = ptap3(PXM(0), PXM(2), 1, wxN);              /* f5 (+x,+y), f7 (-x,-y) */ \
    S[3] = ptap3(PXM(3), PXM(1), 1, wxN);              /* f8 (+x,-y), f6 (-x,+y) */ \
  } while (0)
// y-direction of the separable interpolation; (P0,P1,P2) = stencil rows in ascending y
#define ISLBM_YCOMB2(P0, P1, P2)                          \
  do {                                                    \
    const Pr<AT> q0 = pcomb3(wyN, P0[0], P1[0], P2[0]);   \
    const Pr<AT> q1 = pcomb3(wyN, P0[1], P1[1], P2[1]);   \
    const Pr<AT> q2 = pcomb3(wyN, P0[2], P1[2], P2[2]);   \
    const Pr<AT> q3 = pcomb3(wyS, P0[3], P1[3], P2[3]);   \
    f[2] = lane_a(q0); f[4] = lane_b(q0);                 \
    g[2] = lane_a(q1); g[4] = lane_b(q1);                 \
    f[5] = lane_a(q2); f[7] = lane_b(q2);                 \
    f[8] = lane_a(q3); f[6] = lane_b(q3);                 \
  } while (0)

template <typename ST, int TX, int STAGES, int MINB, int DIR>
__global__ void __launch_bounds__(TX, MINB)
k_step_ymarch(const __grid_constant__ Maps2 mp, DevMesh m, NodeParams np, const ST *__restrict__ src, ST *__restrict__ dst,
              int load_policy, int store_policy, int late_fill) {
  using T = Tile2<ST, TX, STAGES>;
  using AT = typename Acc<ST>::type;   // fp32 storage interpolates the stored deviations in fp32 (islbm_tiled3.cuh)
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *stage0 = smem_raw;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + T::BAR_OFF);
  uint64_t *empty = full + T::STAGES;
  AT *wys = reinterpret_cast<AT *>(smem_raw + T::W_OFF);
  int *claim = reinterpret_cast<int *>(smem_raw + T::BAR_OFF + 2 * T::STAGES * 8);   // refill generation per slot
  pdl_launch_dependents();

  const int x0 = blockIdx.x * T::TX;
  // the emitted rows are split evenly over the gridDim.y chunks (lengths differ by at most one, all <= kMaxChunk):
  // the first rows % chunks chunks are one row longer
  const int rows = m.em_hi - m.em_lo;
  // (32-bit arithmetic: a 64-bit division here cost every thread ~90 instructions per 3-4-row CTA)
  const int cbase = rows / (int)gridDim.y, crem = rows - cbase * (int)gridDim.y;
  const int y0 = m.em_lo + (int)blockIdx.y * cbase + min((int)blockIdx.y, crem);
  const int y1 = y0 + cbase + ((int)blockIdx.y < crem ? 1 : 0);
  const int yf = DIR > 0 ? y0 : y1 - 1;
  const int nstage = 2 + (y1 - y0);
  const bool b_lo = y0 == m.em_lo, b_hi = y1 == m.em_hi;   // slab boundary CTAs (fused exchange; islbm_tiled3.cuh)
  const bool any_peer = m.peer[0] != nullptr || m.peer[1] != nullptr;
  const uint64_t lpol = make_policy(load_policy);
  const uint64_t spol = make_policy(store_policy);
  // thread 0 sets up the ring and (unless late_fill) fills it BEFORE warps 1.. load the weight rows, so the two
  // latencies overlap;
  // griddepcontrol.wait comes before the first access to a population buffer (everything else reads only tables)
  if (threadIdx.x == 0) {
    for (int s = 0; s < T::STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], T::WARPS);
      claim[s] = 0;
    }
    fence_barrier_init();
    tma_prefetch_desc(&mp.c2);
    tma_prefetch_desc(&mp.c4);
    tma_prefetch_desc(&mp.x);
    if (!late_fill) {
      pdl_wait();
      if (b_lo) slab_wait_neighbour(m, 0);
      if (b_hi) slab_wait_neighbour(m, 1);
      for (int s = 0; s < T::STAGES && s < nstage; ++s) issue_stage2<T, DIR>(s, yf, m.ny, x0, stage0, full, empty, mp, lpol);
    }
  }
  for (int i = (int)threadIdx.x - 32; i >= 0 && i < 6 * (y1 - y0); i += T::TX - 32) {   // warps 1..: warp 0 is waiting above
    const int sk = i / (y1 - y0), yi = i - sk * (y1 - y0);
    stage_march_weight<0>(wys, sk, yi, __ldg(wrow(m, 1, sk / 3, sk % 3) + y0 + yi));
  }
  pdl_wait();
  __syncthreads();
  if (late_fill && threadIdx.x == 0) {
    if (b_lo) slab_wait_neighbour(m, 0);
    if (b_hi) slab_wait_neighbour(m, 1);
    for (int s = 0; s < T::STAGES && s < nstage; ++s) issue_stage2<T, DIR>(s, yf, m.ny, x0, stage0, full, empty, mp, lpol);
  }

  const int tx = threadIdx.x;
  const int x = x0 + tx;
  const bool valid = x < m.nx;
  WallFlags wf;
  wf.lo[0] = valid && x == 0;
  wf.hi[0] = valid && x == m.nx - 1;
  wf.lo[2] = wf.hi[2] = false;
  const bool wall_x = wf.lo[0] | wf.hi[0];
  const int sx = wf.lo[0] ? 1 : (wf.hi[0] ? -1 : 0);
  const int o_x = tx + T::XH - 1 + sx;
  Pr<AT> wxN[3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
    wxN[k] = mkpr(valid ? (AT)__ldg(wrow(m, 0, 1, k) + x) : (AT)0, valid ? (AT)__ldg(wrow(m, 0, 0, k) + x) : (AT)0);
  // the node's index in plane 0 at the chunk's first row; advanced by one row (DIR) per emitted row
  long long c = (long long)yf * m.nxp + x;

  // three register sets hold the y-stencil rows; `newest` names the one written last, so the marching order
  // (oldest first) is (newest+1, newest+2, newest) mod 3 and nothing is ever copied between sets
  Pr<AT> S0[4], S1[4], S2[4];
  int newest = 2;
  Pr<AT> *ssm = reinterpret_cast<Pr<AT> *>(smem_raw + T::S_OFF) + threadIdx.x;   // S_IN_SMEM: [slot][pair][thread]
  constexpr int SSLOT = 4 * T::TX;

#pragma unroll 1
  for (int s = 0; s < nstage; ++s) {
    const int st = s % T::STAGES;     // warp-uniform (uniform datapath)
    const uint32_t ph = (uint32_t)(s / T::STAGES) & 1u;
    const int y = yf + DIR * (s - 2);
    const bool has_emit = s >= 2;
    const bool has_mov = s <= 2 || sbase_moves(DIR > 0 ? y : y + 1, m.ny);
    const ST *sb = reinterpret_cast<const ST *>(stage0 + (size_t)st * T::STAGE_BYTES);
    const ST *sbc = sb + tx, *sbx = sb + o_x;
    constexpr int ES = (int)sizeof(ST);
#define PC2(k) (sbc + (T::OFF_C2 + (k) * T::P_C) / ES)
#define PXR(k) (sbx + (T::OFF_XR + (k) * T::P_X) / ES)
#define PC4(k) (sbc + (T::OFF_C4 + (k) * T::P_C) / ES)
#define PXM(k) (sbx + (T::OFF_XM + (k) * T::P_X) / ES)
    mbar_wait(&full[st], ph);

    if (has_mov) {
      newest = newest == 2 ? 0 : newest + 1;
      if constexpr (T::S_IN_SMEM) {
        ISLBM_LOAD_M2(S2);       // S2 = the newest row, in registers for this iteration and in its shared-memory slot
#pragma unroll
        for (int k = 0; k < 4; ++k) ssm[newest * SSLOT + k * T::TX] = S2[k];
      } else {
        if (newest == 0) ISLBM_LOAD_M2(S0);
        else if (newest == 1) ISLBM_LOAD_M2(S1);
        else ISLBM_LOAD_M2(S2);
      }
    }

    AT f[9], g[5];   // fp64, or fp32 deviations (fp32 storage)
    if (has_emit) {
      f[0] = PC2(0)[0];
      g[0] = PC2(1)[0];
      const Pr<AT> p1 = ptap3(PXR(0), PXR(1), 1, wxN);   // f1 (+x), f3 (-x)
      const Pr<AT> p2 = ptap3(PXR(2), PXR(3), 1, wxN);   // g1, g3
      f[1] = lane_a(p1); f[3] = lane_b(p1);
      g[1] = lane_a(p2); g[3] = lane_b(p2);
    }
    // hand the slot back; the warp whose release is the last one refills it at once with stage s + STAGES, so
    // STAGES - 1 stages are in flight whenever one is being consumed
    __syncwarp();
    if ((threadIdx.x & 31) == 0 && mbar_arrive_is_last(&empty[st]) && s + T::STAGES < nstage &&
        atomicCAS(&claim[st], s / T::STAGES, s / T::STAGES + 1) == s / T::STAGES)
      issue_stage2<T, DIR>(s + T::STAGES, yf, m.ny, x0, stage0, full, empty, mp, lpol);

    if (has_emit) {
      Pr<AT> wyN[3], wyS[3];
      load_march_weights<0>(wys, y - y0, wyN, wyS);
      // ascending-y order of the stencil rows: the marching order when DIR = +1, its reverse when DIR = -1
      if constexpr (T::S_IN_SMEM) {
        // marching order = slots (newest+1, newest+2, newest) mod 3; the newest row is still in registers unless the
        // stencil base did not move (first / last two rows of the mesh)
        const Pr<AT> *p0 = ssm + (newest == 2 ? 0 : newest + 1) * SSLOT, *p1 = ssm + (newest == 0 ? 2 : newest - 1) * SSLOT;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          S0[k] = p0[k * T::TX];
          S1[k] = p1[k * T::TX];
        }
        if (!has_mov) {
#pragma unroll
          for (int k = 0; k < 4; ++k) S2[k] = ssm[newest * SSLOT + k * T::TX];
        }
        if (DIR > 0) ISLBM_YCOMB2(S0, S1, S2);
        else ISLBM_YCOMB2(S2, S1, S0);
      } else if (DIR > 0) {
        if (newest == 0) ISLBM_YCOMB2(S1, S2, S0);
        else if (newest == 1) ISLBM_YCOMB2(S2, S0, S1);
        else ISLBM_YCOMB2(S0, S1, S2);
      } else {
        if (newest == 0) ISLBM_YCOMB2(S0, S2, S1);
        else if (newest == 1) ISLBM_YCOMB2(S1, S0, S2);
        else ISLBM_YCOMB2(S2, S1, S0);
      }
      wf.lo[1] = y == 0 && m.wall_mlo;
      wf.hi[1] = y == m.ny - 1 && m.wall_mhi;
      if (valid && (wall_x | wf.lo[1] | wf.hi[1])) wall_fix_node<2>(f, g, wf, src + c, m.nnp, m);
      constexpr bool DEV = Store<ST, 2>::kBiased;   // fp32 storage: collide the deviations as they are
      collide_node<DEV>(f, g, np);
      if (valid) {
        store_node<2, DEV>(dst + c, m.nnp, f, g, spol, std::make_integer_sequence<int, 14>{});
        if (any_peer) peer_store_node<2, ST, DEV>(m, y, x, f, g);   // slab boundary rows only
      }
      c += DIR * (long long)m.nxp;
    }
#undef PC2
#undef PXR
#undef PC4
#undef PXM
  }
  if ((b_lo && m.flag_out[0] != nullptr) || (b_hi && m.flag_out[1] != nullptr)) {   // CTA-uniform
    __syncthreads();
    if (threadIdx.x == 0) {
      if (b_lo) slab_publish(m, 0);
      if (b_hi) slab_publish(m, 1);
    }
  }
}

// ------------------------------ upwind stencil (islbm_set_stencil(h, 1)) ----------------------------------------
// Stage content for the A2-alternative stencil {j-2,j-1,j} / {j,j+1,j+2}: the e_y = +1 half of the y-stencil group
// (f2 g2 | f5 f6) trails the emitted row, the e_y = -1 half (f4 g4 | f7 f8) leads it by two rows.  Marches upwards.
template <typename T>
__device__ __forceinline__ void issue_stage2_up(int s, int yf, int ny, int x0, unsigned char *stage0, uint64_t *full,
                                                const Maps2 &mp, uint64_t pol) {
  const int st = s % T::STAGES;
  int prow = -1, mrow = -1, yrow = -1;
  if (s < 2) {
    prow = ubase_p(yf, ny) + s;
    mrow = ubase_m(yf, ny) + s;
  } else {
    yrow = yf + (s - 2);
    if (s == 2 || ubase_p_moves(yrow, ny)) prow = ubase_p(yrow, ny) + 2;
    if (s == 2 || ubase_m_moves(yrow, ny)) mrow = ubase_m(yrow, ny) + 2;
  }
  uint64_t *bar = &full[st];
  mbar_expect_tx(bar, (prow >= 0 ? T::F_BYTES : 0u) + (mrow >= 0 ? T::F_BYTES : 0u) + (yrow >= 0 ? T::Y_BYTES : 0u));
  unsigned char *sb = stage0 + (size_t)st * T::STAGE_BYTES;
  const int xh = x0 - T::XH;
  if (yrow >= 0) {
    tma_load_3d(sb + T::OFF_C2, &mp.c2, bar, x0, yrow, 0, pol);                    // f0 g0
    tma_load_3d(sb + T::OFF_XR, &mp.x, bar, xh, yrow, 2, pol);                     // f1 f3 g1 g3
  }
  if (prow >= 0) {
    tma_load_3d(sb + T::OFF_C4, &mp.c2, bar, x0, prow, 6, pol);                    // f2 g2
    tma_load_3d(sb + T::OFF_XM, &mp.x2, bar, xh, prow, 10, pol);                   // f5 f6
  }
  if (mrow >= 0) {
    tma_load_3d(sb + T::OFF_C4 + T::H_C, &mp.c2, bar, x0, mrow, 8, pol);           // f4 g4
    tma_load_3d(sb + T::OFF_XM + T::H_X, &mp.x2, bar, xh, mrow, 12, pol);          // f7 f8
  }
}

// family P (e_y = +1): (f2, g2) (f5, f6), rows {y-2, y-1, y}; family M (e_y = -1): (f4, g4) (f8, f7), rows {y, y+1, y+2};
// lane a of the x-interpolated pairs is the +x population (window starts two nodes upstream), lane b the -x one
#define ISLBM_LOAD_U2(S, H)                                                                                     \
  do {                                                                                                          \
    S[0] = mkpr((AT)PC4(2 * H)[tx], (AT)PC4(2 * H + 1)[tx]);                          /* f2 g2 | f4 g4 */        \
    S[1] = H == 0 ? ptap3(PXM(0) + o_xa, PXM(1) + o_xb, 1, wxN)                       /* f5 (+x), f6 (-x) */     \
                  : ptap3(PXM(3) + o_xa, PXM(2) + o_xb, 1, wxN);                      /* f8 (+x), f7 (-x) */     \
  } while (0)
#define ISLBM_YCOMB_U2(W, P0, P1, P2, F0, G0, F1A, F1B)   \
  do {                                                    \
    const Pr<AT> q0 = pcomb3(W, P0[0], P1[0], P2[0]);     \
    const Pr<AT> q1 = pcomb3(W, P0[1], P1[1], P2[1]);     \
    f[F0] = lane_a(q0);  g[G0] = lane_b(q0);              \
    f[F1A] = lane_a(q1); f[F1B] = lane_b(q1);             \
  } while (0)

template <typename ST, int TX, int STAGES, int MINB>
__global__ void __launch_bounds__(TX, MINB)
k_step_ymarch_up(const __grid_constant__ Maps2 mp, DevMesh m, NodeParams np, const ST *__restrict__ src, ST *__restrict__ dst,
                 int load_policy, int store_policy, int late_fill) {
  using T = Tile2<ST, TX, STAGES, 1>;
  using AT = typename Acc<ST>::type;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *stage0 = smem_raw;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + T::BAR_OFF);
  uint64_t *empty = full + T::STAGES;
  AT *wys = reinterpret_cast<AT *>(smem_raw + T::W_OFF);
  int *claim = reinterpret_cast<int *>(smem_raw + T::BAR_OFF + 2 * T::STAGES * 8);
  pdl_launch_dependents();

  const int x0 = blockIdx.x * T::TX;
  const int rows = m.em_hi - m.em_lo;
  // (32-bit arithmetic: a 64-bit division here cost every thread ~90 instructions per 3-4-row CTA)
  const int cbase = rows / (int)gridDim.y, crem = rows - cbase * (int)gridDim.y;
  const int y0 = m.em_lo + (int)blockIdx.y * cbase + min((int)blockIdx.y, crem);
  const int y1 = y0 + cbase + ((int)blockIdx.y < crem ? 1 : 0);
  const int nstage = 2 + (y1 - y0);
  const uint64_t lpol = make_policy(load_policy);
  const uint64_t spol = make_policy(store_policy);
  if (threadIdx.x == 0) {
    for (int s = 0; s < T::STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], T::WARPS);
      claim[s] = 0;
    }
    fence_barrier_init();
    tma_prefetch_desc(&mp.c2);
    tma_prefetch_desc(&mp.x);
    tma_prefetch_desc(&mp.x2);
    if (!late_fill) {
      pdl_wait();
      for (int s = 0; s < T::STAGES && s < nstage; ++s) issue_stage2_up<T>(s, y0, m.ny, x0, stage0, full, mp, lpol);
    }
  }
  for (int i = (int)threadIdx.x - 32; i >= 0 && i < 6 * (y1 - y0); i += T::TX - 32) {
    const int sk = i / (y1 - y0), yi = i - sk * (y1 - y0);
    stage_march_weight<1>(wys, sk, yi, __ldg(wrow(m, 1, sk / 3, sk % 3) + y0 + yi));
  }
  pdl_wait();
  __syncthreads();
  if (late_fill && threadIdx.x == 0) {
    for (int s = 0; s < T::STAGES && s < nstage; ++s) issue_stage2_up<T>(s, y0, m.ny, x0, stage0, full, mp, lpol);
  }

  const int tx = threadIdx.x;
  const int x = x0 + tx;
  const bool valid = x < m.nx;
  WallFlags wf;
  wf.lo[0] = valid && x == 0;
  wf.hi[0] = valid && x == m.nx - 1;
  wf.lo[2] = wf.hi[2] = false;
  const bool wall_x = wf.lo[0] | wf.hi[0];
  const int o_xa = ubase_p(min(x, m.nx - 1), m.nx) - x0 + T::XH, o_xb = ubase_m(min(x, m.nx - 1), m.nx) - x0 + T::XH;
  Pr<AT> wxN[3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
    wxN[k] = mkpr(valid ? (AT)__ldg(wrow(m, 0, 1, k) + x) : (AT)0, valid ? (AT)__ldg(wrow(m, 0, 0, k) + x) : (AT)0);
  long long c = (long long)y0 * m.nxp + x;

  Pr<AT> P0[2], P1[2], P2[2], M0[2], M1[2], M2[2];
  int newest_p = 2, newest_m = 2;
  Pr<AT> *ssm = reinterpret_cast<Pr<AT> *>(smem_raw + T::S_OFF) + threadIdx.x;   // S_IN_SMEM: [family][slot][pair][thread]
  constexpr int SSLOT = 2 * T::TX;

#pragma unroll 1
  for (int s = 0; s < nstage; ++s) {
    const int st = s % T::STAGES;
    const uint32_t ph = (uint32_t)(s / T::STAGES) & 1u;
    const int y = y0 + (s - 2);
    const bool has_emit = s >= 2;
    const bool mov_p = s <= 2 || ubase_p_moves(y, m.ny), mov_m = s <= 2 || ubase_m_moves(y, m.ny);
    const ST *sb = reinterpret_cast<const ST *>(stage0 + (size_t)st * T::STAGE_BYTES);
    constexpr int ES = (int)sizeof(ST);
#define PC2(k) (sb + (T::OFF_C2 + (k) * T::P_C) / ES)
#define PXR(k) (sb + (T::OFF_XR + (k) * T::P_X) / ES)
#define PC4(k) (sb + T::moff(T::OFF_C4, k, T::P_C, T::H_C) / ES)
#define PXM(k) (sb + T::moff(T::OFF_XM, k, T::P_X, T::H_X) / ES)
    mbar_wait(&full[st], ph);

    if (mov_p) {
      newest_p = newest_p == 2 ? 0 : newest_p + 1;
      if constexpr (T::S_IN_SMEM) {
        ISLBM_LOAD_U2(P2, 0);
#pragma unroll
        for (int k = 0; k < 2; ++k) ssm[newest_p * SSLOT + k * T::TX] = P2[k];
      } else {
        if (newest_p == 0) ISLBM_LOAD_U2(P0, 0);
        else if (newest_p == 1) ISLBM_LOAD_U2(P1, 0);
        else ISLBM_LOAD_U2(P2, 0);
      }
    }
    if (mov_m) {
      newest_m = newest_m == 2 ? 0 : newest_m + 1;
      if constexpr (T::S_IN_SMEM) {
        ISLBM_LOAD_U2(M2, 1);
#pragma unroll
        for (int k = 0; k < 2; ++k) ssm[(3 + newest_m) * SSLOT + k * T::TX] = M2[k];
      } else {
        if (newest_m == 0) ISLBM_LOAD_U2(M0, 1);
        else if (newest_m == 1) ISLBM_LOAD_U2(M1, 1);
        else ISLBM_LOAD_U2(M2, 1);
      }
    }

    AT f[9], g[5];
    if (has_emit) {
      f[0] = PC2(0)[tx];
      g[0] = PC2(1)[tx];
      const Pr<AT> p1 = ptap3(PXR(0) + o_xa, PXR(1) + o_xb, 1, wxN);   // f1 (+x), f3 (-x)
      const Pr<AT> p2 = ptap3(PXR(2) + o_xa, PXR(3) + o_xb, 1, wxN);   // g1, g3
      f[1] = lane_a(p1); f[3] = lane_b(p1);
      g[1] = lane_a(p2); g[3] = lane_b(p2);
    }
    __syncwarp();
    if ((threadIdx.x & 31) == 0 && mbar_arrive_is_last(&empty[st]) && s + T::STAGES < nstage &&
        atomicCAS(&claim[st], s / T::STAGES, s / T::STAGES + 1) == s / T::STAGES)
      issue_stage2_up<T>(s + T::STAGES, y0, m.ny, x0, stage0, full, mp, lpol);

    if (has_emit) {
      Pr<AT> wyA[3], wyB[3];    // (c=+1, c=+1) for family P, (c=-1, c=-1) for family M
      load_march_weights<1>(wys, y - y0, wyA, wyB);
      if constexpr (T::S_IN_SMEM) {
        const Pr<AT> *pp0 = ssm + (newest_p == 2 ? 0 : newest_p + 1) * SSLOT, *pp1 = ssm + (newest_p == 0 ? 2 : newest_p - 1) * SSLOT;
        const Pr<AT> *pm0 = ssm + (3 + (newest_m == 2 ? 0 : newest_m + 1)) * SSLOT, *pm1 = ssm + (3 + (newest_m == 0 ? 2 : newest_m - 1)) * SSLOT;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          P0[k] = pp0[k * T::TX];
          P1[k] = pp1[k * T::TX];
          M0[k] = pm0[k * T::TX];
          M1[k] = pm1[k * T::TX];
        }
        if (!mov_p) {
#pragma unroll
          for (int k = 0; k < 2; ++k) P2[k] = ssm[newest_p * SSLOT + k * T::TX];
        }
        if (!mov_m) {
#pragma unroll
          for (int k = 0; k < 2; ++k) M2[k] = ssm[(3 + newest_m) * SSLOT + k * T::TX];
        }
        ISLBM_YCOMB_U2(wyA, P0, P1, P2, 2, 2, 5, 6);
        ISLBM_YCOMB_U2(wyB, M0, M1, M2, 4, 4, 8, 7);
      } else {
        if (newest_p == 0) ISLBM_YCOMB_U2(wyA, P1, P2, P0, 2, 2, 5, 6);
        else if (newest_p == 1) ISLBM_YCOMB_U2(wyA, P2, P0, P1, 2, 2, 5, 6);
        else ISLBM_YCOMB_U2(wyA, P0, P1, P2, 2, 2, 5, 6);
        if (newest_m == 0) ISLBM_YCOMB_U2(wyB, M1, M2, M0, 4, 4, 8, 7);
        else if (newest_m == 1) ISLBM_YCOMB_U2(wyB, M2, M0, M1, 4, 4, 8, 7);
        else ISLBM_YCOMB_U2(wyB, M0, M1, M2, 4, 4, 8, 7);
      }
      wf.lo[1] = y == 0 && m.wall_mlo;
      wf.hi[1] = y == m.ny - 1 && m.wall_mhi;
      if (valid && (wall_x | wf.lo[1] | wf.hi[1])) wall_fix_node<2>(f, g, wf, src + c, m.nnp, m);
      constexpr bool DEV = Store<ST, 2>::kBiased;
      collide_node<DEV>(f, g, np);
      if (valid) store_node<2, DEV>(dst + c, m.nnp, f, g, spol, std::make_integer_sequence<int, 14>{});
      c += m.nxp;
    }
#undef PC2
#undef PXR
#undef PC4
#undef PXM
  }
}

// ------------------------------ host side ---------------------------------
struct Plan2 {
  bool available = false;
  Maps2 maps[2];
  int tx = 128;
  int stages = 3;
  int per_wave = 1;      // chunks per strip in one wave of resident CTAs
  int sk = 0;            // stencil kind the plan was built for: 0 central, 1 upwind (always Cfg2c, marches upwards)
  char why_not[96] = "";
};

// the two instantiated strip widths: (TX, STAGES, min CTAs/SM)
// fp32 storage: five CTAs per SM (96 registers, 16 B spilled) measure 1-3 % above four; six (80 registers) lose 5 %
// 128-wide strip, 3-stage ring: four CTAs per SM in fp64 (128 registers, 47 KB each), five with fp32 storage
template <typename ST> struct Cfg2a { using T = Tile2<ST, 128, 3>; static constexpr int MINB = sizeof(ST) == 4 ? ISLBM_F32_CTAS2D : 4; };
// 128-wide strip, fp64 only: 4-stage ring, three CTAs per SM (62 KB each): three rows in flight per CTA instead of two.
// fp32 storage keeps the 3-stage ring (its stages are half as large; 4 and 5 stages measured 4-10 % slower).
template <typename ST> struct Cfg2c {
  using T = Tile2<ST, 128, sizeof(ST) == 4 ? 3 : 4>;
  static constexpr int MINB = sizeof(ST) == 4 ? ISLBM_F32_CTAS2D : 3;
};
template <typename ST> struct Cfg2b { using T = Tile2<ST, 224, 3>; static constexpr int MINB = 2; };

template <typename ST, typename CFG, int SK = 0>
inline bool plan2_setup(Plan2 &p, const int *n, int nxp, void *buf0, void *buf1, const Tuning &tn) {
  using T = typename CFG::T;
  auto kern = k_step_ymarch<ST, T::TX, T::STAGES, CFG::MINB, 1>;
  auto kern_dn = k_step_ymarch<ST, T::TX, T::STAGES, CFG::MINB, -1>;
  void *bufs[2] = {buf0, buf1};
  const long long dims[3] = {n[0], n[1], 14};
  const int b_c2[3] = {T::TX, 1, 2}, b_c4[3] = {T::TX, 1, 4}, b_x[3] = {T::HX, 1, 4}, b_x2[3] = {T::HX, 1, 2};
  for (int i = 0; i < 2; ++i)
    if (!make_map(&p.maps[i].c2, bufs[i], (int)sizeof(ST), 3, dims, b_c2, tn.l2promo, nxp) ||
        !make_map(&p.maps[i].c4, bufs[i], (int)sizeof(ST), 3, dims, b_c4, tn.l2promo, nxp) ||
        !make_map(&p.maps[i].x, bufs[i], (int)sizeof(ST), 3, dims, b_x, tn.l2promo, nxp) ||
        !make_map(&p.maps[i].x2, bufs[i], (int)sizeof(ST), 3, dims, b_x2, tn.l2promo, nxp))
      return false;
  using TU = Tile2<ST, T::TX, T::STAGES, 1>;   // the upwind kernel's stage layout (padded halves)
  if constexpr (SK == 1) {
    if (cudaFuncSetAttribute(k_step_ymarch_up<ST, T::TX, T::STAGES, CFG::MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)TU::SMEM_BYTES) != cudaSuccess) {
      cudaGetLastError();
      return false;
    }
  } else if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM_BYTES) != cudaSuccess ||
             cudaFuncSetAttribute(kern_dn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM_BYTES) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  int occ = 1, dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const cudaError_t eo = SK == 1 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_step_ymarch_up<ST, T::TX, T::STAGES, CFG::MINB>, T::TX, TU::SMEM_BYTES)
                                 : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, T::TX, T::SMEM_BYTES);
  if (eo != cudaSuccess || occ < 1) {
    cudaGetLastError();
    occ = 1;
  }
  const int strips = (n[0] + T::TX - 1) / T::TX;
  p.per_wave = (sms * occ) / strips;
  if (p.per_wave < 1) p.per_wave = 1;
  p.tx = T::TX;
  p.stages = T::STAGES;
  return true;
}

template <typename ST>
inline bool plan2_create(Plan2 &p, const int *n, int nxp, void *buf0, void *buf1, const Tuning &tn, int sk) {
  p.available = false;
  p.sk = sk;
  auto no = [&](const char *why) { snprintf(p.why_not, sizeof p.why_not, "%s", why); return false; };
  if (n[0] < 3 || n[1] < 3) return no("tiled kernel: n >= 3");
  if ((nxp * (int)sizeof(ST)) % 16) return no("tiled kernel: TMA needs a 16-byte row pitch");
  int dev = 0, cc_major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return no("no device");
  cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev);
  if (cc_major < 10) return no("tiled kernel: needs sm_100");
  const int tx = tn.tx2d ? tn.tx2d : 128;   // a TMA box is at most 256 elements wide: TX + 2*XH <= 256
  // ring depth (measured, profiles/r1_c3_1024sq_ymarch_v5.md): fp64 takes 4 stages x 3 CTAs per SM (512^2 +4 %,
  // 1024^2 +1 %, 1538^2..8193^2 +0.3-2.3 %, 255^2 +20 %; 1026^2/1282^2 -1-2 %, inside the run-to-run spread)
  const int ring = tn.ring2d ? tn.ring2d : 4;
  const bool ok = sk ? plan2_setup<ST, Cfg2c<ST>, 1>(p, n, nxp, buf0, buf1, tn)
                     : (tx == 224 ? plan2_setup<ST, Cfg2b<ST>>(p, n, nxp, buf0, buf1, tn)
                                  : (ring == 4 ? plan2_setup<ST, Cfg2c<ST>>(p, n, nxp, buf0, buf1, tn)
                                               : plan2_setup<ST, Cfg2a<ST>>(p, n, nxp, buf0, buf1, tn)));
  if (!ok) return no("tiled kernel: tensor map / attribute setup failed");
  p.available = true;
  return true;
}

// Number of chunks a strip of `rows` emitted rows is cut into (measured, profiles/): short chunks win (4 rows:
// 0.96-0.97 at 2049^2..8193^2, 8 rows: 0.88-0.93, 60 rows: 0.73-0.87; the doubled prologue rows are found in L2), and
// the CTA count should be a whole number of waves of resident CTAs.  So: one wave if its chunks are at most
// max_single rows (8 with the 3-stage ring, 12 with the 4-stage one; small and medium meshes, down to 1 row), else
// k waves, k the smallest number for which a chunk is at most max_multi = 4 rows.
inline int chunks2(int rows, int per_wave, int forced_chunk, int max_single = 8, int max_multi = 4) {
  int nc;
  if (forced_chunk > 0) {
    nc = (rows + forced_chunk - 1) / forced_chunk;
  } else {
    nc = per_wave;
    if ((rows + nc - 1) / nc > max_single) nc = per_wave * ((rows + max_multi * per_wave - 1) / (max_multi * per_wave));
    if (nc > rows) nc = rows;   // down to ONE row per CTA on tiny meshes: a CTA costs ~2 us + 1.1 us per row (64^2: 4.05 -> 3.08 us per step)
  }
  const int least = (rows + kMaxChunk - 1) / kMaxChunk;
  if (nc < least) nc = least;
  return nc < 1 ? 1 : nc;
}

template <typename ST, typename CFG>
inline void launch2_cfg(const Plan2 &p, const int *n, const DevMesh &m, const NodeParams &np, int cur, void *const *buf,
                        const Tuning &tn, cudaStream_t stream) {
  using T = typename CFG::T;
  const int rows = m.em_hi - m.em_lo;
  // with three rows in flight per CTA a single wave pays up to 12-row chunks (642^2: 0.75 -> 0.82)
  const int nc = chunks2(rows, p.per_wave, tn.chunk, tn.rows2d1 ? tn.rows2d1 : (p.stages >= 4 ? 12 : 8),
                         tn.rows2d ? tn.rows2d : (sizeof(ST) == 4 ? 8 : 4));   // fp32 storage: 8 (1024^2 0.637 -> 0.672, 4096^2 0.71 -> 0.75)
  dim3 grid((n[0] + T::TX - 1) / T::TX, nc, 1);
  // first ring fill (measured, profiles/r1_c3_1024sq_ymarch_v4.md): a single-wave launch is 2-5 % faster with the
  // fill after the CTA barrier, a multi-wave launch 2-6 % faster with the fill first
  const int late = tn.fill ? (tn.fill == 2) : (nc <= p.per_wave);
  DevMesh mm = m;
  mm.bctas = (int)grid.x;   // CTAs that touch one boundary row of a slab
  if (p.sk)
    launch_step(k_step_ymarch_up<ST, T::TX, T::STAGES, CFG::MINB>, grid, dim3(T::TX), Tile2<ST, T::TX, T::STAGES, 1>::SMEM_BYTES, stream, tn.pdl != 0,
                p.maps[cur], m, np, (const ST *)buf[cur], (ST *)buf[1 - cur], tn.load_policy, tn.store_policy, late);
  else if (tn.serpentine && cur)
    launch_step(k_step_ymarch<ST, T::TX, T::STAGES, CFG::MINB, -1>, grid, dim3(T::TX), T::SMEM_BYTES, stream, tn.pdl != 0,
                p.maps[cur], mm, np, (const ST *)buf[cur], (ST *)buf[1 - cur], tn.load_policy, tn.store_policy, late);
  else
    launch_step(k_step_ymarch<ST, T::TX, T::STAGES, CFG::MINB, 1>, grid, dim3(T::TX), T::SMEM_BYTES, stream, tn.pdl != 0,
                p.maps[cur], mm, np, (const ST *)buf[cur], (ST *)buf[1 - cur], tn.load_policy, tn.store_policy, late);
}

template <typename ST>
inline cudaError_t launch2(const Plan2 &p, const int *n, const DevMesh &m, const NodeParams &np, int cur, void *const *buf,
                           const Tuning &tn, cudaStream_t stream) {
  if (p.sk) launch2_cfg<ST, Cfg2c<ST>>(p, n, m, np, cur, buf, tn, stream);
  else if (p.tx == 224) launch2_cfg<ST, Cfg2b<ST>>(p, n, m, np, cur, buf, tn, stream);
  else if (p.stages == Cfg2c<ST>::T::STAGES && p.stages != Cfg2a<ST>::T::STAGES) launch2_cfg<ST, Cfg2c<ST>>(p, n, m, np, cur, buf, tn, stream);
  else launch2_cfg<ST, Cfg2a<ST>>(p, n, m, np, cur, buf, tn, stream);
  return cudaPeekAtLastError();
}

}  // namespace islbmk
