// islbm_uniform.cuh — the uniform-mesh counterpart of the ISLBM step: when every
// spacing equals the lattice unit the departure point x - e*delta is the
// neighbouring node itself, the Lagrange weights are exactly (1,0,0)/(0,0,1)
// (A3, A21) and Eq. 18/20 reduce to a pure shift.
// This is the kernel the paper's "uniform" runs correspond to:
// fused pull-stream + walls (Eq. 21-23) + collide, one thread per node, every
// population read once (26 / 14 independent coalesced loads in flight per
// thread) and written once; no shared memory, no weights.
#pragma once

#include "islbm_kernels.cuh"

namespace islbmk {

template <int DIM, int Q, typename ST>
__device__ __forceinline__ double shift_f(const DevMesh &m, const ST *__restrict__ src, const NodeCtx<DIM> &cx) {
  constexpr int EX = evel<DIM>(Q, 0), EY = evel<DIM>(Q, 1), EZ = evel<DIM>(Q, 2);
  if (crosses<DIM, EX, EY, EZ>(cx)) return ldv(src + (long long)plane_f<DIM>(opposite<DIM>(Q)) * m.nnp + cx.c);
  const long long off = (long long)EX + (long long)EY * m.nxp + (long long)EZ * m.nxp * m.ny;
  return ldv(src + (long long)plane_f<DIM>(Q) * m.nnp + cx.c - off);
}

template <int DIM, int Q, typename ST>
__device__ __forceinline__ double shift_g(const DevMesh &m, const ST *__restrict__ src, const NodeCtx<DIM> &cx) {
  constexpr int EX = evel<DIM>(Q, 0), EY = evel<DIM>(Q, 1), EZ = evel<DIM>(Q, 2);
  if (crosses<DIM, EX, EY, EZ>(cx)) {
    const double gb = ldv(src + (long long)plane_g<DIM>(opposite<DIM>(Q)) * m.nnp + cx.c);
    if (EX != 0) return -gb + m.omega_bc * (cx.lo[0] ? m.T_hot : m.T_cold);   // Eq. 22
    return gb;                                                                // Eq. 23
  }
  const long long off = (long long)EX + (long long)EY * m.nxp + (long long)EZ * m.nxp * m.ny;
  return ldv(src + (long long)plane_g<DIM>(Q) * m.nnp + cx.c - off);
}

template <int DIM, typename ST, int... Qs>
__device__ __forceinline__ void shift_all_f(const DevMesh &m, const ST *src, const NodeCtx<DIM> &cx, double *f,
                                            std::integer_sequence<int, Qs...>) {
  ((f[Qs] = shift_f<DIM, Qs>(m, src, cx)), ...);
}
template <int DIM, typename ST, int... Qs>
__device__ __forceinline__ void shift_all_g(const DevMesh &m, const ST *src, const NodeCtx<DIM> &cx, double *g,
                                            std::integer_sequence<int, Qs...>) {
  ((g[Qs] = shift_g<DIM, Qs>(m, src, cx)), ...);
}

template <int DIM, typename ST>
__global__ void __launch_bounds__(256, 2)
k_step_shift(DevMesh m, NodeParams np, const ST *__restrict__ src, ST *__restrict__ dst) {
  constexpr int QF = Lat<DIM>::QF, QG = Lat<DIM>::QG;
  const int ix = blockIdx.x * blockDim.x + threadIdx.x;
  const int iy = blockIdx.y * blockDim.y + threadIdx.y;
  const int iz = blockIdx.z * blockDim.z + threadIdx.z;
  if (ix >= m.nx || iy >= m.ny || iz >= m.nz) return;
  NodeCtx<DIM> cx;
  cx.i[0] = ix; cx.i[1] = iy; cx.i[2] = iz;
  cx.c = ((long long)iz * m.ny + iy) * m.nxp + ix;
  cx.lo[0] = ix == 0; cx.hi[0] = ix == m.nx - 1;
  cx.lo[1] = iy == 0 && (DIM == 3 || m.wall_mlo); cx.hi[1] = iy == m.ny - 1 && (DIM == 3 || m.wall_mhi);
  cx.lo[2] = DIM == 3 && iz == 0 && m.wall_mlo; cx.hi[2] = DIM == 3 && iz == m.nz - 1 && m.wall_mhi;
  if ((DIM == 3 ? iz : iy) < m.em_lo || (DIM == 3 ? iz : iy) >= m.em_hi) return;   // ghost layer: read, not updated
  double f[QF], g[QG];
  shift_all_f<DIM>(m, src, cx, f, std::make_integer_sequence<int, QF>{});
  shift_all_g<DIM>(m, src, cx, g, std::make_integer_sequence<int, QG>{});
  add_bias<ST, DIM>(f);
  collide_node(f, g, np);
#pragma unroll
  for (int q = 0; q < QF; ++q) dst[(long long)plane_f<DIM>(q) * m.nnp + cx.c] = to_storage<ST, DIM>(f[q], q);
#pragma unroll
  for (int q = 0; q < QG; ++q) dst[(long long)plane_g<DIM>(q) * m.nnp + cx.c] = (ST)g[q];
}

}  // namespace islbmk
