// islbm_reduce.cuh — Nusselt / Reynolds reductions and the steady-state
// residual.  Two passes with a fixed partition and a fixed summation order
// (warp shuffles, then one partial per block, then one block), so results are
// deterministic run to run.
//
// Nu_hot, Nu_cold: Eq. 32 / Eq. 41 with the one-sided wall
// derivative of Eq. 28 and the weighted average of Eq. 29
// normalised by the effective lengths;
// <Re>: Eq. 34 / Eq. 42 with the full speed (A10); <Nu>: Eq. 31 / 40.
#pragma once

#include "islbm_kernels.cuh"

namespace islbmk {

constexpr int kRedSlots = 7;
constexpr int kRedThreads = 256;

struct DiagParams {
  double q_lo, q_hi;   // (x1-x0)/delta, (x_{n-1}-x_{n-2})/delta for Eq. 28
  double T0;
  // Eq. 33 (A23): the two node columns mid_i, mid_i+1 that bracket x* = 0.5, their linear-interpolation
  // weights, and the 3-point derivative coefficients (lattice units) at each of them
  int mid_i;
  double mid_a[2];
  double mid_c[2][3];
};

// Eq. 28, bottom-wall form with Delta = 1 l.u.
__device__ __forceinline__ double wall_derivative(double q, double phi_wall, double phi1, double phi2) {
  const double a = 2.0 * q + 1.0;
  return (-4.0 * q * (q + 1.0) * phi_wall + a * a * phi1 - phi2) / (q * a);
}

__device__ __forceinline__ void block_reduce_store(double (&acc)[kRedSlots], double *__restrict__ partial) {
  __shared__ double sh[kRedSlots][kRedThreads / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int s = 0; s < kRedSlots; ++s) {
    double v = acc[s];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) sh[s][wid] = v;
  }
  __syncthreads();
  if (threadIdx.x < kRedSlots) {
    double v = 0.0;
#pragma unroll
    for (int k = 0; k < kRedThreads / 32; ++k) v += sh[threadIdx.x][k];
    partial[(long long)blockIdx.x * kRedSlots + threadIdx.x] = v;
  }
}

template <int DIM, typename ST>
__device__ __forceinline__ double node_temperature(const DevMesh &m, const ST *__restrict__ S, long long c) {
  constexpr int QG = Lat<DIM>::QG;
  double g[QG];
#pragma unroll
  for (int q = 0; q < QG; ++q) g[q] = ldv(S + (long long)plane_g<DIM>(q) * m.nnp + c);
  if constexpr (DIM == 2) return g[0] + g[1] + g[2] + g[3] + g[4];
  else return g[0] + ((g[1] + g[2]) + (g[3] + g[4]) + (g[5] + g[6]));
}

// pass 1: per-block partial sums of
//   [0] wa*dT/dx|hot  [1] wa*dT/dx|cold  [2] wv*|u|  [3] wv*|u|^2  [4] wv*u*(T-T0)
//   [5] wa*a_k*u*(T-T0) and [6] wa*a_k*dT/dx on the two columns bracketing the centre plane (Eq. 33)
template <int DIM, typename ST>
__global__ void __launch_bounds__(kRedThreads)
k_nusselt_partial(DevMesh m, NodeParams np, DiagParams dp, const ST *__restrict__ S, double *__restrict__ partial) {
  double acc[kRedSlots] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  const long long stride = (long long)gridDim.x * kRedThreads;
  for (long long c = (long long)blockIdx.x * kRedThreads + threadIdx.x; c < m.nn; c += stride) {
    const int ix = (int)(c % m.nx);
    const long long r = c / m.nx;
    const int iy = (int)(r % m.ny), iz = (int)(r / m.ny);
    double f[Lat<DIM>::QF], g[Lat<DIM>::QG];
    const long long cs = (long long)r * m.nxp + ix;
    load_post_node<DIM>(m, S, cs, f, g);
    double rho, u, v, w, T;
    fields_from_post(f, g, np, rho, u, v, w, T);
    const double wa = __ldg(m.avgw + m.npad + iy) * (DIM == 3 ? __ldg(m.avgw + 2 * m.npad + iz) : 1.0);
    const double wv = wa * __ldg(m.avgw + ix);
    const double sp2 = u * u + v * v + w * w;
    acc[2] += wv * sqrt(sp2);
    acc[3] += wv * sp2;
    acc[4] += wv * u * (T - dp.T0);
    if (ix == 0) {
      const double T1 = node_temperature<DIM>(m, S, cs + 1);
      acc[0] += wa * wall_derivative(dp.q_lo, m.T_hot, T, T1);
    }
    if (ix == m.nx - 1) {
      const double T1 = node_temperature<DIM>(m, S, cs - 1);
      acc[1] += wa * (-wall_derivative(dp.q_hi, m.T_cold, T, T1));
    }
    const int km = ix - dp.mid_i;
    if ((km == 0 || km == 1) && dp.mid_a[km] != 0.0) {
      const double Tm = node_temperature<DIM>(m, S, cs - 1), Tp = node_temperature<DIM>(m, S, cs + 1);
      const double dTdx = dp.mid_c[km][0] * Tm + dp.mid_c[km][1] * T + dp.mid_c[km][2] * Tp;
      acc[5] += wa * dp.mid_a[km] * (u * (T - dp.T0));
      acc[6] += wa * dp.mid_a[km] * dTdx;
    }
  }
  block_reduce_store(acc, partial);
}

// pass 2: one block, fixed order
__global__ void __launch_bounds__(kRedThreads)
k_reduce_final(const double *__restrict__ partial, int nblocks, double *__restrict__ out) {
  double acc[kRedSlots] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  for (int b = threadIdx.x; b < nblocks; b += kRedThreads)
#pragma unroll
    for (int s = 0; s < kRedSlots; ++s) acc[s] += partial[(long long)b * kRedSlots + s];
  block_reduce_store(acc, out);   // blockIdx.x == 0 -> out[0..4]
}

// Eq. 30: partial sums of |u-u_prev|_2, |u_prev|_2, |T-T_prev|, |T_prev|;
// the snapshot [u,v,w,T][nn] is overwritten with the current fields.
template <int DIM, typename ST>
__global__ void __launch_bounds__(kRedThreads)
k_residual_partial(DevMesh m, NodeParams np, const ST *__restrict__ S, double *__restrict__ snap,
                   double *__restrict__ partial) {
  double acc[kRedSlots] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  const long long stride = (long long)gridDim.x * kRedThreads;
  for (long long c = (long long)blockIdx.x * kRedThreads + threadIdx.x; c < m.nn; c += stride) {
    {   // ghost layers of a slab are not part of this rank's sums (their snapshot entries stay zero)
      const long long layer = c / ((long long)m.nx * (DIM == 3 ? m.ny : 1));
      if (layer < m.em_lo || layer >= m.em_hi) continue;
    }
    double f[Lat<DIM>::QF], g[Lat<DIM>::QG];
    load_post_node<DIM>(m, S, sidx(m, c), f, g);
    double rho, u, v, w, T;
    fields_from_post(f, g, np, rho, u, v, w, T);
    const double pu = snap[c], pv = snap[m.nn + c], pw = snap[2 * m.nn + c], pT = snap[3 * m.nn + c];
    const double du = u - pu, dv = v - pv, dw = w - pw;
    acc[0] += sqrt(du * du + dv * dv + dw * dw);
    acc[1] += sqrt(pu * pu + pv * pv + pw * pw);
    acc[2] += fabs(T - pT);
    acc[3] += fabs(pT);
    snap[c] = u; snap[m.nn + c] = v; snap[2 * m.nn + c] = w; snap[3 * m.nn + c] = T;
  }
  block_reduce_store(acc, partial);
}

}  // namespace islbmk
