// islbm_lattice.cuh — node-local arithmetic of the ISLBM step for sm_100a.
//
// Hand-factored MRT collisions (no dense M / M^-1 products): the moments of
// Eq. 10/11 and Eq. 15/16 are formed from symmetric /
// antisymmetric partial sums of the populations, relaxed per Eq. 17 / Eq. 19
// with the Guo forcing moments of Eq. 12/13 (PAPER.md:100-
// 104; last entry of Eq. 12 read as u*Fy + v*Fx, A8), and mapped back
// with M^-1 = M^T diag(1/|row|^2) (rows are mutually orthogonal).  The body
// force is F = rho*g*beta*(T - T0)*y^ (T0: DESIGN.md A9), so Fx = Fz = 0
// is folded in.  Relaxation rates: DESIGN.md A7.
//
// Direction ordering: include/islbm.h.  Everything here is fp64.
#pragma once

#include <cmath>

#ifndef ISLBM_HD
#ifdef __CUDACC__
#define ISLBM_HD __host__ __device__ __forceinline__
#else
#define ISLBM_HD inline
#endif
#endif

namespace islbmk {

struct NodeParams {
  double gbeta;   // g*beta in lattice units, times the buoyancy test scale
  double s_nu;    // 1/tau_f         (e, eps, stress moments)
  double s_q;     // 8(2tau-1)/(8tau-1)  (heat-flux-like and third-order moments)
  double hs_nu;   // 1 - s_nu/2
  double hs_q;    // 1 - s_q/2
  double q_k;     // 3 - sqrt(3)     (temperature flux moments)
  double q_e;     // 4 sqrt(3) - 6   (remaining temperature moments)
  double a_T;     // Eq. 15/16
  double T0;      // reference temperature of the buoyancy force
  // relaxation rate x 1/|moment row|^2 (x the forcing factor), folded once on the host by fold_node_params: the
  // kernels read them as constant-bank operands, so Delta m_k / |row_k|^2 is one multiply and one fused multiply-add
  double k[21];
  // the same temperature constants in fp32, for the fp32-storage kernels, which collide the temperature populations in
  // fp32 (ISLBM_G_FP32): kf[0] = -q_k/2, kf[1] = -q_e/20 | -q_e/42, kf[2] = -q_e/12 (3-D), kf[3] = -q_e/4, kf[4] = a_T
  float kf[5];
  // fp32 copies for the all-fp32 3-D collision of the fp32-storage kernels (ISLBM_F_FP32_3D): kq[i] = k[i] for the 17
  // flow constants, kq[17] = gbeta, kq[18] = T0
  float kq[19];
};

// fp32-storage kernels: collide the temperature populations g in fp32 (they are stored in fp32 and T tolerates it:
// BASELINE.json asks 1e-5 on T after 1000 steps, the fp64 collision gives 7e-7, this one the same order; the flow
// populations keep the fp64 collision, whose error on u sits at 4-6e-6 of the same bar).  Saves 14 of the 54
// conversions and 50 of the 293 fp64 instructions per node of the latency-bound fp32-storage step.
#ifndef ISLBM_G_FP32
#define ISLBM_G_FP32 1
#endif
// fp32-storage 3-D kernels: the flow populations (deviations f - w) are collided in fp32 as well, so no fp64
// instruction and no conversion is left in the step: 134 -> 120 registers, which lets 16 instead of 12 warps share an
// SM (256^3 sustained 832 -> 712 us, 0.64 -> 0.75 of the roofline; profiles/attempts.md).  Every parity bar holds as
// it stood (3 steps from a far-from-equilibrium state within 2e-6 of the plane maximum, 1000 steps of
// config 4 / 5 within 1e-5 on u, v, w, T).  The 2-D kernels keep the fp64 flow collision: there the same change
// fails the 3-step bar (6-7e-6).  -DISLBM_F_FP32_3D=0 restores the fp64 flow collision for an A/B build.
#ifndef ISLBM_F_FP32_3D
#define ISLBM_F_FP32_3D 1
#endif

// k[] of NodeParams for the lattice of dimension dim, from s_nu, s_q, hs_nu, hs_q, q_k, q_e (index map: collide_node)
inline void fold_node_params(NodeParams &p, int dim) {
  for (int i = 0; i < 21; ++i) p.k[i] = 0.0;
  if (dim == 2) {
    p.k[0] = -p.s_nu / 36.0;  p.k[1] = 6.0 * p.hs_nu / 36.0;          // e:   k0 (e - e_eq) + k1 vF
    p.k[2] = -p.s_nu / 36.0;  p.k[3] = -6.0 * p.hs_nu / 36.0;         // eps
    p.k[4] = -p.s_q / 12.0;   p.k[5] = -p.hs_q / 12.0;                // q:   k4 (q - q_eq) + k5 Fy
    p.k[6] = -p.s_nu / 4.0;   p.k[7] = -2.0 * p.hs_nu / 4.0;          // pxx: k6 (..) + k7 vF
    p.k[14] = -p.s_nu / 4.0;  p.k[15] = p.hs_nu / 4.0;                // pxy: k14 (..) + k15 u Fy
    p.k[17] = -p.q_k / 2.0;   p.k[18] = -p.q_e / 20.0;  p.k[20] = -p.q_e / 4.0;
    p.kf[2] = 0.f;
  } else {
    p.k[0] = -p.s_nu / 2394.0;  p.k[1] = 38.0 * p.hs_nu / 2394.0;     // e
    p.k[2] = -p.s_nu / 252.0;   p.k[3] = -11.0 * p.hs_nu / 252.0;     // eps
    p.k[4] = -p.s_q / 40.0;     p.k[5] = -p.hs_q * (2.0 / 3.0) / 40.0;  // q
    p.k[6] = -p.s_nu / 36.0;    p.k[7] = -2.0 * p.hs_nu / 36.0;       // 3pxx
    p.k[8] = -p.s_nu / 72.0;    p.k[9] = p.hs_nu / 72.0;              // 3pixx
    p.k[10] = -p.s_nu / 12.0;   p.k[11] = 2.0 * p.hs_nu / 12.0;       // pww
    p.k[12] = -p.s_nu / 24.0;   p.k[13] = -p.hs_nu / 24.0;            // piww
    p.k[14] = -p.s_nu / 4.0;    p.k[15] = p.hs_nu / 4.0;              // pxy, pyz, pxz
    p.k[16] = -p.s_q / 8.0;                                           // m
    p.k[17] = -p.q_k / 2.0;  p.k[18] = -p.q_e / 42.0;  p.k[19] = -p.q_e / 12.0;  p.k[20] = -p.q_e / 4.0;
    p.kf[2] = (float)p.k[19];
  }
  p.kf[0] = (float)p.k[17];
  p.kf[1] = (float)p.k[18];
  p.kf[3] = (float)p.k[20];
  p.kf[4] = (float)p.a_T;
  for (int i = 0; i < 17; ++i) p.kq[i] = (float)p.k[i];
  p.kq[17] = (float)p.gbeta;
  p.kq[18] = (float)p.T0;
}

template <int DIM> struct Lat;
template <> struct Lat<2> { static constexpr int QF = 9, QG = 5; };
template <> struct Lat<3> { static constexpr int QF = 19, QG = 7; };

// velocity component a of flow direction q (temperature directions are the first QG)
template <int DIM>
ISLBM_HD constexpr int evel(int q, int a) {
  if (DIM == 2) {
    constexpr int t[9][3] = {{0, 0, 0}, {1, 0, 0}, {0, 1, 0}, {-1, 0, 0}, {0, -1, 0},
                             {1, 1, 0}, {-1, 1, 0}, {-1, -1, 0}, {1, -1, 0}};
    return t[q][a];
  } else {
    constexpr int t[19][3] = {{0, 0, 0},
                              {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1},
                              {1, 1, 0}, {-1, 1, 0}, {1, -1, 0}, {-1, -1, 0},
                              {1, 0, 1}, {-1, 0, 1}, {1, 0, -1}, {-1, 0, -1},
                              {0, 1, 1}, {0, -1, 1}, {0, 1, -1}, {0, -1, -1}};
    return t[q][a];
  }
}

template <int DIM>
ISLBM_HD constexpr int opposite(int q) {
  if (DIM == 2) {
    constexpr int t[9] = {0, 3, 4, 1, 2, 7, 8, 5, 6};
    return t[q];
  } else {
    constexpr int t[19] = {0, 2, 1, 4, 3, 6, 5, 10, 9, 8, 7, 14, 13, 12, 11, 18, 17, 16, 15};
    return t[q];
  }
}

// Storage plane of flow population q / temperature population q inside a population buffer.  The public
// arrays of include/islbm.h are [q][z][y][x] in direction order; INSIDE the workspace the planes are ordered
// by the halo group the TMA-staged kernels load with one box:
//   2-D: f0 g0 | f1 f3 g1 g3 | f2 g2 f4 g4 | f5 f6 f7 f8
//   3-D: f0 g0 | f1 f2 g1 g2 | f3 f4 g3 g4 | f7..f10 | f5 g5 f6 g6 | f11..f14 | f15..f18
// (inside the last three groups the populations with a positive component along the marching axis come first: the
// upwind-stencil kernels load the two halves of a group from different layers)
template <int DIM>
ISLBM_HD constexpr int plane_f(int q) {
  if (DIM == 2) {
    constexpr int t[9] = {0, 2, 6, 3, 8, 10, 11, 12, 13};
    return t[q];
  } else {
    constexpr int t[19] = {0, 2, 3, 6, 7, 14, 16, 10, 11, 12, 13, 18, 19, 20, 21, 22, 23, 24, 25};
    return t[q];
  }
}
template <int DIM>
ISLBM_HD constexpr int plane_g(int q) {
  if (DIM == 2) {
    constexpr int t[5] = {1, 4, 7, 5, 9};
    return t[q];
  } else {
    constexpr int t[7] = {1, 4, 5, 8, 9, 15, 17};
    return t[q];
  }
}

// the planes whose velocity has a component along the slowest axis (the slab axis) form one contiguous range of
// the storage order: the halo of a slab decomposition
template <int DIM> ISLBM_HD constexpr int halo_first_plane() { return DIM == 2 ? 6 : 14; }
template <int DIM> ISLBM_HD constexpr int halo_plane_count() { return DIM == 2 ? 8 : 12; }

// inverse of plane_f / plane_g: the population stored in plane p (flow q as q, temperature q as QF + q)
template <int DIM>
ISLBM_HD constexpr int pop_of_plane(int p) {
  constexpr int QF = DIM == 2 ? 9 : 19, QG = DIM == 2 ? 5 : 7;
  for (int q = 0; q < QF; ++q)
    if (plane_f<DIM>(q) == p) return q;
  for (int q = 0; q < QG; ++q)
    if (plane_g<DIM>(q) == p) return QF + q;
  return -1;
}

// lattice weights of the rest equilibrium (rho = 1, u = 0): M^-1 m_eq
template <int DIM>
ISLBM_HD constexpr double wflow(int q) {
  if (DIM == 2) return q == 0 ? 4.0 / 9.0 : (q < 5 ? 1.0 / 9.0 : 1.0 / 36.0);
  return q == 0 ? 1.0 / 3.0 : (q < 7 ? 1.0 / 18.0 : 1.0 / 36.0);
}

// ---------------------------------------------------------------------------
// D2Q9 + D2Q5
// ---------------------------------------------------------------------------
// DEV = false: f holds the populations.  DEV = true (fp32 storage): f holds the deviations f_q - w_q from the rest
// equilibrium and stays in that form: M w = m_eq(rho = 1, u = 0), so only rho (= 1 + sum of deviations) and the rho-
// proportional rest parts of e_eq and eps_eq change, and f+ - w = (f - w) + M^T d needs no bias arithmetic at all
// (2 extra additions instead of 2 per flow population).
//
// FT = float (fp32 storage, DEV only): the node's values stay in fp32 registers.  They are widened (exactly) once for
// the moments and once more for the update f+ = fl32(fl64(f) + M^T d), so the result is bit-identical to colliding an
// fp64 copy of the node, but no fp64 copy has to stay live from the interpolation to the end of the collision (the
// compiler re-uses or re-creates the widened values as register pressure allows; measured: 256^3 fp32 storage
// 0.60 -> 0.65, 128^3 0.52 -> 0.58).  Rounding the increment to fp32 and adding it in
// fp32 (26 conversions fewer) measured only 1-2 % faster still and adds a second rounding per value and step, which
// shows on far-from-equilibrium states (2.3e-6 against the 2e-6 bar of test_fp32_storage_every_kernel_three_steps;
// the 1000-step error of 128^3 is unchanged, 4.3e-6): not taken.
ISLBM_HD void upd(double &a, double d) { a += d; }
ISLBM_HD void upd(float &a, double d) { a = (float)((double)a + d); }

// Deviation form with every temporary in fp32 (ISLBM_F_FP32_2D, an A/B switch): the factored M^T D M of collide_node<true>
// below with the host-folded constants rounded to fp32; f holds f_q - w_q, g the temperature populations, in and out.
ISLBM_HD void collide_node_dev_f32(float (&f)[9], float (&g)[5], const NodeParams &p) {
  const float *k = p.kq;
  const float T = g[0] + ((g[1] + g[3]) + (g[2] + g[4]));
  const float p13 = f[1] + f[3], p24 = f[2] + f[4], p57 = f[5] + f[7], p68 = f[6] + f[8];
  const float sa = p13 + p24, sd = p57 + p68;
  const float rsum = f[0] + sa + sd;
  const float rho = 1.0f + rsum;
  const float Fy = rho * k[17] * (T - k[18]);
  const float ax = f[1] - f[3], ay = f[2] - f[4];
  const float d57 = f[5] - f[7], d86 = f[8] - f[6];
  const float dx = d57 + d86, dy = d57 - d86;
  const float jx = ax + dx, jy = ay + dy;
#ifdef __CUDA_ARCH__
  const float inv = __frcp_rn(rho);
#else
  const float inv = 1.0f / rho;
#endif
  const float u = jx * inv, v = (jy + 0.5f * Fy) * inv;
  const float u2 = u * u + v * v;
  const float vF = v * Fy;
  // e - e_eq and eps - eps_eq with the rho-proportional rest parts cancelled before any rounding:
  // (m_e + 2 rsum) = -2 f0 + sa + 4 sd, (m_eps - rsum) = 3 (f0 - sa)
  const float ee = ((4.0f * sd + sa) - 2.0f * f[0]) - rho * (3.0f * u2);
  const float eeps = 3.0f * (f[0] - sa) + rho * (3.0f * u2);
  const float de = fmaf(k[0], ee, k[1] * vF);
  const float deps = fmaf(k[2], eeps, k[3] * vF);
  const float djy = Fy * (1.0f / 6.0f);
  const float dqx = k[4] * ((-2.0f * ax + dx) + rho * u);
  const float dqy = fmaf(k[4], (-2.0f * ay + dy) + rho * v, k[5] * Fy);
  const float dpxx = fmaf(k[6], (p13 - p24) - rho * (u * u - v * v), k[7] * vF);
  const float dpxy = fmaf(k[14], (p57 - p68) - rho * (u * v), k[15] * (u * Fy));
  {
    const float a1 = p.kf[0] * ((g[1] - g[3]) - u * T);
    const float a2 = p.kf[0] * ((g[2] - g[4]) - v * T);
    const float a3 = p.kf[1] * ((-4.0f * g[0] + ((g[1] + g[3]) + (g[2] + g[4]))) - p.kf[4] * T);
    const float a4 = p.kf[3] * ((g[1] + g[3]) - (g[2] + g[4]));
    g[0] += -4.0f * a3;
    const float g1 = g[1] + (a1 + a3 + a4), g2 = g[2] + (a2 + a3 - a4);
    const float g3 = g[3] + (-a1 + a3 + a4), g4 = g[4] + (-a2 + a3 - a4);
    g[1] = g1; g[2] = g2; g[3] = g3; g[4] = g4;
  }
  const float ca = -de - 2.0f * deps;
  const float cd = 2.0f * de + deps;
  const float tx = -2.0f * dqx, ty = djy - 2.0f * dqy;
  const float sx = dqx, sy = djy + dqy;
  f[0] += -4.0f * de + 4.0f * deps;
  f[1] += ca + tx + dpxx;
  f[2] += ca + ty - dpxx;
  f[3] += ca - tx + dpxx;
  f[4] += ca - ty - dpxx;
  f[5] += cd + sx + sy + dpxy;
  f[6] += cd - sx + sy - dpxy;
  f[7] += cd - sx - sy + dpxy;
  f[8] += cd + sx - sy - dpxy;
}

#ifndef ISLBM_F_FP32_2D
#define ISLBM_F_FP32_2D 0
#endif

template <bool DEV = false, typename FT>
ISLBM_HD void collide_node(FT (&fio)[9], FT (&gio)[5], const NodeParams &p) {
  constexpr bool GF = sizeof(FT) == 4 && ISLBM_G_FP32;   // temperature collision in fp32 (fp32 storage)
  if constexpr (DEV && GF && ISLBM_F_FP32_2D) {
    collide_node_dev_f32(fio, gio, p);
    return;
  }
  double f[9], g[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#ifdef __CUDA_ARCH__
#pragma unroll
#endif
  for (int q = 0; q < 9; ++q) f[q] = (double)fio[q];
  float Tf = 0.f;
  if constexpr (GF) {
    Tf = (float)gio[0] + (float)gio[1] + (float)gio[2] + (float)gio[3] + (float)gio[4];
  } else {
#ifdef __CUDA_ARCH__
#pragma unroll
#endif
    for (int q = 0; q < 5; ++q) g[q] = (double)gio[q];
  }
  const double T = GF ? (double)Tf : g[0] + g[1] + g[2] + g[3] + g[4];
  const double sa = (f[1] + f[3]) + (f[2] + f[4]);   // axis shell
  const double sd = (f[5] + f[7]) + (f[6] + f[8]);   // diagonal shell
  const double rsum = f[0] + sa + sd;
  const double rho = DEV ? 1.0 + rsum : rsum;
  const double Fy = rho * p.gbeta * (T - p.T0);
  const double ax = f[1] - f[3], ay = f[2] - f[4];
  const double dx = (f[5] - f[7]) + (f[8] - f[6]);    // sum cx over diagonals
  const double dy = (f[5] - f[7]) + (f[6] - f[8]);    // sum cy over diagonals
  const double jx = ax + dx, jy = ay + dy;
  const double inv = 1.0 / rho;
  const double u = jx * inv, v = (jy + 0.5 * Fy) * inv;
  const double u2 = u * u + v * v;
  // moments (Eq. 10 order): e, eps, qx, qy, pxx, pxy
  const double me = -4.0 * f[0] - sa + 2.0 * sd;
  const double meps = 4.0 * f[0] - 2.0 * sa + sd;
  const double mqx = -2.0 * ax + dx;
  const double mqy = -2.0 * ay + dy;
  const double mpxx = (f[1] + f[3]) - (f[2] + f[4]);
  const double mpxy = (f[5] + f[7]) - (f[6] + f[8]);
  const double vF = v * Fy;
  // Delta m_k / |row_k|^2
  const double ee = DEV ? (me + 2.0 * rsum) - rho * (3.0 * u2) : me - rho * (-2.0 + 3.0 * u2);        // e - e_eq
  const double eeps = DEV ? (meps - rsum) + rho * (3.0 * u2) : meps - rho * (1.0 - 3.0 * u2);        // eps - eps_eq
  const double de = fma(p.k[0], ee, p.k[1] * vF);
  const double deps = fma(p.k[2], eeps, p.k[3] * vF);
  const double djy = Fy * (1.0 / 6.0);
  const double dqx = p.k[4] * (mqx + rho * u);
  const double dqy = fma(p.k[4], mqy + rho * v, p.k[5] * Fy);
  const double dpxx = fma(p.k[6], mpxx - rho * (u * u - v * v), p.k[7] * vF);
  const double dpxy = fma(p.k[14], mpxy - rho * (u * v), p.k[15] * (u * Fy));
  // temperature moments (Eq. 15 order)
  double n1 = 0, n2 = 0, gs = 0, n3 = 0, n4 = 0, e1 = 0, e2 = 0, e3 = 0, e4 = 0;
  if constexpr (GF) {
    const float g0 = (float)gio[0], g1 = (float)gio[1], g2 = (float)gio[2], g3 = (float)gio[3], g4 = (float)gio[4];
    const float uf = (float)u, vf = (float)v;
    const float a1 = p.kf[0] * ((g1 - g3) - uf * Tf);
    const float a2 = p.kf[0] * ((g2 - g4) - vf * Tf);
    const float a3 = p.kf[1] * ((-4.0f * g0 + ((g1 + g3) + (g2 + g4))) - p.kf[4] * Tf);
    const float a4 = p.kf[3] * ((g1 + g3) - (g2 + g4));
    gio[0] = (FT)(g0 + -4.0f * a3);
    gio[1] = (FT)(g1 + (a1 + a3 + a4));
    gio[2] = (FT)(g2 + (a2 + a3 - a4));
    gio[3] = (FT)(g3 + (-a1 + a3 + a4));
    gio[4] = (FT)(g4 + (-a2 + a3 - a4));
  } else {
    n1 = g[1] - g[3], n2 = g[2] - g[4];
    gs = (g[1] + g[3]) + (g[2] + g[4]);
    n3 = -4.0 * g[0] + gs;
    n4 = (g[1] + g[3]) - (g[2] + g[4]);
    e1 = p.k[17] * (n1 - u * T);
    e2 = p.k[17] * (n2 - v * T);
    e3 = p.k[18] * (n3 - p.a_T * T);
    e4 = p.k[20] * n4;
  }
  // f+ = f + M^T d
  const double ca = -de - 2.0 * deps;          // common part, axis shell
  const double cd = 2.0 * de + deps;           // common part, diagonal shell
  const double tx = -2.0 * dqx, ty = djy - 2.0 * dqy;
  const double sx = dqx, sy = djy + dqy;
  upd(fio[0], -4.0 * de + 4.0 * deps);
  upd(fio[1], ca + tx + dpxx);
  upd(fio[2], ca + ty - dpxx);
  upd(fio[3], ca - tx + dpxx);
  upd(fio[4], ca - ty - dpxx);
  upd(fio[5], cd + sx + sy + dpxy);
  upd(fio[6], cd - sx + sy - dpxy);
  upd(fio[7], cd - sx - sy + dpxy);
  upd(fio[8], cd + sx - sy - dpxy);
  if constexpr (!GF) {
    upd(gio[0], -4.0 * e3);
    upd(gio[1], e1 + e3 + e4);
    upd(gio[2], e2 + e3 - e4);
    upd(gio[3], -e1 + e3 + e4);
    upd(gio[4], -e2 + e3 - e4);
  }
}

// macroscopic fields from POST-collision populations: rho and T are collision
// invariants and sum e f+ = sum e f + F, so u = (j+ - F/2)/rho.
ISLBM_HD void fields_from_post(const double (&f)[9], const double (&g)[5], const NodeParams &p,
                               double &rho, double &u, double &v, double &w, double &T) {
  T = g[0] + g[1] + g[2] + g[3] + g[4];
  rho = f[0] + ((f[1] + f[3]) + (f[2] + f[4])) + ((f[5] + f[7]) + (f[6] + f[8]));
  const double Fy = rho * p.gbeta * (T - p.T0);
  const double jx = (f[1] - f[3]) + ((f[5] - f[7]) + (f[8] - f[6]));
  const double jy = (f[2] - f[4]) + ((f[5] - f[7]) + (f[6] - f[8]));
  u = jx / rho;
  v = (jy - 0.5 * Fy) / rho;
  w = 0.0;
}

// ---------------------------------------------------------------------------
// D3Q19 + D3Q7
// ---------------------------------------------------------------------------
// Deviation form, every temporary in fp32 (ISLBM_F_FP32_3D): the same factored M^T D M as collide_node<true> below,
// with the host-folded constants rounded to fp32.  f holds f_q - w_q and g the temperature populations, in and out.
ISLBM_HD void collide_node_dev_f32(float (&f)[19], float (&g)[7], const NodeParams &p) {
  const float *k = p.kq;
  const float T = g[0] + (((g[1] + g[2]) + (g[3] + g[4])) + (g[5] + g[6]));
  const float px = f[1] + f[2], py = f[3] + f[4], pz = f[5] + f[6];
  const float ax = f[1] - f[2], ay = f[3] - f[4], az = f[5] - f[6];
  const float xy_s = (f[7] + f[10]) + (f[8] + f[9]);
  const float xy_x = (f[7] - f[10]) + (f[9] - f[8]);
  const float xy_y = (f[7] - f[10]) + (f[8] - f[9]);
  const float xy_p = (f[7] + f[10]) - (f[8] + f[9]);
  const float xz_s = (f[11] + f[14]) + (f[12] + f[13]);
  const float xz_x = (f[11] - f[14]) + (f[13] - f[12]);
  const float xz_z = (f[11] - f[14]) + (f[12] - f[13]);
  const float xz_p = (f[11] + f[14]) - (f[12] + f[13]);
  const float yz_s = (f[15] + f[18]) + (f[16] + f[17]);
  const float yz_y = (f[15] - f[18]) + (f[17] - f[16]);
  const float yz_z = (f[15] - f[18]) + (f[16] - f[17]);
  const float yz_p = (f[15] + f[18]) - (f[16] + f[17]);
  const float sa = px + py + pz;
  const float sd = xy_s + xz_s + yz_s;
  const float rsum = f[0] + sa + sd;
  const float rho = 1.0f + rsum;
  const float Fy = rho * k[17] * (T - k[18]);
  const float dxs = xy_x + xz_x, dys = xy_y + yz_y, dzs = xz_z + yz_z;
  const float jx = ax + dxs, jy = ay + dys, jz = az + dzs;
#ifdef __CUDA_ARCH__
  const float inv = __frcp_rn(rho);
#else
  const float inv = 1.0f / rho;
#endif
  const float u = jx * inv, v = (jy + 0.5f * Fy) * inv, w = jz * inv;
  const float u2 = u * u + v * v + w * w;
  const float mqx = -4.0f * ax + dxs, mqy = -4.0f * ay + dys, mqz = -4.0f * az + dzs;
  const float a3 = 2.0f * px - py - pz, d3 = xy_s + xz_s - 2.0f * yz_s;
  const float aw = py - pz, dw = xy_s - xz_s;
  const float vF = v * Fy;
  const float q3 = 2.0f * u * u - v * v - w * w, qw = v * v - w * w;
  // e - e_eq and eps - eps_eq with the rho-proportional rest parts cancelled: (m_e + 11 rsum) = 19 (sd - f0),
  // (m_eps - 3 rsum) = 9 f0 - 7 sa - 2 sd
  const float ee = 19.0f * ((sd - f[0]) - rho * u2);
  const float eeps = (9.0f * f[0] - 7.0f * sa - 2.0f * sd) + rho * (5.5f * u2);
  const float r23 = (2.0f / 3.0f) * rho;
  const float djy = Fy * 0.1f;
  const float de = fmaf(k[0], ee, k[1] * vF);
  const float deps = fmaf(k[2], eeps, k[3] * vF);
  const float dqx = k[4] * (mqx + r23 * u);
  const float dqy = fmaf(k[4], mqy + r23 * v, k[5] * Fy);
  const float dqz = k[4] * (mqz + r23 * w);
  const float d3pxx = fmaf(k[6], (a3 + d3) - rho * q3, k[7] * vF);
  const float d3pixx = fmaf(k[8], (-2.0f * a3 + d3) + 0.5f * rho * q3, k[9] * vF);
  const float dpww = fmaf(k[10], (aw + dw) - rho * qw, k[11] * vF);
  const float dpiww = fmaf(k[12], (-2.0f * aw + dw) + 0.5f * rho * qw, k[13] * vF);
  const float dpxy = fmaf(k[14], xy_p - rho * (u * v), k[15] * (u * Fy));
  const float dpyz = fmaf(k[14], yz_p - rho * (v * w), k[15] * (w * Fy));
  const float dpxz = k[14] * (xz_p - rho * (u * w));
  const float dmx = k[16] * (xy_x - xz_x), dmy = k[16] * (yz_y - xy_y), dmz = k[16] * (xz_z - yz_z);
  // temperature (Eq. 16 order), as in the ISLBM_G_FP32 branch of collide_node
  {
    const float hx = g[1] + g[2], hy = g[3] + g[4], hz = g[5] + g[6];
    const float a1 = p.kf[0] * ((g[1] - g[2]) - u * T);
    const float a2 = p.kf[0] * ((g[3] - g[4]) - v * T);
    const float a3g = p.kf[0] * ((g[5] - g[6]) - w * T);
    const float a4 = p.kf[1] * ((-6.0f * g[0] + (hx + hy + hz)) - p.kf[4] * T);
    const float a5 = p.kf[2] * (2.0f * hx - hy - hz);
    const float a6 = p.kf[3] * (hy - hz);
    g[0] += -6.0f * a4;
    g[1] += a1 + a4 + 2.0f * a5;
    g[2] += -a1 + a4 + 2.0f * a5;
    g[3] += a2 + a4 - a5 + a6;
    g[4] += -a2 + a4 - a5 + a6;
    g[5] += a3g + a4 - a5 - a6;
    g[6] += -a3g + a4 - a5 - a6;
  }
  // f+ = f + M^T d
  const float ca = -11.0f * de - 4.0f * deps;
  const float cd = 8.0f * de + deps;
  const float tx = -4.0f * dqx, ty = djy - 4.0f * dqy, tz = -4.0f * dqz;
  const float sx = dqx, sy = djy + dqy, sz = dqz;
  const float nax = 2.0f * d3pxx - 4.0f * d3pixx;
  const float nay = -d3pxx + 2.0f * d3pixx + dpww - 2.0f * dpiww;
  const float naz = -d3pxx + 2.0f * d3pixx - dpww + 2.0f * dpiww;
  const float nxy = d3pxx + d3pixx + dpww + dpiww;
  const float nxz = d3pxx + d3pixx - dpww - dpiww;
  const float nyz = -2.0f * (d3pxx + d3pixx);
  f[0] += -30.0f * de + 12.0f * deps;
  f[1] += ca + tx + nax;
  f[2] += ca - tx + nax;
  f[3] += ca + ty + nay;
  f[4] += ca - ty + nay;
  f[5] += ca + tz + naz;
  f[6] += ca - tz + naz;
  f[7] += cd + nxy + (sx + dmx) + (sy - dmy) + dpxy;
  f[8] += cd + nxy - (sx + dmx) + (sy - dmy) - dpxy;
  f[9] += cd + nxy + (sx + dmx) - (sy - dmy) - dpxy;
  f[10] += cd + nxy - (sx + dmx) - (sy - dmy) + dpxy;
  f[11] += cd + nxz + (sx - dmx) + (sz + dmz) + dpxz;
  f[12] += cd + nxz - (sx - dmx) + (sz + dmz) - dpxz;
  f[13] += cd + nxz + (sx - dmx) - (sz + dmz) - dpxz;
  f[14] += cd + nxz - (sx - dmx) - (sz + dmz) + dpxz;
  f[15] += cd + nyz + (sy + dmy) + (sz - dmz) + dpyz;
  f[16] += cd + nyz - (sy + dmy) + (sz - dmz) - dpyz;
  f[17] += cd + nyz + (sy + dmy) - (sz - dmz) - dpyz;
  f[18] += cd + nyz - (sy + dmy) - (sz - dmz) + dpyz;
}

template <bool DEV = false, typename FT>
ISLBM_HD void collide_node(FT (&fio)[19], FT (&gio)[7], const NodeParams &p) {
  constexpr bool GF = sizeof(FT) == 4 && ISLBM_G_FP32;   // temperature collision in fp32 (fp32 storage)
  if constexpr (DEV && GF && ISLBM_F_FP32_3D) {
    collide_node_dev_f32(fio, gio, p);
    return;
  }
  double f[19], g[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#ifdef __CUDA_ARCH__
#pragma unroll
#endif
  for (int q = 0; q < 19; ++q) f[q] = (double)fio[q];
  float Tf = 0.f;
  if constexpr (GF) {
    Tf = (float)gio[0] + (((float)gio[1] + (float)gio[2]) + ((float)gio[3] + (float)gio[4]) + ((float)gio[5] + (float)gio[6]));
  } else {
#ifdef __CUDA_ARCH__
#pragma unroll
#endif
    for (int q = 0; q < 7; ++q) g[q] = (double)gio[q];
  }
  const double T = GF ? (double)Tf : g[0] + ((g[1] + g[2]) + (g[3] + g[4]) + (g[5] + g[6]));
  // pair sums / differences
  const double px = f[1] + f[2], py = f[3] + f[4], pz = f[5] + f[6];
  const double ax = f[1] - f[2], ay = f[3] - f[4], az = f[5] - f[6];
  // xy diagonals 7(+,+) 8(-,+) 9(+,-) 10(-,-)
  const double xy_s = (f[7] + f[10]) + (f[8] + f[9]);
  const double xy_x = (f[7] - f[10]) + (f[9] - f[8]);    // sum cx
  const double xy_y = (f[7] - f[10]) + (f[8] - f[9]);    // sum cy
  const double xy_p = (f[7] + f[10]) - (f[8] + f[9]);    // sum cx*cy
  // xz diagonals 11(+,+) 12(-,+) 13(+,-) 14(-,-)   (signs: x, z)
  const double xz_s = (f[11] + f[14]) + (f[12] + f[13]);
  const double xz_x = (f[11] - f[14]) + (f[13] - f[12]);
  const double xz_z = (f[11] - f[14]) + (f[12] - f[13]);
  const double xz_p = (f[11] + f[14]) - (f[12] + f[13]);
  // yz diagonals 15(+,+) 16(-,+) 17(+,-) 18(-,-)   (signs: y, z)
  const double yz_s = (f[15] + f[18]) + (f[16] + f[17]);
  const double yz_y = (f[15] - f[18]) + (f[17] - f[16]);
  const double yz_z = (f[15] - f[18]) + (f[16] - f[17]);
  const double yz_p = (f[15] + f[18]) - (f[16] + f[17]);

  const double sa = px + py + pz;
  const double sd = xy_s + xz_s + yz_s;
  const double rsum = f[0] + sa + sd;
  const double rho = DEV ? 1.0 + rsum : rsum;
  const double Fy = rho * p.gbeta * (T - p.T0);
  const double dxs = xy_x + xz_x, dys = xy_y + yz_y, dzs = xz_z + yz_z;
  const double jx = ax + dxs, jy = ay + dys, jz = az + dzs;
  const double inv = 1.0 / rho;
  const double u = jx * inv, v = (jy + 0.5 * Fy) * inv, w = jz * inv;
  const double u2 = u * u + v * v + w * w;
  // moments in the order of Eq. 11
  const double me = -30.0 * f[0] - 11.0 * sa + 8.0 * sd;
  const double meps = 12.0 * f[0] - 4.0 * sa + sd;
  const double mqx = -4.0 * ax + dxs, mqy = -4.0 * ay + dys, mqz = -4.0 * az + dzs;
  const double a3 = 2.0 * px - py - pz;                 // axis part of 3pxx
  const double d3 = xy_s + xz_s - 2.0 * yz_s;           // diagonal part of 3pxx
  const double m3pxx = a3 + d3;
  const double m3pixx = -2.0 * a3 + d3;
  const double aw = py - pz, dw = xy_s - xz_s;
  const double mpww = aw + dw;
  const double mpiww = -2.0 * aw + dw;
  const double mmx = xy_x - xz_x, mmy = yz_y - xy_y, mmz = xz_z - yz_z;
  const double vF = v * Fy;
  const double q3 = 2.0 * u * u - v * v - w * w, qw = v * v - w * w;
  // Delta m_k / |row_k|^2
  const double ee = DEV ? (me + 11.0 * rsum) - rho * (19.0 * u2) : me - rho * (-11.0 + 19.0 * u2);     // e - e_eq
  const double eeps = DEV ? (meps - 3.0 * rsum) + rho * (5.5 * u2) : meps - rho * (3.0 - 5.5 * u2);   // eps - eps_eq
  // Delta m_k / |row_k|^2.  FOLD: with the host-folded constants k[] (one multiply and one fused multiply-add per
  // moment; 256^3 fp64 0.895 -> 0.905, 128^3 0.847 -> 0.859).  FT = float reaches this point only in the A/B build
  // -DISLBM_F_FP32_3D=0 (fp64 flow collision on fp32 storage), which keeps the unfolded expressions: under its
  // 168-register cap the folded form spilled 164 instead of 60 bytes and measured 11 % slower.
  constexpr bool FOLD = sizeof(FT) == 8;
  const double djy = Fy * 0.1;
  double gx = 0, gy = 0, gz = 0;
  if constexpr (!GF) gx = g[1] + g[2], gy = g[3] + g[4], gz = g[5] + g[6];
  if constexpr (GF) {
    const float g0 = (float)gio[0], g1 = (float)gio[1], g2 = (float)gio[2], g3 = (float)gio[3], g4 = (float)gio[4],
                g5 = (float)gio[5], g6 = (float)gio[6];
    const float uf = (float)u, vf = (float)v, wf = (float)w;
    const float hx = g1 + g2, hy = g3 + g4, hz = g5 + g6;
    const float a1 = p.kf[0] * ((g1 - g2) - uf * Tf);
    const float a2 = p.kf[0] * ((g3 - g4) - vf * Tf);
    const float a3 = p.kf[0] * ((g5 - g6) - wf * Tf);
    const float a4 = p.kf[1] * ((-6.0f * g0 + (hx + hy + hz)) - p.kf[4] * Tf);
    const float a5 = p.kf[2] * (2.0f * hx - hy - hz);
    const float a6 = p.kf[3] * (hy - hz);
    gio[0] = (FT)(g0 + -6.0f * a4);
    gio[1] = (FT)(g1 + (a1 + a4 + 2.0f * a5));
    gio[2] = (FT)(g2 + (-a1 + a4 + 2.0f * a5));
    gio[3] = (FT)(g3 + (a2 + a4 - a5 + a6));
    gio[4] = (FT)(g4 + (-a2 + a4 - a5 + a6));
    gio[5] = (FT)(g5 + (a3 + a4 - a5 - a6));
    gio[6] = (FT)(g6 + (-a3 + a4 - a5 - a6));
  }
  double de, deps, dqx, dqy, dqz, d3pxx, d3pixx, dpww, dpiww, dpxy, dpyz, dpxz, dmx, dmy, dmz, e1, e2, e3, e4, e5, e6;
  if constexpr (FOLD) {
    const double r23 = (2.0 / 3.0) * rho;
    de = fma(p.k[0], ee, p.k[1] * vF);
    deps = fma(p.k[2], eeps, p.k[3] * vF);
    dqx = p.k[4] * (mqx + r23 * u);
    dqy = fma(p.k[4], mqy + r23 * v, p.k[5] * Fy);
    dqz = p.k[4] * (mqz + r23 * w);
    d3pxx = fma(p.k[6], m3pxx - rho * q3, p.k[7] * vF);
    d3pixx = fma(p.k[8], m3pixx + 0.5 * rho * q3, p.k[9] * vF);
    dpww = fma(p.k[10], mpww - rho * qw, p.k[11] * vF);
    dpiww = fma(p.k[12], mpiww + 0.5 * rho * qw, p.k[13] * vF);
    dpxy = fma(p.k[14], xy_p - rho * (u * v), p.k[15] * (u * Fy));
    dpyz = fma(p.k[14], yz_p - rho * (v * w), p.k[15] * (w * Fy));
    dpxz = p.k[14] * (xz_p - rho * (u * w));
    dmx = p.k[16] * mmx, dmy = p.k[16] * mmy, dmz = p.k[16] * mmz;
    // temperature moments (Eq. 16 order)
    e1 = p.k[17] * ((g[1] - g[2]) - u * T);
    e2 = p.k[17] * ((g[3] - g[4]) - v * T);
    e3 = p.k[17] * ((g[5] - g[6]) - w * T);
    e4 = p.k[18] * ((-6.0 * g[0] + (gx + gy + gz)) - p.a_T * T);
    e5 = p.k[19] * (2.0 * gx - gy - gz);
    e6 = p.k[20] * (gy - gz);
  } else {
    de = (-p.s_nu * ee + p.hs_nu * (38.0 * vF)) * (1.0 / 2394.0);
    deps = (-p.s_nu * eeps - p.hs_nu * (11.0 * vF)) * (1.0 / 252.0);
    dqx = (-p.s_q * (mqx + (2.0 / 3.0) * rho * u)) * (1.0 / 40.0);
    dqy = (-p.s_q * (mqy + (2.0 / 3.0) * rho * v) - p.hs_q * ((2.0 / 3.0) * Fy)) * (1.0 / 40.0);
    dqz = (-p.s_q * (mqz + (2.0 / 3.0) * rho * w)) * (1.0 / 40.0);
    d3pxx = (-p.s_nu * (m3pxx - rho * q3) - p.hs_nu * (2.0 * vF)) * (1.0 / 36.0);
    d3pixx = (-p.s_nu * (m3pixx + 0.5 * rho * q3) + p.hs_nu * vF) * (1.0 / 72.0);
    dpww = (-p.s_nu * (mpww - rho * qw) + p.hs_nu * (2.0 * vF)) * (1.0 / 12.0);
    dpiww = (-p.s_nu * (mpiww + 0.5 * rho * qw) - p.hs_nu * vF) * (1.0 / 24.0);
    dpxy = (-p.s_nu * (xy_p - rho * (u * v)) + p.hs_nu * (u * Fy)) * 0.25;
    dpyz = (-p.s_nu * (yz_p - rho * (v * w)) + p.hs_nu * (w * Fy)) * 0.25;
    dpxz = (-p.s_nu * (xz_p - rho * (u * w))) * 0.25;
    dmx = (-p.s_q * mmx) * 0.125, dmy = (-p.s_q * mmy) * 0.125, dmz = (-p.s_q * mmz) * 0.125;
    // temperature moments (Eq. 16 order)
    e1 = (-p.q_k * ((g[1] - g[2]) - u * T)) * 0.5;
    e2 = (-p.q_k * ((g[3] - g[4]) - v * T)) * 0.5;
    e3 = (-p.q_k * ((g[5] - g[6]) - w * T)) * 0.5;
    e4 = (-p.q_e * ((-6.0 * g[0] + (gx + gy + gz)) - p.a_T * T)) * (1.0 / 42.0);
    e5 = (-p.q_e * (2.0 * gx - gy - gz)) * (1.0 / 12.0);
    e6 = (-p.q_e * (gy - gz)) * 0.25;
  }
  // f+ = f + M^T d
  const double ca = -11.0 * de - 4.0 * deps;
  const double cd = 8.0 * de + deps;
  const double tx = -4.0 * dqx, ty = djy - 4.0 * dqy, tz = -4.0 * dqz;
  const double sx = dqx, sy = djy + dqy, sz = dqz;
  const double nax = 2.0 * d3pxx - 4.0 * d3pixx;                         // axis x normal-stress part
  const double nay = -d3pxx + 2.0 * d3pixx + dpww - 2.0 * dpiww;         // axis y
  const double naz = -d3pxx + 2.0 * d3pixx - dpww + 2.0 * dpiww;         // axis z
  const double nxy = d3pxx + d3pixx + dpww + dpiww;                      // xy diagonals
  const double nxz = d3pxx + d3pixx - dpww - dpiww;                      // xz diagonals
  const double nyz = -2.0 * (d3pxx + d3pixx);                            // yz diagonals
  upd(fio[0], -30.0 * de + 12.0 * deps);
  upd(fio[1], ca + tx + nax);
  upd(fio[2], ca - tx + nax);
  upd(fio[3], ca + ty + nay);
  upd(fio[4], ca - ty + nay);
  upd(fio[5], ca + tz + naz);
  upd(fio[6], ca - tz + naz);
  // xy: + sx*cx + sy*cy + cx*cy*dpxy + cx*dmx - cy*dmy
  upd(fio[7], cd + nxy + (sx + dmx) + (sy - dmy) + dpxy);
  upd(fio[8], cd + nxy - (sx + dmx) + (sy - dmy) - dpxy);
  upd(fio[9], cd + nxy + (sx + dmx) - (sy - dmy) - dpxy);
  upd(fio[10], cd + nxy - (sx + dmx) - (sy - dmy) + dpxy);
  // xz: + sx*cx + sz*cz + cx*cz*dpxz - cx*dmx + cz*dmz
  upd(fio[11], cd + nxz + (sx - dmx) + (sz + dmz) + dpxz);
  upd(fio[12], cd + nxz - (sx - dmx) + (sz + dmz) - dpxz);
  upd(fio[13], cd + nxz + (sx - dmx) - (sz + dmz) - dpxz);
  upd(fio[14], cd + nxz - (sx - dmx) - (sz + dmz) + dpxz);
  // yz: + sy*cy + sz*cz + cy*cz*dpyz + cy*dmy - cz*dmz
  upd(fio[15], cd + nyz + (sy + dmy) + (sz - dmz) + dpyz);
  upd(fio[16], cd + nyz - (sy + dmy) + (sz - dmz) - dpyz);
  upd(fio[17], cd + nyz + (sy + dmy) - (sz - dmz) - dpyz);
  upd(fio[18], cd + nyz - (sy + dmy) - (sz - dmz) + dpyz);
  if constexpr (!GF) {
    upd(gio[0], -6.0 * e4);
    upd(gio[1], e1 + e4 + 2.0 * e5);
    upd(gio[2], -e1 + e4 + 2.0 * e5);
    upd(gio[3], e2 + e4 - e5 + e6);
    upd(gio[4], -e2 + e4 - e5 + e6);
    upd(gio[5], e3 + e4 - e5 - e6);
    upd(gio[6], -e3 + e4 - e5 - e6);
  }
}

ISLBM_HD void fields_from_post(const double (&f)[19], const double (&g)[7], const NodeParams &p,
                               double &rho, double &u, double &v, double &w, double &T) {
  T = g[0] + ((g[1] + g[2]) + (g[3] + g[4]) + (g[5] + g[6]));
  const double sa = (f[1] + f[2]) + (f[3] + f[4]) + (f[5] + f[6]);
  const double sd = ((f[7] + f[10]) + (f[8] + f[9])) + ((f[11] + f[14]) + (f[12] + f[13])) +
                    ((f[15] + f[18]) + (f[16] + f[17]));
  rho = f[0] + sa + sd;
  const double Fy = rho * p.gbeta * (T - p.T0);
  const double jx = (f[1] - f[2]) + ((f[7] - f[10]) + (f[9] - f[8])) + ((f[11] - f[14]) + (f[13] - f[12]));
  const double jy = (f[3] - f[4]) + ((f[7] - f[10]) + (f[8] - f[9])) + ((f[15] - f[18]) + (f[17] - f[16]));
  const double jz = (f[5] - f[6]) + ((f[11] - f[14]) + (f[12] - f[13])) + ((f[15] - f[18]) + (f[16] - f[17]));
  u = jx / rho;
  v = (jy - 0.5 * Fy) / rho;
  w = jz / rho;
}

// pre-collision macroscopic fields (used by init checks / diagnostics on f_t)
template <int QF, int QG>
ISLBM_HD void rest_equilibrium(double (&f)[QF], double (&g)[QG], double T, double a_T) {
  constexpr int DIM = QF == 9 ? 2 : 3;
#pragma unroll
  for (int q = 0; q < QF; ++q) f[q] = wflow<DIM>(q);
  // N^-1 n_eq(T, u = 0): rest weight (1 - a_T)/5 | (1 - a_T)/7, moving weight (4 + a_T)/20 | (6 + a_T)/42
  const double wm = DIM == 2 ? (4.0 + a_T) * (1.0 / 20.0) : (6.0 + a_T) * (1.0 / 42.0);
  const double w0 = DIM == 2 ? (1.0 - a_T) * 0.2 : (1.0 - a_T) * (1.0 / 7.0);
  g[0] = w0 * T;
#pragma unroll
  for (int q = 1; q < QG; ++q) g[q] = wm * T;
}

}  // namespace islbmk
