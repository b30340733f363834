// islbm_kernels.cuh — device-side data model and the generic (global-memory)
// kernels of the ISLBM step.
//
// State convention: HBM holds POST-collision populations S_t =
// collide(f_t).  One step is  f_{t+1} = stream/interpolate/walls(S_t)  followed,
// in the same kernel, by  S_{t+1} = collide(f_{t+1}),  so each node collides
// once per step and every population is read once and written once
// (PAPER.md:150-154 gives the collide -> stream order this is equivalent to).
//
// Layout: structure-of-arrays planes [plane][z][y][x]; the plane of each
// population is plane_f / plane_g (islbm_lattice.cuh: ordered by TMA halo
// group); storage type ST is double, or float holding the deviation f_q - w_q
// (ISLBM_F32_STORAGE).
#pragma once

#include <cstdint>
#include <utility>

#include "islbm_lattice.cuh"

namespace islbmk {

constexpr int kMaxQ = 26;

struct DevMesh {
  int nx, ny, nz;
  int npad;              // pitch of the per-axis tables
  long long nn;          // nx*ny*nz: nodes (and the pitch of the PUBLIC dense arrays)
  int nxp;               // row pitch of the workspace planes in elements (nx rounded up to 16: TMA needs a
                         // 16-byte pitch, and 128-byte row starts keep the stores coalesced); columns >= nx are padding
  long long nnp;         // plane pitch of the workspace = nxp*ny*nz
  // interpolation weights, [axis 3][sign 2 (0: c=-1, 1: c=+1)][k 3][npad]; the
  // stencil of node j is {b, b+1, b+2}, b = clamp(j-1, 0, n-3) (A2)
  const double *wtab;
  const double *avgw;    // Eq. 29 weights, [axis 3][npad]
  double omega_bc;       // Eq. 22 weight
  double T_hot, T_cold;  // x-lo / x-hi wall temperatures
  // slab decomposition along the slowest axis (y in 2-D, z in 3-D): the local mesh may carry one
  // ghost layer at either end, which is read but not updated; the layers [em_lo, em_hi) are the owned ones, and an
  // end is a wall only if its flag says so.  Whole cavity: em_lo = 0, em_hi = n, both walls.
  int em_lo, em_hi;
  int wall_mlo, wall_mhi;
  long long node_offset; // global linear index of local node 0 (islbm_init draws the noise by global index)
  // fused halo exchange (islbm_slab_set_peer): peer[s] points at the neighbour's ghost layer, in the buffer the
  // neighbour writes during this step, of the FIRST halo plane (plane index kHaloFirst<DIM>); peer_pitch[s] is the
  // neighbour's plane pitch in elements.  The thread that emits this rank's first (s = 0) / last (s = 1) owned layer
  // also stores the halo planes of its node there: NVLink peer stores from inside the step kernel, no separate
  // exchange pass.  nullptr: no neighbour on that side, or the exchange is done outside (islbm_halo).
  void *peer[2];
  long long peer_pitch[2];
  // neighbour-only synchronisation of the fused exchange (include/islbm.h: islbm_slab_set_peer).  flag_in[s]: this
  // rank's step flag of side s, written by that neighbour; flag_out[s]: the neighbour's flag in peer memory; step: the
  // 1-based index of the step this launch performs; done_cnt: two counters of finished boundary CTAs (monotonic);
  // bctas: CTAs of this launch that touch one boundary layer
  unsigned long long *flag_in[2], *flag_out[2];
  unsigned long long *done_cnt;
  unsigned long long step;
  int bctas;
  // the wait for a neighbour's flag is bounded: after wait_ns nanoseconds (0 = wait for ever) the CTA counts a
  // time-out in done_cnt[2] and goes on; the host reports it at the next synchronising slab call instead of hanging
  unsigned long long wait_ns;
  int stencil;           // 0: {j-1,j,j+1} (A2); 1: upwind {j-2,j-1,j} for c=+1, {j,j+1,j+2} for c=-1
                         // (generic kernel; the TMA kernels exist per stencil: k_step_*march / k_step_*march_up)
};

// workspace (padded-row) index of dense node index c
__device__ __forceinline__ long long sidx(const DevMesh &m, long long c) {
  if (m.nxp == m.nx) return c;
  const long long r = c / m.nx;
  return r * m.nxp + (c - r * m.nx);
}

__device__ __forceinline__ const double *wrow(const DevMesh &m, int axis, int sign, int k) {
  return m.wtab + ((axis * 2 + sign) * 3 + k) * (long long)m.npad;
}

// storage <-> fp64 value of flow population q (deviation storage for float)
template <typename ST, int DIM> struct Store;
template <int DIM> struct Store<double, DIM> {
  static constexpr bool kBiased = false;
  static __device__ __forceinline__ double bias(int) { return 0.0; }
};
template <int DIM> struct Store<float, DIM> {
  static constexpr bool kBiased = true;
  static __device__ __forceinline__ double bias(int q) { return wflow<DIM>(q); }
};
// storage form -> value and back (no arithmetic at all for fp64 storage: x + 0.0 is not a no-op for the compiler)
template <typename ST, int DIM, int QF>
__device__ __forceinline__ void add_bias(double (&f)[QF]) {
  if constexpr (Store<ST, DIM>::kBiased) {
#pragma unroll
    for (int q = 0; q < QF; ++q) f[q] += Store<ST, DIM>::bias(q);
  }
}
template <typename ST, int DIM>
__device__ __forceinline__ ST to_storage(double v, int q) {
  if constexpr (Store<ST, DIM>::kBiased) return (ST)(v - Store<ST, DIM>::bias(q));
  else return (ST)v;
}

// DEV = true: v already is the deviation f_q - w_q (collide_node<true>)
template <typename ST, int DIM, bool DEV, typename NT>
__device__ __forceinline__ ST to_storage_from(NT v, int q) {
  if constexpr (DEV) return (ST)v;
  else return to_storage<ST, DIM>(v, q);
}

template <typename ST>
__device__ __forceinline__ double ldv(const ST *p) { return (double)__ldg(p); }
// coherent (L2) load for data another grid may still be writing when this kernel becomes resident (PDL)
template <typename ST>
__device__ __forceinline__ ST ld_coherent(const ST *p) { return __ldcg(p); }

// storage element -> fp64.  (An integer-instruction widening of fp32 - shift, re-bias the exponent - was measured
// against the conversion instruction: 4 instructions instead of 1 on an issue/latency-bound kernel, no gain.)
__device__ __forceinline__ double widen(float x) { return (double)x; }
__device__ __forceinline__ double widen(double x) { return x; }

// SplitMix64 by counter (A15): the (k+1)-th output for `seed`.
__device__ __forceinline__ unsigned long long splitmix64_at(unsigned long long seed, unsigned long long k) {
  unsigned long long z = seed + (k + 1ull) * 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// ---------------------------------------------------------------------------
// per-thread stencil context of the generic kernel
// ---------------------------------------------------------------------------
template <int DIM>
struct NodeCtx {
  int i[3];        // node index
  int b[3][2];     // stencil base per axis and sign (0: c=-1, 1: c=+1)
  bool lo[3], hi[3];
  double w[3][2][3];
  long long c;     // workspace index (padded rows)
  long long cd;    // dense node index (public arrays)
};

template <int DIM>
__device__ __forceinline__ void make_ctx(const DevMesh &m, int ix, int iy, int iz, NodeCtx<DIM> &cx) {
  const int n[3] = {m.nx, m.ny, m.nz};
  cx.i[0] = ix; cx.i[1] = iy; cx.i[2] = iz;
  cx.c = ((long long)iz * m.ny + iy) * m.nxp + ix;
  cx.cd = ((long long)iz * m.ny + iy) * m.nx + ix;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (a < DIM) {
      cx.lo[a] = cx.i[a] == 0 && (a != DIM - 1 || m.wall_mlo);
      cx.hi[a] = cx.i[a] == n[a] - 1 && (a != DIM - 1 || m.wall_mhi);
      cx.b[a][0] = min(max(m.stencil ? cx.i[a] : cx.i[a] - 1, 0), n[a] - 3);
      cx.b[a][1] = min(max(m.stencil ? cx.i[a] - 2 : cx.i[a] - 1, 0), n[a] - 3);
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int k = 0; k < 3; ++k) cx.w[a][s][k] = __ldg(wrow(m, a, s, k) + cx.i[a]);
    } else {
      cx.lo[a] = cx.hi[a] = false;
      cx.b[a][0] = cx.b[a][1] = 0;
    }
  }
}

// Does the departure point of velocity (EX,EY,EZ) lie beyond a wall? (A4)
template <int DIM, int EX, int EY, int EZ>
__device__ __forceinline__ bool crosses(const NodeCtx<DIM> &cx) {
  bool r = false;
  if (EX == 1) r |= cx.lo[0];
  if (EX == -1) r |= cx.hi[0];
  if (EY == 1) r |= cx.lo[1];
  if (EY == -1) r |= cx.hi[1];
  if (DIM == 3 && EZ == 1) r |= cx.lo[2];
  if (DIM == 3 && EZ == -1) r |= cx.hi[2];
  return r;
}

// Separable 3-point Lagrange interpolation of one plane at the departure point
// x - e*delta; x first, then y, then z.
template <int DIM, int EX, int EY, int EZ, typename ST>
__device__ __forceinline__ double interp_plane(const DevMesh &m, const ST *__restrict__ plane,
                                               const NodeCtx<DIM> &cx) {
  constexpr int CX = EX != 0 ? 3 : 1, CY = EY != 0 ? 3 : 1, CZ = (DIM == 3 && EZ != 0) ? 3 : 1;
  constexpr int SX = EX > 0 ? 1 : 0, SY = EY > 0 ? 1 : 0, SZ = EZ > 0 ? 1 : 0;
  const int x0 = EX != 0 ? cx.b[0][SX] : cx.i[0];
  const int y0 = EY != 0 ? cx.b[1][SY] : cx.i[1];
  const int z0 = (DIM == 3 && EZ != 0) ? cx.b[2][SZ] : cx.i[2];
  double accz = 0.0;
#pragma unroll
  for (int kz = 0; kz < CZ; ++kz) {
    double accy = 0.0;
#pragma unroll
    for (int ky = 0; ky < CY; ++ky) {
      const ST *row = plane + ((long long)(z0 + kz) * m.ny + (y0 + ky)) * m.nxp + x0;
      double accx;
      if (CX == 3) {
        accx = cx.w[0][SX][0] * ldv(row);
        accx = fma(cx.w[0][SX][1], ldv(row + 1), accx);
        accx = fma(cx.w[0][SX][2], ldv(row + 2), accx);
      } else {
        accx = ldv(row);
      }
      accy = CY == 3 ? (ky == 0 ? cx.w[1][SY][0] * accx : fma(cx.w[1][SY][ky], accx, accy)) : accx;
    }
    accz = CZ == 3 ? (kz == 0 ? cx.w[2][SZ][0] * accy : fma(cx.w[2][SZ][kz], accy, accz)) : accy;
  }
  return accz;
}

// New value of flow population Q at the node: interpolation, or half-way
// bounce-back f_Q(x,t+1) = f+_opp(Q)(x,t) (Eq. 21).
template <int DIM, int Q, typename ST>
__device__ __forceinline__ double pull_f(const DevMesh &m, const ST *__restrict__ src, const NodeCtx<DIM> &cx) {
  constexpr int EX = evel<DIM>(Q, 0), EY = evel<DIM>(Q, 1), EZ = evel<DIM>(Q, 2);
  if (crosses<DIM, EX, EY, EZ>(cx)) return ldv(src + (long long)plane_f<DIM>(opposite<DIM>(Q)) * m.nnp + cx.c);
  return interp_plane<DIM, EX, EY, EZ>(m, src + (long long)plane_f<DIM>(Q) * m.nnp, cx);
}

// Temperature population Q: interpolation; anti-bounce-back on the isothermal
// x-walls (Eq. 22); bounce-back on the adiabatic walls (Eq. 23).
template <int DIM, int Q, typename ST>
__device__ __forceinline__ double pull_g(const DevMesh &m, const ST *__restrict__ src, const NodeCtx<DIM> &cx) {
  constexpr int EX = evel<DIM>(Q, 0), EY = evel<DIM>(Q, 1), EZ = evel<DIM>(Q, 2);
  if (crosses<DIM, EX, EY, EZ>(cx)) {
    const double gb = ldv(src + (long long)plane_g<DIM>(opposite<DIM>(Q)) * m.nnp + cx.c);
    if (EX != 0) return -gb + m.omega_bc * (cx.lo[0] ? m.T_hot : m.T_cold);
    return gb;
  }
  return interp_plane<DIM, EX, EY, EZ>(m, src + (long long)plane_g<DIM>(Q) * m.nnp, cx);
}

template <int DIM, typename ST, int... Qs>
__device__ __forceinline__ void pull_all_f(const DevMesh &m, const ST *src, const NodeCtx<DIM> &cx,
                                           double *f, std::integer_sequence<int, Qs...>) {
  ((f[Qs] = pull_f<DIM, Qs>(m, src, cx)), ...);
}
template <int DIM, typename ST, int... Qs>
__device__ __forceinline__ void pull_all_g(const DevMesh &m, const ST *src, const NodeCtx<DIM> &cx,
                                           double *g, std::integer_sequence<int, Qs...>) {
  ((g[Qs] = pull_g<DIM, Qs>(m, src, cx)), ...);
}

// fused halo exchange: the halo planes of this node into the neighbour's ghost layer (DevMesh::peer), plain stores
template <int DIM, int K, bool DEV, typename ST, typename NT>
__device__ __forceinline__ void peer_plane(ST *p, const NT *f, const NT *g) {
  constexpr int QF = Lat<DIM>::QF;
  constexpr int code = pop_of_plane<DIM>(halo_first_plane<DIM>() + K);
  if constexpr (code < QF) *p = to_storage_from<ST, DIM, DEV>(f[code], code);
  else *p = (ST)g[code - QF];
}
template <int DIM, typename ST, bool DEV, typename NT, int... Ks>
__device__ __forceinline__ void peer_store(void *base, long long pitch, long long inplane, const NT *f, const NT *g,
                                           std::integer_sequence<int, Ks...>) {
  ST *p = reinterpret_cast<ST *>(base) + inplane;
  (peer_plane<DIM, Ks, DEV>(p + (long long)Ks * pitch, f, g), ...);
}
template <int DIM, typename ST, bool DEV = false, typename NT>
__device__ __forceinline__ void peer_store_node(const DevMesh &m, int layer, long long inplane, const NT *f, const NT *g) {
  if (m.peer[0] != nullptr && layer == m.em_lo)
    peer_store<DIM, ST, DEV, NT>(m.peer[0], m.peer_pitch[0], inplane, f, g, std::make_integer_sequence<int, halo_plane_count<DIM>()>{});
  if (m.peer[1] != nullptr && layer == m.em_hi - 1)
    peer_store<DIM, ST, DEV, NT>(m.peer[1], m.peer_pitch[1], inplane, f, g, std::make_integer_sequence<int, halo_plane_count<DIM>()>{});
}

// ---- neighbour flags of the fused halo exchange -----------------------------------------------------------------
__device__ __forceinline__ unsigned long long ld_acquire_sys(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_sys(unsigned long long *p, unsigned long long v) {
  asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// one thread: wait until the neighbour of `side` has finished step m.step - 1 (its halo of that step is in our ghost
// layer, and it no longer reads the ghost layer we are about to overwrite)
__device__ __forceinline__ void slab_wait_neighbour(const DevMesh &m, int side) {
  if (m.flag_in[side] == nullptr) return;
  if (ld_acquire_sys(m.flag_in[side]) + 1ull >= m.step) return;          // the usual case: already there
  unsigned long long t0;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
  while (ld_acquire_sys(m.flag_in[side]) + 1ull < m.step) {
    __nanosleep(64);
    if (m.wait_ns != 0ull) {
      unsigned long long t1;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
      if (t1 - t0 > m.wait_ns) {
        atomicAdd(m.done_cnt + 2, 1ull);      // gave up: the results of this rank are invalid from here on
        return;
      }
    }
  }
}
// one thread of a CTA whose threads have all finished (after a CTA barrier): count it; the last boundary CTA of this
// launch publishes the step number to the neighbour
__device__ __forceinline__ void slab_publish(const DevMesh &m, int side) {
  if (m.flag_out[side] == nullptr) return;
  __threadfence_system();                                                 // this CTA's peer stores, cumulatively
  const unsigned long long old = atomicAdd(m.done_cnt + side, 1ull);
  if ((old + 1ull) % (unsigned long long)m.bctas == 0ull) {
    __threadfence_system();                                               // ... and those of every CTA counted before
    st_release_sys(m.flag_out[side], m.step);
  }
}
// generic-kernel path: the same protocol as two single-thread kernels around the step
__global__ void k_slab_wait(DevMesh m) {
  slab_wait_neighbour(m, 0);
  slab_wait_neighbour(m, 1);
}
__global__ void k_slab_publish(DevMesh m) {
  for (int side = 0; side < 2; ++side)
    if (m.flag_out[side] != nullptr) {
      __threadfence_system();
      st_release_sys(m.flag_out[side], m.step);
    }
}

// ---------------------------------------------------------------------------
// generic step: one thread per node, neighbours read from global memory
// through L1/L2.  COLLIDE = false writes the pre-collision f_{t+1}, g_{t+1} as
// fp64 to fout/gout (islbm_get_populations).
// ---------------------------------------------------------------------------
template <int DIM, typename ST, bool COLLIDE>
__global__ void __launch_bounds__(256)
k_step_generic(DevMesh m, NodeParams np, const ST *__restrict__ src, ST *__restrict__ dst,
               double *__restrict__ fout, double *__restrict__ gout) {
  constexpr int QF = Lat<DIM>::QF, QG = Lat<DIM>::QG;
  const int ix = blockIdx.x * blockDim.x + threadIdx.x;
  const int iy = blockIdx.y * blockDim.y + threadIdx.y;
  const int iz = blockIdx.z * blockDim.z + threadIdx.z;
  if (ix >= m.nx || iy >= m.ny || iz >= m.nz) return;
  if (COLLIDE && ((DIM == 3 ? iz : iy) < m.em_lo || (DIM == 3 ? iz : iy) >= m.em_hi)) return;   // ghost layer
  NodeCtx<DIM> cx;
  make_ctx<DIM>(m, ix, iy, iz, cx);
  double f[QF], g[QG];
  pull_all_f<DIM>(m, src, cx, f, std::make_integer_sequence<int, QF>{});
  pull_all_g<DIM>(m, src, cx, g, std::make_integer_sequence<int, QG>{});
  add_bias<ST, DIM>(f);
  if (COLLIDE) {
    collide_node(f, g, np);
#pragma unroll
    for (int q = 0; q < QF; ++q) dst[(long long)plane_f<DIM>(q) * m.nnp + cx.c] = to_storage<ST, DIM>(f[q], q);
#pragma unroll
    for (int q = 0; q < QG; ++q) dst[(long long)plane_g<DIM>(q) * m.nnp + cx.c] = (ST)g[q];
    peer_store_node<DIM, ST>(m, DIM == 3 ? iz : iy, DIM == 3 ? (long long)iy * m.nxp + ix : (long long)ix, f, g);
  } else {
#pragma unroll
    for (int q = 0; q < QF; ++q) fout[(long long)q * m.nn + cx.cd] = f[q];
#pragma unroll
    for (int q = 0; q < QG; ++q) gout[(long long)q * m.nn + cx.cd] = g[q];
  }
}

// ---------------------------------------------------------------------------
// state load / init / export
// ---------------------------------------------------------------------------

// pre-collision f,g (fp64, user arrays, or generated) -> `pre` buffer (storage
// form, kept for islbm_get_populations) and collided -> `post` buffer.  The
// kernel handles the node range [c0, c0 + count); fin/gin hold that range with
// a plane pitch of `pitch` elements (pitch = nn, c0 = 0 for whole dense arrays;
// a staged slab for islbm_set_populations_host).
template <int DIM, typename ST, bool GENERATE>
__global__ void __launch_bounds__(256)
k_load_state(DevMesh m, NodeParams np, const double *__restrict__ fin, const double *__restrict__ gin,
             unsigned long long seed, double amp, ST *__restrict__ pre, ST *__restrict__ post, long long pitch,
             long long c0, long long count) {
  constexpr int QF = Lat<DIM>::QF, QG = Lat<DIM>::QG;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  const long long c = c0 + i;
  double f[QF], g[QG];
  if (GENERATE) {
    const unsigned long long z = splitmix64_at(seed, (unsigned long long)(c + m.node_offset));
    const double r = (double)(z >> 11) * (1.0 / 9007199254740992.0);
    rest_equilibrium<QF, QG>(f, g, amp * (2.0 * r - 1.0), np.a_T);
  } else {
#pragma unroll
    for (int q = 0; q < QF; ++q) f[q] = fin[(long long)q * pitch + i];
#pragma unroll
    for (int q = 0; q < QG; ++q) g[q] = gin[(long long)q * pitch + i];
  }
  const long long cs = sidx(m, c);
#pragma unroll
  for (int q = 0; q < QF; ++q) pre[(long long)plane_f<DIM>(q) * m.nnp + cs] = to_storage<ST, DIM>(f[q], q);
#pragma unroll
  for (int q = 0; q < QG; ++q) pre[(long long)plane_g<DIM>(q) * m.nnp + cs] = (ST)g[q];
  collide_node(f, g, np);
#pragma unroll
  for (int q = 0; q < QF; ++q) post[(long long)plane_f<DIM>(q) * m.nnp + cs] = to_storage<ST, DIM>(f[q], q);
#pragma unroll
  for (int q = 0; q < QG; ++q) post[(long long)plane_g<DIM>(q) * m.nnp + cs] = (ST)g[q];
}

// storage-form buffer -> fp64 user arrays
template <int DIM, typename ST>
__global__ void __launch_bounds__(256)
k_export(DevMesh m, const ST *__restrict__ buf, double *__restrict__ fout, double *__restrict__ gout) {
  constexpr int QF = Lat<DIM>::QF, QG = Lat<DIM>::QG;
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= m.nn) return;
  const long long cs = sidx(m, c);
#pragma unroll
  for (int q = 0; q < QF; ++q) fout[(long long)q * m.nn + c] = (double)buf[(long long)plane_f<DIM>(q) * m.nnp + cs] + Store<ST, DIM>::bias(q);
#pragma unroll
  for (int q = 0; q < QG; ++q) gout[(long long)q * m.nn + c] = (double)buf[(long long)plane_g<DIM>(q) * m.nnp + cs];
}

template <int DIM, typename ST>
__device__ __forceinline__ void load_post_node(const DevMesh &m, const ST *__restrict__ S, long long c /* workspace index */,
                                               double (&f)[Lat<DIM>::QF], double (&g)[Lat<DIM>::QG]) {
  constexpr int QF = Lat<DIM>::QF, QG = Lat<DIM>::QG;
#pragma unroll
  for (int q = 0; q < QF; ++q) f[q] = ldv(S + (long long)plane_f<DIM>(q) * m.nnp + c) + Store<ST, DIM>::bias(q);
#pragma unroll
  for (int q = 0; q < QG; ++q) g[q] = ldv(S + (long long)plane_g<DIM>(q) * m.nnp + c);
}

// macroscopic fields from the post-collision state
template <int DIM, typename ST>
__global__ void __launch_bounds__(256)
k_fields(DevMesh m, NodeParams np, const ST *__restrict__ S, double *rho, double *u, double *v, double *w, double *T) {
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= m.nn) return;
  double f[Lat<DIM>::QF], g[Lat<DIM>::QG];
  load_post_node<DIM>(m, S, sidx(m, c), f, g);
  double r, uu, vv, ww, tt;
  fields_from_post(f, g, np, r, uu, vv, ww, tt);
  if (rho) rho[c] = r;
  if (u) u[c] = uu;
  if (v) v[c] = vv;
  if (w && DIM == 3) w[c] = ww;
  if (T) T[c] = tt;
}

}  // namespace islbmk
