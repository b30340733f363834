// Multi-step kernel for very small 2-D meshes: the whole state lives in the shared memory of ONE thread-block cluster
// and n time steps run inside one launch.
//
// A 64^2 mesh is 4096 nodes: one launch per step costs 3-4 us whatever the kernel does (launch latency, ring set-up,
// a DRAM round trip), a CUDA graph of PDL-chained launches still 3.2 us.  Here a cluster of up to 16 CTAs (one band of
// `rows` mesh rows each, one thread per node) keeps both ping-pong buffers of its band in shared memory, with one halo
// row on either side; a step is: interpolate from the local buffer, wall rules (Eq. 21-23),
// collision (Eq. 17, 19), store into the other local buffer, and the two boundary rows of the band ALSO store the
// eight populations with e_y != 0 into the neighbour CTAs' halo rows through distributed shared memory.  Those stores
// are st.async with mbarrier::complete_tx: each CTA has one mbarrier per buffer that counts the bytes its neighbours
// deliver, the rows that read a halo wait on it, and a CTA-local barrier orders the local buffers — a neighbour-only
// hand-shake, no cluster-wide barrier inside the step loop (ISLBM_CLUSTER_MBAR).  Reads are always local.
// The arithmetic is that of k_step_ymarch (same ptap3 / pcomb3 / collide_node, same order): results are bit-identical.
//
// Scope: D2Q9 + D2Q5, fp64 storage, destination-centred stencil, whole cavity (no slab decomposition), ny = ncta * rows
// with rows >= 2 and nx * rows <= 256.  Everything else takes the per-step kernels.
#pragma once
#include "islbm_tiled3.cuh"

namespace islbmk {

constexpr int kClusterThreads = 256;

// Step synchronisation.  1: neighbour-only hand-shake — the halo values travel as st.async stores that complete bytes on
// an mbarrier of the receiving CTA (one per buffer), the receiving boundary rows wait on it, and a CTA-local barrier
// orders the local buffers: no cluster-wide barrier and no memory fence inside the step loop.  0: one
// barrier.cluster.arrive.release / wait.acquire per step (an A/B build; profiles/attempts.md).
#ifndef ISLBM_CLUSTER_MBAR
#define ISLBM_CLUSTER_MBAR 1
#endif

struct PlanC2 {
  bool available = false;
  int ncta = 0, rows = 0;
  size_t smem = 0;
};

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t mapa_shared(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void st_cluster_f64(uint32_t addr, double v) {
  asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}
// remote store that completes 8 bytes on the mbarrier `mbar` of the receiving CTA (both shared::cluster addresses)
__device__ __forceinline__ void st_async_f64(uint32_t addr, double v, uint32_t mbar) {
  asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(addr), "d"(v), "r"(mbar)
               : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release;\n\tbarrier.cluster.wait.acquire;" ::: "memory");
}

// Eq. 21-23 for the populations that cross ONE wall, read from the node's own post-collision values in shared memory
// (planes in natural order: flow q at q, temperature q at 9 + q; pitch PL).  Mirrors wall_fix of islbm_tiled3.cuh.
template <int AXIS, int SIGN, int Q>
__device__ __forceinline__ void cwall_f1(double *f, const double *own, int PL) {
  if constexpr (evel<2>(Q, AXIS) == SIGN) f[Q] = own[opposite<2>(Q) * PL];
}
template <int AXIS, int SIGN, int Q>
__device__ __forceinline__ void cwall_g1(double *g, const double *own, int PL, const DevMesh &m) {
  if constexpr (evel<2>(Q, AXIS) == SIGN) {
    const double gb = own[(9 + opposite<2>(Q)) * PL];
    g[Q] = AXIS == 0 ? -gb + m.omega_bc * (SIGN > 0 ? m.T_hot : m.T_cold) : gb;
  }
}
template <int AXIS, int SIGN, int... Qf, int... Qg>
__device__ __forceinline__ void cwall(double *f, double *g, const double *own, int PL, const DevMesh &m,
                                      std::integer_sequence<int, Qf...>, std::integer_sequence<int, Qg...>) {
  (cwall_f1<AXIS, SIGN, Qf + 1>(f, own, PL), ...);
  (cwall_g1<AXIS, SIGN, Qg + 1>(g, own, PL, m), ...);
}

__global__ void __launch_bounds__(kClusterThreads, 1)
k_multistep_cluster2(DevMesh m, NodeParams np, double *src, double *dst, int rows, int nsteps) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *sm = reinterpret_cast<double *>(smem_raw);
  const int nx = m.nx;
  const int PL = (rows + 2) * nx;     // plane pitch: the band plus one halo row below and above
  const int BUF = 14 * PL;
  const int rank = (int)cluster_ctarank(), nrank = (int)gridDim.x;
  const int r0 = rank * rows;
  const int tid = (int)threadIdx.x;

  // the band with its halo rows, straight from the post-collision buffer in HBM (storage-plane order there)
  const int row_lo = rank > 0 ? 0 : 1, row_hi = rank < nrank - 1 ? rows + 1 : rows;   // local rows that exist
  for (int i = tid + row_lo * nx; i < (row_hi + 1) * nx; i += kClusterThreads) {
    const int lr = i / nx, xx = i - lr * nx;
    const long long gi = (long long)(r0 + lr - 1) * m.nxp + xx;
#pragma unroll
    for (int q = 0; q < 9; ++q) sm[q * PL + i] = src[(long long)plane_f<2>(q) * m.nnp + gi];
#pragma unroll
    for (int q = 0; q < 5; ++q) sm[(9 + q) * PL + i] = src[(long long)plane_g<2>(q) * m.nnp + gi];
  }

  const bool valid = tid < rows * nx;
  const int yl = valid ? tid / nx : 0, x = valid ? tid - yl * nx : 0;
  const int y = r0 + yl;
  const int xs = sbase(x, nx);                       // stencil {xs, xs+1, xs+2}
  const int ysl = sbase(y, m.ny) - r0 + 1;           // local row of the first stencil row
  const int own = (yl + 1) * nx + x;
  WallFlags wf;
  wf.lo[0] = x == 0;  wf.hi[0] = x == nx - 1;
  wf.lo[1] = y == 0;  wf.hi[1] = y == m.ny - 1;
  wf.lo[2] = wf.hi[2] = false;
  const bool wall = wf.lo[0] | wf.hi[0] | wf.lo[1] | wf.hi[1];
  Pr<double> wxN[3], wyN[3], wyS[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    wxN[k] = mkpr(__ldg(wrow(m, 0, 1, k) + x), __ldg(wrow(m, 0, 0, k) + x));
    const double y1 = __ldg(wrow(m, 1, 1, k) + y), y0 = __ldg(wrow(m, 1, 0, k) + y);
    wyN[k] = mkpr(y1, y0);
    wyS[k] = mkpr(y0, y1);
  }
  // halo rows of the neighbours that this thread feeds: the band's first row goes to the upper halo (local row rows+1)
  // of rank-1, its last row to the lower halo (local row 0) of rank+1
  const bool feed_dn = valid && yl == 0 && rank > 0, feed_up = valid && yl == rows - 1 && rank < nrank - 1;
  const uint32_t sm_s = (uint32_t)__cvta_generic_to_shared(sm);
  uint32_t remote = 0;      // shared::cluster address of this node's slot in the neighbour's halo row, plane 0, buffer 0
  if (feed_dn) remote = mapa_shared(sm_s + (uint32_t)(((rows + 1) * nx + x) * 8), (uint32_t)(rank - 1));
  if (feed_up) remote = mapa_shared(sm_s + (uint32_t)(x * 8), (uint32_t)(rank + 1));
  const bool feed = feed_dn | feed_up;
  // which threads READ a halo row: the band's first / last row, and with 2-row bands also the other row of the first and
  // last CTA, whose stencil is clamped at the wall and reaches across the band ({0,1,2} for y = 0)
  const bool reads_halo = valid && ((ysl == 0 && rank > 0) || (ysl + 2 == rows + 1 && rank < nrank - 1));
  // ... in which case a row that does not feed a neighbour reads what that neighbour overwrites two steps later, and the
  // neighbour's go-ahead (this band's boundary row) must not leave before the whole CTA has finished reading
  const bool late_send = rows == 2;
  // halo hand-shake: hfull[k] counts the bytes the neighbours store into the halo rows of buffer k
  uint64_t *hfull = reinterpret_cast<uint64_t *>(sm + 2 * BUF);
  uint32_t rbar = 0;        // the neighbour's hfull[0], shared::cluster address
  const uint32_t halo_bytes = (uint32_t)(((rank > 0) + (rank < nrank - 1)) * 8 * nx * 8);
  if constexpr (ISLBM_CLUSTER_MBAR) {
    if (tid == 0) {
      mbar_init(&hfull[0], 1);
      mbar_init(&hfull[1], 1);
      fence_barrier_init();
    }
    if (feed_dn) rbar = mapa_shared(smem_u32(hfull), (uint32_t)(rank - 1));
    if (feed_up) rbar = mapa_shared(smem_u32(hfull), (uint32_t)(rank + 1));
  }

  cluster_sync_all();       // every CTA of the cluster is running, has its band loaded and its barriers initialised

  int b = 0;
#pragma unroll 1
  for (int s = 0; s < nsteps; ++s) {
    const double *cb = sm + b * BUF;
    double *nb = sm + (1 - b) * BUF;
    if constexpr (ISLBM_CLUSTER_MBAR) {
      // arm this step's phase of the receiving barrier (bytes may already have arrived: the count is signed)
      if (tid == 0) mbar_expect_tx(&hfull[1 - b], halo_bytes);
    }
    double h2 = 0, h4 = 0, h5 = 0, h6 = 0, h7 = 0, h8 = 0, k2 = 0, k4 = 0;   // what the neighbour's halo row takes
    auto send_halo = [&]() {
      const uint32_t rb = remote + (uint32_t)((1 - b) * BUF * 8);
      if constexpr (ISLBM_CLUSTER_MBAR) {
        const uint32_t mb = rbar + (uint32_t)((1 - b) * 8);
        st_async_f64(rb + (uint32_t)(2 * PL * 8), h2, mb);
        st_async_f64(rb + (uint32_t)(4 * PL * 8), h4, mb);
        st_async_f64(rb + (uint32_t)(5 * PL * 8), h5, mb);
        st_async_f64(rb + (uint32_t)(6 * PL * 8), h6, mb);
        st_async_f64(rb + (uint32_t)(7 * PL * 8), h7, mb);
        st_async_f64(rb + (uint32_t)(8 * PL * 8), h8, mb);
        st_async_f64(rb + (uint32_t)(11 * PL * 8), k2, mb);
        st_async_f64(rb + (uint32_t)(13 * PL * 8), k4, mb);
      } else {
        st_cluster_f64(rb + (uint32_t)(2 * PL * 8), h2);
        st_cluster_f64(rb + (uint32_t)(4 * PL * 8), h4);
        st_cluster_f64(rb + (uint32_t)(5 * PL * 8), h5);
        st_cluster_f64(rb + (uint32_t)(6 * PL * 8), h6);
        st_cluster_f64(rb + (uint32_t)(7 * PL * 8), h7);
        st_cluster_f64(rb + (uint32_t)(8 * PL * 8), h8);
        st_cluster_f64(rb + (uint32_t)(11 * PL * 8), k2);
        st_cluster_f64(rb + (uint32_t)(13 * PL * 8), k4);
      }
    };
    if (valid) {
      double f[9], g[5];
      f[0] = cb[own];
      g[0] = cb[9 * PL + own];
      const double *rx = cb + (yl + 1) * nx + xs;
      const Pr<double> p1 = ptap3(rx + 1 * PL, rx + 3 * PL, 1, wxN);     // f1 (+x), f3 (-x)
      const Pr<double> p2 = ptap3(rx + 10 * PL, rx + 12 * PL, 1, wxN);   // g1, g3
      f[1] = lane_a(p1); f[3] = lane_b(p1);
      g[1] = lane_a(p2); g[3] = lane_b(p2);
      Pr<double> S[3][4];     // x-interpolated values of the three y-stencil rows (ascending y), pairs as in islbm_tiled2.cuh
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const double *rc = cb + (ysl + k) * nx + x, *rt = cb + (ysl + k) * nx + xs;
        S[k][0] = mkpr(rc[2 * PL], rc[4 * PL]);                          // f2, f4
        S[k][1] = mkpr(rc[11 * PL], rc[13 * PL]);                        // g2, g4
        S[k][2] = ptap3(rt + 5 * PL, rt + 7 * PL, 1, wxN);               // f5 (+x,+y), f7 (-x,-y)
        S[k][3] = ptap3(rt + 8 * PL, rt + 6 * PL, 1, wxN);               // f8 (+x,-y), f6 (-x,+y)
      }
      const Pr<double> q0 = pcomb3(wyN, S[0][0], S[1][0], S[2][0]);
      const Pr<double> q1 = pcomb3(wyN, S[0][1], S[1][1], S[2][1]);
      const Pr<double> q2 = pcomb3(wyN, S[0][2], S[1][2], S[2][2]);
      const Pr<double> q3 = pcomb3(wyS, S[0][3], S[1][3], S[2][3]);
      f[2] = lane_a(q0); f[4] = lane_b(q0);
      g[2] = lane_a(q1); g[4] = lane_b(q1);
      f[5] = lane_a(q2); f[7] = lane_b(q2);
      f[8] = lane_a(q3); f[6] = lane_b(q3);
      if (wall) {
        using QF = std::make_integer_sequence<int, 8>;
        using QG = std::make_integer_sequence<int, 4>;
        const double *o = cb + own;
        if (wf.lo[0]) cwall<0, 1>(f, g, o, PL, m, QF{}, QG{});
        if (wf.hi[0]) cwall<0, -1>(f, g, o, PL, m, QF{}, QG{});
        if (wf.lo[1]) cwall<1, 1>(f, g, o, PL, m, QF{}, QG{});
        if (wf.hi[1]) cwall<1, -1>(f, g, o, PL, m, QF{}, QG{});
      }
      collide_node<false>(f, g, np);
#pragma unroll
      for (int q = 0; q < 9; ++q) nb[q * PL + own] = f[q];
#pragma unroll
      for (int q = 0; q < 5; ++q) nb[(9 + q) * PL + own] = g[q];
      h2 = f[2]; h4 = f[4]; h5 = f[5]; h6 = f[6]; h7 = f[7]; h8 = f[8]; k2 = g[2]; k4 = g[4];
      if (feed && !(ISLBM_CLUSTER_MBAR && late_send)) send_halo();
    }
    if constexpr (ISLBM_CLUSTER_MBAR) {
      // local rows of the new buffer complete, old buffer free in this CTA; then the rows that read a halo wait for the
      // neighbour's bytes.  A neighbour cannot run two steps ahead (it needs this band's next boundary row first), so
      // the two barriers and the two buffers never alias across steps.
      __syncthreads();
      if (feed && late_send) send_halo();
      if (reads_halo) mbar_wait(&hfull[1 - b], (uint32_t)(s >> 1) & 1u);
    } else {
      cluster_sync_all();   // the new buffer (own rows and halo rows) is complete everywhere; the old one is free
    }
    b ^= 1;
  }
  if constexpr (ISLBM_CLUSTER_MBAR) cluster_sync_all();   // nobody leaves while a neighbour could still store into it

  // The library's two HBM buffers hold the post-collision states of the last two time levels (the newer one is the
  // state, the older one is what islbm_get_populations streams to recover f_t): dst takes level n, src level n-1.
  // (Every CTA read its rows of src before the first cluster barrier, and each thread rewrites only its own node.)
  if (valid) {
    const double *cb = sm + b * BUF, *pb = sm + (1 - b) * BUF;
    const long long gi = (long long)y * m.nxp + x;
#pragma unroll
    for (int q = 0; q < 9; ++q) {
      dst[(long long)plane_f<2>(q) * m.nnp + gi] = cb[q * PL + own];
      src[(long long)plane_f<2>(q) * m.nnp + gi] = pb[q * PL + own];
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      dst[(long long)plane_g<2>(q) * m.nnp + gi] = cb[(9 + q) * PL + own];
      src[(long long)plane_g<2>(q) * m.nnp + gi] = pb[(9 + q) * PL + own];
    }
  }
}

// largest cluster (16, 8, 4, 2 CTAs) whose bands are whole rows, at least two of them, one thread per node
inline bool planc2_create(PlanC2 &p, const int *n) {
  p.available = false;
  int cc_major = 0, dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return false;
  cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev);
  if (cc_major < 9) return false;
  for (int c = 16; c >= 2; c >>= 1) {
    if (n[1] % c) continue;
    const int rows = n[1] / c;
    if (rows < 2 || (long long)rows * n[0] > kClusterThreads) continue;
    const size_t smem = (size_t)2 * 14 * (rows + 2) * n[0] * sizeof(double) + 16;   // + two mbarriers
    if (cudaFuncSetAttribute(k_multistep_cluster2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
        (c > 8 && cudaFuncSetAttribute(k_multistep_cluster2, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess)) {
      cudaGetLastError();
      continue;
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(c);
    cfg.blockDim = dim3(kClusterThreads);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = c; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, k_multistep_cluster2, &cfg) != cudaSuccess || nclusters < 1) {
      cudaGetLastError();
      continue;
    }
    p.ncta = c; p.rows = rows; p.smem = smem; p.available = true;
    return true;
  }
  return false;
}

inline cudaError_t launch_cluster2(const PlanC2 &p, const DevMesh &m, const NodeParams &np, double *src, double *dst,
                                   int nsteps, cudaStream_t stream) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(p.ncta);
  cfg.blockDim = dim3(kClusterThreads);
  cfg.dynamicSmemBytes = p.smem;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = p.ncta; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, k_multistep_cluster2, m, np, src, dst, p.rows, nsteps);
}

}  // namespace islbmk
