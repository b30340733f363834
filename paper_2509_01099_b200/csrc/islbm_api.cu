// islbm_api.cu — C-ABI of the ISLBM hot path (include/islbm.h): host-side
// setup (parameter map, interpolation tables, workspace carving) and kernel
// dispatch.  No torch types, no CPU fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/islbm.h"
#include "islbm_kernels.cuh"
#include "islbm_reduce.cuh"
#include "islbm_tiled2.cuh"
#include "islbm_tiled3.cuh"
#include "islbm_cluster2.cuh"
#include "islbm_uniform.cuh"

using namespace islbmk;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string &msg) {
  g_err = msg;
  return code;
}

#define CUDA_TRY(expr)                                                                 \
  do {                                                                                 \
    cudaError_t e_ = (expr);                                                           \
    if (e_ != cudaSuccess)                                                             \
      return fail(ISLBM_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_)); \
  } while (0)

constexpr size_t kAlign = 256;
size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

constexpr int kMaxRedBlocks = 2048;   // capacity of the partial-sum area; the launch takes 8 blocks per SM (red_blocks)

struct Carve {
  size_t buf[2], wtab, avgw, partial, red_out, flags, snap, total;
};

// row pitch of the workspace planes: nx rounded up to 16 elements (see DevMesh::nxp)
int row_pitch(int nx) { return (nx + 15) / 16 * 16; }

Carve carve(long long nn, long long nnp, int q, size_t st_bytes, int npad) {
  Carve c{};
  size_t off = 0;
  for (int i = 0; i < 2; ++i) {
    c.buf[i] = off;
    off = align_up(off + (size_t)q * (size_t)nnp * st_bytes);
  }
  c.wtab = off;    off = align_up(off + sizeof(double) * 18 * (size_t)npad);
  c.avgw = off;    off = align_up(off + sizeof(double) * 3 * (size_t)npad);
  c.partial = off; off = align_up(off + sizeof(double) * kRedSlots * kMaxRedBlocks);
  c.red_out = off; off = align_up(off + sizeof(double) * 8);
  c.flags = off;   off = align_up(off + 256);   // neighbour step flags [2] (u64, written by the neighbours) + done counters [2]
  c.snap = off;    off = align_up(off + sizeof(double) * 4 * (size_t)nn);
  c.total = off;
  return c;
}

int check_mesh_args(const islbm_mesh *mesh, int lattice, int precision) {
  if (!mesh) return fail(ISLBM_ERR_ARG, "mesh is NULL");
  if (mesh->dim != 2 && mesh->dim != 3) return fail(ISLBM_ERR_ARG, "dim must be 2 or 3");
  if ((mesh->dim == 2) != (lattice == ISLBM_D2Q9_D2Q5) || (mesh->dim == 3) != (lattice == ISLBM_D3Q19_D3Q7))
    return fail(ISLBM_ERR_ARG, "lattice does not match dim (2-D: D2Q9+D2Q5, 3-D: D3Q19+D3Q7)");
  if (precision != ISLBM_F64 && precision != ISLBM_F32_STORAGE) return fail(ISLBM_ERR_ARG, "unknown precision");
  for (int a = 0; a < mesh->dim; ++a)
    if (mesh->n[a] < 3) return fail(ISLBM_ERR_ARG, "need at least 3 nodes per axis");
  return ISLBM_OK;
}

int npad_of(const islbm_mesh *mesh) {
  int mx = 0;
  for (int a = 0; a < mesh->dim; ++a) mx = mesh->n[a] > mx ? mesh->n[a] : mx;
  return (mx + 31) / 32 * 32;
}

}  // namespace

struct islbm {
  int dim, precision;
  int n[3];
  long long nn;
  int q, qf, qg;
  size_t st_bytes;
  double Ra, Pr, Ma, delta;
  std::vector<double> xs[3];   // node coordinates (kept for islbm_set_stencil)
  int stencil;                 // 0 central, 1 upwind
  int npad;
  bool is_slab;                // slab of a larger cavity along the slowest axis (islbm_create_slab)
  islbm_slab slab;
  // fused halo exchange: the neighbour's workspace as mapped in this process, the byte offsets of its ghost layer
  // (first halo plane) in its two ping-pong buffers, and its plane pitch in bytes
  char *peer_base[2];
  size_t peer_ghost_off[2][2];
  size_t peer_pitch_bytes[2];
  size_t peer_flag_off[2];     // the neighbour's step flag of its facing side
  int peer_flip[2];            // neighbour's `cur` XOR ours at connect time (both flip once per step)
  long long steps;             // steps since the last islbm_init / islbm_set_populations
  cudaGraphExec_t graph_exec;  // kGraphSteps captured step kernels (small meshes), valid for buffer parity graph_cur
  int graph_cur;
  cudaStream_t cap_stream;     // private stream the graph is captured on (the caller's may be the legacy stream, which cannot capture)
  islbm_params prm;
  double buoy;
  double T0;               // reference temperature of the buoyancy force
  DevMesh dm;
  NodeParams np;
  DiagParams dp;
  bool uniform;            // every spacing == delta (pure-shift kernel valid)
  char *ws;
  Carve cv;
  cudaStream_t stream;
  int cur;                 // buf[cur] holds S_t (post-collision)
  bool has_state;
  bool other_is_pre;       // buf[1-cur] holds f_t itself (right after init / set)
  bool snap_valid;
  int kernel_choice;       // 0 auto, 1 generic, 2 tiled, 3 uniform shift
  long long launches;
  Tuning tune;
  Plan2 plan2;
  Plan3 plan3;
  PlanC2 planc2;           // multi-step cluster kernel for tiny 2-D fp64 meshes (islbm_cluster2.cuh)
  bool tiled_ok() const { return dim == 2 ? plan2.available : plan3.available; }
  const char *tiled_why_not() const { return dim == 2 ? plan2.why_not : plan3.why_not; }
};

// (re)build the TMA plan of the tiled kernel for the current tuning
static void drop_graph(islbm *h);
static void make_tiled_plan(islbm *h) {
  drop_graph(h);     // the captured launches hold the old tensor maps and launch configuration
  void *b0 = h->ws + h->cv.buf[0], *b1 = h->ws + h->cv.buf[1];
  if (h->dim == 2) {
    if (h->precision == ISLBM_F64) plan2_create<double>(h->plan2, h->n, h->dm.nxp, b0, b1, h->tune, h->stencil);
    else plan2_create<float>(h->plan2, h->n, h->dm.nxp, b0, b1, h->tune, h->stencil);
    h->planc2.available = false;
    if (h->precision == ISLBM_F64 && h->stencil == 0 && !h->is_slab && h->tune.cluster != 2) planc2_create(h->planc2, h->n);
  } else {
    if (h->precision == ISLBM_F64) plan3_create<double>(h->plan3, h->n, h->dm.nxp, b0, b1, h->tune, h->stencil);
    else plan3_create<float>(h->plan3, h->n, h->dm.nxp, b0, b1, h->tune, h->stencil);
  }
}

extern "C" const char *islbm_last_error(void) { return g_err.c_str(); }
extern "C" const char *islbm_version(void) { return "islbm-b200 0.1 (sm_100a)"; }

extern "C" int islbm_workspace_bytes(const islbm_mesh *mesh, int lattice, int precision, size_t *bytes) {
  if (!bytes) return fail(ISLBM_ERR_ARG, "bytes is NULL");
  int rc = check_mesh_args(mesh, lattice, precision);
  if (rc) return rc;
  long long nn = 1;
  for (int a = 0; a < mesh->dim; ++a) nn *= mesh->n[a];
  const int q = mesh->dim == 2 ? 14 : 26;
  const long long nnp = nn / mesh->n[0] * row_pitch(mesh->n[0]);
  *bytes = carve(nn, nnp, q, precision == ISLBM_F64 ? 8 : 4, npad_of(mesh)).total;
  return ISLBM_OK;
}

// Parameter map: PAPER.md:53-72 (free-fall scaling), :248 (Ma = u_f/c_s, c_s = 1/sqrt 3), Table 1
// (:206-212, characteristic length = effective height / minimal resolution), :124 (a_T), :177 (omega).
static int derive_params(islbm *h, const islbm_mesh *mesh) {
  islbm_params &p = h->prm;
  for (int a = 0; a < 3; ++a)
    p.L_eff[a] = a < h->dim ? mesh->x[a][h->n[a] - 1] - mesh->x[a][0] + h->delta : 1.0;
  if (h->is_slab) p.L_eff[h->dim - 1] = h->slab.L_eff_global;   // the whole cavity's extent, not this slab's
  p.U = h->Ma / std::sqrt(3.0);
  p.H_lu = p.L_eff[1] / h->delta;
  p.nu = p.U * p.H_lu * std::sqrt(h->Pr / h->Ra);
  p.alpha = p.nu / h->Pr;
  p.gbeta = p.U * p.U / p.H_lu;
  p.tau_f = 3.0 * p.nu + 0.5;
  p.a_T = h->dim == 2 ? 20.0 * std::sqrt(3.0) * p.alpha - 4.0 : 42.0 * std::sqrt(3.0) * p.alpha - 6.0;
  p.omega_bc = h->dim == 2 ? (4.0 + p.a_T) / 10.0 : (6.0 + p.a_T) / 21.0;
  p.dt_star = p.U / p.H_lu;
  if (!(p.tau_f > 0.5) || !std::isfinite(p.tau_f)) return fail(ISLBM_ERR_PARAM, "tau_f <= 1/2");
  const double lo = h->dim == 2 ? -4.0 : -6.0;
  if (!(p.a_T > lo && p.a_T < 1.0)) {
    char b[160];
    snprintf(b, sizeof b, "a_T = %.6g outside (%g, 1): temperature equilibrium weights would be negative", p.a_T, lo);
    return fail(ISLBM_ERR_PARAM, b);
  }
  return ISLBM_OK;
}

static void drop_graph(islbm *h);
static void set_node_params(islbm *h) {
  drop_graph(h);     // captured launches hold the node parameters by value
  const double tau = h->prm.tau_f;
  NodeParams &np = h->np;
  np.gbeta = h->prm.gbeta * h->buoy;
  np.s_nu = 1.0 / tau;                                   // DESIGN.md A7
  np.s_q = 8.0 * (2.0 * tau - 1.0) / (8.0 * tau - 1.0);
  np.hs_nu = 1.0 - 0.5 * np.s_nu;
  np.hs_q = 1.0 - 0.5 * np.s_q;
  np.q_k = 3.0 - std::sqrt(3.0);
  np.q_e = 4.0 * std::sqrt(3.0) - 6.0;
  np.a_T = h->prm.a_T;
  np.T0 = h->T0;
  fold_node_params(np, h->dim);
  h->dp.T0 = h->T0;
}

// 3-point Lagrange weights of the departure point x_j - c*delta on the
// destination-centred stencil (A2, A3).  Offsets are
// taken relative to x_j so that an exact unit spacing gives exactly (1,0,0)/(0,0,1).
static void build_tables(const islbm *h, const double *const *xs, int stencil, int npad, std::vector<double> &wtab,
                         std::vector<double> &avgw) {
  wtab.assign((size_t)18 * npad, 0.0);
  avgw.assign((size_t)3 * npad, 1.0);
  for (int a = 0; a < h->dim; ++a) {
    const int n = h->n[a];
    const double *x = xs[a];
    for (int s = 0; s < 2; ++s) {
      const double xi = s == 0 ? h->delta : -h->delta;   // c = -1 -> +delta ; c = +1 -> -delta
      for (int j = 0; j < n; ++j) {
        int b = stencil == 0 ? j - 1 : (s == 1 ? j - 2 : j);   // s = 1 is c = +1 (A2 and its alternative)
        if (b < 0) b = 0;
        if (b > n - 3) b = n - 3;
        const double d0 = x[b] - x[j], d1 = x[b + 1] - x[j], d2 = x[b + 2] - x[j];
        double *w = &wtab[(size_t)((a * 2 + s) * 3) * npad + j];
        w[0] = ((xi - d1) * (xi - d2)) / ((d0 - d1) * (d0 - d2));
        w[(size_t)npad] = ((xi - d0) * (xi - d2)) / ((d1 - d0) * (d1 - d2));
        w[(size_t)2 * npad] = ((xi - d0) * (xi - d1)) / ((d2 - d0) * (d2 - d1));
      }
    }
    const bool slab_axis = h->is_slab && a == h->dim - 1;
    for (int j = 0; j < n; ++j) {   // Eq. 29 with ghost points one lattice unit outside (A14)
      const double xm = j == 0 ? x[0] - h->delta : x[j - 1];
      const double xp = j == n - 1 ? x[n - 1] + h->delta : x[j + 1];
      avgw[(size_t)a * npad + j] = 0.5 * (xp - xm);
      // a slab's ghost layers belong to the neighbouring rank: weight 0, so every weighted sum is this rank's share
      if (slab_axis && ((j == 0 && !h->slab.lo_is_wall) || (j == n - 1 && !h->slab.hi_is_wall)))
        avgw[(size_t)a * npad + j] = 0.0;
    }
  }
}

static int upload_tables(islbm *h) {
  std::vector<double> wtab, avgw;
  const double *xs[3] = {h->xs[0].data(), h->xs[1].data(), h->xs[2].data()};
  build_tables(h, xs, h->stencil, h->npad, wtab, avgw);
  CUDA_TRY(cudaMemcpy(h->ws + h->cv.wtab, wtab.data(), wtab.size() * sizeof(double), cudaMemcpyHostToDevice));
  CUDA_TRY(cudaMemcpy(h->ws + h->cv.avgw, avgw.data(), avgw.size() * sizeof(double), cudaMemcpyHostToDevice));
  return ISLBM_OK;
}

static int create_impl(islbm_t **out, const islbm_mesh *mesh, int lattice, double Ra, double Pr, double Ma, int precision,
                       void *dev_workspace, size_t bytes, void *cuda_stream, const islbm_slab *slab);

extern "C" int islbm_create(islbm_t **out, const islbm_mesh *mesh, int lattice, double Ra, double Pr, double Ma,
                            int precision, void *dev_workspace, size_t bytes, void *cuda_stream) {
  return create_impl(out, mesh, lattice, Ra, Pr, Ma, precision, dev_workspace, bytes, cuda_stream, nullptr);
}

extern "C" int islbm_create_slab(islbm_t **out, const islbm_mesh *mesh, int lattice, double Ra, double Pr, double Ma,
                                 int precision, void *dev_workspace, size_t bytes, void *cuda_stream,
                                 const islbm_slab *slab) {
  if (!slab) return fail(ISLBM_ERR_ARG, "slab is NULL");
  if (!(slab->L_eff_global > 0.0) || slab->node_offset < 0) return fail(ISLBM_ERR_ARG, "bad slab description");
  if (mesh && mesh->dim >= 2 && mesh->dim <= 3 &&
      mesh->n[mesh->dim - 1] - (slab->lo_is_wall ? 0 : 1) - (slab->hi_is_wall ? 0 : 1) < 1)
    return fail(ISLBM_ERR_ARG, "a slab needs at least one owned layer besides its ghost layers");
  return create_impl(out, mesh, lattice, Ra, Pr, Ma, precision, dev_workspace, bytes, cuda_stream, slab);
}

static int create_impl(islbm_t **out, const islbm_mesh *mesh, int lattice, double Ra, double Pr, double Ma, int precision,
                       void *dev_workspace, size_t bytes, void *cuda_stream, const islbm_slab *slab) {
  if (!out) return fail(ISLBM_ERR_ARG, "out is NULL");
  *out = nullptr;
  int rc = check_mesh_args(mesh, lattice, precision);
  if (rc) return rc;
  if (!(Ra > 0.0) || !(Pr > 0.0) || !(Ma > 0.0) || !std::isfinite(Ra + Pr + Ma))
    return fail(ISLBM_ERR_PARAM, "Ra, Pr, Ma must be positive and finite");
  if (!(mesh->delta > 0.0)) return fail(ISLBM_ERR_MESH, "delta must be positive");
  bool uniform = true;
  for (int a = 0; a < mesh->dim; ++a) {
    if (!mesh->x[a]) return fail(ISLBM_ERR_ARG, "coordinate array is NULL");
    for (int j = 1; j < mesh->n[a]; ++j) {
      const double d = mesh->x[a][j] - mesh->x[a][j - 1];
      if (!(d > 0.0)) return fail(ISLBM_ERR_MESH, "coordinates must be strictly increasing");
      if (!(d >= mesh->delta * (1.0 - 1e-12)))
        return fail(ISLBM_ERR_MESH, "a mesh spacing is smaller than delta: the departure point would leave the adjacent cell");
      // "uniform" enables the pure-shift kernel on request: spacings equal to delta to within 1e-10 relative (exactly
      // equal for power-of-two N; otherwise the shift differs from the interpolation by that much per step)
      if (std::fabs(d - mesh->delta) > 1e-10 * mesh->delta) uniform = false;
    }
  }
  islbm *h = new islbm();
  h->dim = mesh->dim;
  h->precision = precision;
  h->nn = 1;
  for (int a = 0; a < 3; ++a) {
    h->n[a] = a < mesh->dim ? mesh->n[a] : 1;
    h->nn *= h->n[a];
  }
  h->qf = h->dim == 2 ? 9 : 19;
  h->qg = h->dim == 2 ? 5 : 7;
  h->q = h->qf + h->qg;
  h->st_bytes = precision == ISLBM_F64 ? 8 : 4;
  h->Ra = Ra; h->Pr = Pr; h->Ma = Ma; h->delta = mesh->delta;
  h->is_slab = slab != nullptr;
  if (slab) h->slab = *slab;
  h->buoy = 1.0;
  h->T0 = 0.0;             // BASELINE.json configs: walls at +-0.5, reference = their mean (A9)
  h->uniform = uniform;
  rc = derive_params(h, mesh);
  if (rc) { delete h; return rc; }
  set_node_params(h);
  const int npad = npad_of(mesh);
  const int nxp = row_pitch(h->n[0]);
  const long long nnp = h->nn / h->n[0] * nxp;
  h->cv = carve(h->nn, nnp, h->q, h->st_bytes, npad);
  if (!dev_workspace) { delete h; return fail(ISLBM_ERR_WORKSPACE, "workspace is NULL"); }
  if ((uintptr_t)dev_workspace % kAlign) { delete h; return fail(ISLBM_ERR_WORKSPACE, "workspace must be 256-byte aligned"); }
  if (bytes < h->cv.total) {
    char b[128];
    snprintf(b, sizeof b, "workspace too small: %zu < %zu bytes", bytes, h->cv.total);
    delete h;
    return fail(ISLBM_ERR_WORKSPACE, b);
  }
  h->ws = (char *)dev_workspace;
  h->stream = (cudaStream_t)cuda_stream;
  for (int a = 0; a < h->dim; ++a) h->xs[a].assign(mesh->x[a], mesh->x[a] + h->n[a]);
  h->stencil = 0;
  h->npad = npad;
  rc = upload_tables(h);
  if (rc) { delete h; return rc; }
  DevMesh &dm = h->dm;
  dm.nx = h->n[0]; dm.ny = h->n[1]; dm.nz = h->n[2];
  dm.npad = npad;
  dm.nn = h->nn;
  dm.nxp = nxp;
  dm.nnp = nnp;
  dm.wtab = (const double *)(h->ws + h->cv.wtab);
  dm.avgw = (const double *)(h->ws + h->cv.avgw);
  dm.omega_bc = h->prm.omega_bc;
  dm.T_hot = 0.5;      // PAPER.md:237, 430; BASELINE.json configs (A11)
  dm.T_cold = -0.5;
  dm.stencil = 0;
  dm.peer[0] = dm.peer[1] = nullptr;
  dm.peer_pitch[0] = dm.peer_pitch[1] = 0;
  h->peer_base[0] = h->peer_base[1] = nullptr;
  h->peer_flip[0] = h->peer_flip[1] = 0;
  h->steps = 0;
  h->graph_exec = nullptr;
  h->graph_cur = 0;
  h->cap_stream = nullptr;
  dm.flag_in[0] = dm.flag_in[1] = dm.flag_out[0] = dm.flag_out[1] = nullptr;
  dm.done_cnt = (unsigned long long *)(h->ws + h->cv.flags + 64);
  dm.step = 0;
  dm.bctas = 1;
  {
    const int nm = h->n[h->dim - 1];
    dm.wall_mlo = !slab || slab->lo_is_wall;
    dm.wall_mhi = !slab || slab->hi_is_wall;
    dm.em_lo = dm.wall_mlo ? 0 : 1;
    dm.em_hi = dm.wall_mhi ? nm : nm - 1;
    dm.node_offset = slab ? slab->node_offset : 0;
  }
  h->dp.q_lo = (mesh->x[0][1] - mesh->x[0][0]) / mesh->delta;
  h->dp.q_hi = (mesh->x[0][h->n[0] - 1] - mesh->x[0][h->n[0] - 2]) / mesh->delta;
  h->dp.T0 = h->T0;
  {   // Eq. 33 tables (A23)
    const double *x = mesh->x[0];
    const int nx = h->n[0];
    const double xmid = 0.5 * ((x[0] - 0.5 * mesh->delta) + (x[nx - 1] + 0.5 * mesh->delta));
    int i0 = 1;
    while (i0 < nx - 3 && x[i0 + 1] <= xmid) ++i0;
    double a1 = (xmid - x[i0]) / (x[i0 + 1] - x[i0]);
    if (a1 < 0.0 || nx < 4) a1 = 0.0;
    if (a1 > 1.0) a1 = 1.0;
    h->dp.mid_i = i0;
    h->dp.mid_a[0] = 1.0 - a1;
    h->dp.mid_a[1] = a1;
    for (int k = 0; k < 2; ++k) {
      const int i = i0 + k;
      if (i + 1 > nx - 1) { h->dp.mid_c[k][0] = h->dp.mid_c[k][1] = h->dp.mid_c[k][2] = 0.0; continue; }
      const double hm = (x[i] - x[i - 1]) / mesh->delta, hp = (x[i + 1] - x[i]) / mesh->delta;
      h->dp.mid_c[k][0] = -hp / (hm * (hm + hp));
      h->dp.mid_c[k][1] = (hp - hm) / (hm * hp);
      h->dp.mid_c[k][2] = hm / (hp * (hm + hp));
    }
  }
  h->cur = 0;
  h->has_state = false;
  h->other_is_pre = false;
  h->snap_valid = false;
  h->kernel_choice = 0;
  h->launches = 0;
  if (h->dim == 2) {          // measured on 1024^2 (profiles/): the 2-D states are of the order of the L2
    h->tune.serpentine = 1;   // start each step on the rows the previous step wrote last
    h->tune.store_policy = 2; // keep freshly written populations in L2 (evict_last)
  }
  make_tiled_plan(h);
  *out = h;
  return ISLBM_OK;
}

static void drop_graph(islbm *h);
extern "C" void islbm_destroy(islbm_t *h) {
  if (h) {
    drop_graph(h);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  }
  delete h;
}

extern "C" int islbm_get_params(const islbm_t *h, islbm_params *out) {
  if (!h || !out) return fail(ISLBM_ERR_ARG, "NULL argument");
  *out = h->prm;
  return ISLBM_OK;
}

extern "C" int islbm_set_buoyancy_scale(islbm_t *h, double s) {
  if (!h) return fail(ISLBM_ERR_ARG, "NULL handle");
  if (h->has_state && s != h->buoy)
    return fail(ISLBM_ERR_STATE, "set the buoyancy scale before islbm_init / islbm_set_populations "
                                 "(the stored post-collision state already contains the force)");
  h->buoy = s;
  set_node_params(h);
  return ISLBM_OK;
}

extern "C" int islbm_set_reference_temperature(islbm_t *h, double T0) {
  if (!h) return fail(ISLBM_ERR_ARG, "NULL handle");
  if (!std::isfinite(T0)) return fail(ISLBM_ERR_ARG, "T0 must be finite");
  if (h->has_state && T0 != h->T0)
    return fail(ISLBM_ERR_STATE, "set the reference temperature before islbm_init / islbm_set_populations "
                                 "(the stored post-collision state already contains the force)");
  h->T0 = T0;
  set_node_params(h);
  return ISLBM_OK;
}

extern "C" int islbm_set_stencil(islbm_t *h, int kind) {
  if (!h) return fail(ISLBM_ERR_ARG, "NULL handle");
  if (kind != 0 && kind != 1) return fail(ISLBM_ERR_ARG, "stencil must be 0 (central) or 1 (upwind)");
  if (h->has_state && kind != h->stencil)
    return fail(ISLBM_ERR_STATE, "set the stencil before islbm_init / islbm_set_populations");
  if (kind == 1 && h->is_slab)
    return fail(ISLBM_ERR_ARG, "the upwind stencil reaches two layers upstream: not available on slab handles (one ghost layer)");
  if (kind == 1 && h->kernel_choice == 3) return fail(ISLBM_ERR_ARG, "the pure-shift kernel has no stencil");
  h->stencil = kind;
  h->dm.stencil = kind;
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  make_tiled_plan(h);     // the TMA kernels of the chosen stencil (2-row halo and split z-stencil groups for the upwind one)
  return upload_tables(h);
}

extern "C" long long islbm_launch_count(const islbm_t *h) { return h ? h->launches : 0; }

// ---------------------------------------------------------------------------
// dispatch helpers
// ---------------------------------------------------------------------------
#define DISPATCH(h, CALL)                                                     \
  do {                                                                        \
    if ((h)->dim == 2) {                                                      \
      if ((h)->precision == ISLBM_F64) { CALL(2, double); } else { CALL(2, float); } \
    } else {                                                                  \
      if ((h)->precision == ISLBM_F64) { CALL(3, double); } else { CALL(3, float); } \
    }                                                                         \
  } while (0)

static inline unsigned cdiv(long long a, long long b) { return (unsigned)((a + b - 1) / b); }

static void generic_geometry(const islbm *h, dim3 &grid, dim3 &block) {
  block = h->dim == 2 ? dim3(64, 4, 1) : dim3(32, 4, 2);
  grid = dim3(cdiv(h->n[0], block.x), cdiv(h->n[1], block.y), cdiv(h->n[2], block.z));
}

template <int DIM, typename ST>
static void launch_load(islbm *h, const double *f, const double *g, bool generate, unsigned long long seed, double amp) {
  ST *pre = (ST *)(h->ws + h->cv.buf[1 - h->cur]);
  ST *post = (ST *)(h->ws + h->cv.buf[h->cur]);
  const unsigned blocks = cdiv(h->nn, 256);
  if (generate)
    k_load_state<DIM, ST, true><<<blocks, 256, 0, h->stream>>>(h->dm, h->np, nullptr, nullptr, seed, amp, pre, post, h->nn, 0, h->nn);
  else
    k_load_state<DIM, ST, false><<<blocks, 256, 0, h->stream>>>(h->dm, h->np, f, g, 0ull, 0.0, pre, post, h->nn, 0, h->nn);
  h->launches++;
}

// one staged slab of islbm_set_populations_host: nodes [c0, c0 + count), staging planes at pitch `pitch`
template <int DIM, typename ST>
static void launch_load_slab(islbm *h, const double *stage_f, const double *stage_g, long long pitch, long long c0,
                             long long count) {
  ST *pre = (ST *)(h->ws + h->cv.buf[1 - h->cur]);
  ST *post = (ST *)(h->ws + h->cv.buf[h->cur]);
  k_load_state<DIM, ST, false><<<cdiv(count, 256), 256, 0, h->stream>>>(h->dm, h->np, stage_f, stage_g, 0ull, 0.0, pre, post,
                                                                      pitch, c0, count);
  h->launches++;
}

static int load_state(islbm *h, const double *f, const double *g, bool generate, unsigned long long seed, double amp) {
#define CALL(D, T) launch_load<D, T>(h, f, g, generate, seed, amp)
  DISPATCH(h, CALL);
#undef CALL
  CUDA_TRY(cudaPeekAtLastError());
  h->has_state = true;
  h->other_is_pre = true;
  h->snap_valid = false;
  h->steps = 0;
  h->peer_base[0] = h->peer_base[1] = nullptr;   // a new state: the neighbours must be connected again
  return ISLBM_OK;
}

extern "C" int islbm_init(islbm_t *h, unsigned long long seed, double noise_amp) {
  if (!h) return fail(ISLBM_ERR_ARG, "NULL handle");
  return load_state(h, nullptr, nullptr, true, seed, noise_amp);
}

extern "C" int islbm_set_populations(islbm_t *h, const double *f, const double *g) {
  if (!h || !f || !g) return fail(ISLBM_ERR_ARG, "NULL argument");
  return load_state(h, f, g, false, 0ull, 0.0);
}

// HOST arrays: staged through the snapshot area of the workspace (4*nn doubles) in slabs of nodes; per slab one
// H2D copy per plane and one conversion + collision kernel, all on the handle's stream.
extern "C" int islbm_set_populations_host(islbm_t *h, const double *f, const double *g) {
  if (!h || !f || !g) return fail(ISLBM_ERR_ARG, "NULL argument");
  double *stage = (double *)(h->ws + h->cv.snap);
  long long slab = (4 * h->nn) / h->q;              // nodes per slab: q planes of `slab` doubles fit the staging area
  if (slab < 1) return fail(ISLBM_ERR_WORKSPACE, "staging area too small");
  if (slab > h->nn) slab = h->nn;
  for (long long c0 = 0; c0 < h->nn; c0 += slab) {
    const long long count = c0 + slab <= h->nn ? slab : h->nn - c0;
    for (int q = 0; q < h->qf; ++q)
      CUDA_TRY(cudaMemcpyAsync(stage + (long long)q * slab, f + (long long)q * h->nn + c0, sizeof(double) * count,
                               cudaMemcpyHostToDevice, h->stream));
    for (int q = 0; q < h->qg; ++q)
      CUDA_TRY(cudaMemcpyAsync(stage + (long long)(h->qf + q) * slab, g + (long long)q * h->nn + c0, sizeof(double) * count,
                               cudaMemcpyHostToDevice, h->stream));
#define CALL(D, T) launch_load_slab<D, T>(h, stage, stage + (long long)h->qf * slab, slab, c0, count)
    DISPATCH(h, CALL);
#undef CALL
  }
  CUDA_TRY(cudaPeekAtLastError());
  h->has_state = true;
  h->other_is_pre = true;
  h->snap_valid = false;
  h->steps = 0;
  h->peer_base[0] = h->peer_base[1] = nullptr;
  return ISLBM_OK;
}

template <int DIM, typename ST>
static void launch_generic_step(islbm *h, bool collide, double *fout, double *gout) {
  dim3 grid, block;
  generic_geometry(h, grid, block);
  if (collide) {
    const ST *src = (const ST *)(h->ws + h->cv.buf[h->cur]);
    ST *dst = (ST *)(h->ws + h->cv.buf[1 - h->cur]);
    k_step_generic<DIM, ST, true><<<grid, block, 0, h->stream>>>(h->dm, h->np, src, dst, nullptr, nullptr);
  } else {
    const ST *src = (const ST *)(h->ws + h->cv.buf[1 - h->cur]);
    k_step_generic<DIM, ST, false><<<grid, block, 0, h->stream>>>(h->dm, h->np, src, nullptr, fout, gout);
  }
  h->launches++;
}

template <int DIM, typename ST>
static void launch_shift_step(islbm *h) {
  dim3 grid, block;
  generic_geometry(h, grid, block);
  const ST *src = (const ST *)(h->ws + h->cv.buf[h->cur]);
  ST *dst = (ST *)(h->ws + h->cv.buf[1 - h->cur]);
  k_step_shift<DIM, ST><<<grid, block, 0, h->stream>>>(h->dm, h->np, src, dst);
  h->launches++;
}

static int effective_kernel(const islbm *h) {
  if (h->kernel_choice != 0) return h->kernel_choice;
  return h->tiled_ok() ? 2 : 1;
}

extern "C" const char *islbm_kernel_name(const islbm_t *h) {
  if (!h) return "";
  switch (effective_kernel(h)) {
    case 2:
      if (h->stencil) return h->dim == 2 ? "tiled_ymarch_tma_upwind" : "tiled_zmarch_tma_upwind";
      return h->dim == 2 ? (h->plan2.tx == 224 ? "tiled_ymarch_tma_tx224" : "tiled_ymarch_tma_tx128") : "tiled_zmarch_tma";
    case 3: return "uniform_shift";
    default: return "generic_global";
  }
}

extern "C" int islbm_set_kernel(islbm_t *h, int which) {
  if (!h) return fail(ISLBM_ERR_ARG, "NULL handle");
  if (which < 0 || which > 3) return fail(ISLBM_ERR_ARG, "kernel selector must be 0..3");
  if (which == 3 && h->stencil != 0) return fail(ISLBM_ERR_ARG, "the pure-shift kernel has no stencil");
  if (which == 2 && !h->tiled_ok()) return fail(ISLBM_ERR_ARG, std::string("tiled kernel not available: ") + h->tiled_why_not());
  if (which == 3 && !h->uniform) return fail(ISLBM_ERR_ARG, "uniform-shift kernel needs every spacing to equal delta");
  h->kernel_choice = which;
  return ISLBM_OK;
}

extern "C" int islbm_set_tuning(islbm_t *h, const char *key, int value) {
  if (!h || !key) return fail(ISLBM_ERR_ARG, "NULL argument");
  const std::string k(key);
  if (value < 0) return fail(ISLBM_ERR_ARG, "tuning values are non-negative");
  Tuning &t = h->tune;
  if (k == "chunk") t.chunk = value;
  else if (k == "l2promo") t.l2promo = value;
  else if (k == "load_policy") t.load_policy = value;
  else if (k == "store_policy") t.store_policy = value;
  else if (k == "tx2d") { if (value != 0 && value != 128 && value != 224) return fail(ISLBM_ERR_ARG, "tx2d must be 0, 128 or 224"); t.tx2d = value; }
  else if (k == "serpentine") t.serpentine = value;
  else if (k == "shape3d") { if (value > 5) return fail(ISLBM_ERR_ARG, "shape3d must be 0 (automatic) .. 5"); t.shape3d = value; }
  else if (k == "pdl") t.pdl = value;
  else if (k == "fill") { if (value > 2) return fail(ISLBM_ERR_ARG, "fill must be 0 (automatic), 1 (early) or 2 (late)"); t.fill = value; }
  else if (k == "ring2d") { if (value != 0 && value != 3 && value != 4) return fail(ISLBM_ERR_ARG, "ring2d must be 0 (automatic), 3 or 4"); t.ring2d = value; }
  else if (k == "rows2d") { if (value > kMaxChunk) return fail(ISLBM_ERR_ARG, "rows2d must be at most 64"); t.rows2d = value; }
  else if (k == "rows2d1") { if (value > kMaxChunk) return fail(ISLBM_ERR_ARG, "rows2d1 must be at most 64"); t.rows2d1 = value; }
  else if (k == "graph") { if (value > 2) return fail(ISLBM_ERR_ARG, "graph must be 0 (automatic), 1 (always) or 2 (never)"); t.graph = value; }
  else if (k == "slab_wait_ms") t.slab_wait_ms = value;
  else if (k == "cluster") { if (value != 0 && value != 2) return fail(ISLBM_ERR_ARG, "cluster must be 0 (automatic) or 2 (never)"); t.cluster = value; }
  else if (k == "walls") { if (value > 1) return fail(ISLBM_ERR_ARG, "walls must be 0 (fused) or 1 (separate boundary kernel)"); t.walls = value; }
  else return fail(ISLBM_ERR_ARG, "unknown tuning key: " + k);
  make_tiled_plan(h);
  return ISLBM_OK;
}

// enqueue ONE time step on the handle's stream (kernel `which` of effective_kernel)
static int enqueue_one_step(islbm *h, int which, bool fused) {
  // fused halo exchange: this step writes buffer 1 - cur; the neighbour's `cur` is ours XOR the parity difference
  // recorded at connect time (both flip once per step), and it reads the ghost layer we store from ITS buffer
  // 1 - cur in its next step
  for (int sd = 0; sd < 2; ++sd) {
    const bool on = h->peer_base[sd] != nullptr;
    const int peer_cur = h->cur ^ h->peer_flip[sd];
    h->dm.peer[sd] = on ? (void *)(h->peer_base[sd] + h->peer_ghost_off[sd][1 - peer_cur]) : nullptr;
    h->dm.peer_pitch[sd] = on ? (long long)(h->peer_pitch_bytes[sd] / h->st_bytes) : 0;
    h->dm.flag_in[sd] = on ? (unsigned long long *)(h->ws + h->cv.flags) + sd : nullptr;
    h->dm.flag_out[sd] = on ? (unsigned long long *)(h->peer_base[sd] + h->peer_flag_off[sd]) : nullptr;
  }
  h->dm.step = (unsigned long long)h->steps + 1ull;
  h->dm.wait_ns = (unsigned long long)h->tune.slab_wait_ms * 1000000ull;
  if (fused && which != 2) {
    k_slab_wait<<<1, 1, 0, h->stream>>>(h->dm);
    h->launches++;
  }
  if (which == 2) {
    void *bufs[2] = {h->ws + h->cv.buf[0], h->ws + h->cv.buf[1]};
    cudaError_t e;
    if (h->dim == 2)
      e = h->precision == ISLBM_F64 ? launch2<double>(h->plan2, h->n, h->dm, h->np, h->cur, bufs, h->tune, h->stream)
                                    : launch2<float>(h->plan2, h->n, h->dm, h->np, h->cur, bufs, h->tune, h->stream);
    else
      e = h->precision == ISLBM_F64 ? launch3<double>(h->plan3, h->n, h->dm, h->np, h->cur, bufs, h->tune, h->stream)
                                    : launch3<float>(h->plan3, h->n, h->dm, h->np, h->cur, bufs, h->tune, h->stream);
    if (e != cudaSuccess) return fail(ISLBM_ERR_CUDA, std::string("tiled step launch: ") + cudaGetErrorString(e));
    h->launches += (h->dim == 3 && h->tune.walls == 1 && !h->is_slab && h->stencil == 0) ? 2 : 1;
  } else if (which == 3) {
#define CALL(D, T) launch_shift_step<D, T>(h)
    DISPATCH(h, CALL);
#undef CALL
  } else {
#define CALL(D, T) launch_generic_step<D, T>(h, true, nullptr, nullptr)
    DISPATCH(h, CALL);
#undef CALL
  }
  if (fused && which != 2) {
    k_slab_publish<<<1, 1, 0, h->stream>>>(h->dm);
    h->launches++;
  }
  h->cur ^= 1;
  h->steps++;
  h->other_is_pre = false;
  return ISLBM_OK;
}

static void drop_graph(islbm *h) {
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  h->graph_exec = nullptr;
}

// Small meshes (a step kernel of a few microseconds): kGraphSteps consecutive step kernels, PDL-chained, are captured
// once into a CUDA graph and replayed, so that islbm_step(n) costs n / kGraphSteps host launches instead of n (the
// 64^2 mesh of BASELINE.json config 1 is bound by the host's launch rate otherwise).  The graph holds an even number
// of steps, so it always starts on the same ping-pong buffer parity it was captured on.  Automatic up to 2^20 nodes:
// measured gain 13-23 % at 64^2, 6-8 % at 512^2, 1-3 % at 1024^2, none from 128^3 on (profiles/attempts.md).
constexpr int kGraphSteps = 32;
static bool graph_eligible(const islbm *h, int which, bool fused) {
  return which == 2 && !fused && h->tune.graph != 2 && (h->tune.graph == 1 || h->nn <= (1LL << 20));
}

extern "C" int islbm_step(islbm_t *h, int n) {
  if (!h) return fail(ISLBM_ERR_ARG, "NULL handle");
  if (n < 0) return fail(ISLBM_ERR_ARG, "n < 0");
  if (!h->has_state) return fail(ISLBM_ERR_STATE, "islbm_step before islbm_init / islbm_set_populations");
  const int which = effective_kernel(h);
  if ((h->peer_base[0] || h->peer_base[1]) && which == 3)
    return fail(ISLBM_ERR_STATE, "the fused halo exchange is not available with the pure-shift kernel");
  const bool fused = h->peer_base[0] || h->peer_base[1];
  int left = n;
  // tiny 2-D fp64 meshes: all n steps in ONE launch of a thread-block cluster, state in distributed shared memory
  if (left >= 2 && which == 2 && !fused && h->dim == 2 && h->planc2.available && h->tune.cluster != 2) {
    double *srcb = (double *)(h->ws + h->cv.buf[h->cur]);     // rewritten at the end with the state of step n-1
    double *dstb = (double *)(h->ws + h->cv.buf[1 - h->cur]);
    const cudaError_t e = launch_cluster2(h->planc2, h->dm, h->np, srcb, dstb, left, h->stream);
    if (e != cudaSuccess) return fail(ISLBM_ERR_CUDA, std::string("cluster step launch: ") + cudaGetErrorString(e));
    h->launches++;
    h->cur ^= 1;
    h->steps += left;
    h->other_is_pre = false;
    left = 0;
  }
  if (left >= kGraphSteps && graph_eligible(h, which, fused)) {
    if (h->graph_exec && h->graph_cur != h->cur) drop_graph(h);
    if (!h->graph_exec) {
      cudaGraph_t g = nullptr;
      const long long l0 = h->launches, s0 = h->steps;
      const int c0 = h->cur;
      const bool pre0 = h->other_is_pre;
      if (!h->cap_stream) CUDA_TRY(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
      cudaStream_t user = h->stream;
      CUDA_TRY(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
      h->stream = h->cap_stream;       // the launches of the capture go to the private stream ...
      int rc = ISLBM_OK;
      for (int s = 0; s < kGraphSteps && rc == ISLBM_OK; ++s) rc = enqueue_one_step(h, which, false);
      h->stream = user;                // ... the graph itself is launched on the caller's
      const cudaError_t ec = cudaStreamEndCapture(h->cap_stream, &g);
      h->launches = l0; h->steps = s0; h->cur = c0; h->other_is_pre = pre0;      // nothing has run yet
      if (rc != ISLBM_OK || ec != cudaSuccess || !g) {
        if (g) cudaGraphDestroy(g);
        cudaGetLastError();
        return rc != ISLBM_OK ? rc : fail(ISLBM_ERR_CUDA, std::string("graph capture: ") + cudaGetErrorString(ec));
      }
      const cudaError_t ei = cudaGraphInstantiate(&h->graph_exec, g, 0);
      cudaGraphDestroy(g);
      if (ei != cudaSuccess) { h->graph_exec = nullptr; return fail(ISLBM_ERR_CUDA, std::string("graph instantiate: ") + cudaGetErrorString(ei)); }
      h->graph_cur = h->cur;
    }
    while (left >= kGraphSteps) {
      CUDA_TRY(cudaGraphLaunch(h->graph_exec, h->stream));
      h->launches += kGraphSteps;
      h->steps += kGraphSteps;
      h->other_is_pre = false;
      left -= kGraphSteps;           // an even number of steps: `cur` is unchanged
    }
  }
  for (int s = 0; s < left; ++s) {
    const int rc = enqueue_one_step(h, which, fused);
    if (rc) return rc;
  }
  CUDA_TRY(cudaPeekAtLastError());
  return ISLBM_OK;
}

template <int DIM, typename ST>
static void launch_export(islbm *h, double *f, double *g) {
  const ST *buf = (const ST *)(h->ws + h->cv.buf[1 - h->cur]);
  k_export<DIM, ST><<<cdiv(h->nn, 256), 256, 0, h->stream>>>(h->dm, buf, f, g);
  h->launches++;
}

extern "C" int islbm_get_populations(islbm_t *h, double *f, double *g) {
  if (!h || !f || !g) return fail(ISLBM_ERR_ARG, "NULL argument");
  if (!h->has_state) return fail(ISLBM_ERR_STATE, "no state");
  if (h->other_is_pre) {
#define CALL(D, T) launch_export<D, T>(h, f, g)
    DISPATCH(h, CALL);
#undef CALL
  } else {
    // f_t = stream/interpolate/walls(S_{t-1}); the previous ping-pong buffer is intact
#define CALL(D, T) launch_generic_step<D, T>(h, false, f, g)
    DISPATCH(h, CALL);
#undef CALL
  }
  CUDA_TRY(cudaPeekAtLastError());
  return ISLBM_OK;
}

template <int DIM, typename ST>
static void launch_fields(islbm *h, double *rho, double *u, double *v, double *w, double *T) {
  const ST *S = (const ST *)(h->ws + h->cv.buf[h->cur]);
  k_fields<DIM, ST><<<cdiv(h->nn, 256), 256, 0, h->stream>>>(h->dm, h->np, S, rho, u, v, w, T);
  h->launches++;
}

extern "C" int islbm_fields(islbm_t *h, double *rho, double *u, double *v, double *w, double *T) {
  if (!h) return fail(ISLBM_ERR_ARG, "NULL handle");
  if (!h->has_state) return fail(ISLBM_ERR_STATE, "no state");
#define CALL(D, T_) launch_fields<D, T_>(h, rho, u, v, w, T)
  DISPATCH(h, CALL);
#undef CALL
  CUDA_TRY(cudaPeekAtLastError());
  return ISLBM_OK;
}

static int red_blocks(const islbm *h) {
  long long b = (h->nn + kRedThreads - 1) / kRedThreads;
  const long long cap = std::min<long long>(kMaxRedBlocks, 8LL * sm_count());
  return (int)(b < cap ? b : cap);
}

template <int DIM, typename ST>
static void launch_nusselt(islbm *h, int nb) {
  const ST *S = (const ST *)(h->ws + h->cv.buf[h->cur]);
  double *partial = (double *)(h->ws + h->cv.partial);
  k_nusselt_partial<DIM, ST><<<nb, kRedThreads, 0, h->stream>>>(h->dm, h->np, h->dp, S, partial);
  k_reduce_final<<<1, kRedThreads, 0, h->stream>>>(partial, nb, (double *)(h->ws + h->cv.red_out));
  h->launches += 2;
}

// one pass of the Nu / Re reduction; s[kRedSlots] on the host, stream synchronised
static int run_diag_reduction(islbm *h, double *s) {
  const int nb = red_blocks(h);
#define CALL(D, T) launch_nusselt<D, T>(h, nb)
  DISPATCH(h, CALL);
#undef CALL
  CUDA_TRY(cudaPeekAtLastError());
  CUDA_TRY(cudaMemcpyAsync(s, h->ws + h->cv.red_out, sizeof(double) * kRedSlots, cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return ISLBM_OK;
}

// ---- slab decomposition: halo layout, partial sums -----------------------------------------------------------
extern "C" int islbm_halo(islbm_t *h, int side, islbm_halo_info *out) {
  if (!h || !out) return fail(ISLBM_ERR_ARG, "NULL argument");
  if (side != 0 && side != 1) return fail(ISLBM_ERR_ARG, "side must be 0 (low) or 1 (high)");
  const int nm = h->n[h->dim - 1];
  const size_t layer = (size_t)h->dm.nxp * (h->dim == 3 ? h->n[1] : 1) * h->st_bytes;
  out->first_plane = h->dim == 2 ? 6 : 14;     // the planes with a velocity component along the slab axis
  out->n_planes = h->dim == 2 ? 8 : 12;
  out->plane_pitch_bytes = (size_t)h->dm.nnp * h->st_bytes;
  out->layer_bytes = layer;
  out->is_wall = side == 0 ? h->dm.wall_mlo : h->dm.wall_mhi;
  const size_t base = h->cv.buf[h->cur] + (size_t)out->first_plane * out->plane_pitch_bytes;
  const int send_layer = side == 0 ? h->dm.em_lo : h->dm.em_hi - 1;
  const int recv_layer = side == 0 ? 0 : nm - 1;
  out->send_offset = base + (size_t)send_layer * layer;
  out->recv_offset = base + (size_t)recv_layer * layer;
  return ISLBM_OK;
}

extern "C" int islbm_halo_layout(islbm_t *h, int side, islbm_halo_layout_info *out) {
  if (!h || !out) return fail(ISLBM_ERR_ARG, "NULL argument");
  if (side != 0 && side != 1) return fail(ISLBM_ERR_ARG, "side must be 0 (low) or 1 (high)");
  const int nm = h->n[h->dim - 1];
  const size_t layer = (size_t)h->dm.nxp * (h->dim == 3 ? h->n[1] : 1) * h->st_bytes;
  const size_t pitch = (size_t)h->dm.nnp * h->st_bytes;
  const int first = h->dim == 2 ? 6 : 14;
  out->is_wall = side == 0 ? h->dm.wall_mlo : h->dm.wall_mhi;
  out->plane_pitch_bytes = pitch;
  out->layer_bytes = layer;
  out->cur = h->cur;
  out->steps = h->steps;
  out->flag_offset = h->cv.flags + 8 * (size_t)side;
  for (int b = 0; b < 2; ++b)
    out->ghost_offset[b] = h->cv.buf[b] + (size_t)first * pitch + (size_t)(side == 0 ? 0 : nm - 1) * layer;
  return ISLBM_OK;
}

extern "C" int islbm_slab_set_peer(islbm_t *h, int side, void *peer_workspace, const islbm_halo_layout_info *pl) {
  if (!h) return fail(ISLBM_ERR_ARG, "NULL handle");
  if (side != 0 && side != 1) return fail(ISLBM_ERR_ARG, "side must be 0 (low) or 1 (high)");
  if (!h->is_slab) return fail(ISLBM_ERR_STATE, "not a slab handle");
  if (side == 0 ? h->dm.wall_mlo : h->dm.wall_mhi) return fail(ISLBM_ERR_ARG, "this side is a wall: it has no neighbour");
  if (!peer_workspace) {                               // detach (exchange outside the kernel again)
    h->peer_base[side] = nullptr;
    return ISLBM_OK;
  }
  if (!pl || pl->plane_pitch_bytes == 0 || pl->plane_pitch_bytes % h->st_bytes || pl->is_wall || (pl->cur != 0 && pl->cur != 1))
    return fail(ISLBM_ERR_ARG, "bad peer layout");
  if (pl->steps != h->steps)
    return fail(ISLBM_ERR_STATE, "the neighbour has taken a different number of steps: both slabs must be connected "
                                 "at the same step count (the step flags count steps)");
  // our flag of this side starts at the common step count: "the neighbour has finished step `steps`"
  const unsigned long long init = (unsigned long long)h->steps;
  CUDA_TRY(cudaMemcpyAsync(h->ws + h->cv.flags + 8 * (size_t)side, &init, 8, cudaMemcpyHostToDevice, h->stream));
  CUDA_TRY(cudaMemsetAsync(h->ws + h->cv.flags + 64 + 8 * (size_t)side, 0, 8, h->stream));   // done counter
  CUDA_TRY(cudaMemsetAsync(h->ws + h->cv.flags + 64 + 16, 0, 8, h->stream));                  // time-out counter
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  h->peer_base[side] = (char *)peer_workspace;
  h->peer_ghost_off[side][0] = pl->ghost_offset[0];
  h->peer_ghost_off[side][1] = pl->ghost_offset[1];
  h->peer_pitch_bytes[side] = pl->plane_pitch_bytes;
  h->peer_flag_off[side] = pl->flag_offset;
  h->peer_flip[side] = pl->cur ^ h->cur;
  return ISLBM_OK;
}

// fused slab exchange: did a step kernel give up waiting for a neighbour's flag?  (stream already synchronised)
static int check_slab_timeouts(islbm *h) {
  if (!h->peer_base[0] && !h->peer_base[1]) return ISLBM_OK;
  unsigned long long n = 0;
  CUDA_TRY(cudaMemcpyAsync(&n, h->ws + h->cv.flags + 64 + 16, 8, cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (n) {
    char b[256];
    snprintf(b, sizeof b, "fused slab exchange: %llu boundary CTA(s) gave up waiting for a neighbour's step flag after %d ms "
                          "(neighbour not stepping, or connected at a different step count): this rank's state is invalid", n,
             h->tune.slab_wait_ms);
    return fail(ISLBM_ERR_STATE, b);
  }
  return ISLBM_OK;
}

extern "C" int islbm_diag_sums(islbm_t *h, double s[8]) {
  if (!h || !s) return fail(ISLBM_ERR_ARG, "NULL argument");
  if (!h->has_state) return fail(ISLBM_ERR_STATE, "no state");
  double t[kRedSlots];
  int rc = run_diag_reduction(h, t);
  if (rc) return rc;
  rc = check_slab_timeouts(h);
  if (rc) return rc;
  for (int i = 0; i < 8; ++i) s[i] = i < kRedSlots ? t[i] : 0.0;
  return ISLBM_OK;
}

extern "C" int islbm_diag_from_sums(const islbm_t *h, const double s[8], double out[6]) {
  if (!h || !s || !out) return fail(ISLBM_ERR_ARG, "NULL argument");
  const islbm_params &p = h->prm;
  const double area = p.L_eff[1] * (h->dim == 3 ? p.L_eff[2] : 1.0);
  const double vol = area * p.L_eff[0];
  out[0] = -p.H_lu * s[0] / area;
  out[1] = -p.H_lu * s[1] / area;
  out[2] = std::sqrt(h->Ra / h->Pr) * (s[2] / vol) / p.U;
  out[3] = (s[3] / vol) / (p.U * p.U);
  out[4] = std::sqrt(h->Ra * h->Pr) * (s[4] / vol) / p.U + 1.0;
  out[5] = std::sqrt(h->Ra * h->Pr) * (s[5] / area) / p.U - p.H_lu * (s[6] / area);
  for (int i = 0; i < 6; ++i)
    if (!std::isfinite(out[i])) return fail(ISLBM_ERR_NONFINITE, "non-finite diagnostic: the run has diverged");
  return ISLBM_OK;
}

extern "C" int islbm_nusselt_middle(islbm_t *h, double *out) {
  if (!h || !out) return fail(ISLBM_ERR_ARG, "NULL argument");
  if (h->is_slab) return fail(ISLBM_ERR_STATE, "slab handle: use islbm_diag_sums, sum over ranks, islbm_diag_from_sums");
  if (!h->has_state) return fail(ISLBM_ERR_STATE, "no state");
  double s[kRedSlots];
  int rc = run_diag_reduction(h, s);
  if (rc) return rc;
  const islbm_params &p = h->prm;
  const double area = p.L_eff[1] * (h->dim == 3 ? p.L_eff[2] : 1.0);
  *out = std::sqrt(h->Ra * h->Pr) * (s[5] / area) / p.U - p.H_lu * (s[6] / area);
  if (!std::isfinite(*out)) return fail(ISLBM_ERR_NONFINITE, "non-finite diagnostic: the run has diverged");
  return ISLBM_OK;
}

extern "C" int islbm_nusselt(islbm_t *h, double out[5]) {
  if (!h || !out) return fail(ISLBM_ERR_ARG, "NULL argument");
  if (h->is_slab) return fail(ISLBM_ERR_STATE, "slab handle: use islbm_diag_sums, sum over ranks, islbm_diag_from_sums");
  if (!h->has_state) return fail(ISLBM_ERR_STATE, "no state");
  double s[kRedSlots];
  int rc = run_diag_reduction(h, s);
  if (rc) return rc;
  const islbm_params &p = h->prm;
  const double area = p.L_eff[1] * (h->dim == 3 ? p.L_eff[2] : 1.0);
  const double vol = area * p.L_eff[0];
  out[0] = -p.H_lu * s[0] / area;
  out[1] = -p.H_lu * s[1] / area;
  out[2] = std::sqrt(h->Ra / h->Pr) * (s[2] / vol) / p.U;
  out[3] = (s[3] / vol) / (p.U * p.U);
  out[4] = std::sqrt(h->Ra * h->Pr) * (s[4] / vol) / p.U + 1.0;
  for (int i = 0; i < 5; ++i)
    if (!std::isfinite(out[i])) return fail(ISLBM_ERR_NONFINITE, "non-finite diagnostic: the run has diverged");
  return ISLBM_OK;
}

// ---------------------------------------------------------------------------
// islbm_nusselt_static: the Nu / Re reduction with NO allocation and no use of the workspace's scratch areas.
// Its scratch (one partial sum per block and slot, and the 8 result slots) is the file-scope array below, which every
// GPU that loads this library holds until exit: kStaticRedBlocks * kRedSlots + 8 doubles = 114 752 bytes.
// Each block reduces a FIXED share of kStaticNodesPerBlock nodes, so the number of blocks (and with it the order of
// the summation) depends on the mesh alone, not on the GPU; meshes beyond kStaticRedBlocks * kStaticNodesPerBlock
// = 33 554 432 nodes are refused.  Every partial and result slot is written by each call before it is read, so
// nothing has to start at zero; the array keeps the last call's contents.  All calls on a device share the array:
// calls that overlap on the GPU (different streams, different handles) race.
// ---------------------------------------------------------------------------
constexpr int kStaticRedBlocks = 2048;
constexpr long long kStaticNodesPerBlock = 16384;     // 64 nodes per thread of a 256-thread block
static __device__ __align__(256) double g_static_red[kStaticRedBlocks * kRedSlots + 8];

// Device address of g_static_red on the CURRENT device.  In host code the array's name is only a stand-in for the
// symbol, not a device address: it is resolved once per device with cudaGetSymbolAddress (no allocation) and cached.
static int static_scratch_ptr(double **out) {
  constexpr int kMaxDev = 64;
  static double *cache[kMaxDev] = {};
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDev) return fail(ISLBM_ERR_CUDA, "device ordinal beyond the static-scratch table");
  if (!cache[dev]) {
    double *p = nullptr;
    CUDA_TRY(cudaGetSymbolAddress((void **)&p, g_static_red));
    if (!p) return fail(ISLBM_ERR_CUDA, "cudaGetSymbolAddress returned a null address for the static scratch");
    cache[dev] = p;      // racing first calls on one device write the same value
  }
  *out = cache[dev];
  return ISLBM_OK;
}

template <int DIM, typename ST>
static void launch_nusselt_static(islbm *h, int nb, double *scratch) {
  const ST *S = (const ST *)(h->ws + h->cv.buf[h->cur]);
  double *partial = scratch, *result = scratch + (size_t)kStaticRedBlocks * kRedSlots;
  k_nusselt_partial<DIM, ST><<<nb, kRedThreads, 0, h->stream>>>(h->dm, h->np, h->dp, S, partial);
  k_reduce_final<<<1, kRedThreads, 0, h->stream>>>(partial, nb, result);
  h->launches += 2;
}

extern "C" int islbm_nusselt_static(islbm_t *h, double out[5]) {
  if (!h || !out) return fail(ISLBM_ERR_ARG, "NULL argument");
  if (h->is_slab) return fail(ISLBM_ERR_STATE, "slab handle: use islbm_diag_sums, sum over ranks, islbm_diag_from_sums");
  if (h->nn > (long long)kStaticRedBlocks * kStaticNodesPerBlock) {
    char b[160];
    snprintf(b, sizeof b, "islbm_nusselt_static: %lld nodes exceed the static scratch (at most %lld nodes); use islbm_nusselt",
             h->nn, (long long)kStaticRedBlocks * kStaticNodesPerBlock);
    return fail(ISLBM_ERR_ARG, b);
  }
  if (!h->has_state) return fail(ISLBM_ERR_STATE, "no state");
  double *scratch = nullptr;
  int rc = static_scratch_ptr(&scratch);
  if (rc) return rc;
  const int nb = (int)((h->nn + kStaticNodesPerBlock - 1) / kStaticNodesPerBlock);
#define CALL(D, T) launch_nusselt_static<D, T>(h, nb, scratch)
  DISPATCH(h, CALL);
#undef CALL
  CUDA_TRY(cudaPeekAtLastError());
  double s[kRedSlots];
  CUDA_TRY(cudaMemcpyAsync(s, scratch + (size_t)kStaticRedBlocks * kRedSlots, sizeof s, cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  const islbm_params &p = h->prm;
  const double area = p.L_eff[1] * (h->dim == 3 ? p.L_eff[2] : 1.0);
  const double vol = area * p.L_eff[0];
  out[0] = -p.H_lu * s[0] / area;
  out[1] = -p.H_lu * s[1] / area;
  out[2] = std::sqrt(h->Ra / h->Pr) * (s[2] / vol) / p.U;
  out[3] = (s[3] / vol) / (p.U * p.U);
  out[4] = std::sqrt(h->Ra * h->Pr) * (s[4] / vol) / p.U + 1.0;
  for (int i = 0; i < 5; ++i)
    if (!std::isfinite(out[i])) return fail(ISLBM_ERR_NONFINITE, "non-finite diagnostic: the run has diverged");
  return ISLBM_OK;
}

template <int DIM, typename ST>
static void launch_residual(islbm *h, int nb) {
  const ST *S = (const ST *)(h->ws + h->cv.buf[h->cur]);
  double *partial = (double *)(h->ws + h->cv.partial);
  k_residual_partial<DIM, ST><<<nb, kRedThreads, 0, h->stream>>>(h->dm, h->np, S, (double *)(h->ws + h->cv.snap), partial);
  k_reduce_final<<<1, kRedThreads, 0, h->stream>>>(partial, nb, (double *)(h->ws + h->cv.red_out));
  h->launches += 2;
}

// Eq. 30 sums between the current fields and the snapshot (which the kernel then overwrites): s[0..3] =
// sum|u-u_prev|_2, sum|u_prev|_2, sum|T-T_prev|, sum|T_prev| over the owned nodes; *first = no snapshot existed.
static int run_residual(islbm *h, double s[4], bool *first) {
  if (!h->snap_valid) CUDA_TRY(cudaMemsetAsync(h->ws + h->cv.snap, 0, sizeof(double) * 4 * (size_t)h->nn, h->stream));
  const int nb = red_blocks(h);
#define CALL(D, T) launch_residual<D, T>(h, nb)
  DISPATCH(h, CALL);
#undef CALL
  CUDA_TRY(cudaPeekAtLastError());
  double t[kRedSlots];
  CUDA_TRY(cudaMemcpyAsync(t, h->ws + h->cv.red_out, sizeof t, cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  for (int i = 0; i < 4; ++i) s[i] = t[i];
  *first = !h->snap_valid;
  h->snap_valid = true;
  return ISLBM_OK;
}

extern "C" int islbm_residual_sums(islbm_t *h, double s[4], int *first) {
  if (!h || !s || !first) return fail(ISLBM_ERR_ARG, "NULL argument");
  if (!h->has_state) return fail(ISLBM_ERR_STATE, "no state");
  bool f = false;
  int rc = run_residual(h, s, &f);
  *first = f ? 1 : 0;
  if (rc == ISLBM_OK) rc = check_slab_timeouts(h);
  return rc;
}

extern "C" int islbm_steady_residual(islbm_t *h, double out[2]) {
  if (!h || !out) return fail(ISLBM_ERR_ARG, "NULL argument");
  if (h->is_slab) return fail(ISLBM_ERR_STATE, "slab handle: use islbm_residual_sums and add the sums over ranks");
  if (!h->has_state) return fail(ISLBM_ERR_STATE, "no state");
  double s[4];
  bool first = false;
  int rc = run_residual(h, s, &first);
  if (rc) return rc;
  if (first) {
    out[0] = out[1] = 1.0;
  } else {
    out[0] = s[1] > 0.0 ? s[0] / s[1] : (s[0] > 0.0 ? 1.0 : 0.0);
    out[1] = s[3] > 0.0 ? s[2] / s[3] : (s[2] > 0.0 ? 1.0 : 0.0);
  }
  return ISLBM_OK;
}
