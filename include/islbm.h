/*
 * islbm.h — C-ABI boundary of the B200-native ISLBM hot path.
 *
 * The library implements ONE thing: the per-timestep double-distribution
 * update of the interpolation-supplemented lattice Boltzmann method for the
 * side-heated cavity of arXiv 2509.01099 ("PAPER.md" below is
 * /root/reference/PAPER.md), on a tensor-product non-uniform mesh:
 *
 *   collision of the flow (D2Q9 / D3Q19, MRT + Guo forcing, Eq. 9-13, 17) and
 *   temperature (D2Q5 / D3Q7, MRT, Eq. 14-16, 19) populations with the
 *   Boussinesq force, virtual streaming by one lattice
 *   displacement (Eq. 18, 20), separable quadratic interpolation back onto the
 *   mesh nodes, half-way bounce-back / anti-bounce-back
 *   walls (Eq. 21-23), and the Nusselt / Reynolds reductions (Eq. 27-34, 40-42).
 *
 * Every step of that path runs in CUDA kernels compiled for sm_100a.  There is
 * no CPU fallback: a call that needs the device and finds none returns
 * ISLBM_ERR_CUDA.
 *
 * Conventions
 *   - plain C types only; pointers are marked HOST or DEVICE below.
 *   - every function returns 0 (ISLBM_OK) or a negative ISLBM_ERR_* code and
 *     never aborts or throws; islbm_last_error() returns a thread-local,
 *     human-readable message for the last failing call on this thread.
 *   - population arrays: [q][z][y][x], x fastest, fp64, dense (no padding);
 *     field arrays: [z][y][x], fp64.  nz = 1 in 2-D.
 *   - direction ordering (reading A5; the paper prints only the
 *     moment ordering of Eq. 10/11/15/16):
 *       D2Q9 : 0 (0,0) 1 (1,0) 2 (0,1) 3 (-1,0) 4 (0,-1) 5 (1,1) 6 (-1,1)
 *              7 (-1,-1) 8 (1,-1);                     D2Q5 = first five.
 *       D3Q19: 0 rest; 1..6 (+x)(-x)(+y)(-y)(+z)(-z);
 *              7..10 (1,1,0)(-1,1,0)(1,-1,0)(-1,-1,0);
 *              11..14 (1,0,1)(-1,0,1)(1,0,-1)(-1,0,-1);
 *              15..18 (0,1,1)(0,-1,1)(0,1,-1)(0,-1,-1);  D3Q7 = first seven.
 *   - the problem is fixed (BASELINE.json configs): x-lo
 *     wall isothermal T = +0.5, x-hi wall isothermal T = -0.5, all other walls
 *     adiabatic, all walls no-slip, T0 = 0, buoyancy along +y.
 *   - all device work is enqueued on the CUDA stream given to islbm_create and
 *     is asynchronous unless stated otherwise.
 */
#ifndef ISLBM_H
#define ISLBM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct islbm islbm_t; /* opaque; owned by the library */

typedef struct {
  int dim;            /* 2 or 3 */
  int n[3];           /* FLUID nodes per axis (n[2] = 1 in 2-D); every node is updated */
  const double *x[3]; /* HOST; strictly increasing node coordinates per axis;
                         borrowed for the call and copied; x[2] ignored in 2-D */
  double delta;       /* lattice unit in mesh units (1 l.u. = minimal
                         spacing); the walls sit at x[a][0] - delta/2 and
                         x[a][n-1] + delta/2 (half-way schemes) */
} islbm_mesh;

enum { ISLBM_D2Q9_D2Q5 = 0, ISLBM_D3Q19_D3Q7 = 1 };
/* ISLBM_F32_STORAGE: the workspace holds f_q - w_q and g_q as fp32; the TMA kernels interpolate those stored
 * deviations in fp32 (one or two more fp32 roundings of the deviation per step, the size of the storage rounding
 * itself) and collide the temperature populations in fp32; the flow populations are collided in fp64 by the 2-D
 * kernels and in fp32 by the 3-D kernels (the precision is the cheapest one that holds the parity bars
 * of each lattice); everything else (API arrays, diagnostics, weights) is fp64.  Tolerance against the
 * fp64 oracle: 1e-5 on u and T after 1000 steps (BASELINE.json). */
enum { ISLBM_F64 = 0, ISLBM_F32_STORAGE = 1 };

enum {
  ISLBM_OK = 0,
  ISLBM_ERR_ARG = -1,       /* NULL pointer, bad dim / lattice / precision combination, n < 3 */
  ISLBM_ERR_MESH = -2,      /* non-monotone coordinates or a spacing < delta (the departure
                               point must stay inside the adjacent cell) */
  ISLBM_ERR_PARAM = -3,     /* Ra, Pr, Ma <= 0; tau_f <= 1/2; a_T outside (-4,1) / (-6,1) */
  ISLBM_ERR_WORKSPACE = -4, /* workspace NULL, misaligned (256 B) or too small */
  ISLBM_ERR_CUDA = -5,      /* a CUDA runtime call failed (message has the CUDA error) */
  ISLBM_ERR_STATE = -6,     /* call not valid in the current state (e.g. step before init) */
  ISLBM_ERR_NONFINITE = -7  /* islbm_nusselt found a non-finite result */
};

/* Parameters derived by islbm_create (Table 1). */
typedef struct {
  double U;        /* free-fall velocity in lattice units = Ma * c_s              */
  double H_lu;     /* characteristic length in lattice units = L_eff,y / delta    */
  double nu;       /* U * H_lu * sqrt(Pr/Ra)                                      */
  double alpha;    /* nu / Pr                                                     */
  double gbeta;    /* U^2 / H_lu  (Delta_T = 1)                                   */
  double tau_f;    /* 3 nu + 1/2                                                  */
  double a_T;      /* 20 sqrt3 alpha - 4  (2-D),  42 sqrt3 alpha - 6  (3-D)       */
  double omega_bc; /* (4 + a_T)/10 (2-D), (6 + a_T)/21 (3-D)                      */
  double dt_star;  /* free-fall time advanced by one step = U / H_lu              */
  double L_eff[3]; /* x[n-1] - x[0] + delta per axis (1 for the unused axis)      */
} islbm_params;

/* A slab of a larger cavity along its slowest axis (y in 2-D, z in 3-D), for a one-rank-per-GPU decomposition
 * (DESIGN.md 8).  The mesh given to islbm_create_slab holds the slab's owned layers plus ONE ghost layer at each
 * end that is not a wall; the other axes are complete. */
typedef struct {
  int lo_is_wall, hi_is_wall; /* is the first / last layer of this mesh a cavity wall (no ghost layer there)? */
  double L_eff_global;        /* effective length of the slab axis of the WHOLE cavity (x[n-1] - x[0] + delta) */
  long long node_offset;      /* global linear index of this mesh's node 0 (islbm_init draws noise by global index) */
} islbm_slab;

/* Where the halo of one side lives in the workspace, for the CURRENT state (call again after islbm_step). */
typedef struct {
  int is_wall;                /* 1: this side is a wall, nothing to exchange */
  int first_plane, n_planes;  /* the storage planes whose velocity has a component along the slab axis */
  size_t plane_pitch_bytes;   /* distance between consecutive planes */
  size_t layer_bytes;         /* contiguous bytes of one layer of one plane */
  size_t send_offset;         /* workspace byte offset of the first/last OWNED layer of plane first_plane */
  size_t recv_offset;         /* ... of the ghost layer on this side */
} islbm_halo_info;

/* Bytes of DEVICE workspace islbm_create needs for this mesh / lattice /
 * precision: two ping-pong population buffers (rows padded to 16 elements, planes
 * in the storage order of DESIGN.md 5) + interpolation tables + reduction scratch
 * + a 4*nn-double area used as the Eq. 30 snapshot and as the staging buffer of
 * islbm_set_populations_host.  Pure host arithmetic. */
int islbm_workspace_bytes(const islbm_mesh *mesh, int lattice, int precision,
                          size_t *bytes);

/* Create a solver.  mesh: HOST.  Ma = U / c_s (BASELINE.json's U = 0.1 l.u. is
 * Ma = 0.1*sqrt(3); the paper's runs use Ma = 0.1).
 * dev_workspace: DEVICE, 256-byte aligned, >= islbm_workspace_bytes; owned by
 * the caller and kept alive until islbm_destroy.  cuda_stream: a cudaStream_t
 * (NULL = the legacy default stream).  Uploads the tables; state is undefined
 * until islbm_init or islbm_set_populations. */
int islbm_create(islbm_t **out, const islbm_mesh *mesh, int lattice, double Ra,
                 double Pr, double Ma, int precision, void *dev_workspace,
                 size_t bytes, void *cuda_stream);

/* As islbm_create for a slab (see islbm_slab).  After every islbm_step(h, 1) the caller copies, for each plane
 * first_plane .. first_plane + n_planes - 1, the neighbour's send layer into this handle's recv layer (NCCL
 * send/recv or a peer copy on the handle's stream; islbm_halo gives the offsets).  islbm_nusselt,
 * islbm_nusselt_middle and islbm_steady_residual refuse slab handles: use islbm_diag_sums on every rank, add the
 * arrays, and islbm_diag_from_sums.  islbm_get_populations / islbm_fields return the local mesh; their ghost
 * layers are undefined. */
int islbm_create_slab(islbm_t **out, const islbm_mesh *mesh, int lattice, double Ra, double Pr, double Ma,
                      int precision, void *dev_workspace, size_t bytes, void *cuda_stream, const islbm_slab *slab);
int islbm_halo(islbm_t *h, int side /* 0 low, 1 high */, islbm_halo_info *out);
/* Fused halo exchange over peer memory, synchronised between NEIGHBOURS on the device (no collective per step).
 * islbm_halo_layout describes where this handle's ghost layer of `side` lives in ITS workspace, for both ping-pong
 * buffers, where its step flag of that side lives, which buffer holds its current state and how many steps it has
 * taken; the neighbour passes that description, together with this workspace as mapped in the neighbour's process
 * (same process: the pointer itself; another process on the node: a CUDA IPC mapping, peer access over NVLink), to
 * islbm_slab_set_peer on its facing side.  From then on
 *   - the neighbour's step kernel stores the halo planes of its boundary layer straight into this ghost layer as it
 *     emits them (no pack / unpack, no exchange pass);
 *   - when the last of the neighbour's CTAs that touch the boundary has finished step t, it publishes t into this
 *     handle's flag (st.release.sys after its peer stores); this handle's CTAs that read the ghost layer in step t+1,
 *     or store into the neighbour's ghost layer, first wait for it (ld.acquire.sys).  With ping-pong buffers that one
 *     flag per side and step orders both the ghost-layer reads (data of step t) and the peer stores of step t+1 (into
 *     the buffer the neighbour read during step t);
 *   - islbm_step(h, n) therefore enqueues its n step kernels back to back, with no host or NCCL synchronisation.
 * Both handles must have taken the same number of steps since their last islbm_init / islbm_set_populations when
 * they are connected (checked), and both must then be stepped the same number of times; islbm_init /
 * islbm_set_populations detach the peers (connect again).  The kernels of different ranks wait on one another, so
 * every rank must run on its OWN GPU (or the caller must order the steps on the host so that no kernel ever has to
 * wait, as the single-GPU tests do).  peer_workspace = NULL detaches. */
typedef struct {
  int is_wall;
  int cur;                    /* index of the buffer that holds the current state (the next step writes 1 - cur) */
  size_t ghost_offset[2];     /* byte offset of the ghost layer of the first halo plane, per ping-pong buffer */
  size_t plane_pitch_bytes;
  size_t layer_bytes;
  size_t flag_offset;         /* byte offset of this handle's 8-byte step flag of `side` (written by the neighbour) */
  long long steps;            /* steps taken since the last islbm_init / islbm_set_populations */
} islbm_halo_layout_info;
int islbm_halo_layout(islbm_t *h, int side, islbm_halo_layout_info *out);
int islbm_slab_set_peer(islbm_t *h, int side, void *peer_workspace /* DEVICE */,
                        const islbm_halo_layout_info *peer_layout /* HOST: the neighbour's layout of its facing side */);

/* HOST s[8]: this handle's Eq. 29-weighted partial sums (ghost layers weigh 0); synchronises the stream. */
int islbm_diag_sums(islbm_t *h, double s[8]);
/* HOST out[6] = Nu_hot, Nu_cold, <Re>, <u*^2>_V, <Nu>, Nu_middle from sums added over all slabs (pure host). */
int islbm_diag_from_sums(const islbm_t *h, const double s[8], double out[6]);
/* HOST s[4]: the four sums of Eq. 30 over this handle's owned nodes against the snapshot of the previous call
 * (then overwritten); *first = 1 if there was no snapshot (sums meaningless).  Residuals of the whole cavity:
 * (sum of s[0]) / (sum of s[1]) and (sum of s[2]) / (sum of s[3]) over the ranks.  Synchronises the stream. */
int islbm_residual_sums(islbm_t *h, double s[4], int *first);

void islbm_destroy(islbm_t *h);

/* Derived parameters (HOST out). */
int islbm_get_params(const islbm_t *h, islbm_params *out);

/* Rest state: rho = 1, u = 0, T = noise_amp * (2 r_k - 1) with r_k in [0,1) the
 * top 53 bits of the (k+1)-th SplitMix64 output for `seed`, k the linear node
 * index (reading A15); populations are the equilibria of that state. */
int islbm_init(islbm_t *h, unsigned long long seed, double noise_amp);

/* Load / read the PRE-collision populations f_t, g_t (the paper's state
 * variable).  f: DEVICE [qf][z][y][x], g: DEVICE [qg][z][y][x],
 * fp64, dense.  Internally the library keeps post-collision populations
 * (DESIGN.md "state convention"); set collides once, get re-runs the streaming
 * half of the last step on the previous buffer. */
int islbm_set_populations(islbm_t *h, const double *f, const double *g);
int islbm_get_populations(islbm_t *h, double *f, double *g);
/* As islbm_set_populations with HOST arrays (pinned memory makes the copies asynchronous): the library stages them
 * slab by slab through the Eq. 30 snapshot area of the workspace (which it invalidates) with cudaMemcpyAsync on
 * the handle's stream.  The arrays must stay valid until the stream has passed the call. */
int islbm_set_populations_host(islbm_t *h, const double *f, const double *g);

/* Advance n time steps: n x (collide, stream + interpolate + walls). */
int islbm_step(islbm_t *h, int n);

/* Macroscopic fields of the current state: rho = sum f,
 * u = (sum e f + F/2)/rho, T = sum g.  DEVICE outputs [z][y][x]; any of them
 * may be NULL (w is ignored in 2-D). */
int islbm_fields(islbm_t *h, double *rho, double *u, double *v, double *w,
                 double *T);

/* HOST out[5]: Nu_hot (Eq. 32/41), Nu_cold (Eq. 41), <Re> (Eq. 34/42),
 * <u*^2>_V, <Nu> (Eq. 31/40); wall derivative per Eq. 28, averages per Eq. 29
 * normalised by the effective lengths.  Synchronises the stream.
 * Returns ISLBM_ERR_NONFINITE (out still written) if any entry is not finite. */
int islbm_nusselt(islbm_t *h, double out[5]);

/* As islbm_nusselt (same five diagnostics, Eq. 27-29, 31-34, 40-42), for callers that must not allocate or hand out
 * scratch memory (code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc): the block
 * partial sums go to a file-scope __device__ array of the library (114 752 bytes, held by every GPU that loads the
 * library until exit), not to the workspace, and the call allocates nothing (no cudaMalloc / cudaFree, no allocating
 * library routine; the first call on a device resolves the array's address with cudaGetSymbolAddress).
 * LIMIT: at most 2048 * 16384 = 33 554 432 nodes (256^3 is 16 777 216); a larger mesh returns ISLBM_ERR_ARG, and
 * islbm_nusselt remains the path for it.  Each block reduces a fixed share of 16 384 nodes, so the summation order
 * depends on the mesh only (results agree with islbm_nusselt to summation-order round-off, 1e-12 relative).
 * The array is shared by every call on the device and keeps the last call's contents (each call overwrites all the
 * slots it reads, so nothing needs clearing): calls that overlap on the GPU — other streams, other handles — RACE;
 * serialise them.  Synchronises the handle's stream.  HOST out[5]; ISLBM_ERR_NONFINITE as for islbm_nusselt. */
int islbm_nusselt_static(islbm_t *h, double out[5]);

/* HOST *out = Nu_middle (Eq. 33): average over the vertical centre plane x* = 0.5 of
 * sqrt(Ra Pr) u* T* - dT* / dx*; the derivative at a node column is that of the parabola through the column and
 * its two neighbours, and the flux is interpolated linearly between the two columns bracketing the midpoint of
 * the x-walls (reading A23).  Synchronises the stream.  ISLBM_ERR_NONFINITE as for islbm_nusselt. */
int islbm_nusselt_middle(islbm_t *h, double *out);

/* Steady-state residuals of Eq. 30 between the current fields and the fields
 * saved by the previous call (first call saves and returns 1, 1):
 * HOST out[2] = { sum|u - u_prev|_2 / sum|u_prev|_2, sum|T - T_prev| / sum|T_prev| }.
 * Needs the optional snapshot area (requested with islbm_workspace_bytes'
 * default sizing).  Synchronises the stream. */
int islbm_steady_residual(islbm_t *h, double out[2]);

/* Test / study hooks (not part of the four-call contract). */
int islbm_set_buoyancy_scale(islbm_t *h, double s); /* multiplies g*beta; 0 for pin P5 */
/* Reference temperature T0 of the buoyancy force F = rho g beta (T - T0) y^ and of T* in
 * Eq. 31/33.  Default 0 = the mean of the wall temperatures (BASELINE.json configs).  The paper's own runs have
 * T* = (T - T0)/Delta_T in [0,1], i.e. T0 = the cold-wall temperature = -0.5 here (reading A9): in the
 * weakly compressible model that breaks the centro-symmetry of the solution, which is what Table 3 prints.
 * Must be called before islbm_init / islbm_set_populations. */
int islbm_set_reference_temperature(islbm_t *h, double T0);
/* Interpolation stencil: 0 = destination-centred {j-1,j,j+1} (default, reading A2), 1 = upwind
 * {j-2,j-1,j} for c = +1 and {j,j+1,j+2} for c = -1 (the A2 alternative; TMA kernels of its own and the generic kernel;
 * not on slab handles, whose single ghost layer is one short of its reach).
 * Before islbm_init / islbm_set_populations. */
int islbm_set_stencil(islbm_t *h, int kind);
/* 0 = auto (fastest kernel for this mesh), 1 = generic global-memory kernel,
 * 2 = TMA-staged shared-memory kernel (y-marching in 2-D, z-marching in 3-D),
 * 3 = uniform-mesh pure-shift kernel (only valid when every spacing equals
 * delta to within 1e-10 relative; Eq. 17-20 on the uniform mesh of Eq. 24-25;
 * identical to the interpolating kernels when the spacings are bit-exact,
 * e.g. N a power of two, otherwise to that relative accuracy per step). */
int islbm_set_kernel(islbm_t *h, int which);
/* Run-time knobs of the TMA-staged kernels.  key: "chunk" (marching
 * chunk length, 0 = automatic), "l2promo" (tensor-map L2 promotion 0 none, 1 64 B,
 * 2 128 B, 3 256 B), "load_policy" / "store_policy" (L2 eviction policy 0 normal,
 * 1 evict_first, 2 evict_last), "tx2d" (2-D strip width 0 auto, 128, 224),
 * "serpentine" (2-D: march downwards on odd steps), "shape3d" (3-D tile 0 automatic, 1 64x4, 2 128x2, 3 32x6, 4 32x4, 5 32x8), "pdl" (programmatic
 * dependent launch of consecutive step kernels, default 1), "fill" (first fill of the TMA
 * ring: 1 before the weight rows and the CTA barrier, 2 after them, 0 automatic), "ring2d" (2-D fp64
 * ring: 3 stages with four CTAs per SM or 4 stages with three, 0 automatic), "rows2d" / "rows2d1"
 * (2-D chunk rule: longest chunk of a multi-wave launch / longest chunk for which a single wave
 * of CTAs is taken, 0 automatic), "graph" (islbm_step(n) with n >= 32 replays a captured CUDA graph of 32 PDL-chained
 * step kernels: 0 automatic = meshes of at most 2^20 nodes, whose steps are short enough for the host's launch rate to show, 1 always,
 * 2 never), "slab_wait_ms" (fused slab exchange: the longest a boundary CTA waits for its neighbour's step flag, default
 * 10 000 ms, 0 = for ever; a CTA that gives up is counted, and islbm_diag_sums / islbm_residual_sums then return
 * ISLBM_ERR_STATE instead of the GPU hanging on a neighbour that never steps), "cluster" (2-D fp64 meshes of at most 16 bands of 256
 * nodes: islbm_step(n >= 2) runs all n steps in one launch of a thread-block cluster with the state in distributed shared
 * memory; 0 automatic, 2 never), "walls" (3-D whole cavity: 0 wall rules inside the step kernel, 1 a separate
 * boundary kernel over the shell of wall-adjacent nodes: the design BASELINE.json names, measured slower).  Results
 * do not depend on any of them.  Unknown key or negative value: ISLBM_ERR_ARG. */
int islbm_set_tuning(islbm_t *h, const char *key, int value);
/* Number of kernels launched by this handle since creation. */
long long islbm_launch_count(const islbm_t *h);
/* Name of the step kernel variant that islbm_step currently dispatches to. */
const char *islbm_kernel_name(const islbm_t *h);

const char *islbm_last_error(void);
const char *islbm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ISLBM_H */
