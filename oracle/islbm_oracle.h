/*
 * islbm_oracle.h — plain CPU oracle for the ISLBM double-distribution step.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call
 * this.  It shares no code, header, table or constant generator with the CUDA
 * path under paper_2509_01099_b200/csrc (the direction ordering below is
 * retyped there, not included).
 *
 * What it computes, in the paper's order (Sec. 2.2):
 *   collide at every node (Eq. 17, Eq. 19)  ->  virtual streaming by one
 *   lattice displacement (Eq. 18, Eq. 20)   ->  quadratic interpolation back
 *   onto the mesh nodes  ->  half-way bounce-back /
 *   anti-bounce-back at the walls (Eq. 21-23).
 * fp64 throughout, dense M / N mat-vecs, no blocking, no fusion.
 *
 * Parity status of the readings this file takes:
 *   pinned   : lattice algebra (P3), interpolation weights (P1), uniform-mesh
 *              reduction to textbook streaming (P2), mass (P4), conduction
 *              fixed point (P5), wall derivative (P6), brute-force step (P7),
 *              parameter map (P8), q_kappa (closed form from a_T),
 *              normalisation of <Re>, <u*^2>, <Nu> (P12), Nu_middle (P13: exact on
 *              quadratic T and uniform advection, = 1 on the conduction state).
 *   parity unpinned : the choice of the destination-centred stencil
 *              {j-1,j,j+1} (A2; Fig. 1 and ref [28] are not in PAPER.md) and
 *              the relaxation rates s_e, s_eps, s_q, q_e, q_nu (A7; refs
 *              [8,37,38] are not in PAPER.md).  End-to-end evidence only
 *              (Table 2 / Table 4 reproduction on the GPU path: DESIGN.md 3.1).  The
 *              alternative upwind stencil (oracle_set_stencil) is pinned the same way as
 *              the central one; which of the two the authors used stays undecided.
 *   readings without a formula to pin: the reference temperature T0 of the buoyancy force
 *              (A9: 0 by default, T_cold in the paper's mode) and the form of <Re> the tables
 *              print (A22) are choices of input / output convention, not of arithmetic.
 *
 * Layout of every population array: [q][z][y][x], x fastest, fp64.
 * Layout of every field array:      [z][y][x].
 */
#ifndef ISLBM_ORACLE_H
#define ISLBM_ORACLE_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle oracle_t;

/* dim = 2 (D2Q9 + D2Q5) or 3 (D3Q19 + D3Q7).  x/y/z: strictly increasing
 * fluid-node coordinates (copied).  delta: lattice unit in mesh units; walls
 * sit delta/2 outside the first/last node.  Returns NULL
 * on invalid input. */
oracle_t *oracle_create(int dim, int nx, int ny, int nz,
                        const double *x, const double *y, const double *z,
                        double delta, double Ra, double Pr, double Ma);
void oracle_destroy(oracle_t *h);

/* threads used by collide/stream (OpenMP over rows; bit-identical to 1). */
void oracle_set_threads(oracle_t *h, int nthreads);
int  oracle_get_threads(const oracle_t *h);

/* reference temperature T0 of the buoyancy force and of T* (default 0; the paper's runs: T_cold, reading A9). */
void oracle_set_reference_temperature(oracle_t *h, double T0);

/* interpolation stencil: 0 destination-centred {j-1,j,j+1} (reading A2, default), 1 upwind {j-2,j-1,j} for
 * c = +1 and {j,j+1,j+2} for c = -1 (the A2 alternative of SURVEY.md 8(f)-3).  Rebuilds the tables. */
void oracle_set_stencil(oracle_t *h, int kind);

/* test hook: scale on the buoyancy force (1 = paper; 0 = pin P5). */
void oracle_set_buoyancy_scale(oracle_t *h, double s);

/* rest state rho=1, u=0, T = amp*(2r-1), r from SplitMix64(seed) indexed by
 * the linear node index (reading A15). */
void oracle_init(oracle_t *h, unsigned long long seed, double amp);

void oracle_set_populations(oracle_t *h, const double *f, const double *g);
void oracle_get_populations(const oracle_t *h, double *f, double *g);
/* post-collision populations of the LAST oracle_collide / oracle_step. */
void oracle_get_post_collision(const oracle_t *h, double *fp, double *gp);
/* test hook: load f+,g+ directly so that oracle_stream can be pinned alone. */
void oracle_set_post_collision(oracle_t *h, const double *fp, const double *gp);

void oracle_collide(oracle_t *h);          /* f,g -> f+,g+   (Eq. 17, 19)   */
void oracle_stream(oracle_t *h);           /* f+,g+ -> f,g at t+1 (Eq.18-23) */
void oracle_step(oracle_t *h, int nsteps); /* nsteps x (collide; stream)    */

/* one node of the next state, computed from the CURRENT f,g by colliding the
 * nodes of its stencil on the fly (for sampled parity at full size).
 * out_f[qf], out_g[qg]. */
void oracle_step_node(const oracle_t *h, int ix, int iy, int iz,
                      double *out_f, double *out_g);

/* macroscopic fields of the current f,g. w may be NULL. */
void oracle_fields(const oracle_t *h, double *rho, double *u, double *v,
                   double *w, double *T);

/* out[0]=Nu_hot (Eq. 32/41), out[1]=Nu_cold (Eq. 41), out[2]=<Re> (Eq. 34/42),
 * out[3]=<u*^2>_V, out[4]=<Nu> (Eq. 31/40). */
void oracle_nusselt(const oracle_t *h, double out[5]);

/* Nu_middle, Eq. 33: average over the vertical centre plane of sqrt(RaPr) u.T - dT/dx in free-fall units (reading A23). */
double oracle_nusselt_middle(const oracle_t *h);

/* Eq. 29-weighted total mass  sum rho * wx*wy(*wz)  and plain sum rho. */
void oracle_mass(const oracle_t *h, double out[2]);

/* introspection for the pins */
int  oracle_qf(const oracle_t *h);
int  oracle_qg(const oracle_t *h);
void oracle_get_velocities(const oracle_t *h, int *ef /*[qf*3]*/, int *eg /*[qg*3]*/);
void oracle_get_matrices(const oracle_t *h, double *M /*[qf*qf]*/, double *Minv,
                         double *S /*[qf]*/, double *N /*[qg*qg]*/, double *Ninv,
                         double *Q /*[qg]*/);
/* out: U, H_lu, nu, alpha, gbeta, tau_f, a_T, omega_bc, dt_star, L_eff_x, L_eff_y, L_eff_z */
void oracle_get_params(const oracle_t *h, double out[12]);
/* axis 0..2, sign index 0 (c=-1) / 1 (c=+1): base[n], w[3*n] */
void oracle_get_weights(const oracle_t *h, int axis, int sign_idx, int *base, double *w);
/* equilibrium moments Eq. 10/11 and Eq. 15/16, forcing moments Eq. 12/13 */
void oracle_meq(const oracle_t *h, double rho, const double u[3], double *meq);
void oracle_neq(const oracle_t *h, double T, const double u[3], double *neq);
void oracle_mforce(const oracle_t *h, const double u[3], const double F[3], double *mF);
/* collide one node: in f[qf], g[qg] -> out fp[qf], gp[qg] */
void oracle_collide_node(const oracle_t *h, const double *f, const double *g,
                         double *fp, double *gp);
/* wall derivative Eq. 28 (lattice units, Delta = 1 l.u.) */
double oracle_wall_derivative(double q, double phi_wall, double phi1, double phi2);

#ifdef __cplusplus
}
#endif
#endif
