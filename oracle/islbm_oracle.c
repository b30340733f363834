/*
 * islbm_oracle.c — plain, slow, fp64 CPU oracle of the ISLBM step.
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE (see islbm_oracle.h).
 *
 * Every function cites the passage of /root/reference/PAPER.md it restates
 * ("PAPER.md:<line>") or the DESIGN.md reading (A1..A21) it takes where the
 * paper is silent.  Nothing here is blocked, fused or reordered beyond what
 * the paper's algorithm states: collide every node, then pull every population
 * through its interpolation stencil or its wall rule.
 */
#include "islbm_oracle.h"

#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define QF_MAX 19
#define QG_MAX 7

/* Discrete velocities, reading A5 (the paper prints only the moment
 * ordering, Eq. 10/11/15/16).  D2Q5 / D3Q7 are the first 5 / 7 entries. */
static const int E_D2Q9[9][3] = {
    {0, 0, 0}, {1, 0, 0}, {0, 1, 0}, {-1, 0, 0}, {0, -1, 0},
    {1, 1, 0}, {-1, 1, 0}, {-1, -1, 0}, {1, -1, 0}};
static const int E_D3Q19[19][3] = {
    {0, 0, 0},
    {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1},
    {1, 1, 0}, {-1, 1, 0}, {1, -1, 0}, {-1, -1, 0},
    {1, 0, 1}, {-1, 0, 1}, {1, 0, -1}, {-1, 0, -1},
    {0, 1, 1}, {0, -1, 1}, {0, 1, -1}, {0, -1, -1}};

struct oracle {
  int dim, n[3];
  double *x[3];
  double delta;
  int qf, qg;
  int ef[QF_MAX][3], eg[QG_MAX][3];
  int opp_f[QF_MAX], opp_g[QG_MAX];
  double M[QF_MAX][QF_MAX], Minv[QF_MAX][QF_MAX], S[QF_MAX];
  double N[QG_MAX][QG_MAX], Ninv[QG_MAX][QG_MAX], Q[QG_MAX];
  double Ra, Pr, Ma;
  double U, H_lu, nu, alpha, gbeta, tau_f, a_T, omega_bc;
  double L_eff[3];
  double T_hot, T_cold, T0, buoy;
  int stencil; /* 0: destination-centred {j-1,j,j+1} (reading A2); 1: upwind {j-2,j-1,j} / {j,j+1,j+2} (A2 alternative) */
  /* interpolation tables: axis a, sign index s (0: c=-1, 1: c=+1) */
  int *base[3][2];
  double *wgt[3][2];
  /* Eq. 29 averaging weights per axis */
  double *avgw[3];
  size_t nn;
  double *f, *g, *fp, *gp;
  int nthreads;
};

/* a strided window onto population storage: value(q, ix,iy,iz) */
typedef struct {
  const double *p;
  long sq, sz, sy;
  int ox, oy, oz;
} view_t;

static inline double view_at(const view_t *v, int q, int ix, int iy, int iz) {
  return v->p[(long)q * v->sq + (long)(iz - v->oz) * v->sz +
              (long)(iy - v->oy) * v->sy + (long)(ix - v->ox)];
}

/* ------------------------------------------------------------------------ */
/* lattice algebra                                                          */
/* ------------------------------------------------------------------------ */

/* Rows of M and N written as polynomials of the discrete velocity, in the
 * moment order of Eq. 10/11 and Eq. 15/16;
 * DESIGN.md reading A6.  M^-1 follows from mutual orthogonality of the rows
 * (checked by pin P3): Minv[i][k] = M[k][i] / sum_j M[k][j]^2. */
static double m_row(int dim, int k, const int c[3]) {
  double cx = c[0], cy = c[1], cz = c[2];
  double c2 = cx * cx + cy * cy + cz * cz;
  if (dim == 2) {
    switch (k) {
      case 0: return 1.0;
      case 1: return -4.0 + 3.0 * c2;
      case 2: return 4.0 - 10.5 * c2 + 4.5 * c2 * c2;
      case 3: return cx;
      case 4: return (-5.0 + 3.0 * c2) * cx;
      case 5: return cy;
      case 6: return (-5.0 + 3.0 * c2) * cy;
      case 7: return cx * cx - cy * cy;
      case 8: return cx * cy;
    }
  } else {
    switch (k) {
      case 0: return 1.0;
      case 1: return 19.0 * c2 - 30.0;
      case 2: return (21.0 * c2 * c2 - 53.0 * c2 + 24.0) / 2.0;
      case 3: return cx;
      case 4: return (5.0 * c2 - 9.0) * cx;
      case 5: return cy;
      case 6: return (5.0 * c2 - 9.0) * cy;
      case 7: return cz;
      case 8: return (5.0 * c2 - 9.0) * cz;
      case 9: return 3.0 * cx * cx - c2;
      case 10: return (3.0 * c2 - 5.0) * (3.0 * cx * cx - c2);
      case 11: return cy * cy - cz * cz;
      case 12: return (3.0 * c2 - 5.0) * (cy * cy - cz * cz);
      case 13: return cx * cy;
      case 14: return cy * cz;
      case 15: return cx * cz;
      case 16: return (cy * cy - cz * cz) * cx;
      case 17: return (cz * cz - cx * cx) * cy;
      case 18: return (cx * cx - cy * cy) * cz;
    }
  }
  return 0.0;
}

static double n_row(int dim, int k, const int c[3]) {
  double cx = c[0], cy = c[1], cz = c[2];
  double c2 = cx * cx + cy * cy + cz * cz;
  if (dim == 2) {
    switch (k) {
      case 0: return 1.0;
      case 1: return cx;
      case 2: return cy;
      case 3: return -4.0 + 5.0 * c2;
      case 4: return cx * cx - cy * cy;
    }
  } else {
    switch (k) {
      case 0: return 1.0;
      case 1: return cx;
      case 2: return cy;
      case 3: return cz;
      case 4: return -6.0 + 7.0 * c2;
      case 5: return 3.0 * cx * cx - c2;
      case 6: return cy * cy - cz * cz;
    }
  }
  return 0.0;
}

static void build_lattice(oracle_t *h) {
  int dim = h->dim;
  h->qf = dim == 2 ? 9 : 19;
  h->qg = dim == 2 ? 5 : 7;
  for (int i = 0; i < h->qf; ++i)
    for (int a = 0; a < 3; ++a)
      h->ef[i][a] = dim == 2 ? E_D2Q9[i][a] : E_D3Q19[i][a];
  for (int i = 0; i < h->qg; ++i)
    for (int a = 0; a < 3; ++a) h->eg[i][a] = h->ef[i][a];
  for (int i = 0; i < h->qf; ++i)
    for (int j = 0; j < h->qf; ++j)
      if (h->ef[i][0] == -h->ef[j][0] && h->ef[i][1] == -h->ef[j][1] &&
          h->ef[i][2] == -h->ef[j][2])
        h->opp_f[i] = j;
  for (int i = 0; i < h->qg; ++i)
    for (int j = 0; j < h->qg; ++j)
      if (h->eg[i][0] == -h->eg[j][0] && h->eg[i][1] == -h->eg[j][1] &&
          h->eg[i][2] == -h->eg[j][2])
        h->opp_g[i] = j;
  for (int k = 0; k < h->qf; ++k) {
    double nrm = 0.0;
    for (int i = 0; i < h->qf; ++i) {
      h->M[k][i] = m_row(dim, k, h->ef[i]);
      nrm += h->M[k][i] * h->M[k][i];
    }
    for (int i = 0; i < h->qf; ++i) h->Minv[i][k] = h->M[k][i] / nrm;
  }
  for (int k = 0; k < h->qg; ++k) {
    double nrm = 0.0;
    for (int i = 0; i < h->qg; ++i) {
      h->N[k][i] = n_row(dim, k, h->eg[i]);
      nrm += h->N[k][i] * h->N[k][i];
    }
    for (int i = 0; i < h->qg; ++i) h->Ninv[i][k] = h->N[k][i] / nrm;
  }
}

/* Parameter map.  PAPER.md:53-72 (free-fall scaling), PAPER.md:248 (Ma = u_f /
 * c_s, c_s = 1/sqrt 3), Table 1 PAPER.md:206-212 (characteristic length =
 * effective height / minimal resolution), PAPER.md:124 (a_T)
 * (omega); relaxation rates: DESIGN.md reading A7. */
static void build_params(oracle_t *h) {
  const double cs = 1.0 / sqrt(3.0);
  for (int a = 0; a < h->dim; ++a)
    h->L_eff[a] = h->x[a][h->n[a] - 1] - h->x[a][0] + h->delta;
  if (h->dim == 2) h->L_eff[2] = 1.0;
  h->U = h->Ma * cs;
  h->H_lu = h->L_eff[1] / h->delta; /* H = cavity height, y is vertical */
  h->nu = h->U * h->H_lu * sqrt(h->Pr / h->Ra);
  h->alpha = h->nu / h->Pr;
  h->gbeta = h->U * h->U / h->H_lu; /* Delta_T = 1 */
  h->tau_f = 3.0 * h->nu + 0.5;
  if (h->dim == 2) {
    h->a_T = 20.0 * sqrt(3.0) * h->alpha - 4.0;
    h->omega_bc = (4.0 + h->a_T) / 10.0;
  } else {
    h->a_T = 42.0 * sqrt(3.0) * h->alpha - 6.0;
    h->omega_bc = (6.0 + h->a_T) / 21.0;
  }
  double tau = h->tau_f;
  double s_nu = 1.0 / tau;
  double s_q = 8.0 * (2.0 * tau - 1.0) / (8.0 * tau - 1.0);
  double q_k = 3.0 - sqrt(3.0);
  double q_e = 4.0 * sqrt(3.0) - 6.0;
  if (h->dim == 2) {
    double S[9] = {0.0, s_nu, s_nu, 0.0, s_q, 0.0, s_q, s_nu, s_nu};
    double Q[5] = {0.0, q_k, q_k, q_e, q_e};
    memcpy(h->S, S, sizeof S);
    memcpy(h->Q, Q, sizeof Q);
  } else {
    double S[19] = {0.0, s_nu, s_nu, 0.0, s_q, 0.0, s_q, 0.0, s_q, s_nu,
                    s_nu, s_nu, s_nu, s_nu, s_nu, s_nu, s_q, s_q, s_q};
    double Q[7] = {0.0, q_k, q_k, q_k, q_e, q_e, q_e};
    memcpy(h->S, S, sizeof S);
    memcpy(h->Q, Q, sizeof Q);
  }
  /* Side-heated cavity, BASELINE.json configs: x-lo wall hot, x-hi wall cold,
   * T0 = mean; reading A11. */
  h->T_hot = 0.5;
  h->T_cold = -0.5;
  h->T0 = 0.0;
  h->buoy = 1.0;
}

/* Interpolation tables ("quadratic interpolation"; weights
 * are the 3-point Lagrange coefficients PAPER.md:160 names).  Readings A2, A3:
 * population with velocity component c along this axis arrives at node j from
 * the departure point x_j - c*delta; the stencil is the destination-centred
 * triple {j-1, j, j+1}, shifted inward at the first/last node.  Offsets are
 * taken relative to x_j so that a bit-exact unit spacing gives weights that
 * are bit-exactly (1,0,0) / (0,0,1). */
static void build_weights(oracle_t *h) {
  for (int a = 0; a < h->dim; ++a) {
    int n = h->n[a];
    const double *x = h->x[a];
    for (int s = 0; s < 2; ++s) {
      double c = s == 0 ? -1.0 : 1.0;
      h->base[a][s] = (int *)malloc(sizeof(int) * (size_t)n);
      h->wgt[a][s] = (double *)malloc(sizeof(double) * 3 * (size_t)n);
      for (int j = 0; j < n; ++j) {
        /* central: {j-1,j,j+1}.  upwind (A2 alternative): the triple that ends at j on the side the population
         * comes from, {j-2,j-1,j} for c = +1 and {j,j+1,j+2} for c = -1.  Either way the departure point lies in
         * [x_{j-1}, x_j] (c = +1) or [x_j, x_{j+1}] (c = -1), inside the triple after clamping to the mesh. */
        int b = h->stencil == 0 ? j - 1 : (s == 1 ? j - 2 : j);
        if (b < 0) b = 0;
        if (b > n - 3) b = n - 3;
        h->base[a][s][j] = b;
        double xi = -c * h->delta; /* departure point relative to x_j */
        double d[3];
        for (int k = 0; k < 3; ++k) d[k] = x[b + k] - x[j];
        for (int k = 0; k < 3; ++k) {
          double num = 1.0, den = 1.0;
          for (int m = 0; m < 3; ++m) {
            if (m == k) continue;
            num *= (xi - d[m]);
            den *= (d[k] - d[m]);
          }
          h->wgt[a][s][3 * j + k] = num / den;
        }
      }
    }
    /* Eq. 29: w_j = (x_{j+1} - x_{j-1}) / 2 with the ghost
     * coordinates one lattice unit outside the end nodes (reading A14), so
     * that the weights sum to the effective length L_eff. */
    h->avgw[a] = (double *)malloc(sizeof(double) * (size_t)n);
    for (int j = 0; j < n; ++j) {
      double xm = j == 0 ? x[0] - h->delta : x[j - 1];
      double xp = j == n - 1 ? x[n - 1] + h->delta : x[j + 1];
      h->avgw[a][j] = (xp - xm) / 2.0;
    }
  }
  for (int a = h->dim; a < 3; ++a) {
    h->base[a][0] = h->base[a][1] = NULL;
    h->wgt[a][0] = h->wgt[a][1] = NULL;
    h->avgw[a] = (double *)malloc(sizeof(double));
    h->avgw[a][0] = 1.0;
  }
}

oracle_t *oracle_create(int dim, int nx, int ny, int nz, const double *x,
                        const double *y, const double *z, double delta,
                        double Ra, double Pr, double Ma) {
  if (dim != 2 && dim != 3) return NULL;
  if (dim == 2) nz = 1;
  const double *xs[3] = {x, y, z};
  int n[3] = {nx, ny, nz};
  if (!(delta > 0.0) || !(Ra > 0.0) || !(Pr > 0.0) || !(Ma > 0.0)) return NULL;
  for (int a = 0; a < dim; ++a) {
    if (n[a] < 3 || xs[a] == NULL) return NULL;
    for (int j = 1; j < n[a]; ++j)
      if (!(xs[a][j] - xs[a][j - 1] >= delta * (1.0 - 1e-12))) return NULL;
  }
  oracle_t *h = (oracle_t *)calloc(1, sizeof(oracle_t));
  h->dim = dim;
  for (int a = 0; a < 3; ++a) h->n[a] = n[a];
  for (int a = 0; a < dim; ++a) {
    h->x[a] = (double *)malloc(sizeof(double) * (size_t)n[a]);
    memcpy(h->x[a], xs[a], sizeof(double) * (size_t)n[a]);
  }
  h->delta = delta;
  h->Ra = Ra;
  h->Pr = Pr;
  h->Ma = Ma;
  h->nthreads = 1;
  build_lattice(h);
  build_params(h);
  build_weights(h);
  h->nn = (size_t)n[0] * (size_t)n[1] * (size_t)n[2];
  h->f = (double *)calloc(h->nn * (size_t)h->qf, sizeof(double));
  h->fp = (double *)calloc(h->nn * (size_t)h->qf, sizeof(double));
  h->g = (double *)calloc(h->nn * (size_t)h->qg, sizeof(double));
  h->gp = (double *)calloc(h->nn * (size_t)h->qg, sizeof(double));
  if (!h->f || !h->fp || !h->g || !h->gp) {
    oracle_destroy(h);
    return NULL;
  }
  return h;
}

void oracle_destroy(oracle_t *h) {
  if (!h) return;
  for (int a = 0; a < 3; ++a) {
    free(h->x[a]);
    free(h->avgw[a]);
    for (int s = 0; s < 2; ++s) {
      free(h->base[a][s]);
      free(h->wgt[a][s]);
    }
  }
  free(h->f);
  free(h->g);
  free(h->fp);
  free(h->gp);
  free(h);
}

void oracle_set_threads(oracle_t *h, int nthreads) {
#ifdef _OPENMP
  h->nthreads = nthreads < 1 ? 1 : nthreads;
#else
  (void)nthreads;
  h->nthreads = 1;
#endif
}
int oracle_get_threads(const oracle_t *h) { return h->nthreads; }
/* reference temperature T0 of F = rho g beta (T - T0) y^ and of T* = (T - T0)/Delta_T.
 * Default 0 (mean of the walls, BASELINE.json); the paper's T* in [0,1] corresponds to T0 = T_cold (reading A9). */
void oracle_set_reference_temperature(oracle_t *h, double T0) { h->T0 = T0; }

/* A2 alternative stencil: rebuilds the interpolation tables.  kind 0 central (default), 1 upwind. */
void oracle_set_stencil(oracle_t *h, int kind) {
  for (int a = 0; a < 3; ++a) {
    for (int s = 0; s < 2; ++s) {
      free(h->base[a][s]);
      free(h->wgt[a][s]);
    }
    free(h->avgw[a]);
  }
  h->stencil = kind ? 1 : 0;
  build_weights(h);
}

void oracle_set_buoyancy_scale(oracle_t *h, double s) { h->buoy = s; }

/* ------------------------------------------------------------------------ */
/* equilibria, forcing, collision at one node                               */
/* ------------------------------------------------------------------------ */

/* Eq. 10 and Eq. 11; full rho multiplies every
 * entry (weakly compressible form). */
void oracle_meq(const oracle_t *h, double rho, const double uu[3], double *meq) {
  double u = uu[0], v = uu[1], w = uu[2];
  if (h->dim == 2) {
    double u2 = u * u + v * v;
    meq[0] = rho;
    meq[1] = rho * (-2.0 + 3.0 * u2);
    meq[2] = rho * (1.0 - 3.0 * u2);
    meq[3] = rho * u;
    meq[4] = rho * (-u);
    meq[5] = rho * v;
    meq[6] = rho * (-v);
    meq[7] = rho * (u * u - v * v);
    meq[8] = rho * (u * v);
  } else {
    double u2 = u * u + v * v + w * w;
    meq[0] = rho;
    meq[1] = rho * (-11.0 + 19.0 * u2);
    meq[2] = rho * (3.0 - 11.0 / 2.0 * u2);
    meq[3] = rho * u;
    meq[4] = rho * (-2.0 / 3.0 * u);
    meq[5] = rho * v;
    meq[6] = rho * (-2.0 / 3.0 * v);
    meq[7] = rho * w;
    meq[8] = rho * (-2.0 / 3.0 * w);
    meq[9] = rho * (2.0 * u * u - v * v - w * w);
    meq[10] = rho * (-0.5 * (2.0 * u * u - v * v - w * w));
    meq[11] = rho * (v * v - w * w);
    meq[12] = rho * (-0.5 * (v * v - w * w));
    meq[13] = rho * (u * v);
    meq[14] = rho * (v * w);
    meq[15] = rho * (u * w);
    meq[16] = 0.0;
    meq[17] = 0.0;
    meq[18] = 0.0;
  }
}

/* Eq. 15 and Eq. 16. */
void oracle_neq(const oracle_t *h, double T, const double uu[3], double *neq) {
  if (h->dim == 2) {
    neq[0] = T;
    neq[1] = uu[0] * T;
    neq[2] = uu[1] * T;
    neq[3] = h->a_T * T;
    neq[4] = 0.0;
  } else {
    neq[0] = T;
    neq[1] = uu[0] * T;
    neq[2] = uu[1] * T;
    neq[3] = uu[2] * T;
    neq[4] = h->a_T * T;
    neq[5] = 0.0;
    neq[6] = 0.0;
  }
}

/* Eq. 12 and Eq. 13.  The last entry of Eq. 12
 * is printed "uF_x + vF_y"; the 3-D analogue (entry 13 of Eq. 13) prints
 * "uF_y + vF_x", which is what Guo's velocity-space forcing projects to
 * (pin P3) — DESIGN.md reading A8. */
void oracle_mforce(const oracle_t *h, const double uu[3], const double F[3],
                   double *mF) {
  double u = uu[0], v = uu[1], w = uu[2];
  double Fx = F[0], Fy = F[1], Fz = F[2];
  if (h->dim == 2) {
    double uF = u * Fx + v * Fy;
    mF[0] = 0.0;
    mF[1] = 6.0 * uF;
    mF[2] = -6.0 * uF;
    mF[3] = Fx;
    mF[4] = -Fx;
    mF[5] = Fy;
    mF[6] = -Fy;
    mF[7] = 2.0 * u * Fx - 2.0 * v * Fy;
    mF[8] = u * Fy + v * Fx;
  } else {
    double uF = u * Fx + v * Fy + w * Fz;
    mF[0] = 0.0;
    mF[1] = 38.0 * uF;
    mF[2] = -11.0 * uF;
    mF[3] = Fx;
    mF[4] = -2.0 / 3.0 * Fx;
    mF[5] = Fy;
    mF[6] = -2.0 / 3.0 * Fy;
    mF[7] = Fz;
    mF[8] = -2.0 / 3.0 * Fz;
    mF[9] = 4.0 * u * Fx - 2.0 * v * Fy - 2.0 * w * Fz;
    mF[10] = -2.0 * u * Fx + v * Fy + w * Fz;
    mF[11] = 2.0 * v * Fy - 2.0 * w * Fz;
    mF[12] = -v * Fy + w * Fz;
    mF[13] = u * Fy + v * Fx;
    mF[14] = v * Fz + w * Fy;
    mF[15] = u * Fz + w * Fx;
    mF[16] = 0.0;
    mF[17] = 0.0;
    mF[18] = 0.0;
  }
}

/* Moments at one node.  PAPER.md:124 (T = sum g), PAPER.md:106 (rho = sum f,
 * F = rho g beta (T - T0) y^, u = (sum e f + F/2) / rho); order per reading
 * A16: T and rho first, then F, then u; buoyancy along +y (reading A9). */
static void node_moments(const oracle_t *h, const double *f, const double *g,
                         double *rho, double u[3], double *T, double F[3]) {
  double t = 0.0, r = 0.0, j[3] = {0.0, 0.0, 0.0};
  for (int i = 0; i < h->qg; ++i) t += g[i];
  for (int i = 0; i < h->qf; ++i) {
    r += f[i];
    for (int a = 0; a < 3; ++a) j[a] += h->ef[i][a] * f[i];
  }
  F[0] = 0.0;
  F[1] = h->buoy * r * h->gbeta * (t - h->T0);
  F[2] = 0.0;
  for (int a = 0; a < 3; ++a) u[a] = (j[a] + F[a] / 2.0) / r;
  *rho = r;
  *T = t;
}

/* Eq. 17 with F' = M^-1 (I - S/2) M F~, and
 * Eq. 19. */
void oracle_collide_node(const oracle_t *h, const double *f, const double *g,
                         double *fp, double *gp) {
  double rho, u[3], T, F[3];
  double m[QF_MAX], meq[QF_MAX], mF[QF_MAX], r[QF_MAX];
  double n[QG_MAX], neq[QG_MAX], rg[QG_MAX];
  node_moments(h, f, g, &rho, u, &T, F);
  oracle_meq(h, rho, u, meq);
  oracle_mforce(h, u, F, mF);
  for (int k = 0; k < h->qf; ++k) {
    double s = 0.0;
    for (int i = 0; i < h->qf; ++i) s += h->M[k][i] * f[i];
    m[k] = s;
    r[k] = h->S[k] * (m[k] - meq[k]) - (1.0 - h->S[k] / 2.0) * mF[k];
  }
  for (int i = 0; i < h->qf; ++i) {
    double s = 0.0;
    for (int k = 0; k < h->qf; ++k) s += h->Minv[i][k] * r[k];
    fp[i] = f[i] - s;
  }
  oracle_neq(h, T, u, neq);
  for (int k = 0; k < h->qg; ++k) {
    double s = 0.0;
    for (int i = 0; i < h->qg; ++i) s += h->N[k][i] * g[i];
    n[k] = s;
    rg[k] = h->Q[k] * (n[k] - neq[k]);
  }
  for (int i = 0; i < h->qg; ++i) {
    double s = 0.0;
    for (int k = 0; k < h->qg; ++k) s += h->Ninv[i][k] * rg[k];
    gp[i] = g[i] - s;
  }
}

void oracle_collide(oracle_t *h) {
  const long nn = (long)h->nn;
#ifdef _OPENMP
#pragma omp parallel for num_threads(h->nthreads) schedule(static)
#endif
  for (long c = 0; c < nn; ++c) {
    double f[QF_MAX], g[QG_MAX], fp[QF_MAX], gp[QG_MAX];
    for (int i = 0; i < h->qf; ++i) f[i] = h->f[(long)i * nn + c];
    for (int i = 0; i < h->qg; ++i) g[i] = h->g[(long)i * nn + c];
    oracle_collide_node(h, f, g, fp, gp);
    for (int i = 0; i < h->qf; ++i) h->fp[(long)i * nn + c] = fp[i];
    for (int i = 0; i < h->qg; ++i) h->gp[(long)i * nn + c] = gp[i];
  }
}

/* ------------------------------------------------------------------------ */
/* streaming + interpolation + walls at one node                            */
/* ------------------------------------------------------------------------ */

/* Does the departure point x - e*delta of velocity e leave the fluid at node
 * idx?  The walls sit half a lattice unit outside the first/last node
 * (PAPER.md:191, 198), so it does exactly when the node is the first one and
 * e points away from the low wall, or the last one and e points away from the
 * high wall.  Returns the axis of the first wall crossed, -1 if none. */
static int crosses_wall(const oracle_t *h, const int e[3], const int idx[3]) {
  for (int a = 0; a < h->dim; ++a) {
    if (e[a] == 1 && idx[a] == 0) return a;
    if (e[a] == -1 && idx[a] == h->n[a] - 1) return a;
  }
  return -1;
}

/* Separable quadratic interpolation of post-collision plane q at the departure
 * point of velocity e for node idx; axes with e_a = 0 take
 * the node itself.  Sum over x first, then y, then z (reading A3). */
static double interp_pull(const oracle_t *h, const view_t *v, int q,
                          const int e[3], const int idx[3]) {
  int b[3], cnt[3];
  const double *w[3];
  static const double one[3] = {1.0, 0.0, 0.0};
  for (int a = 0; a < 3; ++a) {
    if (a < h->dim && e[a] != 0) {
      int s = e[a] > 0 ? 1 : 0;
      b[a] = h->base[a][s][idx[a]];
      w[a] = &h->wgt[a][s][3 * idx[a]];
      cnt[a] = 3;
    } else {
      b[a] = idx[a];
      w[a] = one;
      cnt[a] = 1;
    }
  }
  double sz = 0.0;
  for (int kz = 0; kz < cnt[2]; ++kz) {
    double sy = 0.0;
    for (int ky = 0; ky < cnt[1]; ++ky) {
      double sx = 0.0;
      for (int kx = 0; kx < cnt[0]; ++kx)
        sx += w[0][kx] * view_at(v, q, b[0] + kx, b[1] + ky, b[2] + kz);
      sy += w[1][ky] * sx;
    }
    sz += w[2][kz] * sy;
  }
  return sz;
}

/* New populations of one node from post-collision views vf, vg.
 * Interior: interpolation.  Wall: Eq. 21 for f; Eq. 22
 * on the isothermal x-walls and Eq. 23 on the
 * adiabatic walls for g.  A population bounces back as soon as any component
 * of its departure point crosses a wall (reading A4). */
static void pull_node(const oracle_t *h, const view_t *vf, const view_t *vg,
                      const int idx[3], double *nf, double *ng) {
  for (int i = 0; i < h->qf; ++i) {
    if (crosses_wall(h, h->ef[i], idx) >= 0)
      nf[i] = view_at(vf, h->opp_f[i], idx[0], idx[1], idx[2]);
    else
      nf[i] = interp_pull(h, vf, i, h->ef[i], idx);
  }
  for (int i = 0; i < h->qg; ++i) {
    int a = crosses_wall(h, h->eg[i], idx);
    if (a < 0) {
      ng[i] = interp_pull(h, vg, i, h->eg[i], idx);
    } else {
      double gb = view_at(vg, h->opp_g[i], idx[0], idx[1], idx[2]);
      if (a == 0) {
        double Tw = idx[0] == 0 ? h->T_hot : h->T_cold;
        ng[i] = -gb + h->omega_bc * Tw;
      } else {
        ng[i] = gb;
      }
    }
  }
}

void oracle_stream(oracle_t *h) {
  const long nn = (long)h->nn;
  const int nx = h->n[0], ny = h->n[1], nz = h->n[2];
  view_t vf = {h->fp, nn, (long)nx * ny, nx, 0, 0, 0};
  view_t vg = {h->gp, nn, (long)nx * ny, nx, 0, 0, 0};
  const long rows = (long)ny * nz;
#ifdef _OPENMP
#pragma omp parallel for num_threads(h->nthreads) schedule(static)
#endif
  for (long r = 0; r < rows; ++r) {
    int iz = (int)(r / ny), iy = (int)(r % ny);
    for (int ix = 0; ix < nx; ++ix) {
      int idx[3] = {ix, iy, iz};
      double nf[QF_MAX], ng[QG_MAX];
      pull_node(h, &vf, &vg, idx, nf, ng);
      long c = ((long)iz * ny + iy) * nx + ix;
      for (int i = 0; i < h->qf; ++i) h->f[(long)i * nn + c] = nf[i];
      for (int i = 0; i < h->qg; ++i) h->g[(long)i * nn + c] = ng[i];
    }
  }
}

void oracle_step(oracle_t *h, int nsteps) {
  for (int s = 0; s < nsteps; ++s) {
    oracle_collide(h);
    oracle_stream(h);
  }
}

void oracle_step_node(const oracle_t *h, int ix, int iy, int iz, double *out_f,
                      double *out_g) {
  /* collide the clamped 3x3(x3) box around the node into a local window */
  int idx[3] = {ix, iy, iz}, lo[3], cnt[3];
  for (int a = 0; a < 3; ++a) {
    if (a < h->dim) {
      lo[a] = idx[a] - 1;
      if (lo[a] < 0) lo[a] = 0;
      if (lo[a] > h->n[a] - 3) lo[a] = h->n[a] - 3;
      cnt[a] = 3;
    } else {
      lo[a] = 0;
      cnt[a] = 1;
    }
  }
  double bf[QF_MAX * 27], bg[QG_MAX * 27];
  const long nn = (long)h->nn;
  const int nx = h->n[0], ny = h->n[1];
  int box = cnt[0] * cnt[1] * cnt[2];
  for (int kz = 0; kz < cnt[2]; ++kz)
    for (int ky = 0; ky < cnt[1]; ++ky)
      for (int kx = 0; kx < cnt[0]; ++kx) {
        long c = ((long)(lo[2] + kz) * ny + (lo[1] + ky)) * nx + (lo[0] + kx);
        int lc = (kz * cnt[1] + ky) * cnt[0] + kx;
        double f[QF_MAX], g[QG_MAX], fp[QF_MAX], gp[QG_MAX];
        for (int i = 0; i < h->qf; ++i) f[i] = h->f[(long)i * nn + c];
        for (int i = 0; i < h->qg; ++i) g[i] = h->g[(long)i * nn + c];
        oracle_collide_node(h, f, g, fp, gp);
        for (int i = 0; i < h->qf; ++i) bf[i * box + lc] = fp[i];
        for (int i = 0; i < h->qg; ++i) bg[i * box + lc] = gp[i];
      }
  view_t vf = {bf, box, (long)cnt[0] * cnt[1], cnt[0], lo[0], lo[1], lo[2]};
  view_t vg = {bg, box, (long)cnt[0] * cnt[1], cnt[0], lo[0], lo[1], lo[2]};
  pull_node(h, &vf, &vg, idx, out_f, out_g);
}

/* ------------------------------------------------------------------------ */
/* init, I/O                                                                */
/* ------------------------------------------------------------------------ */

/* SplitMix64, random access by counter: state = seed + (k+1)*gamma
 * (reading A15). */
static uint64_t splitmix64_at(uint64_t seed, uint64_t k) {
  uint64_t z = seed + (k + 1u) * 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

/* Rest state: f = equilibrium at rho = 1, u = 0; g = equilibrium at
 * T = amp (2r - 1), u = 0; both obtained as M^-1 m_eq, N^-1 n_eq
 * (BASELINE.json configs: "rest, rho=1, T=0 plus uniform noise"). */
void oracle_init(oracle_t *h, unsigned long long seed, double amp) {
  const long nn = (long)h->nn;
  double u0[3] = {0.0, 0.0, 0.0};
  double meq[QF_MAX], feq[QF_MAX];
  oracle_meq(h, 1.0, u0, meq);
  for (int i = 0; i < h->qf; ++i) {
    double s = 0.0;
    for (int k = 0; k < h->qf; ++k) s += h->Minv[i][k] * meq[k];
    feq[i] = s;
  }
  for (long c = 0; c < nn; ++c) {
    uint64_t z = splitmix64_at((uint64_t)seed, (uint64_t)c);
    double r = (double)(z >> 11) * (1.0 / 9007199254740992.0);
    double T = amp * (2.0 * r - 1.0);
    double neq[QG_MAX];
    oracle_neq(h, T, u0, neq);
    for (int i = 0; i < h->qf; ++i) h->f[(long)i * nn + c] = feq[i];
    for (int i = 0; i < h->qg; ++i) {
      double s = 0.0;
      for (int k = 0; k < h->qg; ++k) s += h->Ninv[i][k] * neq[k];
      h->g[(long)i * nn + c] = s;
    }
  }
}

void oracle_set_populations(oracle_t *h, const double *f, const double *g) {
  memcpy(h->f, f, sizeof(double) * h->nn * (size_t)h->qf);
  memcpy(h->g, g, sizeof(double) * h->nn * (size_t)h->qg);
}
void oracle_get_populations(const oracle_t *h, double *f, double *g) {
  memcpy(f, h->f, sizeof(double) * h->nn * (size_t)h->qf);
  memcpy(g, h->g, sizeof(double) * h->nn * (size_t)h->qg);
}
void oracle_get_post_collision(const oracle_t *h, double *fp, double *gp) {
  memcpy(fp, h->fp, sizeof(double) * h->nn * (size_t)h->qf);
  memcpy(gp, h->gp, sizeof(double) * h->nn * (size_t)h->qg);
}

void oracle_set_post_collision(oracle_t *h, const double *fp, const double *gp) {
  memcpy(h->fp, fp, sizeof(double) * h->nn * (size_t)h->qf);
  memcpy(h->gp, gp, sizeof(double) * h->nn * (size_t)h->qg);
}

/* ------------------------------------------------------------------------ */
/* diagnostics                                                              */
/* ------------------------------------------------------------------------ */

void oracle_fields(const oracle_t *h, double *rho, double *u, double *v,
                   double *w, double *T) {
  const long nn = (long)h->nn;
  for (long c = 0; c < nn; ++c) {
    double f[QF_MAX], g[QG_MAX], r, uu[3], t, F[3];
    for (int i = 0; i < h->qf; ++i) f[i] = h->f[(long)i * nn + c];
    for (int i = 0; i < h->qg; ++i) g[i] = h->g[(long)i * nn + c];
    node_moments(h, f, g, &r, uu, &t, F);
    if (rho) rho[c] = r;
    if (u) u[c] = uu[0];
    if (v) v[c] = uu[1];
    if (w) w[c] = uu[2];
    if (T) T[c] = t;
  }
}

/* Eq. 28, bottom-wall form, Delta = 1 l.u.; the top-wall form
 * is its mirror image: d/dn(top) = -oracle_wall_derivative(q, wall, N, N-1). */
double oracle_wall_derivative(double q, double phi_wall, double phi1,
                              double phi2) {
  return (-4.0 * q * (q + 1.0) * phi_wall +
          (2.0 * q + 1.0) * (2.0 * q + 1.0) * phi1 - phi2) /
         (q * (2.0 * q + 1.0));
}

/* Nu_hot, Nu_cold: Eq. 32 / Eq. 41 with the wall
 * derivative of Eq. 28 and the weighted average of Eq. 29 normalised by the
 * effective length.  <Re>: Eq. 34 / Eq. 42 with the full speed
 * (reading A10).  <Nu>: Eq. 31 / Eq. 40.  Lattice -> free-fall units:
 * u* = u/U, x* = x_lu/H_lu, T* = (T - T0)/Delta_T with Delta_T = 1. */
void oracle_nusselt(const oracle_t *h, double out[5]) {
  const long nn = (long)h->nn;
  const int nx = h->n[0], ny = h->n[1], nz = h->n[2];
  double *T = (double *)malloc(sizeof(double) * (size_t)nn);
  double *u = (double *)malloc(sizeof(double) * (size_t)nn);
  double *v = (double *)malloc(sizeof(double) * (size_t)nn);
  double *w = (double *)malloc(sizeof(double) * (size_t)nn);
  oracle_fields(h, NULL, u, v, w, T);
  double q_lo = (h->x[0][1] - h->x[0][0]) / h->delta;
  double q_hi = (h->x[0][nx - 1] - h->x[0][nx - 2]) / h->delta;
  double area = h->L_eff[1] * (h->dim == 3 ? h->L_eff[2] : 1.0);
  double vol = area * h->L_eff[0];
  double s_hot = 0.0, s_cold = 0.0, s_spd = 0.0, s_u2 = 0.0, s_uT = 0.0;
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy) {
      double wa = h->avgw[1][iy] * h->avgw[2][iz];
      long r = ((long)iz * ny + iy) * nx;
      double d_hot = oracle_wall_derivative(q_lo, h->T_hot, T[r], T[r + 1]);
      double d_cold = -oracle_wall_derivative(q_hi, h->T_cold, T[r + nx - 1],
                                              T[r + nx - 2]);
      s_hot += wa * d_hot;
      s_cold += wa * d_cold;
      for (int ix = 0; ix < nx; ++ix) {
        double wv = wa * h->avgw[0][ix];
        double uu = u[r + ix], vv = v[r + ix], ww = w[r + ix];
        double sp2 = uu * uu + vv * vv + ww * ww;
        s_spd += wv * sqrt(sp2);
        s_u2 += wv * sp2;
        s_uT += wv * uu * (T[r + ix] - h->T0);
      }
    }
  out[0] = -h->H_lu * s_hot / area;
  out[1] = -h->H_lu * s_cold / area;
  out[2] = sqrt(h->Ra / h->Pr) * (s_spd / vol) / h->U;
  out[3] = (s_u2 / vol) / (h->U * h->U);
  out[4] = sqrt(h->Ra * h->Pr) * (s_uT / vol) / h->U + 1.0;
  free(T);
  free(u);
  free(v);
  free(w);
}

/* Nu_middle, Eq. 33: line (area) average over the vertical centre plane x* = 0.5 of
 * sqrt(Ra Pr) u* T* - dT* / dx*.  The paper does not say how the derivative is taken or what happens when
 * no node column sits at x* = 0.5 (reading A23): dT/dx at a node column is the derivative of the
 * parabola through the column and its two neighbours (second order on the stretched mesh), and the flux is
 * interpolated linearly between the two columns that bracket the midpoint of the two x-walls.  Averaging
 * weights and normalisation as for Nu_hot (Eq. 29). */
double oracle_nusselt_middle(const oracle_t *h) {
  const long nn = (long)h->nn;
  const int nx = h->n[0], ny = h->n[1], nz = h->n[2];
  double *T = (double *)malloc(sizeof(double) * (size_t)nn);
  double *u = (double *)malloc(sizeof(double) * (size_t)nn);
  oracle_fields(h, NULL, u, NULL, NULL, T);
  const double *x = h->x[0];
  double xmid = 0.5 * ((x[0] - 0.5 * h->delta) + (x[nx - 1] + 0.5 * h->delta));
  int i0 = 1;
  while (i0 < nx - 3 && x[i0 + 1] <= xmid) ++i0;          /* x[i0] <= xmid < x[i0+1], 1 <= i0 <= nx-3 */
  double a1 = (xmid - x[i0]) / (x[i0 + 1] - x[i0]);
  if (a1 < 0.0 || nx < 4) a1 = 0.0;                        /* nx = 3: the only interior column */
  if (a1 > 1.0) a1 = 1.0;
  double a[2] = {1.0 - a1, a1};
  double area = h->L_eff[1] * (h->dim == 3 ? h->L_eff[2] : 1.0);
  double s = 0.0;
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy) {
      double wa = h->avgw[1][iy] * h->avgw[2][iz];
      long r = ((long)iz * ny + iy) * nx;
      for (int k = 0; k < 2; ++k) {
        int i = i0 + k;
        if (a[k] == 0.0) continue;
        double hm = (x[i] - x[i - 1]) / h->delta, hp = (x[i + 1] - x[i]) / h->delta;   /* lattice units */
        double dTdx = -hp / (hm * (hm + hp)) * T[r + i - 1] + (hp - hm) / (hm * hp) * T[r + i] +
                      hm / (hp * (hm + hp)) * T[r + i + 1];
        double flux = sqrt(h->Ra * h->Pr) * (u[r + i] / h->U) * (T[r + i] - h->T0) - h->H_lu * dTdx;
        s += wa * a[k] * flux;
      }
    }
  free(T);
  free(u);
  return s / area;
}

void oracle_mass(const oracle_t *h, double out[2]) {
  const long nn = (long)h->nn;
  const int nx = h->n[0], ny = h->n[1], nz = h->n[2];
  double sw = 0.0, sp = 0.0;
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy)
      for (int ix = 0; ix < nx; ++ix) {
        long c = ((long)iz * ny + iy) * nx + ix;
        double r = 0.0;
        for (int i = 0; i < h->qf; ++i) r += h->f[(long)i * nn + c];
        sw += r * h->avgw[0][ix] * h->avgw[1][iy] * h->avgw[2][iz];
        sp += r;
      }
  out[0] = sw;
  out[1] = sp;
}

/* ------------------------------------------------------------------------ */
/* introspection                                                            */
/* ------------------------------------------------------------------------ */

int oracle_qf(const oracle_t *h) { return h->qf; }
int oracle_qg(const oracle_t *h) { return h->qg; }

void oracle_get_velocities(const oracle_t *h, int *ef, int *eg) {
  for (int i = 0; i < h->qf; ++i)
    for (int a = 0; a < 3; ++a) ef[3 * i + a] = h->ef[i][a];
  for (int i = 0; i < h->qg; ++i)
    for (int a = 0; a < 3; ++a) eg[3 * i + a] = h->eg[i][a];
}

void oracle_get_matrices(const oracle_t *h, double *M, double *Minv, double *S,
                         double *N, double *Ninv, double *Q) {
  for (int k = 0; k < h->qf; ++k) {
    S[k] = h->S[k];
    for (int i = 0; i < h->qf; ++i) {
      M[k * h->qf + i] = h->M[k][i];
      Minv[k * h->qf + i] = h->Minv[k][i];
    }
  }
  for (int k = 0; k < h->qg; ++k) {
    Q[k] = h->Q[k];
    for (int i = 0; i < h->qg; ++i) {
      N[k * h->qg + i] = h->N[k][i];
      Ninv[k * h->qg + i] = h->Ninv[k][i];
    }
  }
}

void oracle_get_params(const oracle_t *h, double out[12]) {
  out[0] = h->U;
  out[1] = h->H_lu;
  out[2] = h->nu;
  out[3] = h->alpha;
  out[4] = h->gbeta;
  out[5] = h->tau_f;
  out[6] = h->a_T;
  out[7] = h->omega_bc;
  out[8] = h->U / h->H_lu; /* dt* of one step: delta_t / t_f */
  out[9] = h->L_eff[0];
  out[10] = h->L_eff[1];
  out[11] = h->L_eff[2];
}

void oracle_get_weights(const oracle_t *h, int axis, int sign_idx, int *base,
                        double *w) {
  int n = h->n[axis];
  memcpy(base, h->base[axis][sign_idx], sizeof(int) * (size_t)n);
  memcpy(w, h->wgt[axis][sign_idx], sizeof(double) * 3 * (size_t)n);
}
