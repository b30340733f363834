// Test-only host build of the node-local device functions (csrc/islbm_lattice.cuh)
// so that the hand-factored collisions can be compared with the oracle on a box
// without a GPU.  Not linked into the product library.
#include "../../paper_2509_01099_b200/csrc/islbm_lattice.cuh"

extern "C" void harness_collide(int dim, double *f, double *g, const double *prm) {
  islbmk::NodeParams p;
  p.gbeta = prm[0]; p.s_nu = prm[1]; p.s_q = prm[2];
  p.hs_nu = 1.0 - 0.5 * p.s_nu; p.hs_q = 1.0 - 0.5 * p.s_q;
  p.q_k = prm[3]; p.q_e = prm[4]; p.a_T = prm[5]; p.T0 = 0.0;
  islbmk::fold_node_params(p, dim);
  if (dim == 2) {
    double ff[9], gg[5];
    for (int i = 0; i < 9; ++i) ff[i] = f[i];
    for (int i = 0; i < 5; ++i) gg[i] = g[i];
    islbmk::collide_node(ff, gg, p);
    for (int i = 0; i < 9; ++i) f[i] = ff[i];
    for (int i = 0; i < 5; ++i) g[i] = gg[i];
  } else {
    double ff[19], gg[7];
    for (int i = 0; i < 19; ++i) ff[i] = f[i];
    for (int i = 0; i < 7; ++i) gg[i] = g[i];
    islbmk::collide_node(ff, gg, p);
    for (int i = 0; i < 19; ++i) f[i] = ff[i];
    for (int i = 0; i < 7; ++i) g[i] = gg[i];
  }
}

// deviation form used by the fp32-storage kernels: collide f - w in place, return (f - w)+ + w
extern "C" void harness_collide_dev(int dim, double *f, double *g, const double *prm) {
  islbmk::NodeParams p;
  p.gbeta = prm[0]; p.s_nu = prm[1]; p.s_q = prm[2];
  p.hs_nu = 1.0 - 0.5 * p.s_nu; p.hs_q = 1.0 - 0.5 * p.s_q;
  p.q_k = prm[3]; p.q_e = prm[4]; p.a_T = prm[5]; p.T0 = 0.0;
  islbmk::fold_node_params(p, dim);
  if (dim == 2) {
    double ff[9], gg[5];
    for (int i = 0; i < 9; ++i) ff[i] = f[i] - islbmk::wflow<2>(i);
    for (int i = 0; i < 5; ++i) gg[i] = g[i];
    islbmk::collide_node<true>(ff, gg, p);
    for (int i = 0; i < 9; ++i) f[i] = ff[i] + islbmk::wflow<2>(i);
    for (int i = 0; i < 5; ++i) g[i] = gg[i];
  } else {
    double ff[19], gg[7];
    for (int i = 0; i < 19; ++i) ff[i] = f[i] - islbmk::wflow<3>(i);
    for (int i = 0; i < 7; ++i) gg[i] = g[i];
    islbmk::collide_node<true>(ff, gg, p);
    for (int i = 0; i < 19; ++i) f[i] = ff[i] + islbmk::wflow<3>(i);
    for (int i = 0; i < 7; ++i) g[i] = gg[i];
  }
}

// the fp32-storage kernels' form: fp32 deviations in, fp32 deviations out (collide_node<true, float>)
extern "C" void harness_collide_dev_f32(int dim, float *fdev, float *g, const double *prm) {
  islbmk::NodeParams p;
  p.gbeta = prm[0]; p.s_nu = prm[1]; p.s_q = prm[2];
  p.hs_nu = 1.0 - 0.5 * p.s_nu; p.hs_q = 1.0 - 0.5 * p.s_q;
  p.q_k = prm[3]; p.q_e = prm[4]; p.a_T = prm[5]; p.T0 = 0.0;
  islbmk::fold_node_params(p, dim);
  if (dim == 2) {
    float ff[9], gg[5];
    for (int i = 0; i < 9; ++i) ff[i] = fdev[i];
    for (int i = 0; i < 5; ++i) gg[i] = g[i];
    islbmk::collide_node<true>(ff, gg, p);
    for (int i = 0; i < 9; ++i) fdev[i] = ff[i];
    for (int i = 0; i < 5; ++i) g[i] = gg[i];
  } else {
    float ff[19], gg[7];
    for (int i = 0; i < 19; ++i) ff[i] = fdev[i];
    for (int i = 0; i < 7; ++i) gg[i] = g[i];
    islbmk::collide_node<true>(ff, gg, p);
    for (int i = 0; i < 19; ++i) fdev[i] = ff[i];
    for (int i = 0; i < 7; ++i) g[i] = gg[i];
  }
}

// the all-fp32 deviation-form collisions called directly (3-D: what the fp32-storage kernels run; 2-D: the A/B switch
// ISLBM_F_FP32_2D, off by default)
extern "C" void harness_collide_dev_allf32(int dim, float *fdev, float *g, const double *prm) {
  islbmk::NodeParams p;
  p.gbeta = prm[0]; p.s_nu = prm[1]; p.s_q = prm[2];
  p.hs_nu = 1.0 - 0.5 * p.s_nu; p.hs_q = 1.0 - 0.5 * p.s_q;
  p.q_k = prm[3]; p.q_e = prm[4]; p.a_T = prm[5]; p.T0 = 0.0;
  islbmk::fold_node_params(p, dim);
  if (dim == 2) {
    float ff[9], gg[5];
    for (int i = 0; i < 9; ++i) ff[i] = fdev[i];
    for (int i = 0; i < 5; ++i) gg[i] = g[i];
    islbmk::collide_node_dev_f32(ff, gg, p);
    for (int i = 0; i < 9; ++i) fdev[i] = ff[i];
    for (int i = 0; i < 5; ++i) g[i] = gg[i];
  } else {
    float ff[19], gg[7];
    for (int i = 0; i < 19; ++i) ff[i] = fdev[i];
    for (int i = 0; i < 7; ++i) gg[i] = g[i];
    islbmk::collide_node_dev_f32(ff, gg, p);
    for (int i = 0; i < 19; ++i) fdev[i] = ff[i];
    for (int i = 0; i < 7; ++i) g[i] = gg[i];
  }
}

// out: rho,u,v,w,T from post-collision populations
extern "C" void harness_fields_post(int dim, const double *f, const double *g, const double *prm, double *out) {
  islbmk::NodeParams p{};
  p.gbeta = prm[0];
  if (dim == 2) {
    double ff[9], gg[5];
    for (int i = 0; i < 9; ++i) ff[i] = f[i];
    for (int i = 0; i < 5; ++i) gg[i] = g[i];
    islbmk::fields_from_post(ff, gg, p, out[0], out[1], out[2], out[3], out[4]);
  } else {
    double ff[19], gg[7];
    for (int i = 0; i < 19; ++i) ff[i] = f[i];
    for (int i = 0; i < 7; ++i) gg[i] = g[i];
    islbmk::fields_from_post(ff, gg, p, out[0], out[1], out[2], out[3], out[4]);
  }
}

extern "C" void harness_tables(int dim, int *e, int *opp, double *w) {
  int qf = dim == 2 ? 9 : 19;
  for (int q = 0; q < qf; ++q) {
    for (int a = 0; a < 3; ++a) e[3 * q + a] = dim == 2 ? islbmk::evel<2>(q, a) : islbmk::evel<3>(q, a);
    opp[q] = dim == 2 ? islbmk::opposite<2>(q) : islbmk::opposite<3>(q);
    w[q] = dim == 2 ? islbmk::wflow<2>(q) : islbmk::wflow<3>(q);
  }
}

// storage-plane permutation of the workspace (plane_f / plane_g) and its inverse
extern "C" void harness_planes(int dim, int *pf, int *pg, int *inv) {
  const int qf = dim == 2 ? 9 : 19, qg = dim == 2 ? 5 : 7;
  for (int q = 0; q < qf; ++q) pf[q] = dim == 2 ? islbmk::plane_f<2>(q) : islbmk::plane_f<3>(q);
  for (int q = 0; q < qg; ++q) pg[q] = dim == 2 ? islbmk::plane_g<2>(q) : islbmk::plane_g<3>(q);
  for (int p = 0; p < qf + qg; ++p) inv[p] = dim == 2 ? islbmk::pop_of_plane<2>(p) : islbmk::pop_of_plane<3>(p);
}
