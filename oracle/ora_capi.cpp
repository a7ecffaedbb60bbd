// ora_capi.cpp — extern "C" surface of the CPU ORACLE (test infrastructure, not the product).
// See ora.h.  Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
#include <cstdio>
#include <cstdlib>
#include <new>
#ifdef _OPENMP
#include <omp.h>
#endif
#include "ora.h"
#include "ora_solver.hpp"
#include "ora_naive.hpp"

struct ora_solver {
  ora::Config c;
  int dtype;
};

extern "C" {

int ora_create(ora_solver** out, const ora_grid* g, int dtype, double gamma, double R_gas, double Pr,
               const ora_mu_law* mu, const ora_bc* bc, const double body_accel[3]) {
  if (!out) return ORA_EINVAL;
  *out = nullptr;
  if (!g || !mu || !bc) return ORA_EINVAL;
  if (g->nx < 4 || g->ny < 4 || g->nz < 4 || !g->xf || !g->yf || !g->zf) return ORA_EINVAL;
  if (!(gamma > 1.0) || !(Pr > 0.0) || !(mu->mu_ref >= 0.0) || !(R_gas > 0.0)) return ORA_EINVAL;
  if (dtype != ORA_F64 && dtype != ORA_F32 && dtype != ORA_F80) return ORA_EINVAL;
  const double* xf[3] = {g->xf, g->yf, g->zf};
  int n[3] = {g->nx, g->ny, g->nz};
  for (int a = 0; a < 3; ++a)
    for (int i = 0; i < n[a]; ++i)
      if (!(xf[a][i + 1] > xf[a][i])) return ORA_EINVAL;
  for (int a = 0; a < 3; ++a) {
    bool lo = bc->face[2 * a].type == ORA_BC_PERIODIC, hi = bc->face[2 * a + 1].type == ORA_BC_PERIODIC;
    if (lo != hi) return ORA_EINVAL;
  }
  for (int f = 0; f < 6; ++f) {
    int t = bc->face[f].type;
    if (t < 0 || t > 4) return ORA_EINVAL;
    if (t == ORA_BC_DIRICHLET && !bc->face[f].dirichlet) return ORA_EINVAL;
    if (t == ORA_BC_WALL_ISOTHERMAL && !(bc->face[f].T_wall > 0.0)) return ORA_EINVAL;
  }
  ora_solver* s = new (std::nothrow) ora_solver;
  if (!s) return ORA_EINVAL;
  ora::Config& c = s->c;
  for (int a = 0; a < 3; ++a) { c.n[a] = n[a]; c.xf[a].assign(xf[a], xf[a] + n[a] + 1); }
  c.gamma = gamma; c.Rgas = R_gas; c.Pr = Pr; c.mu = *mu; c.bc = *bc;
  for (int a = 0; a < 3; ++a) c.g[a] = body_accel ? body_accel[a] : 0.0;
  c.viscous = mu->mu_ref > 0.0;
  for (int f = 0; f < 6; ++f) {
    if (bc->face[f].type == ORA_BC_DIRICHLET) {
      int a = f / 2;
      int t1a = (a == 0) ? 1 : 0, t2a = (a == 2) ? 1 : 2;
      size_t cnt = (size_t)5 * n[t1a] * n[t2a];
      c.dirichlet[f].assign(bc->face[f].dirichlet, bc->face[f].dirichlet + cnt);
    }
    c.bc.face[f].dirichlet = nullptr;
  }
  ora::build_metrics(c);
  s->dtype = dtype;
  *out = s;
  return ORA_OK;
}

int ora_set_visc_order(ora_solver* s, int order) {
  if (!s || (order != 4 && order != 6)) return ORA_EINVAL;
  s->c.visc_order = order;
  ora::build_metrics(s->c);
  return ORA_OK;
}

void ora_destroy(ora_solver* s) { delete s; }

size_t ora_state_elems(const ora_solver* s) { return (size_t)5 * s->c.P[0] * s->c.P[1] * s->c.P[2]; }

int ora_fill_halo(ora_solver* s, void* U) {
  if (!s || !U) return ORA_EINVAL;
  if (s->dtype == ORA_F64) ora::fill_halo<double>(s->c, (double*)U);
  else if (s->dtype == ORA_F80) ora::fill_halo<long double>(s->c, (long double*)U);
  else ora::fill_halo<float>(s->c, (float*)U);
  return ORA_OK;
}

int ora_rhs(ora_solver* s, const void* U, void* R) {
  if (!s || !U || !R) return ORA_EINVAL;
  if (s->dtype == ORA_F64) ora::rhs<double>(s->c, (const double*)U, (double*)R, true, true, true);
  else if (s->dtype == ORA_F80) ora::rhs<long double>(s->c, (const long double*)U, (long double*)R, true, true, true);
  else ora::rhs<float>(s->c, (const float*)U, (float*)R, true, true, true);
  return ORA_OK;
}

int ora_rhs_parts(ora_solver* s, const void* U, void* R, int inviscid, int viscous, int source) {
  if (!s || !U || !R || s->dtype != ORA_F64) return ORA_EINVAL;
  ora::rhs<double>(s->c, (const double*)U, (double*)R, inviscid != 0, viscous != 0, source != 0);
  return ORA_OK;
}

int ora_rhs_naive(ora_solver* s, const void* U, void* R) {
  if (!s || !U || !R || s->dtype != ORA_F64) return ORA_EINVAL;
  ora_naive::rhs(s->c, (const double*)U, (double*)R, true, true, true);
  return ORA_OK;
}

int ora_rk3_step(ora_solver* s, void* U, double dt) {
  if (!s || !U) return ORA_EINVAL;
  if (s->dtype == ORA_F64) ora::rk3_step<double>(s->c, (double*)U, dt);
  else if (s->dtype == ORA_F80) ora::rk3_step<long double>(s->c, (long double*)U, (long double)dt);
  else ora::rk3_step<float>(s->c, (float*)U, (float)dt);
  return ORA_OK;
}

int ora_cfl_dt(ora_solver* s, const void* U, double cfl, double* dt) {
  if (!s || !U || !dt) return ORA_EINVAL;
  if (s->dtype == ORA_F64) return ora::cfl_dt<double>(s->c, (const double*)U, cfl, dt);
  if (s->dtype == ORA_F80) return ora::cfl_dt<long double>(s->c, (const long double*)U, cfl, dt);
  return ora::cfl_dt<float>(s->c, (const float*)U, cfl, dt);
}

int ora_count_flops_step(ora_solver* s, const void* U, double dt, double counts[4]) {
  if (!s || !U || !counts || s->dtype != ORA_F64) return ORA_EINVAL;
  size_t ne = ora_state_elems(s);
  std::vector<ora::Cnt> Uc(ne);
  const double* Ud = (const double*)U;
  for (size_t i = 0; i < ne; ++i) Uc[i].v = Ud[i];
  ora::Cnt::n_basic = ora::Cnt::n_div = ora::Cnt::n_sqrt = 0;
  int saved = 1;
#ifdef _OPENMP
  saved = omp_get_max_threads();
  omp_set_num_threads(1);  // the counters are plain globals
#endif
  ora::rk3_step<ora::Cnt>(s->c, Uc.data(), ora::Cnt(dt));
#ifdef _OPENMP
  omp_set_num_threads(saved);
#endif
  (void)saved;
  counts[0] = ora::Cnt::n_basic; counts[1] = ora::Cnt::n_div; counts[2] = ora::Cnt::n_sqrt;
  counts[3] = counts[0] + counts[1] + counts[2];
  return ORA_OK;
}

int ora_count_flops_part(ora_solver* s, const void* U, int what, double counts[4]) {
  // what: 1 = cons->prim over the padded box, 2 = centre gradients, 3 = one full RHS (Eq. 6)
  if (!s || !U || !counts || s->dtype != ORA_F64 || what < 1 || what > 3) return ORA_EINVAL;
  size_t ne = ora_state_elems(s);
  std::vector<ora::Cnt> Uc(ne), Rc(ne);
  const double* Ud = (const double*)U;
  for (size_t i = 0; i < ne; ++i) Uc[i].v = Ud[i];
  int saved = 1;
#ifdef _OPENMP
  saved = omp_get_max_threads();
  omp_set_num_threads(1);
#endif
  ora::Prim<ora::Cnt> P;
  ora::Cnt::n_basic = ora::Cnt::n_div = ora::Cnt::n_sqrt = 0;
  if (what == 1) ora::compute_prims<ora::Cnt>(s->c, Uc.data(), P);
  if (what == 2) {
    ora::compute_prims<ora::Cnt>(s->c, Uc.data(), P);
    ora::Cnt::n_basic = ora::Cnt::n_div = ora::Cnt::n_sqrt = 0;
    ora::compute_gradients<ora::Cnt>(s->c, P);
  }
  if (what == 3) ora::rhs<ora::Cnt>(s->c, Uc.data(), Rc.data(), true, true, true);
#ifdef _OPENMP
  omp_set_num_threads(saved);
#endif
  (void)saved;
  counts[0] = ora::Cnt::n_basic; counts[1] = ora::Cnt::n_div; counts[2] = ora::Cnt::n_sqrt;
  counts[3] = counts[0] + counts[1] + counts[2];
  return ORA_OK;
}

int ora_metrics(const ora_solver* s, int axis, double* delta, double* centre) {
  if (!s || axis < 0 || axis > 2) return ORA_EINVAL;
  for (int p = 0; p < s->c.P[axis]; ++p) {
    if (delta) delta[p] = s->c.dl[axis][p];
    if (centre) centre[p] = s->c.xc[axis][p];
  }
  return ORA_OK;
}

int ora_metrics_index(const ora_solver* s, int axis, double* Xc, double* Xf) {
  if (!s || axis < 0 || axis > 2) return ORA_EINVAL;
  for (int p = 0; p < s->c.P[axis]; ++p) {
    if (Xc) Xc[p] = s->c.Xc[axis][p];
    if (Xf) Xf[p] = s->c.Xf[axis][p];
  }
  return ORA_OK;
}

double ora_weno5(const double v[5]) { return ora::weno5<double>(v[0], v[1], v[2], v[3], v[4]); }
void ora_weno5_detail(const double v[5], double beta[3], double omega[3], double p[3]) {
  ora::weno5<double>(v[0], v[1], v[2], v[3], v[4], beta, omega, p);
}
void ora_hllc(int dir, double gamma, const double WL[5], const double WR[5], double F[5]) {
  ora::hllc<double>(dir, gamma, WL, WR, F);
}
void ora_flux_phys(int dir, double gamma, const double W[5], double F[5]) { ora::flux_phys<double>(dir, gamma, W, F); }
void ora_cons_to_prim(double gamma, const double U[5], double W[5]) { ora::cons_to_prim<double>(gamma, U, W); }
void ora_prim_to_cons(double gamma, const double W[5], double U[5]) { ora::prim_to_cons<double>(gamma, W, U); }
double ora_viscosity(const ora_mu_law* mu, double T) {
  return ora::viscosity<double>(mu->sutherland, mu->mu_ref, mu->T_ref, mu->S, T);
}
double ora_dc(const double phi[5], double Xc) { return ora::d_centre<double>(phi[0], phi[1], phi[3], phi[4], Xc); }
double ora_df(const double phi[4], double Xf) { return ora::d_face<double>(phi[0], phi[1], phi[2], phi[3], Xf); }
double ora_if(const double phi[4]) { return ora::i_face<double>(phi[0], phi[1], phi[2], phi[3]); }
double ora_dc6(const double phi[7], double Xc) { return ora::d_centre6<double>(phi[0], phi[1], phi[2], phi[4], phi[5], phi[6], Xc); }
double ora_df6(const double phi[6], double Xf) { return ora::d_face6<double>(phi[0], phi[1], phi[2], phi[3], phi[4], phi[5], Xf); }
double ora_if6(const double phi[6]) { return ora::i_face6<double>(phi[0], phi[1], phi[2], phi[3], phi[4], phi[5]); }

int ora_viscous_face(ora_solver* s, const void* U, int dir, int i, int j, int k, double Fd[5]) {
  if (!s || !U || s->dtype != ORA_F64 || dir < 0 || dir > 2) return ORA_EINVAL;
  ora::Prim<double> P;
  ora::compute_prims<double>(s->c, (const double*)U, P);
  ora::compute_gradients<double>(s->c, P);
  int pc[3] = {i + ora::NH, j + ora::NH, k + ora::NH};
  ora::viscous_face<double>(s->c, P, dir, pc, Fd);
  return ORA_OK;
}

}  // extern "C"
