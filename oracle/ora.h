/* ora.h — C interface of the CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU implementation of the hot path of
 * arxiv/paper_2406_19494 (Eq. 1-6; halo layout PAPER.md:80;
 * boundary conditions by halo assignment PAPER.md:100-104; Eq. 8), with the
 * schemes BASELINE.json:north_star names (WENO5-JS, HLLC, 4th-order central viscous/heat
 * flux with Sutherland viscosity, SSP-RK3, CFL step).  Formulas the paper does not print
 * follow SURVEY.md §8(c) O1-O9 and are listed as "readings" in DESIGN.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may load this library.  It shares no code with paper_2406_19494_b200/csrc.
 *
 * Layout (Nh = 3): U[5][nz+6][ny+6][nx+6], x fastest,
 *   index ((q*(nz+6)+k+3)*(ny+6)+j+3)*(nx+6)+i+3, q in {rho, rho*u, rho*v, rho*w, E}.
 * All pointers are HOST pointers.  dtype 0 = double, 1 = float, 2 = long double (the arbiter:
 * same text instantiated on a 64-bit mantissa, rational constants formed in that precision).
 */
#ifndef ORA_H
#define ORA_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ora_solver ora_solver;

enum { ORA_OK = 0, ORA_EINVAL = 1, ORA_ENOTFINITE = 5 };
enum { ORA_F64 = 0, ORA_F32 = 1,
       ORA_F80 = 2 /* x87 long double (16-byte elements): the arbiter instantiation, tests only */ };
enum { ORA_BC_PERIODIC = 0, ORA_BC_ZEROGRAD = 1, ORA_BC_DIRICHLET = 2,
       ORA_BC_WALL_ISOTHERMAL = 3, ORA_BC_WALL_ADIABATIC = 4 };

typedef struct {
  int nx, ny, nz;
  const double *xf, *yf, *zf; /* nx+1, ny+1, nz+1 face coordinates, strictly increasing */
} ora_grid;

typedef struct { int sutherland; double mu_ref, T_ref, S; } ora_mu_law;

typedef struct {
  int enabled;
  double A, kappa;     /* v_w(t1) = A*sin(2*pi*kappa*t1), Eq. 8 */
  double t1_lo, t1_hi; /* active where t1_lo <= t1 <= t1_hi               */
} ora_disturbance;

typedef struct {
  int type;
  double T_wall;
  double u_wall[3];        /* wall velocity vector (u,v,w)                              */
  const double *dirichlet; /* prim[5][n_t2][n_t1] (rho,u,v,w,p), interior tangential sizes */
  ora_disturbance dist;
} ora_bc_face;

typedef struct { ora_bc_face face[6]; } ora_bc; /* x-, x+, y-, y+, z-, z+ */

/* --- the five calls (same meaning as include/jf.h, on host arrays) --- */
int ora_create(ora_solver **out, const ora_grid *g, int dtype, double gamma, double R_gas,
               double Pr, const ora_mu_law *mu, const ora_bc *bc, const double body_accel[3]);
/* order of the central dissipative-flux stencils: 4 (default; north_star) or 6:
   centre / face derivatives, face interpolation and the index-space metrics all switch together */
int ora_set_visc_order(ora_solver *s, int order);
void ora_destroy(ora_solver *s);
size_t ora_state_elems(const ora_solver *s);
int ora_fill_halo(ora_solver *s, void *U);
int ora_rhs(ora_solver *s, const void *U, void *R);        /* halos of U must be filled */
int ora_rk3_step(ora_solver *s, void *U, double dt);
int ora_cfl_dt(ora_solver *s, const void *U, double cfl, double *dt);

/* second, deliberately naive RHS (per cell, six fluxes from scratch, Toro's four-branch
   HLLC): brute-force pin for the face-loop ora_rhs on tiny grids. double only. */
int ora_rhs_naive(ora_solver *s, const void *U, void *R);

/* separate inviscid / viscous parts of R (double only; for pins) */
int ora_rhs_parts(ora_solver *s, const void *U, void *R, int inviscid, int viscous, int source);

/* flop counting: runs one RK3 step on a counting scalar type (data in double).
   counts[0]=add/sub/mul/min/max (1 each), [1]=div, [2]=sqrt, [3]=total. */
int ora_count_flops_step(ora_solver *s, const void *U, double dt, double counts[4]);

/* same convention; what: 1 = cons->prim over the padded box, 2 = centre gradients, 3 = one RHS */
int ora_count_flops_part(ora_solver *s, const void *U, int what, double counts[4]);

/* grid metrics (padded arrays of length n+6 for axis a in 0..2): widths and centres */
int ora_metrics(const ora_solver *s, int axis, double *delta, double *centre);
/* index-space metrics of O2: Xc[p] = X_xi^c at padded cell p (interior p; 0 elsewhere), Xf[p] = X_xi^f of
   the face on the high side of padded cell p (p = 2 .. n+2; 0 elsewhere) */
int ora_metrics_index(const ora_solver *s, int axis, double *Xc, double *Xf);

/* --- unit-level functions for the pins (double) --- */
/* WENO5-JS value at the face between v[2] and v[3], stencil v[0..4] */
double ora_weno5(const double v[5]);
void ora_weno5_detail(const double v[5], double beta[3], double omega[3], double p[3]);
/* HLLC flux in direction dir (0,1,2) from primitive states (rho,u,v,w,p) */
void ora_hllc(int dir, double gamma, const double WL[5], const double WR[5], double F[5]);
/* physical convective flux of Eq. 3 in direction dir from a primitive state */
void ora_flux_phys(int dir, double gamma, const double W[5], double F[5]);
void ora_cons_to_prim(double gamma, const double U[5], double W[5]);
void ora_prim_to_cons(double gamma, const double W[5], double U[5]);
double ora_viscosity(const ora_mu_law *mu, double T);
/* central stencils on 4 (face) or 4 (centre, i-2,i-1,i+1,i+2) samples; metric passed in */
double ora_dc(const double phi[5], double Xc);  /* phi[0..4] = i-2..i+2 */
double ora_df(const double phi[4], double Xf);  /* phi[0..3] = i-1..i+2, face i+1/2 */
double ora_if(const double phi[4]);
/* sixth-order members: phi[0..6] = i-3..i+3 (centre), phi[0..5] = i-2..i+3 (face i+1/2) */
double ora_dc6(const double phi[7], double Xc);
double ora_df6(const double phi[6], double Xf);
double ora_if6(const double phi[6]);
/* dissipative flux of one face (dir, face index (i,j,k) = the cell on its low side) */
int ora_viscous_face(ora_solver *s, const void *U, int dir, int i, int j, int k, double Fd[5]);

#ifdef __cplusplus
}
#endif
#endif
