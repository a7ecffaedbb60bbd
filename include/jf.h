/* jf.h — C ABI of libjf: B200-native (sm_100a) finite-volume right-hand side of the 3-D
 * compressible Navier-Stokes equations on a structured, optionally stretched Cartesian grid,
 * after arxiv/paper_2406_19494.
 *
 * What the calls compute (citations are PAPER.md line numbers):
 *   state U = [rho, rho u, rho v, rho w, E], E = rho e + 1/2 rho u.u         Eq. 2, :44-46
 *   dU/dt = R_NSE(U): flux divergence of convective (Eq. 3, :50) minus dissipative (Eq. 4-5,
 *   :54-62) face fluxes with per-cell widths, plus sources                   Eq. 6, :64-69
 *   convective face flux: WENO-type reconstruction + approximate Riemann solver (:72) —
 *   here WENO5-JS on primitive variables + HLLC (:88); dissipative flux: central finite
 *   differences (:72) — here 4th order (6th order, the paper's DNS, :90, by jf_set_visc_order),
 *   Sutherland viscosity (:108), Fourier heat flux (:62)
 *   time integration: explicit TVD Runge-Kutta (:72) — here SSP-RK3
 *   arrays carry Nh = 3 halo cells per side, shape [N+2Nh]^3 (:80); boundary conditions are
 *   imposed by assigning the halo cells (:100): periodic, zero-gradient, Dirichlet, no-slip wall
 *   (isothermal / adiabatic) and the paper's "Disturbance Wall" v = A sin(2 pi kappa x)
 *   (:102-104, Eq. 8 :112), which with A = 0 is exactly the no-slip wall (:104).
 * Formulas the paper does not print are fixed in DESIGN.md ("Readings").
 *
 * Conventions
 *   - All functions return jf_status (0 = success) unless noted; no exception crosses the ABI.
 *   - "dev" pointers are DEVICE pointers owned by the caller (e.g. torch tensors); "host"
 *     pointers are host memory.  The library allocates no device memory for fields: scratch
 *     is the caller's workspace (jf_workspace_bytes).  Small metric/BC tables are carved out of
 *     the same workspace.
 *   - State layout: jf_state_elems() contiguous elements of the solver's dtype,
 *       index ((q*(nz+6) + k+3)*(ny+6) + j+3)*(nx+6) + i+3,  q in {rho, rho u, rho v, rho w, E},
 *     x fastest; base address 16-byte aligned (JF_EALIGN otherwise).
 *   - Every launch goes to the cuda_stream given to jf_create (a cudaStream_t passed as
 *     void*; NULL = default stream).  Only jf_cfl_dt, jf_dev_time, jf_set_visc_order, jf_set_tangent_seed and
 *     jf_diag_* synchronise that stream.
 *   - A solver belongs to the CUDA device that was current at jf_create (its workspace must live there: JF_EINVAL
 *     otherwise); every call makes that device current for its duration and restores the caller's.
 *   - One jf_solver per host thread / stream (thread-compatible, not thread-safe).
 *   - There is no CPU fallback: without a CUDA device every compute call fails with JF_ECUDA.
 */
#ifndef JF_H
#define JF_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct jf_solver jf_solver; /* opaque */

typedef enum {
  JF_OK = 0, JF_EINVAL = 1, JF_EALIGN = 2, JF_EWORKSPACE = 3, JF_ECUDA = 4, JF_ENOTFINITE = 5
} jf_status;
/* JF_F64_TANGENT: forward-mode (tangent) solver.  Every state element is a pair of doubles
 * (value, tangent), i.e. U_dev / R_dev hold jf_state_elems() pairs = 2*jf_state_elems() doubles,
 * element e at doubles [2e] (value) and [2e+1] (directional derivative); the same kernels run on a
 * dual-number scalar, so the value part follows the JF_F64 formulas.  See jf_set_tangent_seed. */
typedef enum { JF_F64 = 0, JF_F32 = 1, JF_F64_TANGENT = 2 } jf_dtype;
/* JF_BC_EXCHANGE: the face adjoins another block of a block-decomposed domain (equal
 * blocks, one per device, halo exchange with exactly one neighbour per face).  jf_fill_halo leaves its
 * halo layers alone; the caller fills them from the neighbour with jf_pull_face or jf_pack_face /
 * jf_unpack_face, axis by axis (see "Block decomposition" below). */
typedef enum {
  JF_BC_PERIODIC = 0, JF_BC_ZEROGRAD = 1, JF_BC_DIRICHLET = 2,
  JF_BC_WALL_ISOTHERMAL = 3, JF_BC_WALL_ADIABATIC = 4, JF_BC_EXCHANGE = 5
} jf_bc_type;

/* Grid: face coordinates per axis (host pointers, copied by jf_create), strictly increasing.
 * Stretched meshes (:31, :104) are given through these arrays; Delta x_{i,j,k} of Eq. 6 is
 * xf[i+1]-xf[i].  Each n >= 4, and (nx+6)(ny+6)(nz+6) < 2^32 (cells of one variable are addressed with a
 * 32-bit offset; a 1600^3 box is 33 GB per variable, beyond one GPU anyway); otherwise JF_EINVAL. */
typedef struct {
  int nx, ny, nz;
  const double *xf, *yf, *zf; /* nx+1, ny+1, nz+1 entries */
} jf_grid;

/* Viscosity law (:108): sutherland != 0: mu = mu_ref (T/T_ref)^1.5 (T_ref+S)/(T+S);
 * sutherland == 0: mu = mu_ref.  mu_ref == 0 means inviscid (dissipative flux skipped). */
typedef struct { int sutherland; double mu_ref, T_ref, S; } jf_mu_law;

/* Disturbance ("porous") segment on a wall face, Eq. 8 (:112): wall-normal wall velocity
 * v_w(t1) = A sin(2 pi kappa t1) added where t1_lo <= t1 <= t1_hi, t1 = the ghost cell's own
 * centre coordinate along the first tangential axis (x for y and z faces, y for x faces);
 * positive = along the + axis.  Elsewhere the plain wall. */
typedef struct { int enabled; double A, kappa, t1_lo, t1_hi; } jf_disturbance;

typedef struct {
  jf_bc_type type;
  double T_wall;           /* isothermal walls                                            */
  double u_wall[3];        /* wall velocity vector (u,v,w); 0 for a wall at rest          */
  const double *dirichlet; /* JF_BC_DIRICHLET: host array prim[5][n_t2][n_t1] of
                              (rho,u,v,w,p) over the interior tangential sizes (x faces:
                              t1=y,t2=z; y faces: t1=x,t2=z; z faces: t1=x,t2=y); copied     */
  jf_disturbance dist;     /* walls only */
  double nb_width[3];      /* JF_BC_EXCHANGE: widths of the neighbouring block's three cells next to
                              this face, nearest first (> 0): the halo cells then carry the geometry
                              they have on the undivided grid (stretched axes included)              */
  int nb_has_face;         /* JF_BC_EXCHANGE across an interior cut (not a periodic wrap): nb_face holds  */
  double nb_face[3];       /* the coordinates of the neighbour's three faces beyond this one, nearest
                              first; widths and centres of the halo cells are then formed from them as
                              for interior cells (xf[i+1]-xf[i], (xf[i]+xf[i+1])/2: the undivided grid's
                              values bit for bit) and nb_width is ignored.  Across a periodic wrap
                              (nb_has_face = 0) the undivided grid itself copies widths and accumulates
                              centres outward, which is what nb_width reproduces                      */
} jf_bc_face;
typedef struct { jf_bc_face face[6]; } jf_bc; /* x-, x+, y-, y+, z-, z+; periodic must pair */

/* Bytes of device workspace jf_create needs for this grid and dtype (0 on invalid input). */
size_t jf_workspace_bytes(const jf_grid *grid, jf_dtype dtype);

/* Create a solver.  Validates: n >= 4, monotone faces, gamma > 1, R_gas > 0, Pr > 0,
 * mu_ref >= 0, periodic faces paired, Dirichlet pointer non-null, T_wall > 0 on isothermal
 * walls (else JF_EINVAL, *out = NULL); workspace_dev 256-byte aligned (JF_EALIGN) and at least
 * jf_workspace_bytes() (JF_EWORKSPACE).  body_accel = constant acceleration g of the source
 * term S = [0, rho g, rho u.g] (Eq. 1 :39-42), may be NULL (= 0).  Copies the metric and BC
 * tables to the workspace (synchronous small copies).  The workspace must outlive the solver. */
jf_status jf_create(jf_solver **out, const jf_grid *grid, jf_dtype dtype, double gamma,
                    double R_gas, double Pr, const jf_mu_law *mu, const jf_bc *bc,
                    const double body_accel[3], void *workspace_dev, size_t workspace_bytes,
                    void *cuda_stream);
jf_status jf_destroy(jf_solver *s);

/* 5*(nz+6)*(ny+6)*(nx+6) */
size_t jf_state_elems(const jf_solver *s);

/* Halo / boundary fill (:80, :100-104, Eq. 8), in place, asynchronous.  Order x, y, z; the y
 * pass runs over all padded i and the z pass over all padded (i,j), which defines every edge
 * and corner cell.  Without a JF_BC_EXCHANGE face the three passes are ONE launch that composes them
 * per ghost cell (each pass maps one source cell to one ghost cell); the result is bitwise that of
 * jf_fill_halo_axis(0), (1), (2). */
jf_status jf_fill_halo(jf_solver *s, void *U_dev);

/* R = R_NSE(U) of Eq. 6 on interior cells (halo cells of R are left untouched).  The halos of
 * U must already be filled.  U and R must not alias.  Asynchronous. */
jf_status jf_rhs(jf_solver *s, const void *U_dev, void *R_dev);

/* One SSP-RK3 step in place: 3 x (halo fill, R_NSE, stage update)
 *   U1 = U + dt L(U);  U2 = 3/4 U + 1/4 (U1 + dt L(U1));  U <- 1/3 U + 2/3 (U2 + dt L(U2)).
 * On return the interior of U is U^{n+1}; its halo cells hold the fill of U^n.  Asynchronous. */
jf_status jf_rk3_step(jf_solver *s, void *U_dev, double dt);

/* CFL time step over interior cells (not in the paper; reading O9):
 *   dt = cfl * min( min_d Delta_d/(|u_d|+c), 3/14 Dmin^2 rho/mu, 1/10 Dmin^2 rho Pr/mu ).
 * Writes *dt_host and synchronises the stream.  JF_ENOTFINITE (and *dt_host = NaN) if any
 * interior cell is non-finite or has rho <= 0 or p <= 0. */
jf_status jf_cfl_dt(jf_solver *s, const void *U_dev, double cfl, double *dt_host);

/* Order of the central stencils of the dissipative flux (a5): 4 (default; north_star) or 6 — the "6th-order central"
 * dissipative fluxes the paper's DNS used.  The coefficients are fixed by
 * polynomial exactness on the symmetric stencils: D^c_6 = (-1,9,-45,0,45,-9,1)/60, D^f_6 = (75/64, -25/384, 3/640)
 * on the three cell pairs about the face, I^f_6 = (150,-25,3)/256; difference form, transverse derivatives = I^f_6
 * of D^c_6, index-space metrics rebuilt with the same stencils.  A face then reads cells -3..2 about it: the same
 * three halo layers as WENO5 (N_h of PAPER.md:80 stays 3).  Synchronises; rewrites the metric tables.  JF_EINVAL for
 * other orders and for JF_F64_TANGENT with order 6.  (The paper's TENO6-A reconstruction is NOT provided: its
 * constants are not in PAPER.md.) */
jf_status jf_set_visc_order(jf_solver *s, int order);

/* Device-resident time step: the same reduction, finished on the device (the last block forms dt), with NO host
 * synchronisation:   dt = min(jf_cfl_dt's value, t_end - t)   (t_end = NaN: no clipping),
 * stored in the solver's workspace together with the running time t <- t + dt (t starts at 0; jf_dev_time sets it).
 * jf_rk3_step_dev then advances U by that dt (its z + RK kernels read it from device memory), so a CFL-driven loop
 *     for (...) { jf_cfl_dt_dev(s, U, cfl, t_end); jf_rk3_step_dev(s, U); }
 * queues steps without ever waiting for the GPU; the host reads dt and t when it wants them (jf_dev_time), e.g.
 * one step late.  An inadmissible state makes dt NaN (it then spreads through U) and jf_dev_time returns
 * JF_ENOTFINITE from then on.  Asynchronous. */
jf_status jf_cfl_dt_dev(jf_solver *s, const void *U_dev, double cfl, double t_end);
jf_status jf_rk3_step_dev(jf_solver *s, void *U_dev);
/* set == 0: synchronise, then *dt_host = last device-side dt, *t_host = device-side time (either may be NULL).
 * set != 0: device-side time <- *t_host, dt <- 0, status cleared. */
jf_status jf_dev_time(jf_solver *s, int set, double *dt_host, double *t_host);

/* Launch mechanics of jf_rk3_step / jf_rk3_step_dev: the 15 launches of a step are captured once per state-array
 * address into a CUDA graph owned by the solver (on a private stream) and replayed into the caller's stream; their
 * z + RK kernels read dt from the device scalar, which jf_rk3_step sets with a one-thread kernel.  Environment
 * JF_GRAPH=0 at jf_create time turns this off (plain launches; also used while jf_diag_timing is on).
 *
 * Environment variables read once, at jf_create (tuning / A-B measurements; none changes a result beyond round-off):
 *   JF_GRAPH=0      plain launches instead of the CUDA-graph replay
 *   JF_GRAD_TMA=0|1 centre-gradient pass with plain loads | TMA-staged (cp.async.bulk.tensor + mbarrier ring; fp64, even nx
 *                   only).  Default: TMA for fields of at most 40 M padded cells per variable, where it is 6-8 % faster;
 *                   plain loads above (at 448^3 and more TMA is 15-22 % slower; profiles/r2_tma_sass.md)
 *   JF_F32X2=1      fp32 solvers: y / z sweeps with two columns per thread on packed FP32x2 arithmetic (FFMA2): 2-4 % faster on
 *                   the periodic boxes, slower on the channel, hence not the default (profiles/r2_experiments.md)
 *   JF_YZ_PC=1      producer / consumer form of the y / z sweeps (fp64, viscous, fourth-order flux): 20 % slower, kept as a
 *                   measured variant (profiles/r2_experiments.md) */

/* ---- Block decomposition ------------------------------------------
 * One solver per block; faces between blocks are JF_BC_EXCHANGE.  One RK stage of a decomposed step is
 *   for axis in x, y, z:   every block: jf_fill_halo_axis(axis)            (its physical faces)
 *                          every block: for its exchange faces of that axis: jf_pull_face from the
 *                                       neighbour's stage input (or pack -> transport -> unpack)
 *   every block: jf_rk3_stage_advance(stage)
 * with the stage inputs given by jf_rk3_stage_input.  The axis order and the tangential extents of each
 * pass (x: interior (j,k); y: all padded i, interior k; z: all padded (i,j)) are those of jf_fill_halo, so
 * edges and corners come out exactly as on the undivided grid: a decomposed run reproduces the undivided
 * one cell for cell.  All calls are asynchronous on the solver's stream; ordering BETWEEN blocks (the
 * neighbour must have finished the previous axis pass, and must not overwrite the array before it was
 * read) is the caller's: same stream, events, or a barrier between ranks. */

/* Boundary pass of one axis (0 x, 1 y, 2 z) only; jf_fill_halo = axes 0, 1, 2 in this order. */
jf_status jf_fill_halo_axis(jf_solver *s, void *U_dev, int axis);

/* Elements (of the solver dtype; pairs for tangent solvers) of one packed face buffer:
 * 5 * 3 * (tangential cells of that axis' pass); 0 on bad arguments. */
size_t jf_face_elems(const jf_solver *s, int face);

/* Pack the three interior layers next to `face` (0..5 = x-, x+, y-, y+, z-, z+) into buf_dev
 * [5][3][n_t2][n_t1] - what the neighbour across that face needs for ITS opposite face; unpack writes
 * such a buffer (packed by the neighbour across `face` for its opposite face) into the halo layers of
 * `face`.  Layer m = 1..3 counts outward from the face on both sides. */
jf_status jf_pack_face(jf_solver *s, const void *U_dev, int face, void *buf_dev);
jf_status jf_unpack_face(jf_solver *s, void *U_dev, int face, const void *buf_dev);

/* Fill the halo layers of `face` directly from the neighbouring block's state array U_peer_dev (same
 * layout and dtype; a pointer on this device or a peer-mapped one: the loads then cross NVLink inside
 * the kernel, no staging buffer).  n_peer = the peer block's interior sizes: equal to this block's in the
 * two tangential axes (else JF_EINVAL). */
jf_status jf_pull_face(jf_solver *s, void *U_dev, int face, const void *U_peer_dev, const int n_peer[3]);

/* The array whose halos stage 1, 2, 3 of jf_rk3_step reads: U_dev itself (stage 1) or one of the
 * solver's two stage buffers inside the workspace; NULL on bad arguments.  jf_rk3_stage_advance runs
 * R_NSE and the SSP-RK3 update of that stage, assuming the halos of its input are filled:
 * jf_rk3_step(U, dt) == for stage 1..3: jf_fill_halo(jf_rk3_stage_input(U, stage)); advance(U, stage, dt). */
void *jf_rk3_stage_input(jf_solver *s, void *U_dev, int stage);
jf_status jf_rk3_stage_advance(jf_solver *s, void *U_dev, int stage, double dt);

/* ---- Plane statistics (Fig. 1: profiles averaged over the two homogeneous directions) --
 * For every interior plane p of `axis` (0 x, 1 y, 2 z) the area-weighted sums over the plane's interior cells,
 *   sums_dev[q * n_axis + p] = sum_{t1,t2} phi_q dA,   dA = Delta_t1 Delta_t2,
 * of the JF_NSTATS quantities  phi = 1, rho, T, u, v, w, uu, vv, ww, uv, uw, vw, rho^2, T^2  (T = p/(rho R)).
 * The caller forms means S_q/S_0 and Reynolds stresses <u_i u_j> - <u_i><u_j>.  sums_dev: DEVICE array of
 * JF_NSTATS * n_axis doubles (double for every solver dtype; tangent solvers: value parts).  Deterministic
 * (fixed reduction order for a given grid).  Asynchronous on the solver's stream. */
#define JF_NSTATS 14
jf_status jf_plane_sums(jf_solver *s, const void *U_dev, int axis, double *sums_dev);

/* jf_plane_sums for callers that must not allocate and have no workspace to spare for it (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): the same two kernels and the same summation
 * order (the same bits as jf_plane_sums), but the per-block partial sums go to a STATIC device array inside the
 * library (14 x 1024 x 16 doubles = 1.75 MiB per GPU that loads the library, held until the process exits) instead of
 * the solver's workspace.  The call allocates nothing on host or device (no cudaMalloc / cudaFree, no allocating
 * library routine; the array's device address is looked up once per device with cudaGetSymbolAddress and cached).
 * Limit: at most jf_plane_sums_static_max_planes() = 1024 interior planes along `axis`; larger grids get JF_EINVAL
 * with the reason in jf_last_error (use jf_plane_sums).  sums_dev as for jf_plane_sums (DEVICE, JF_NSTATS * n_axis
 * doubles, caller-owned).  The array is shared by every solver and every call on that GPU and keeps the last call's
 * contents; nothing in it needs clearing (each call writes every partial it reads), but two calls that OVERLAP on the
 * GPU (different streams, no ordering between them) race on it: order them on one stream or with events.
 * Asynchronous on the solver's stream. */
jf_status jf_plane_sums_static(jf_solver *s, const void *U_dev, int axis, double *sums_dev);
int jf_plane_sums_static_max_planes(void);

/* Tangent solvers (JF_F64_TANGENT) only; JF_EINVAL otherwise.  The paper introduces the Disturbance
 * Wall so that its parameters can be differentiated through the solver.
 * Sets the direction (dA, dkappa) in the parameter space of Eq. 8 (:112), applied to every disturbance
 * segment: jf_fill_halo then seeds the wall-velocity tangent
 *   d v_w = dA sin(2 pi kappa t1) + dkappa A 2 pi t1 cos(2 pi kappa t1),
 * and jf_fill_halo / jf_rhs / jf_rk3_step propagate (value, tangent) pairs, so that after a step the
 * tangent part of U is the directional derivative of the value part with respect to (A, kappa) along
 * (dA, dkappa) (plus the propagated input tangent), at FIXED dt: jf_cfl_dt uses the value parts only
 * and the tangent of dt is not propagated.  Non-smooth selections (min / max / sign in HLLC, the
 * wall-temperature floor) take the derivative of the selected branch.  Default seed (0, 0). */
jf_status jf_set_tangent_seed(jf_solver *s, double dA, double dkappa);

/* Last error text of this solver ("" if none); never NULL. */
const char *jf_last_error(const jf_solver *s);

/* Number of kernel launches issued by this solver since jf_create (for bench accounting). */
unsigned long long jf_launch_count(const jf_solver *s);

/* Diagnostics (not on the hot path): register-resident FMA loop on the plain FP64 (dtype
 * JF_F64) or FP32 ALUs; writes the achieved FLOP/s (2 per FMA) to *flops_host.  Used by
 * bench.py as the measured ALU peak of the roofline.  Synchronises the device. */
jf_status jf_diag_alu_peak(jf_dtype dtype, int iters, double *flops_host, double *ms_host);

/* Per-kernel device timing (diagnostic).  jf_diag_timing(s, 1) makes every launch of this solver
 * record a CUDA-event pair on its stream; jf_diag_kernel_times synchronises the stream, writes the
 * accumulated milliseconds and launch counts per kernel class since the previous call (6 classes:
 * 0 halo (one fused launch per fill; three per-axis passes for decomposed blocks), 1 gradient, 2 x sweep, 3 y sweep, 4 z sweep + RK3 stage, 5 CFL)
 * and resets them.  jf_diag_kernel_name(k) names class k ("" if out of range). */
jf_status jf_diag_timing(jf_solver *s, int enable);
jf_status jf_diag_kernel_times(jf_solver *s, double ms[6], unsigned long long launches[6]);
const char *jf_diag_kernel_name(int k);

/* Unit-level diagnostic of the per-face arithmetic the sweep kernels use (not on the hot path):
 * total face flux F = F^c - F^d (Eq. 6) along dir for n_faces independent faces.  HOST arrays:
 * W[n][6][6] primitives (rho,u,v,w,p,T) of the six cells i-2..i+3 around each face, Gt[n][4][4]
 * transverse centre derivatives at cells i-1..i+2 (d_t1 u_n, d_t1 u_t1, d_t2 u_n, d_t2 u_t2;
 * may be NULL = 0), Xf[n] face metric X_xi^f (NULL = 1), F[n][5] output.  Dissipative part only
 * if mu->mu_ref > 0.  Allocates its own scratch; synchronises. */
jf_status jf_diag_face_flux(jf_dtype dtype, int dir, double gamma, double R_gas, double Pr,
                            const jf_mu_law *mu, int n_faces, const double *W, const double *Gt,
                            const double *Xf, double *F);

/* Geometry tables the kernels read, copied back from the workspace (diagnostic; synchronises): for axis
 * a in 0..2, HOST arrays of n_a + 6 doubles (padded index p = i + 3; any pointer may be NULL):
 *   inv_delta[p] = 1/Delta_p,  centre[p] = cell centre,  i12Xc[p] = 1/(12 X_xi^c) (interior p only, else 1/12),
 *   i24Xf[p] = 1/(24 X_xi^f) of the face on the high side of cell p (p = 2 .. n+2, else 1/24)
 * (reading O2; halo geometry: periodic copy, mirror, or the neighbour widths of a JF_BC_EXCHANGE
 * face).  Values are those of the solver dtype converted to double.  tests/test_gpu_units.py compares them with
 * the oracle's own tables. */
jf_status jf_diag_metrics(jf_solver *s, int axis, double *inv_delta, double *centre, double *i12Xc, double *i24Xf);

/* Library version / build info string (static storage). */
const char *jf_version(void);

#ifdef __cplusplus
}
#endif
#endif
