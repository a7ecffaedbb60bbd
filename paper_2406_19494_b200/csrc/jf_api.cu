// jf_api.cu — C ABI of libjf (include/jf.h): argument validation, metric / BC tables, workspace
// carving, kernel launches.  Host logic only; every step of the path runs in jf_kernels.cuh.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>
#include <cuda_runtime.h>
#include "../../include/jf.h"
#include "jf_kernels.cuh"
#include "jf_tma.cuh"
#include "jf_pc.cuh"
#include "jf_f32x2.cuh"
#include <type_traits>
#include <cstdlib>
#include <unordered_map>

namespace {

using jf::NH;

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
constexpr int STATS_NB = 16;  // at most this many partial blocks per plane in jf_plane_sums

// Grid geometry (reading O2): widths, centres, halo geometry, index-space metrics.
struct Metrics {
  std::vector<double> dl[3], xc[3], Xc[3], Xf[3];
};

// nbw[f]: for a JF_BC_EXCHANGE face f, the widths of the neighbouring block's three cells next to the
// face (nearest first) - the halo cells then have the geometry they have on the undivided grid; else null.
// nbf[f]: for an exchange face across an interior cut, the neighbour's three face coordinates beyond the face.
void build_metrics(const int n[3], const double* const xf[3], const bool periodic[3], const double* const nbw[6],
                   const double* const nbf[6], int order, Metrics& M) {
  for (int a = 0; a < 3; ++a) {
    const int N = n[a], P = N + 2 * NH;
    std::vector<double>&d = M.dl[a], &x = M.xc[a];
    d.assign(P, 0.0); x.assign(P, 0.0); M.Xc[a].assign(P, 1.0); M.Xf[a].assign(P, 1.0);
    for (int i = 0; i < N; ++i) { d[i + NH] = xf[a][i + 1] - xf[a][i]; x[i + NH] = 0.5 * (xf[a][i] + xf[a][i + 1]); }
    for (int m = 1; m <= NH; ++m) {
      d[NH - m] = nbw[2 * a] ? nbw[2 * a][m - 1] : (periodic[a] ? d[NH + N - m] : d[NH + m - 1]);
      d[NH + N - 1 + m] = nbw[2 * a + 1] ? nbw[2 * a + 1][m - 1] : (periodic[a] ? d[NH + m - 1] : d[NH + N - m]);
    }
    double e = xf[a][0];
    for (int m = 1; m <= NH; ++m) { x[NH - m] = e - 0.5 * d[NH - m]; e -= d[NH - m]; }
    e = xf[a][N];
    for (int m = 1; m <= NH; ++m) { x[NH + N - 1 + m] = e + 0.5 * d[NH + N - 1 + m]; e += d[NH + N - 1 + m]; }
    if (nbf[2 * a]) {                      // interior cut on the low side: the undivided grid's own expressions
      double g0 = xf[a][0];
      for (int m = 1; m <= NH; ++m) { const double g1 = nbf[2 * a][m - 1]; d[NH - m] = g0 - g1; x[NH - m] = 0.5 * (g1 + g0); g0 = g1; }
    }
    if (nbf[2 * a + 1]) {
      double g0 = xf[a][N];
      for (int m = 1; m <= NH; ++m) { const double g1 = nbf[2 * a + 1][m - 1]; d[NH + N - 1 + m] = g1 - g0; x[NH + N - 1 + m] = 0.5 * (g0 + g1); g0 = g1; }
    }
    // index-space metrics: the derivative stencils of the dissipative flux (fourth or sixth order) applied to the centres
    if (order == 6) {
      for (int p = NH; p < NH + N; ++p)
        M.Xc[a][p] = (45.0 * (x[p + 1] - x[p - 1]) - 9.0 * (x[p + 2] - x[p - 2]) + (x[p + 3] - x[p - 3])) / 60.0;
      for (int p = NH - 1; p < NH + N; ++p)
        M.Xf[a][p] = (2250.0 * (x[p + 1] - x[p]) - 125.0 * (x[p + 2] - x[p - 1]) + 9.0 * (x[p + 3] - x[p - 2])) / 1920.0;
    } else {
      for (int p = NH; p < NH + N; ++p) M.Xc[a][p] = (x[p - 2] - 8.0 * x[p - 1] + 8.0 * x[p + 1] - x[p + 2]) / 12.0;
      for (int p = NH - 1; p < NH + N; ++p) M.Xf[a][p] = (x[p - 1] - 27.0 * x[p] + 27.0 * x[p + 1] - x[p + 2]) / 24.0;
    }
  }
}

struct Layout {  // byte offsets into the workspace
  size_t tab_T[3][4];   // inv_dl, dl, i12Xc, i24Xf per axis (dtype)
  size_t tab_xc[3];     // double
  size_t dirichlet[6];  // double
  size_t cfl;           // 8 x u64: three minima, flag, block counter, then (as doubles) dt, t, and a sticky status word
  size_t stats;         // NSTAT x max(n) x STATS_NB doubles (plane-sum partials)
  size_t R, A, B, G;    // fields (dtype)
  size_t total;
};

Layout make_layout(const int n[3], size_t esz) {
  Layout L;
  size_t off = 0;
  for (int a = 0; a < 3; ++a) {
    for (int t = 0; t < 4; ++t) { L.tab_T[a][t] = off; off = align_up(off + (size_t)(n[a] + 6) * esz); }
    L.tab_xc[a] = off; off = align_up(off + (size_t)(n[a] + 6) * sizeof(double));
  }
  for (int f = 0; f < 6; ++f) {
    int a = f / 2, t1 = (a == 0) ? 1 : 0, t2 = (a == 2) ? 1 : 2;
    L.dirichlet[f] = off; off = align_up(off + (size_t)5 * n[t1] * n[t2] * sizeof(double));
  }
  L.cfl = off; off = align_up(off + 8 * sizeof(unsigned long long));
  L.stats = off; off = align_up(off + (size_t)jf::NSTAT * std::max(n[0], std::max(n[1], n[2])) * STATS_NB * sizeof(double));
  size_t vol = (size_t)(n[0] + 6) * (n[1] + 6) * (n[2] + 6);
  L.R = off; off = align_up(off + 5 * vol * esz);
  L.A = off; off = align_up(off + 5 * vol * esz);
  L.B = off; off = align_up(off + 5 * vol * esz);
  L.G = off; off = align_up(off + 9 * vol * esz);
  L.total = off;
  return L;
}

bool grid_ok(const jf_grid* g) {
  if (!g || g->nx < 4 || g->ny < 4 || g->nz < 4 || !g->xf || !g->yf || !g->zf) return false;
  const double* xf[3] = {g->xf, g->yf, g->zf};
  const int n[3] = {g->nx, g->ny, g->nz};
  for (int a = 0; a < 3; ++a)
    for (int i = 0; i < n[a]; ++i)
      if (!(xf[a][i + 1] > xf[a][i])) return false;
  // the kernels address a cell inside one variable's array with a 32-bit offset
  if ((double)(g->nx + 6) * (double)(g->ny + 6) * (double)(g->nz + 6) >= 4294967296.0) return false;
  return true;
}

template <class T>
struct Impl {
  jf::Params<T> P;
  jf::FaceBC<T> bc[6];
  T *R, *A, *B, *G;
  unsigned long long* cfl_out;
  double* stats;
};

}  // namespace
namespace jf {
inline double value_of(double a) { return a; }
inline double value_of(float a) { return (double)a; }
inline double value_of(Dual a) { return a.v; }
}  // namespace jf
namespace {

bool dtype_ok(jf_dtype d) { return d == JF_F64 || d == JF_F32 || d == JF_F64_TANGENT; }
size_t elem_size(jf_dtype d) { return d == JF_F64 ? sizeof(double) : (d == JF_F32 ? sizeof(float) : sizeof(jf::Dual)); }

}  // namespace

// ---- scratch of the allocation-free entry point jf_plane_sums_static (include/jf.h) ----------------------------
// Partial sums of plane_sums_kernel: NSTAT quantities x planes x STATS_NB partial blocks, for at most
// JF_STATIC_MAX_PLANES planes: 14 x 1024 x 16 doubles = 1.75 MiB.  Lives in every GPU context that loads the library
// until the process exits.  In HOST code the name `jf_static_scratch` is a host-side stand-in, not a device address:
// host code takes the address once per device with cudaGetSymbolAddress (static_scratch_ptr below) and hands THAT to
// the kernels.  All calls on one device share the array and it keeps the last call's contents; nothing in it has to
// start at zero (every partial a call reads is written by that call first).
#define JF_STATIC_MAX_PLANES 1024
static __device__ __align__(256) double jf_static_scratch[(size_t)jf::NSTAT * JF_STATIC_MAX_PLANES * STATS_NB];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex static_scratch_mutex;
double* static_scratch_addr[STATIC_MAX_DEVICES] = {};

// Device address of jf_static_scratch on the CURRENT device; resolved once per device, then cached.
cudaError_t static_scratch_ptr(double** out) {
  int dev = -1;
  cudaError_t ce = cudaGetDevice(&dev);
  if (ce != cudaSuccess) return ce;
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(static_scratch_mutex);
  if (!static_scratch_addr[dev]) {
    double* ptr = nullptr;
    ce = cudaGetSymbolAddress((void**)&ptr, jf_static_scratch);
    if (ce != cudaSuccess) return ce;
    static_scratch_addr[dev] = ptr;
  }
  *out = static_scratch_addr[dev];
  return cudaSuccess;
}
}  // namespace

struct jf_solver {
  jf_dtype dtype;
  Impl<double> d;
  Impl<float> f;
  Impl<jf::Dual> t;              // JF_F64_TANGENT: (value, tangent) pairs
  cudaStream_t stream;
  int device;                    // the CUDA device current at jf_create: workspace, stream and every launch live there
  bool viscous;
  double Pr;
  std::string err;
  unsigned long long launches;
  int seg_len[3];
  // geometry inputs kept for jf_set_visc_order (the metric tables depend on the order of the derivative stencils)
  int visc_order = 4;
  int n[3];
  std::vector<double> xfh[3];
  jf_bc bc_host;
  char* ws = nullptr;
  // TMA-staged gradient pass (jf_tma.cuh): tensor maps per state-array base address (U, stage buffers A, B, ...)
  bool grad_tma = false;
  bool f32x2 = false;            // fp32 solver: marching sweeps with two columns per thread on packed FP32x2 arithmetic (jf_f32x2.cuh)
  int seg_len2[3] = {0, 0, 0};   // their segment lengths (half as many warps per layer)
  bool yz_pc = false;            // producer / consumer form of the marching sweeps (jf_pc.cuh; fp64, viscous, fourth order)
  std::unordered_map<const void*, CUtensorMap> maps;
  // CUDA graphs of one RK3 step (the 15 launches), one per state-array address, captured on first use on a private
  // stream and launched into the caller's stream.  The kernels of a graph read dt from the device scalar
  // (RKArgs::dt_dev), so the same graph serves every dt (jf_rk3_step sets it, jf_cfl_dt_dev computes it).
  bool use_graph = true;
  cudaStream_t cap_stream = nullptr;
  struct GraphEntry { const void* U; cudaGraphExec_t exec; unsigned kernels; };
  std::vector<GraphEntry> graphs;
  // optional per-kernel timing (jf_diag_timing): CUDA events around every launch
  bool timing = false;
  struct Ev { cudaEvent_t a, b; int cls; };
  std::vector<Ev> ev_used, ev_free;
};

enum { K_HALO = 0, K_GRAD = 1, K_SWEEP_X = 2, K_SWEEP_Y = 3, K_SWEEP_Z = 4, K_CFL = 5, K_COUNT = 6 };

namespace {

jf_status fail(jf_solver* s, jf_status st, const char* what, cudaError_t ce = cudaSuccess) {
  if (s) {
    s->err = what;
    if (ce != cudaSuccess) { s->err += ": "; s->err += cudaGetErrorString(ce); }
  }
  return st;
}

// RAII: records an event pair around one kernel launch when timing is on.
struct Timed {
  jf_solver* s; jf_solver::Ev e; bool on;
  Timed(jf_solver* s_, int cls) : s(s_), on(s_->timing) {
    if (!on) return;
    if (!s->ev_free.empty()) { e = s->ev_free.back(); s->ev_free.pop_back(); }
    else { cudaEventCreate(&e.a); cudaEventCreate(&e.b); }
    e.cls = cls;
    cudaEventRecord(e.a, s->stream);
  }
  ~Timed() {
    if (!on) return;
    cudaEventRecord(e.b, s->stream);
    s->ev_used.push_back(e);
  }
};

// Makes the solver's device current for the duration of one API call (a process driving several GPUs
// may have another device current) and restores the caller's device on return.
struct DeviceGuard {
  int prev = -1; bool sw = false;
  explicit DeviceGuard(const jf_solver* s) {
    if (s && cudaGetDevice(&prev) == cudaSuccess && prev != s->device) sw = cudaSetDevice(s->device) == cudaSuccess;
  }
  ~DeviceGuard() { if (sw) cudaSetDevice(prev); }
};

#define JF_CUDA(s, call)                                                  \
  do {                                                                    \
    cudaError_t ce_ = (call);                                             \
    if (ce_ != cudaSuccess) return fail((s), JF_ECUDA, #call, ce_);       \
  } while (0)

template <class T>
void fill_gas(jf::Gas<T>& G, double gamma, double R_gas, double Pr, const jf_mu_law* mu, const double* ga) {
  G.gamma = T(gamma); G.gm1 = T(gamma - 1.0); G.inv_gm1 = T(1.0 / (gamma - 1.0));
  G.Rgas = T(R_gas); G.inv_Rgas = T(1.0 / R_gas);
  G.mu_ref = T(mu->mu_ref); G.inv_T_ref = T(1.0 / mu->T_ref); G.S = T(mu->S); G.TrefS = T(mu->T_ref + mu->S);
  G.lam_fac = T(gamma * R_gas / (gamma - 1.0) / Pr); G.Pr = T(Pr);
  G.sutherland = mu->sutherland != 0; G.viscous = mu->mu_ref > 0.0;
  for (int a = 0; a < 3; ++a) G.g[a] = T(ga ? ga[a] : 0.0);
  G.has_g = ga && (ga[0] != 0.0 || ga[1] != 0.0 || ga[2] != 0.0);
}

template <class T>
jf_status diag_face_flux(int dir, double gamma, double R_gas, double Pr, const jf_mu_law* mu, int nf,
                         const double* W, const double* Gt, const double* Xf, double* F) {
  jf::Gas<T> gas;
  fill_gas<T>(gas, gamma, R_gas, Pr, mu, nullptr);
  std::vector<T> hW((size_t)nf * 36), hG((size_t)nf * 16), hX(nf), hF((size_t)nf * 5);
  for (size_t i = 0; i < hW.size(); ++i) hW[i] = T(W[i]);
  for (size_t i = 0; i < hG.size(); ++i) hG[i] = T(Gt ? Gt[i] : 0.0);
  for (int i = 0; i < nf; ++i) hX[i] = T(1.0 / (24.0 * (Xf ? Xf[i] : 1.0)));
  T *dW = nullptr, *dG = nullptr, *dX = nullptr, *dF = nullptr;
  bool ok = cudaMalloc(&dW, hW.size() * sizeof(T)) == cudaSuccess && cudaMalloc(&dG, hG.size() * sizeof(T)) == cudaSuccess &&
            cudaMalloc(&dX, hX.size() * sizeof(T)) == cudaSuccess && cudaMalloc(&dF, hF.size() * sizeof(T)) == cudaSuccess;
  if (ok) {
    cudaMemcpy(dW, hW.data(), hW.size() * sizeof(T), cudaMemcpyHostToDevice);
    cudaMemcpy(dG, hG.data(), hG.size() * sizeof(T), cudaMemcpyHostToDevice);
    cudaMemcpy(dX, hX.data(), hX.size() * sizeof(T), cudaMemcpyHostToDevice);
    const int blocks = (nf + 127) / 128;
    if (dir == 0) jf::face_flux_kernel<T, 0><<<blocks, 128>>>(gas, dW, dG, dX, dF, nf);
    else if (dir == 1) jf::face_flux_kernel<T, 1><<<blocks, 128>>>(gas, dW, dG, dX, dF, nf);
    else jf::face_flux_kernel<T, 2><<<blocks, 128>>>(gas, dW, dG, dX, dF, nf);
    ok = cudaMemcpy(hF.data(), dF, hF.size() * sizeof(T), cudaMemcpyDeviceToHost) == cudaSuccess;
  }
  cudaFree(dW); cudaFree(dG); cudaFree(dX); cudaFree(dF);
  if (!ok) return JF_ECUDA;
  for (size_t i = 0; i < hF.size(); ++i) F[i] = (double)hF[i];
  return JF_OK;
}

// Geometry tables of the solver's grid for the current order of the dissipative stencils -> workspace
// (1/Delta, Delta, 1/(12 X_xi^c) | 1/(60 X_xi^c), 1/(24 X_xi^f) | 1/(1920 X_xi^f), centres).  Synchronous copies.
template <class T>
jf_status upload_tables(jf_solver* s, Impl<T>& I) {
  const int* n = s->n;
  const double* xf[3] = {s->xfh[0].data(), s->xfh[1].data(), s->xfh[2].data()};
  const jf_bc* bc = &s->bc_host;
  char* ws = s->ws;
  bool per[3];
  for (int a = 0; a < 3; ++a) per[a] = bc->face[2 * a].type == JF_BC_PERIODIC;
  const double* nbw[6];
  const double* nbf[6];
  for (int f = 0; f < 6; ++f) {
    const bool ex = bc->face[f].type == JF_BC_EXCHANGE;
    nbf[f] = ex && bc->face[f].nb_has_face ? bc->face[f].nb_face : nullptr;
    nbw[f] = ex && !nbf[f] ? bc->face[f].nb_width : nullptr;
  }
  Metrics M;
  build_metrics(n, xf, per, nbw, nbf, s->visc_order, M);
  Layout L = make_layout(n, sizeof(T));
  jf::Params<T>& P = I.P;
  const double kc = s->visc_order == 6 ? 60.0 : 12.0, kf = s->visc_order == 6 ? 1920.0 : 24.0;
  for (int a = 0; a < 3; ++a) {
    const int Pn = n[a] + 6;
    std::vector<T> t[4];
    for (int k = 0; k < 4; ++k) t[k].resize(Pn);
    for (int p = 0; p < Pn; ++p) {
      t[0][p] = T(1.0 / M.dl[a][p]); t[1][p] = T(M.dl[a][p]);
      t[2][p] = T(1.0 / (kc * M.Xc[a][p])); t[3][p] = T(1.0 / (kf * M.Xf[a][p]));
    }
    for (int k = 0; k < 4; ++k)
      JF_CUDA(s, cudaMemcpy(ws + L.tab_T[a][k], t[k].data(), Pn * sizeof(T), cudaMemcpyHostToDevice));
    JF_CUDA(s, cudaMemcpy(ws + L.tab_xc[a], M.xc[a].data(), Pn * sizeof(double), cudaMemcpyHostToDevice));
    P.inv_dl[a] = (const T*)(ws + L.tab_T[a][0]); P.dl[a] = (const T*)(ws + L.tab_T[a][1]);
    P.i12Xc[a] = (const T*)(ws + L.tab_T[a][2]); P.i24Xf[a] = (const T*)(ws + L.tab_T[a][3]);
    P.xc[a] = (const double*)(ws + L.tab_xc[a]);
  }
  return JF_OK;
}

template <class T>
jf_status setup(jf_solver* s, Impl<T>& I, const jf_grid* g, double gamma, double R_gas, double Pr,
                const jf_mu_law* mu, const jf_bc* bc, const double* ga, char* ws) {
  const int n[3] = {g->nx, g->ny, g->nz};
  const double* xf[3] = {g->xf, g->yf, g->zf};
  for (int a = 0; a < 3; ++a) { s->n[a] = n[a]; s->xfh[a].assign(xf[a], xf[a] + n[a] + 1); }
  s->bc_host = *bc;
  s->ws = ws;
  Layout L = make_layout(n, sizeof(T));
  jf::Params<T>& P = I.P;
  for (int a = 0; a < 3; ++a) { P.n[a] = n[a]; P.P[a] = n[a] + 6; }
  P.sy = P.P[0]; P.sz = (long long)P.P[0] * P.P[1]; P.vol = P.sz * P.P[2];
  fill_gas<T>(P.gas, gamma, R_gas, Pr, mu, ga);
  {
    const jf_status st = upload_tables<T>(s, I);
    if (st != JF_OK) return st;
  }
  for (int f = 0; f < 6; ++f) {
    const jf_bc_face& b = bc->face[f];
    jf::FaceBC<T>& o = I.bc[f];
    o.type = (int)b.type; o.T_wall = T(b.T_wall);
    for (int d = 0; d < 3; ++d) o.uw[d] = T(b.u_wall[d]);
    const bool wall = b.type == JF_BC_WALL_ISOTHERMAL || b.type == JF_BC_WALL_ADIABATIC;
    o.dist_on = wall && b.dist.enabled;
    o.A = b.dist.A; o.kappa = b.dist.kappa; o.lo = b.dist.t1_lo; o.hi = b.dist.t1_hi;
    o.dA = 0.0; o.dkappa = 0.0;
    o.dirichlet = nullptr;
    if (b.type == JF_BC_DIRICHLET) {
      int a = f / 2, t1 = (a == 0) ? 1 : 0, t2 = (a == 2) ? 1 : 2;
      JF_CUDA(s, cudaMemcpy(ws + L.dirichlet[f], b.dirichlet, (size_t)5 * n[t1] * n[t2] * sizeof(double),
                            cudaMemcpyHostToDevice));
      o.dirichlet = (const double*)(ws + L.dirichlet[f]);
    }
  }
  I.R = (T*)(ws + L.R); I.A = (T*)(ws + L.A); I.B = (T*)(ws + L.B); I.G = (T*)(ws + L.G);
  I.cfl_out = (unsigned long long*)(ws + L.cfl);
  {
    // armed once; every finalising reduction re-arms it (jf_cfl_dt_dev), jf_cfl_dt re-arms by memset
    unsigned long long h[8] = {~0ULL, ~0ULL, ~0ULL, 0, 0, 0, 0, 0};
    JF_CUDA(s, cudaMemcpy(I.cfl_out, h, sizeof(h), cudaMemcpyHostToDevice));
  }
  I.stats = (double*)(ws + L.stats);
  return JF_OK;
}

// Segment length of the marching (y / z) sweeps.  Each segment costs two extra WENO steps, one extra
// face and a window prologue, so segments should be long; but the grid must still fill the 148 SMs
// (12 resident warps each) for several waves.  Small grids: equal segments for about 2.5 waves of warps
// (measured best on the 192x128x128 channel, 128^3 and 192^3: L = 22, 15, 48; fewer, longer segments
// leave SMs idle in the last wave, shorter ones pay the per-segment extras), never below 8 cells.  When
// that length reaches 64 the extras are below 4 % and the old rule is kept: largest power-of-two length
// (<= N) that leaves at least JF_SEG_WAVES waves (256^3: 64; 37...86 measured within 1 %).
#ifndef JF_GM_WAVES
#define JF_GM_WAVES 8
#endif
#ifndef JF_SEG_WAVES
#define JF_SEG_WAVES 4
#endif
int pick_segment(long long warps_per_layer, int N) {
#ifdef JF_SEG_FORCE
  return JF_SEG_FORCE < N ? JF_SEG_FORCE : N;
#endif
  const long long cap = 148 * 12;
  {
    const long long nseg = (5 * cap / 2 + warps_per_layer - 1) / warps_per_layer;
    const int Ls = (int)std::max<long long>((N + nseg - 1) / nseg, 8);
    if (Ls < 64) return Ls < N ? Ls : N;
  }
  const long long want = (long long)JF_SEG_WAVES * cap;
  int L = 8;
  while (L < N) L *= 2;                      // one segment
  while (L > 8 && warps_per_layer * ((N + L - 1) / L) < want) L /= 2;
  return L < N ? L : N;
}

// boundary pass of one axis (both sides, 3 layers); JF_BC_EXCHANGE faces are left to the face transfer
template <class T>
jf_status launch_halo_axis(jf_solver* s, Impl<T>& I, T* U, int axis) {
  const jf::Params<T>& P = I.P;
  Timed t(s, K_HALO);
  if (axis == 0) {
    long long tot = (long long)P.n[1] * P.n[2] * 6;
    jf::halo_kernel<T, 0><<<(unsigned)((tot + 255) / 256), 256, 0, s->stream>>>(P, I.bc[0], I.bc[1], U);
  } else if (axis == 1) {
    long long tot = (long long)P.P[0] * P.n[2] * 6;
    jf::halo_kernel<T, 1><<<(unsigned)((tot + 255) / 256), 256, 0, s->stream>>>(P, I.bc[2], I.bc[3], U);
  } else {
    long long tot = (long long)P.P[0] * P.P[1] * 6;
    jf::halo_kernel<T, 2><<<(unsigned)((tot + 255) / 256), 256, 0, s->stream>>>(P, I.bc[4], I.bc[5], U);
  }
  s->launches += 1;
  JF_CUDA(s, cudaPeekAtLastError());
  return JF_OK;
}

// all three passes: one fused launch (halo_all_kernel), or the per-axis passes when a face is JF_BC_EXCHANGE
// (those are driven pass by pass with the face transfers in between)
template <class T>
jf_status launch_halo(jf_solver* s, Impl<T>& I, T* U) {
  jf_status st;
  bool exchange = false;
  for (int f = 0; f < 6; ++f) exchange = exchange || I.bc[f].type == 5;
#ifdef JF_HALO_PER_AXIS
  exchange = true;
#endif
  if (!exchange) {
    const jf::Params<T>& P = I.P;
    const long long tot = 6LL * ((long long)P.n[1] * P.n[2] + (long long)P.P[0] * P.n[2] + (long long)P.P[0] * P.P[1]);
    jf::HaloFaces<T> B;
    for (int f = 0; f < 6; ++f) B.f[f] = I.bc[f];
    Timed t(s, K_HALO);
    jf::halo_all_kernel<T><<<(unsigned)((tot + 255) / 256), 256, 0, s->stream>>>(P, B, U);
    s->launches += 1;
    JF_CUDA(s, cudaPeekAtLastError());
    return JF_OK;
  }
  for (int a = 0; a < 3; ++a)
    if ((st = launch_halo_axis<T>(s, I, U, a))) return st;
  return JF_OK;
}

// tangential cell counts of the boundary pass of `axis` (reading O3): x: interior (j,k); y: all padded i,
// interior k; z: all padded (i,j)
template <class T>
long long face_cells(const jf::Params<T>& P, int axis) {
  const long long n1 = axis == 0 ? P.n[1] : P.P[0], n2 = axis == 2 ? P.P[1] : P.n[2];
  return n1 * n2;
}

// MODE 0 pack / 1 unpack / 2 pull of one face (jf_kernels.cuh: face_xfer_kernel)
template <class T, int MODE>
jf_status launch_xfer(jf_solver* s, Impl<T>& I, int face, T* U, T* buf, const T* peer, const int* np) {
  const jf::Params<T>& P = I.P;
  const int axis = face / 2, side = face % 2;
  const long long tot = face_cells<T>(P, axis) * 3;
  long long psy = 0, psz = 0, pvol = 0;
  int Np = 0;
  if (MODE == 2) {
    psy = np[0] + 6; psz = psy * (np[1] + 6); pvol = psz * (np[2] + 6); Np = np[axis];
  }
  const unsigned blocks = (unsigned)((tot + 255) / 256);
  Timed t(s, K_HALO);
  if (axis == 0) jf::face_xfer_kernel<T, 0, MODE><<<blocks, 256, 0, s->stream>>>(P, side, U, buf, peer, Np, psy, psz, pvol);
  else if (axis == 1) jf::face_xfer_kernel<T, 1, MODE><<<blocks, 256, 0, s->stream>>>(P, side, U, buf, peer, Np, psy, psz, pvol);
  else jf::face_xfer_kernel<T, 2, MODE><<<blocks, 256, 0, s->stream>>>(P, side, U, buf, peer, Np, psy, psz, pvol);
  s->launches += 1;
  JF_CUDA(s, cudaPeekAtLastError());
  return JF_OK;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time dependency on libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
      f = nullptr;
    return (EncodeTiledFn)f;
  }();
  return fn;
}

// Tensor map of one state array U[5][Pz][Py][Px] (x fastest) for boxes {GM_SX, GM_SY, 1, 4}: the (x,y) tile of one
// plane with its 2-cell rim, variables rho .. rho w.  Out-of-range box cells are zero-filled.  Cached per base address.
template <class T>
const CUtensorMap* grad_map(jf_solver* s, const jf::Params<T>& P, const T* U) {
  auto it = s->maps.find((const void*)U);
  if (it != s->maps.end()) return &it->second;
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return nullptr;
  CUtensorMap m;
  const cuuint64_t dims[4] = {(cuuint64_t)P.P[0], (cuuint64_t)P.P[1], (cuuint64_t)P.P[2], 5};
  const cuuint64_t strides[3] = {(cuuint64_t)P.sy * sizeof(T), (cuuint64_t)P.sz * sizeof(T), (cuuint64_t)P.vol * sizeof(T)};
  const cuuint32_t box[4] = {(cuuint32_t)jf::GM_SX, (cuuint32_t)jf::GM_SY, 1, 4};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const CUtensorMapDataType dt = sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
  if (enc(&m, dt, 4, (void*)U, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
          CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return nullptr;
  if (s->maps.size() > 64) s->maps.clear();
  return &(s->maps[(const void*)U] = m);
}

template <class T>
bool launch_grad_tma(jf_solver* s, Impl<T>& I, const T* U, dim3 grid, int Lz) {
  const CUtensorMap* m = grad_map<T>(s, I.P, U);
  if (!m) return false;
  jf::gradient_tma_kernel<T><<<grid, dim3(jf::GM_TX, jf::GM_TY), sizeof(jf::GradTmaSmem<T>), s->stream>>>(I.P, *m, I.G, Lz);
  return true;
}
template <>
bool launch_grad_tma<jf::Dual>(jf_solver*, Impl<jf::Dual>&, const jf::Dual*, dim3, int) { return false; }
template <>
bool launch_grad_tma<float>(jf_solver*, Impl<float>&, const float*, dim3, int) { return false; }

// R_NSE of Eq. 6.  rk == nullptr: R <- R_NSE(U).  Otherwise the z sweep applies the RK stage.
template <class T, bool VISC, int ORD = 4>
jf_status launch_rhs_t(jf_solver* s, Impl<T>& I, const T* U, T* R, const jf::RKArgs<T>* rk) {
  const jf::Params<T>& P = I.P;
  const T* G = VISC ? I.G : nullptr;
  if (VISC) {
    Timed t(s, K_GRAD);
    // plane march: z segments long enough to amortise the 4-plane prologue, short enough for JF_GM_WAVES waves
    const int tiles = ((P.P[0] + jf::GM_TX - 1) / jf::GM_TX) * ((P.P[1] + jf::GM_TY - 1) / jf::GM_TY);
    int nseg = (JF_GM_WAVES * 148 * 4 + tiles - 1) / tiles;
    if (nseg > P.P[2] / 8) nseg = P.P[2] / 8;
    if (nseg < 1) nseg = 1;
    const int Lz = (P.P[2] + nseg - 1) / nseg;
    dim3 grid((P.P[0] + jf::GM_TX - 1) / jf::GM_TX, (P.P[1] + jf::GM_TY - 1) / jf::GM_TY, (P.P[2] + Lz - 1) / Lz);
    if constexpr (ORD == 6) {
      jf::gradient6_kernel<T><<<grid, dim3(jf::GM_TX, jf::GM_TY), 0, s->stream>>>(P, U, I.G, Lz);
    } else {
      if (!(s->grad_tma && launch_grad_tma<T>(s, I, U, grid, Lz)))
        jf::gradient_kernel<T><<<grid, dim3(jf::GM_TX, jf::GM_TY), 0, s->stream>>>(P, U, I.G, Lz);
    }
    s->launches += 1;
  }
  {
    Timed t(s, K_SWEEP_X);
    const int groups = (P.n[1] * P.n[2] + jf::XS_LINES - 1) / jf::XS_LINES;   // one warp per group of lines
    const size_t sh = (size_t)jf::XS_WARPS * (jf::XS<VISC>::NV * jf::XS_RING + jf::XS_CARRY) * sizeof(T);
    jf::sweep_x_kernel<T, VISC, ORD><<<(groups + jf::XS_WARPS - 1) / jf::XS_WARPS, jf::XS_WARPS * 32, sh, s->stream>>>(P, U, G, R);
  }
  jf::RKArgs<T> none{nullptr, nullptr, T(0), T(0), T(0), nullptr};
  if constexpr (std::is_same<T, double>::value && VISC && ORD == 4) {
    if (s->yz_pc) {
      const size_t shp = jf::pc_smem_bytes();
      {
        Timed t(s, K_SWEEP_Y);
        const int L = s->seg_len[1];
        dim3 grid((P.n[0] + 31) / 32, (P.n[2] + 3) / 4, (P.n[1] + L - 1) / L);
        jf::sweep_yz_pc_kernel<1, 0><<<grid, 256, shp, s->stream>>>(P, U, G, R, none, L);
      }
      {
        Timed t(s, K_SWEEP_Z);
        const int L = s->seg_len[2];
        dim3 grid((P.n[0] + 31) / 32, (P.n[1] + 3) / 4, (P.n[2] + L - 1) / L);
        if (rk) jf::sweep_yz_pc_kernel<2, 2><<<grid, 256, shp, s->stream>>>(P, U, G, R, *rk, L);
        else jf::sweep_yz_pc_kernel<2, 1><<<grid, 256, shp, s->stream>>>(P, U, G, R, none, L);
      }
      s->launches += 3;
      JF_CUDA(s, cudaPeekAtLastError());
      return JF_OK;
    }
  }
  if constexpr (std::is_same<T, float>::value) {
    if (s->f32x2) {
      const size_t sh2 = jf::yz2_smem_bytes<VISC, ORD>();
      const dim3 blk2(jf::YZ_TX, jf::YZ_TY);
      auto rows = [](int n) { return ((n + 1) / 2 + jf::YZ_TY - 1) / jf::YZ_TY; };   // blocks over pairs of columns
      {
        Timed t(s, K_SWEEP_Y);
        const int L = s->seg_len2[1];
        dim3 grid((P.n[0] + jf::YZ_TX - 1) / jf::YZ_TX, rows(P.n[2]), (P.n[1] + L - 1) / L);
        jf::sweep_yz2_kernel<1, VISC, 0, ORD><<<grid, blk2, sh2, s->stream>>>(P, U, G, R, none, L);
      }
      {
        Timed t(s, K_SWEEP_Z);
        const int L = s->seg_len2[2];
        dim3 grid((P.n[0] + jf::YZ_TX - 1) / jf::YZ_TX, rows(P.n[1]), (P.n[2] + L - 1) / L);
        if (rk) jf::sweep_yz2_kernel<2, VISC, 2, ORD><<<grid, blk2, sh2, s->stream>>>(P, U, G, R, *rk, L);
        else jf::sweep_yz2_kernel<2, VISC, 1, ORD><<<grid, blk2, sh2, s->stream>>>(P, U, G, R, none, L);
      }
      s->launches += 3;
      JF_CUDA(s, cudaPeekAtLastError());
      return JF_OK;
    }
  }
  const size_t sh = jf::yz_smem_bytes<T, VISC, ORD>();
  const dim3 blk(jf::YZ_TX, jf::YZ_TY);
  {
    Timed t(s, K_SWEEP_Y);
    const int L = s->seg_len[1];
    dim3 grid((P.n[0] + jf::YZ_TX - 1) / jf::YZ_TX, (P.n[2] + jf::YZ_TY - 1) / jf::YZ_TY, (P.n[1] + L - 1) / L);
    jf::sweep_yz_kernel<T, 1, VISC, 0, ORD><<<grid, blk, sh, s->stream>>>(P, U, G, R, none, L);
  }
  {
    Timed t(s, K_SWEEP_Z);
    const int L = s->seg_len[2];
    dim3 grid((P.n[0] + jf::YZ_TX - 1) / jf::YZ_TX, (P.n[1] + jf::YZ_TY - 1) / jf::YZ_TY, (P.n[2] + L - 1) / L);
    if (rk) jf::sweep_yz_kernel<T, 2, VISC, 2, ORD><<<grid, blk, sh, s->stream>>>(P, U, G, R, *rk, L);
    else jf::sweep_yz_kernel<T, 2, VISC, 1, ORD><<<grid, blk, sh, s->stream>>>(P, U, G, R, none, L);
  }
  s->launches += 3;
  JF_CUDA(s, cudaPeekAtLastError());
  return JF_OK;
}

// The viscous y/z sweeps keep a 5-cell window of 10 values per thread in shared memory (50 KB per
// 128-thread block in fp64): above the 48 KB default, so opt in once per solver.
template <class T, bool VISC, int ORD = 4>
cudaError_t opt_in_smem() {
  const int sh = (int)jf::yz_smem_bytes<T, VISC, ORD>();
  cudaError_t e = cudaSuccess;
  auto set = [&](const void* f) {
    if (e == cudaSuccess) e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, sh);
#ifdef JF_YZ_CARVEOUT
    // (measured: with the largest carve-out the L1 shrinks and the re-read of U_s in the z + RK sweep misses it:
    // z + RK 2.15 -> 2.93 ms per step at 256^3; the default carve-out is kept)
    if (e == cudaSuccess) e = cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, JF_YZ_CARVEOUT);
#endif
  };
  set((const void*)jf::sweep_yz_kernel<T, 1, VISC, 0, ORD>);
  set((const void*)jf::sweep_yz_kernel<T, 2, VISC, 1, ORD>);
  set((const void*)jf::sweep_yz_kernel<T, 2, VISC, 2, ORD>);
  return e;
}

// sixth-order dissipative flux: fp64 / fp32 only (jf_set_visc_order refuses the tangent type)
template <class T>
jf_status launch_rhs_o6(jf_solver* s, Impl<T>& I, const T* U, T* R, const jf::RKArgs<T>* rk) {
  return launch_rhs_t<T, true, 6>(s, I, U, R, rk);
}
template <>
jf_status launch_rhs_o6<jf::Dual>(jf_solver* s, Impl<jf::Dual>&, const jf::Dual*, jf::Dual*, const jf::RKArgs<jf::Dual>*) {
  return fail(s, JF_EINVAL, "sixth-order dissipative flux: not built for the tangent type");
}

template <bool VISC, int ORD>
cudaError_t opt_in_smem_yz2() {
  const int sh = (int)jf::yz2_smem_bytes<VISC, ORD>();
  cudaError_t e = cudaFuncSetAttribute((const void*)jf::sweep_yz2_kernel<1, VISC, 0, ORD>, cudaFuncAttributeMaxDynamicSharedMemorySize, sh);
  if (e == cudaSuccess) e = cudaFuncSetAttribute((const void*)jf::sweep_yz2_kernel<2, VISC, 1, ORD>, cudaFuncAttributeMaxDynamicSharedMemorySize, sh);
  if (e == cudaSuccess) e = cudaFuncSetAttribute((const void*)jf::sweep_yz2_kernel<2, VISC, 2, ORD>, cudaFuncAttributeMaxDynamicSharedMemorySize, sh);
  return e;
}

template <class T>
jf_status launch_rhs(jf_solver* s, Impl<T>& I, const T* U, T* R, const jf::RKArgs<T>* rk) {
  if (s->viscous && s->visc_order == 6) return launch_rhs_o6<T>(s, I, U, R, rk);
  return s->viscous ? launch_rhs_t<T, true>(s, I, U, R, rk) : launch_rhs_t<T, false>(s, I, U, R, rk);
}

// SSP-RK3 (reading O8) stage by stage.  Stage input (the array whose halos must be filled): 1: U, 2: A, 3: B.
//   1: A = U + dt L(U);  2: B = 3/4 U + 1/4 (A + dt L(A));  3: U = 1/3 U + 2/3 (B + dt L(B)) (pointwise in
//   place: each thread reads U^n of its cell before writing it)
template <class T>
T* stage_input(Impl<T>& I, T* U, int stage) { return stage == 1 ? U : (stage == 2 ? I.A : I.B); }

template <class T>
jf_status stage_advance(jf_solver* s, Impl<T>& I, T* U, int stage, double dt, const double* dt_dev = nullptr) {
  if (stage == 1) { jf::RKArgs<T> r{U, I.A, T(0), T(1), T(dt), dt_dev}; return launch_rhs<T>(s, I, U, I.R, &r); }
  if (stage == 2) { jf::RKArgs<T> r{U, I.B, T(0.75), T(0.25), T(dt), dt_dev}; return launch_rhs<T>(s, I, I.A, I.R, &r); }
  jf::RKArgs<T> r{U, U, T(1.0 / 3.0), T(2.0 / 3.0), T(dt), dt_dev};
  return launch_rhs<T>(s, I, I.B, I.R, &r);
}

template <class T>
jf_status rk3_launches(jf_solver* s, Impl<T>& I, T* U, double dt, const double* dt_dev) {
  jf_status st;
  for (int stage = 1; stage <= 3; ++stage) {
    if ((st = launch_halo<T>(s, I, stage_input<T>(I, U, stage)))) return st;
    if ((st = stage_advance<T>(s, I, U, stage, dt, dt_dev))) return st;
  }
  return JF_OK;
}

__global__ void set_dt_kernel(double* st, double dt) { st[5] = dt; }

// One RK3 step.  dev_dt: take the step from the device scalar cfl_out[5] (jf_cfl_dt_dev) instead of `dt`.
// With graphs on (default; off while per-launch timing is enabled) the 15 launches are replayed from a graph whose
// kernels read the device scalar; a host dt is written there first by a one-thread kernel.
template <class T>
jf_status rk3(jf_solver* s, Impl<T>& I, T* U, double dt, bool dev_dt) {
  double* dt_dev = reinterpret_cast<double*>(I.cfl_out) + 5;
  if (!s->use_graph || s->timing) return rk3_launches<T>(s, I, U, dt, dev_dt ? dt_dev : nullptr);
  jf_solver::GraphEntry* ge = nullptr;
  for (auto& g : s->graphs)
    if (g.U == (const void*)U) ge = &g;
  if (!ge) {
    if (!s->cap_stream) JF_CUDA(s, cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking));
    const cudaStream_t user = s->stream;
    const unsigned long long l0 = s->launches;
    JF_CUDA(s, cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal));
    s->stream = s->cap_stream;
    const jf_status st = rk3_launches<T>(s, I, U, 0.0, dt_dev);
    s->stream = user;
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(s->cap_stream, &graph);
    const unsigned nk = (unsigned)(s->launches - l0);
    s->launches = l0;
    if (st != JF_OK) { if (graph) cudaGraphDestroy(graph); return st; }
    if (ce != cudaSuccess) return fail(s, JF_ECUDA, "cudaStreamEndCapture", ce);
    cudaGraphExec_t exec = nullptr;
    const cudaError_t ci = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ci != cudaSuccess) return fail(s, JF_ECUDA, "cudaGraphInstantiate", ci);
    if (s->graphs.size() >= 8) { cudaGraphExecDestroy(s->graphs.front().exec); s->graphs.erase(s->graphs.begin()); }
    s->graphs.push_back({(const void*)U, exec, nk});
    ge = &s->graphs.back();
  }
  if (!dev_dt) {
    set_dt_kernel<<<1, 1, 0, s->stream>>>(reinterpret_cast<double*>(I.cfl_out), dt);
    s->launches += 1;
  }
  JF_CUDA(s, cudaGraphLaunch(ge->exec, s->stream));
  s->launches += ge->kernels;
  return JF_OK;
}

template <class T>
int cfl_blocks(const Impl<T>& I) {
  // one warp per 32-cell chunk of a grid line; at most 8 resident blocks of 8 warps on each of the 148 SMs
  const long long ntask = (long long)((I.P.n[0] + 31) / 32) * I.P.n[1] * I.P.n[2];
  return (int)std::max<long long>(1, std::min<long long>((ntask + 7) / 8, 148LL * 8));
}

// reduction + finalize on the device (no host synchronisation): dt -> cfl_out[5], t += dt -> cfl_out[6]
template <class T>
jf_status cfl_dev(jf_solver* s, Impl<T>& I, const T* U, double cflnum, double t_end) {
  {
    Timed t(s, K_CFL);
    jf::cfl_kernel<T><<<cfl_blocks<T>(I), 256, 0, s->stream>>>(I.P, U, I.cfl_out, 1, cflnum, t_end);
  }
  s->launches += 1;
  JF_CUDA(s, cudaPeekAtLastError());
  return JF_OK;
}

template <class T>
jf_status cfl(jf_solver* s, Impl<T>& I, const T* U, double cflnum, double* dt_host) {
  JF_CUDA(s, cudaMemsetAsync(I.cfl_out, 0xFF, 3 * sizeof(unsigned long long), s->stream));
  JF_CUDA(s, cudaMemsetAsync(I.cfl_out + 3, 0, 2 * sizeof(unsigned long long), s->stream));
  int blocks = cfl_blocks<T>(I);
  {
    Timed t(s, K_CFL);
    jf::cfl_kernel<T><<<blocks, 256, 0, s->stream>>>(I.P, U, I.cfl_out, 0, 0.0, 0.0);
  }
  s->launches += 1;
  JF_CUDA(s, cudaPeekAtLastError());
  unsigned long long h[4];
  JF_CUDA(s, cudaMemcpyAsync(h, I.cfl_out, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
  JF_CUDA(s, cudaMemsetAsync(I.cfl_out, 0xFF, 3 * sizeof(unsigned long long), s->stream));   // leave it armed for jf_cfl_dt_dev
  JF_CUDA(s, cudaMemsetAsync(I.cfl_out + 3, 0, 2 * sizeof(unsigned long long), s->stream));
  JF_CUDA(s, cudaStreamSynchronize(s->stream));
  if (h[3]) { *dt_host = std::nan(""); return fail(s, JF_ENOTFINITE, "jf_cfl_dt: non-finite state or rho <= 0 or p <= 0"); }
  double v[3];
  std::memcpy(v, h, sizeof(v));
  double dt = v[0];
  if (s->viscous) dt = std::fmin(dt, std::fmin((3.0 / 14.0) * v[1], (1.0 / 10.0) * v[2]));
  *dt_host = cflnum * dt;
  return JF_OK;
}

template <class T>
jf_status plane_sums(jf_solver* s, Impl<T>& I, const T* U, int axis, double* out) {
  const jf::Params<T>& P = I.P;
  const int np = P.n[axis];
  const long long ntang = (long long)P.n[(axis + 1) % 3] * P.n[(axis + 2) % 3];
  int NB = (int)std::min<long long>(STATS_NB, std::max<long long>(1, std::min<long long>((148LL * 8 + np - 1) / np, (ntang + 1023) / 1024)));
  const dim3 grid(np, NB);
  if (axis == 0) jf::plane_sums_kernel<T, 0><<<grid, 256, 0, s->stream>>>(P, U, I.stats, NB);
  else if (axis == 1) jf::plane_sums_kernel<T, 1><<<grid, 256, 0, s->stream>>>(P, U, I.stats, NB);
  else jf::plane_sums_kernel<T, 2><<<grid, 256, 0, s->stream>>>(P, U, I.stats, NB);
  jf::plane_sums_final<<<(jf::NSTAT * np + 127) / 128, 128, 0, s->stream>>>(I.stats, out, np, NB);
  s->launches += 2;
  JF_CUDA(s, cudaPeekAtLastError());
  return JF_OK;
}

// jf_plane_sums with the partial sums in the library's static device array instead of the caller's workspace: same
// kernels, same launch configuration, same summation order => the same bits as plane_sums above.  Allocates nothing.
template <class T>
jf_status plane_sums_static(jf_solver* s, Impl<T>& I, const T* U, int axis, double* out) {
  const jf::Params<T>& P = I.P;
  const int np = P.n[axis];
  if (np > JF_STATIC_MAX_PLANES)
    return fail(s, JF_EINVAL, "jf_plane_sums_static: more than JF_STATIC_MAX_PLANES = 1024 planes along this axis "
                              "(the static scratch array holds 14 x 1024 x 16 partial sums); use jf_plane_sums");
  double* scratch = nullptr;
  {
    const cudaError_t ce = static_scratch_ptr(&scratch);
    if (ce != cudaSuccess || !scratch) return fail(s, JF_ECUDA, "jf_plane_sums_static: cudaGetSymbolAddress(jf_static_scratch)", ce);
  }
  const long long ntang = (long long)P.n[(axis + 1) % 3] * P.n[(axis + 2) % 3];
  int NB = (int)std::min<long long>(STATS_NB, std::max<long long>(1, std::min<long long>((148LL * 8 + np - 1) / np, (ntang + 1023) / 1024)));
  const dim3 grid(np, NB);
  if (axis == 0) jf::plane_sums_kernel<T, 0><<<grid, 256, 0, s->stream>>>(P, U, scratch, NB);
  else if (axis == 1) jf::plane_sums_kernel<T, 1><<<grid, 256, 0, s->stream>>>(P, U, scratch, NB);
  else jf::plane_sums_kernel<T, 2><<<grid, 256, 0, s->stream>>>(P, U, scratch, NB);
  jf::plane_sums_final<<<(jf::NSTAT * np + 127) / 128, 128, 0, s->stream>>>(scratch, out, np, NB);
  s->launches += 2;
  JF_CUDA(s, cudaPeekAtLastError());
  return JF_OK;
}

template <class T>
jf_status diag_metrics(jf_solver* s, Impl<T>& I, int axis, double* inv_delta, double* centre, double* i12Xc, double* i24Xf) {
  const int Pn = I.P.P[axis];
  JF_CUDA(s, cudaStreamSynchronize(s->stream));
  std::vector<T> t(Pn);
  const T* src[3] = {I.P.inv_dl[axis], I.P.i12Xc[axis], I.P.i24Xf[axis]};
  double* dst[3] = {inv_delta, i12Xc, i24Xf};
  for (int k = 0; k < 3; ++k) {
    if (!dst[k]) continue;
    JF_CUDA(s, cudaMemcpy(t.data(), src[k], Pn * sizeof(T), cudaMemcpyDeviceToHost));
    for (int p = 0; p < Pn; ++p) dst[k][p] = jf::value_of(t[p]);
  }
  if (centre) JF_CUDA(s, cudaMemcpy(centre, I.P.xc[axis], Pn * sizeof(double), cudaMemcpyDeviceToHost));
  return JF_OK;
}

}  // namespace

extern "C" {

size_t jf_workspace_bytes(const jf_grid* g, jf_dtype dtype) {
  if (!grid_ok(g) || !dtype_ok(dtype)) return 0;
  const int n[3] = {g->nx, g->ny, g->nz};
  return make_layout(n, elem_size(dtype)).total;
}

jf_status jf_create(jf_solver** out, const jf_grid* g, jf_dtype dtype, double gamma, double R_gas, double Pr,
                    const jf_mu_law* mu, const jf_bc* bc, const double body_accel[3], void* workspace_dev,
                    size_t workspace_bytes, void* cuda_stream) {
  if (!out) return JF_EINVAL;
  *out = nullptr;
  if (!grid_ok(g) || !mu || !bc) return JF_EINVAL;
  if (!dtype_ok(dtype)) return JF_EINVAL;
  if (!(gamma > 1.0) || !(R_gas > 0.0) || !(Pr > 0.0) || !(mu->mu_ref >= 0.0)) return JF_EINVAL;
  if (mu->sutherland && !(mu->T_ref > 0.0)) return JF_EINVAL;
  for (int a = 0; a < 3; ++a)
    if ((bc->face[2 * a].type == JF_BC_PERIODIC) != (bc->face[2 * a + 1].type == JF_BC_PERIODIC)) return JF_EINVAL;
  for (int f = 0; f < 6; ++f) {
    const jf_bc_face& b = bc->face[f];
    if ((int)b.type < 0 || (int)b.type > 5) return JF_EINVAL;
    if (b.type == JF_BC_EXCHANGE && !b.nb_has_face && !(b.nb_width[0] > 0.0 && b.nb_width[1] > 0.0 && b.nb_width[2] > 0.0)) return JF_EINVAL;
    if (b.type == JF_BC_EXCHANGE && b.nb_has_face) {      // strictly monotone away from the face
      const double e = (f % 2 == 0) ? (f / 2 == 0 ? g->xf : f / 2 == 1 ? g->yf : g->zf)[0]
                                    : (f / 2 == 0 ? g->xf[g->nx] : f / 2 == 1 ? g->yf[g->ny] : g->zf[g->nz]);
      const double sg = (f % 2 == 0) ? -1.0 : 1.0;
      if (!(sg * (b.nb_face[0] - e) > 0.0 && sg * (b.nb_face[1] - b.nb_face[0]) > 0.0 && sg * (b.nb_face[2] - b.nb_face[1]) > 0.0)) return JF_EINVAL;
    }
    if (b.type == JF_BC_DIRICHLET && !b.dirichlet) return JF_EINVAL;
    if (b.type == JF_BC_WALL_ISOTHERMAL && !(b.T_wall > 0.0)) return JF_EINVAL;
  }
  if (!workspace_dev) return JF_EWORKSPACE;
  if (((uintptr_t)workspace_dev) % 256 != 0) return JF_EALIGN;
  if (workspace_bytes < jf_workspace_bytes(g, dtype)) return JF_EWORKSPACE;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return JF_ECUDA;  // no CPU fallback
  jf_solver* s = new (std::nothrow) jf_solver();
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  s->dtype = dtype;
  s->stream = (cudaStream_t)cuda_stream;
  if (cudaGetDevice(&s->device) != cudaSuccess) { delete s; return JF_ECUDA; }
  {
    // the workspace must live on the current device: the kernels are launched there
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, workspace_dev) == cudaSuccess && at.type == cudaMemoryTypeDevice && at.device != s->device) {
      delete s;
      return JF_EINVAL;
    }
  }
  s->viscous = mu->mu_ref > 0.0;
  s->Pr = Pr;
  s->launches = 0;
  jf_status st = dtype == JF_F64   ? setup<double>(s, s->d, g, gamma, R_gas, Pr, mu, bc, body_accel, (char*)workspace_dev)
                 : dtype == JF_F32 ? setup<float>(s, s->f, g, gamma, R_gas, Pr, mu, bc, body_accel, (char*)workspace_dev)
                                   : setup<jf::Dual>(s, s->t, g, gamma, R_gas, Pr, mu, bc, body_accel, (char*)workspace_dev);
  if (st != JF_OK) { delete s; return st; }
  {
    cudaError_t ce = dtype == JF_F64   ? (s->viscous ? opt_in_smem<double, true>() : opt_in_smem<double, false>())
                     : dtype == JF_F32 ? (s->viscous ? opt_in_smem<float, true>() : opt_in_smem<float, false>())
                                       : (s->viscous ? opt_in_smem<jf::Dual, true>() : opt_in_smem<jf::Dual, false>());
    if (ce != cudaSuccess) { delete s; return JF_ECUDA; }
  }
  {
    // TMA needs 16-byte global strides: (nx+6) * 8 bytes, i.e. even nx.  fp64 only: the tangent type has no tensor-map
    // data type, and the fp32 instantiation (pitch aligned only for nx = 2 mod 4) faulted on the box copy in the one
    // run it got ("illegal instruction", 70x35x67) and is not worth a second kernel.
    // JF_GRAD_TMA=0/1 overrides the default (tuning / A-B measurements).
    const size_t esz = elem_size(dtype);
    bool ok = dtype == JF_F64 && ((size_t)(g->nx + 6) * esz) % 16 == 0 && encode_tiled_fn() != nullptr;
    const char* e = std::getenv("JF_GRAD_TMA");
    // Default by size: the TMA-staged pass is 6-8 % faster than the plain-load pass up to 320^3, equal at 384^3 and
    // 15 % slower at 448^3 and above (profiles/r2_tma_sass.md), so it is used for fields of at most JF_GRAD_TMA_MAX_CELLS
    // padded cells per variable (40 M: up to ~335^3).
#ifndef JF_GRAD_TMA_MAX_CELLS
#define JF_GRAD_TMA_MAX_CELLS 40000000.0
#endif
    bool want = (double)(g->nx + 6) * (double)(g->ny + 6) * (double)(g->nz + 6) <= JF_GRAD_TMA_MAX_CELLS;
    if (e) want = std::atoi(e) != 0;
    s->grad_tma = ok && want;
    if (s->grad_tma) {
      cudaError_t ce = cudaFuncSetAttribute((const void*)jf::gradient_tma_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(jf::GradTmaSmem<double>));
      if (ce != cudaSuccess) s->grad_tma = false;
    }
  }
  if (const char* e = std::getenv("JF_GRAPH")) s->use_graph = std::atoi(e) != 0;
  {
    bool want = false;
#ifdef JF_YZ_PC_DEFAULT
    want = JF_YZ_PC_DEFAULT != 0;
#endif
    if (const char* e = std::getenv("JF_YZ_PC")) want = std::atoi(e) != 0;
    s->yz_pc = want && dtype == JF_F64 && s->viscous;
    if (s->yz_pc) {
      const int shp = (int)jf::pc_smem_bytes();
      cudaError_t ce = cudaFuncSetAttribute((const void*)jf::sweep_yz_pc_kernel<1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, shp);
      if (ce == cudaSuccess) ce = cudaFuncSetAttribute((const void*)jf::sweep_yz_pc_kernel<2, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, shp);
      if (ce == cudaSuccess) ce = cudaFuncSetAttribute((const void*)jf::sweep_yz_pc_kernel<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, shp);
      if (ce != cudaSuccess) s->yz_pc = false;
    }
  }
  const int n[3] = {g->nx, g->ny, g->nz};
  s->seg_len[0] = 0;
  auto cdiv = [](int a, int b) { return (long long)((a + b - 1) / b); };
  s->seg_len[1] = pick_segment(cdiv(n[0], jf::YZ_TX) * cdiv(n[2], jf::YZ_TY) * jf::YZ_TY, n[1]);
  s->seg_len[2] = pick_segment(cdiv(n[0], jf::YZ_TX) * cdiv(n[1], jf::YZ_TY) * jf::YZ_TY, n[2]);
  {
    bool want = false;
#ifdef JF_F32X2_DEFAULT
    want = JF_F32X2_DEFAULT != 0;
#endif
    if (const char* e = std::getenv("JF_F32X2")) want = std::atoi(e) != 0;
    s->f32x2 = want && dtype == JF_F32;
    if (s->f32x2) {
      cudaError_t ce = s->viscous ? opt_in_smem_yz2<true, 4>() : opt_in_smem_yz2<false, 4>();
      if (ce == cudaSuccess && s->viscous) ce = opt_in_smem_yz2<true, 6>();
      if (ce != cudaSuccess) s->f32x2 = false;
      s->seg_len2[1] = pick_segment(cdiv(n[0], jf::YZ_TX) * cdiv((n[2] + 1) / 2, jf::YZ_TY) * jf::YZ_TY, n[1]);
      s->seg_len2[2] = pick_segment(cdiv(n[0], jf::YZ_TX) * cdiv((n[1] + 1) / 2, jf::YZ_TY) * jf::YZ_TY, n[2]);
    }
  }
  *out = s;
  return JF_OK;
}

jf_status jf_destroy(jf_solver* s) {
  if (s) {
    for (auto& e : s->ev_used) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    for (auto& e : s->ev_free) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    for (auto& g : s->graphs) cudaGraphExecDestroy(g.exec);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
  }
  delete s;
  return JF_OK;
}

jf_status jf_diag_timing(jf_solver* s, int enable) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  s->timing = enable != 0;
  return JF_OK;
}

jf_status jf_diag_kernel_times(jf_solver* s, double ms[6], unsigned long long launches[6]) {
  if (!s || !ms || !launches) return JF_EINVAL;
  for (int k = 0; k < K_COUNT; ++k) { ms[k] = 0.0; launches[k] = 0; }
  JF_CUDA(s, cudaStreamSynchronize(s->stream));
  for (auto& e : s->ev_used) {
    float t = 0.f;
    JF_CUDA(s, cudaEventElapsedTime(&t, e.a, e.b));
    ms[e.cls] += t; launches[e.cls] += 1;
    s->ev_free.push_back(e);
  }
  s->ev_used.clear();
  return JF_OK;
}

const char* jf_diag_kernel_name(int k) {
  static const char* names[K_COUNT] = {"halo_all_kernel", "gradient_kernel", "sweep_x_kernel", "sweep_yz_kernel<y>",
                                       "sweep_yz_kernel<z>+rk", "cfl_kernel"};
  return (k >= 0 && k < K_COUNT) ? names[k] : "";
}

size_t jf_state_elems(const jf_solver* s) {
  if (!s) return 0;
  return (size_t)5 * (s->dtype == JF_F64 ? s->d.P.vol : s->dtype == JF_F32 ? s->f.P.vol : s->t.P.vol);
}

static bool aligned16(const void* p) { return ((uintptr_t)p) % 16 == 0; }

jf_status jf_fill_halo(jf_solver* s, void* U) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U) return fail(s, JF_EINVAL, "jf_fill_halo: null pointer");
  if (!aligned16(U)) return fail(s, JF_EALIGN, "jf_fill_halo: U not 16-byte aligned");
  return s->dtype == JF_F64   ? launch_halo<double>(s, s->d, (double*)U)
         : s->dtype == JF_F32 ? launch_halo<float>(s, s->f, (float*)U)
                              : launch_halo<jf::Dual>(s, s->t, (jf::Dual*)U);
}

jf_status jf_rhs(jf_solver* s, const void* U, void* R) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || !R || U == R) return fail(s, JF_EINVAL, "jf_rhs: null or aliased pointers");
  if (!aligned16(U) || !aligned16(R)) return fail(s, JF_EALIGN, "jf_rhs: pointer not 16-byte aligned");
  return s->dtype == JF_F64   ? launch_rhs<double>(s, s->d, (const double*)U, (double*)R, nullptr)
         : s->dtype == JF_F32 ? launch_rhs<float>(s, s->f, (const float*)U, (float*)R, nullptr)
                              : launch_rhs<jf::Dual>(s, s->t, (const jf::Dual*)U, (jf::Dual*)R, nullptr);
}

jf_status jf_rk3_step(jf_solver* s, void* U, double dt) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || !(dt == dt)) return fail(s, JF_EINVAL, "jf_rk3_step: null pointer or NaN dt");
  if (!aligned16(U)) return fail(s, JF_EALIGN, "jf_rk3_step: U not 16-byte aligned");
  return s->dtype == JF_F64   ? rk3<double>(s, s->d, (double*)U, dt, false)
         : s->dtype == JF_F32 ? rk3<float>(s, s->f, (float*)U, dt, false)
                              : rk3<jf::Dual>(s, s->t, (jf::Dual*)U, dt, false);
}

jf_status jf_set_visc_order(jf_solver* s, int order) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (order != 4 && order != 6) return fail(s, JF_EINVAL, "jf_set_visc_order: order must be 4 or 6");
  if (order == 6 && s->dtype == JF_F64_TANGENT) return fail(s, JF_EINVAL, "jf_set_visc_order: order 6 is not built for the tangent type");
  if (order == s->visc_order) return JF_OK;
  JF_CUDA(s, cudaStreamSynchronize(s->stream));
  s->visc_order = order;
  for (auto& g : s->graphs) cudaGraphExecDestroy(g.exec);      // the captured steps launch the other kernels
  s->graphs.clear();
  if (order == 6 && s->viscous) {
    const cudaError_t ce = s->dtype == JF_F64 ? opt_in_smem<double, true, 6>() : opt_in_smem<float, true, 6>();
    if (ce != cudaSuccess) return fail(s, JF_ECUDA, "cudaFuncSetAttribute", ce);
  }
  return s->dtype == JF_F64 ? upload_tables<double>(s, s->d) : s->dtype == JF_F32 ? upload_tables<float>(s, s->f)
                                                                                  : upload_tables<jf::Dual>(s, s->t);
}

jf_status jf_cfl_dt_dev(jf_solver* s, const void* U, double cflnum, double t_end) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || !(cflnum > 0.0)) return fail(s, JF_EINVAL, "jf_cfl_dt_dev: null pointer or cfl <= 0");
  if (!aligned16(U)) return fail(s, JF_EALIGN, "jf_cfl_dt_dev: U not 16-byte aligned");
  return s->dtype == JF_F64   ? cfl_dev<double>(s, s->d, (const double*)U, cflnum, t_end)
         : s->dtype == JF_F32 ? cfl_dev<float>(s, s->f, (const float*)U, cflnum, t_end)
                              : cfl_dev<jf::Dual>(s, s->t, (const jf::Dual*)U, cflnum, t_end);
}

jf_status jf_rk3_step_dev(jf_solver* s, void* U) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U) return fail(s, JF_EINVAL, "jf_rk3_step_dev: null pointer");
  if (!aligned16(U)) return fail(s, JF_EALIGN, "jf_rk3_step_dev: U not 16-byte aligned");
  return s->dtype == JF_F64   ? rk3<double>(s, s->d, (double*)U, 0.0, true)
         : s->dtype == JF_F32 ? rk3<float>(s, s->f, (float*)U, 0.0, true)
                              : rk3<jf::Dual>(s, s->t, (jf::Dual*)U, 0.0, true);
}

jf_status jf_dev_time(jf_solver* s, int set, double* dt_host, double* t_host) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  unsigned long long* out = s->dtype == JF_F64 ? s->d.cfl_out : s->dtype == JF_F32 ? s->f.cfl_out : s->t.cfl_out;
  if (set) {
    if (!t_host) return fail(s, JF_EINVAL, "jf_dev_time: null pointer");
    unsigned long long h[3] = {0, 0, 0};
    std::memcpy(&h[1], t_host, sizeof(double));
    JF_CUDA(s, cudaMemcpyAsync(out + 5, h, sizeof(h), cudaMemcpyHostToDevice, s->stream));
    JF_CUDA(s, cudaStreamSynchronize(s->stream));
    return JF_OK;
  }
  unsigned long long h[3];
  JF_CUDA(s, cudaMemcpyAsync(h, out + 5, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
  JF_CUDA(s, cudaStreamSynchronize(s->stream));
  if (dt_host) std::memcpy(dt_host, &h[0], sizeof(double));
  if (t_host) std::memcpy(t_host, &h[1], sizeof(double));
  if (h[2]) return fail(s, JF_ENOTFINITE, "jf_dev_time: a device-side CFL reduction met a non-finite state or rho <= 0 or p <= 0");
  return JF_OK;
}

jf_status jf_cfl_dt(jf_solver* s, const void* U, double cflnum, double* dt_host) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || !dt_host) return fail(s, JF_EINVAL, "jf_cfl_dt: null pointer");
  if (!aligned16(U)) return fail(s, JF_EALIGN, "jf_cfl_dt: U not 16-byte aligned");
  return s->dtype == JF_F64   ? cfl<double>(s, s->d, (const double*)U, cflnum, dt_host)
         : s->dtype == JF_F32 ? cfl<float>(s, s->f, (const float*)U, cflnum, dt_host)
                              : cfl<jf::Dual>(s, s->t, (const jf::Dual*)U, cflnum, dt_host);
}

// dispatch on the solver's scalar type: F(Impl<T>&, T tag)
#define JF_DISPATCH(s, EXPR_D, EXPR_F, EXPR_T) \
  ((s)->dtype == JF_F64 ? (EXPR_D) : (s)->dtype == JF_F32 ? (EXPR_F) : (EXPR_T))

jf_status jf_fill_halo_axis(jf_solver* s, void* U, int axis) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || axis < 0 || axis > 2) return fail(s, JF_EINVAL, "jf_fill_halo_axis: null pointer or bad axis");
  if (!aligned16(U)) return fail(s, JF_EALIGN, "jf_fill_halo_axis: U not 16-byte aligned");
  return JF_DISPATCH(s, launch_halo_axis<double>(s, s->d, (double*)U, axis), launch_halo_axis<float>(s, s->f, (float*)U, axis),
                     launch_halo_axis<jf::Dual>(s, s->t, (jf::Dual*)U, axis));
}

size_t jf_face_elems(const jf_solver* s, int face) {
  if (!s || face < 0 || face > 5) return 0;
  return (size_t)(15 * JF_DISPATCH(s, face_cells<double>(s->d.P, face / 2), face_cells<float>(s->f.P, face / 2),
                                   face_cells<jf::Dual>(s->t.P, face / 2)));
}

jf_status jf_pack_face(jf_solver* s, const void* U, int face, void* buf) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || !buf || face < 0 || face > 5) return fail(s, JF_EINVAL, "jf_pack_face: null pointer or bad face");
  return JF_DISPATCH(s, (launch_xfer<double, 0>(s, s->d, face, (double*)U, (double*)buf, nullptr, nullptr)),
                     (launch_xfer<float, 0>(s, s->f, face, (float*)U, (float*)buf, nullptr, nullptr)),
                     (launch_xfer<jf::Dual, 0>(s, s->t, face, (jf::Dual*)U, (jf::Dual*)buf, nullptr, nullptr)));
}

jf_status jf_unpack_face(jf_solver* s, void* U, int face, const void* buf) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || !buf || face < 0 || face > 5) return fail(s, JF_EINVAL, "jf_unpack_face: null pointer or bad face");
  return JF_DISPATCH(s, (launch_xfer<double, 1>(s, s->d, face, (double*)U, (double*)buf, nullptr, nullptr)),
                     (launch_xfer<float, 1>(s, s->f, face, (float*)U, (float*)buf, nullptr, nullptr)),
                     (launch_xfer<jf::Dual, 1>(s, s->t, face, (jf::Dual*)U, (jf::Dual*)buf, nullptr, nullptr)));
}

jf_status jf_pull_face(jf_solver* s, void* U, int face, const void* U_peer, const int n_peer[3]) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || !U_peer || !n_peer || face < 0 || face > 5) return fail(s, JF_EINVAL, "jf_pull_face: null pointer or bad face");
  const int a = face / 2;
  const int* n = JF_DISPATCH(s, s->d.P.n, s->f.P.n, s->t.P.n);
  for (int b = 0; b < 3; ++b)
    if (n_peer[b] < 4 || (b != a && n_peer[b] != n[b]))
      return fail(s, JF_EINVAL, "jf_pull_face: the peer block must match this block's tangential extents");
  return JF_DISPATCH(s, (launch_xfer<double, 2>(s, s->d, face, (double*)U, nullptr, (const double*)U_peer, n_peer)),
                     (launch_xfer<float, 2>(s, s->f, face, (float*)U, nullptr, (const float*)U_peer, n_peer)),
                     (launch_xfer<jf::Dual, 2>(s, s->t, face, (jf::Dual*)U, nullptr, (const jf::Dual*)U_peer, n_peer)));
}

void* jf_rk3_stage_input(jf_solver* s, void* U, int stage) {
  if (!s || !U || stage < 1 || stage > 3) return nullptr;
  return JF_DISPATCH(s, (void*)stage_input<double>(s->d, (double*)U, stage), (void*)stage_input<float>(s->f, (float*)U, stage),
                     (void*)stage_input<jf::Dual>(s->t, (jf::Dual*)U, stage));
}

jf_status jf_rk3_stage_advance(jf_solver* s, void* U, int stage, double dt) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || stage < 1 || stage > 3 || !(dt == dt)) return fail(s, JF_EINVAL, "jf_rk3_stage_advance: bad argument");
  if (!aligned16(U)) return fail(s, JF_EALIGN, "jf_rk3_stage_advance: U not 16-byte aligned");
  return JF_DISPATCH(s, stage_advance<double>(s, s->d, (double*)U, stage, dt), stage_advance<float>(s, s->f, (float*)U, stage, dt),
                     stage_advance<jf::Dual>(s, s->t, (jf::Dual*)U, stage, dt));
}

jf_status jf_plane_sums(jf_solver* s, const void* U, int axis, double* sums) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || !sums || axis < 0 || axis > 2) return fail(s, JF_EINVAL, "jf_plane_sums: null pointer or bad axis");
  if (!aligned16(U)) return fail(s, JF_EALIGN, "jf_plane_sums: U not 16-byte aligned");
  return JF_DISPATCH(s, plane_sums<double>(s, s->d, (const double*)U, axis, sums), plane_sums<float>(s, s->f, (const float*)U, axis, sums),
                     plane_sums<jf::Dual>(s, s->t, (const jf::Dual*)U, axis, sums));
}

jf_status jf_plane_sums_static(jf_solver* s, const void* U, int axis, double* sums) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (!U || !sums || axis < 0 || axis > 2) return fail(s, JF_EINVAL, "jf_plane_sums_static: null pointer or bad axis");
  if (!aligned16(U)) return fail(s, JF_EALIGN, "jf_plane_sums_static: U not 16-byte aligned");
  return JF_DISPATCH(s, plane_sums_static<double>(s, s->d, (const double*)U, axis, sums),
                     plane_sums_static<float>(s, s->f, (const float*)U, axis, sums),
                     plane_sums_static<jf::Dual>(s, s->t, (const jf::Dual*)U, axis, sums));
}

int jf_plane_sums_static_max_planes(void) { return JF_STATIC_MAX_PLANES; }

jf_status jf_set_tangent_seed(jf_solver* s, double dA, double dkappa) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (s->dtype != JF_F64_TANGENT) return fail(s, JF_EINVAL, "jf_set_tangent_seed: not a tangent solver");
  if (!(dA == dA) || !(dkappa == dkappa)) return fail(s, JF_EINVAL, "jf_set_tangent_seed: NaN seed");
  for (int f = 0; f < 6; ++f) { s->t.bc[f].dA = dA; s->t.bc[f].dkappa = dkappa; }
  // the halo kernels take the face tables by value: captured steps would replay the old seed
  JF_CUDA(s, cudaStreamSynchronize(s->stream));
  for (auto& g : s->graphs) cudaGraphExecDestroy(g.exec);
  s->graphs.clear();
  return JF_OK;
}

const char* jf_last_error(const jf_solver* s) { return s ? s->err.c_str() : ""; }

unsigned long long jf_launch_count(const jf_solver* s) { return s ? s->launches : 0ULL; }

jf_status jf_diag_alu_peak(jf_dtype dtype, int iters, double* flops_host, double* ms_host) {
  if (!flops_host || iters <= 0 || (dtype != JF_F64 && dtype != JF_F32)) return JF_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return JF_ECUDA;
  void* buf = nullptr;
  if (cudaMalloc(&buf, 256) != cudaSuccess) return JF_ECUDA;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = 148 * 8, threads = 256;
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0);
    if (dtype == JF_F64) jf::alu_peak_kernel<double><<<blocks, threads>>>((double*)buf, iters, 1.0);
    else jf::alu_peak_kernel<float><<<blocks, threads>>>((float*)buf, iters, 1.0f);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(buf); return JF_ECUDA; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(buf);
  double fl = 2.0 * 64.0 * (double)iters * (double)blocks * threads;
  *flops_host = fl / (best * 1e-3);
  if (ms_host) *ms_host = best;
  return cudaGetLastError() == cudaSuccess ? JF_OK : JF_ECUDA;
}

jf_status jf_diag_face_flux(jf_dtype dtype, int dir, double gamma, double R_gas, double Pr, const jf_mu_law* mu,
                            int n_faces, const double* W, const double* Gt, const double* Xf, double* F) {
  if (!mu || !W || !F || n_faces <= 0 || dir < 0 || dir > 2 || (dtype != JF_F64 && dtype != JF_F32)) return JF_EINVAL;
  if (!(gamma > 1.0) || !(R_gas > 0.0) || !(Pr > 0.0)) return JF_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return JF_ECUDA;
  return dtype == JF_F64 ? diag_face_flux<double>(dir, gamma, R_gas, Pr, mu, n_faces, W, Gt, Xf, F)
                         : diag_face_flux<float>(dir, gamma, R_gas, Pr, mu, n_faces, W, Gt, Xf, F);
}

jf_status jf_diag_metrics(jf_solver* s, int axis, double* inv_delta, double* centre, double* i12Xc, double* i24Xf) {
  if (!s) return JF_EINVAL;
  DeviceGuard dev_guard(s);
  if (axis < 0 || axis > 2) return fail(s, JF_EINVAL, "jf_diag_metrics: bad axis");
  return JF_DISPATCH(s, diag_metrics<double>(s, s->d, axis, inv_delta, centre, i12Xc, i24Xf),
                     diag_metrics<float>(s, s->f, axis, inv_delta, centre, i12Xc, i24Xf),
                     diag_metrics<jf::Dual>(s, s->t, axis, inv_delta, centre, i12Xc, i24Xf));
}

const char* jf_version(void) { return "libjf 0.2 (sm_100a; WENO5-JS + HLLC + 4th- or 6th-order central viscous flux + SSP-RK3; CUDA-graph step, device-resident dt)"; }

}  // extern "C"
