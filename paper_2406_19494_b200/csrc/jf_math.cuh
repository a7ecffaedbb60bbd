// jf_math.cuh — per-face device arithmetic of the hot path (sm_100a).
//
// Written for the plain FP64/FP32 ALUs (nothing here is a dense contraction, so no tensor
// cores): the formulas of DESIGN.md "Readings" (WENO5-JS, HLLC with Roe-average wave speeds,
// 4th-order central dissipative flux, Sutherland) restructured to cut divisions — the FP64
// pipe pays ~10 issue slots per division:
//   * WENO5 is evaluated per CELL, not per face: the left-biased state at face i+1/2 and the
//     right-biased state at face i-1/2 are both built from cells i-2..i+2 with the SAME three
//     smoothness indicators (the mirrored stencil of Jiang & Shu only swaps beta_0 and beta_2
//     and the linear weights), so the indicators are computed once for two reconstructions;
//   * the three non-linear weights are formed as products n_k = d_k e_l e_m with
//     e_k = (beta_k + eps)^2, so one reconstruction costs ONE reciprocal instead of four
//     divisions; reciprocal / square roots are a hardware seed plus one cubic Newton step;
//   * HLLC: only the star state on the side selected by sign(S*) is evaluated (the other is
//     multiplied by an exact zero in the closed form), reciprocals are shared.
// Results agree with the closed forms to a few ulp, not bit-wise (tolerance: DESIGN.md).
#pragma once
#include <cuda_runtime.h>
#include "jf_dual.cuh"

namespace jf {

template <class T> struct Num;
template <> struct Num<double> {
  static __device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
  // reciprocal for normal, finite a: hardware seed (MUFU.RCP64H, rel. error <= 2^-23) and one
  // cubic step x (1 + e + e^2), e = 1 - a x  =>  error ~ e^3 < 2^-66: a few ulp-fractions, not
  // correctly rounded; 3 DFMA instead of the ~10-instruction 1.0/a.
  static __device__ __forceinline__ double rcp(double a) {
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(a));
    double e = fma(-a, x, 1.0);
    return fma(x, fma(e, e, e), x);
  }
  // 1/sqrt(a), normal finite a > 0: seed (MUFU.RSQ64H) and one cubic step
  // y (1 + e/2 + 3 e^2/8), e = 1 - a y^2.
  static __device__ __forceinline__ double rsqrt_(double a) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double e = fma(-(a * y), y, 1.0);
    return fma(y, e * fma(0.375, e, 0.5), y);
  }
  static __device__ __forceinline__ double sqrt_(double a) { return a * rsqrt_(a); }
  static __device__ __forceinline__ double min_(double a, double b) { return fmin(a, b); }
  static __device__ __forceinline__ double max_(double a, double b) { return fmax(a, b); }
  static __device__ __forceinline__ double abs_(double a) { return fabs(a); }
};
template <> struct Num<float> {
  static __device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
  // MUFU seeds (rel. error ~2^-22) refined by one Newton step: ~1 ulp, a fraction of the IEEE sequences
  static __device__ __forceinline__ float rcp(float a) {
    float x;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(x) : "f"(a));
    return fmaf(x, fmaf(-a, x, 1.0f), x);
  }
  static __device__ __forceinline__ float rsqrt_(float a) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(a));
    float e = fmaf(-(a * y), y, 1.0f);
    return fmaf(y, 0.5f * e, y);
  }
  static __device__ __forceinline__ float sqrt_(float a) { return a * rsqrt_(a); }
  static __device__ __forceinline__ float min_(float a, float b) { return fminf(a, b); }
  static __device__ __forceinline__ float max_(float a, float b) { return fmaxf(a, b); }
  static __device__ __forceinline__ float abs_(float a) { return fabsf(a); }
};

// tangent scalar: value part by the same formulas as Num<double>, tangent by the chain rule
template <> struct Num<Dual> {
  using D = Num<double>;
  static __device__ __forceinline__ Dual fma_(Dual a, Dual b, Dual c) {
    return Dual(fma(a.v, b.v, c.v), fma(a.v, b.d, fma(a.d, b.v, c.d)));
  }
  static __device__ __forceinline__ Dual rcp(Dual a) { const double r = D::rcp(a.v); return Dual(r, -a.d * r * r); }
  static __device__ __forceinline__ Dual rsqrt_(Dual a) {
    const double y = D::rsqrt_(a.v);
    return Dual(y, -0.5 * a.d * y * y * y);
  }
  static __device__ __forceinline__ Dual sqrt_(Dual a) {
    const double y = D::rsqrt_(a.v);
    return Dual(a.v * y, 0.5 * a.d * y);
  }
  static __device__ __forceinline__ Dual min_(Dual a, Dual b) { return b.v < a.v ? b : a; }
  static __device__ __forceinline__ Dual max_(Dual a, Dual b) { return b.v > a.v ? b : a; }
  static __device__ __forceinline__ Dual abs_(Dual a) { return a.v < 0.0 ? -a : a; }
};

// warp shuffles / finiteness / (value, tangent) construction, generic over the scalar type
template <class T> __device__ __forceinline__ T shfl(unsigned m, T a, int src) { return __shfl_sync(m, a, src); }
__device__ __forceinline__ Dual shfl(unsigned m, Dual a, int src) {
  return Dual(__shfl_sync(m, a.v, src), __shfl_sync(m, a.d, src));
}
template <class T> __device__ __forceinline__ T shfl_xor(unsigned m, T a, int lm) { return __shfl_xor_sync(m, a, lm); }
__device__ __forceinline__ Dual shfl_xor(unsigned m, Dual a, int lm) {
  return Dual(__shfl_xor_sync(m, a.v, lm), __shfl_xor_sync(m, a.d, lm));
}
template <class T> __device__ __forceinline__ bool finite_(T a) { return isfinite(a); }
__device__ __forceinline__ bool finite_(Dual a) { return isfinite(a.v) && isfinite(a.d); }
template <class T> __device__ __forceinline__ T with_tangent(double v, double) { return T(v); }
template <> __device__ __forceinline__ Dual with_tangent<Dual>(double v, double d) { return Dual(v, d); }

// gas / transport constants handed to every kernel
template <class T>
struct Gas {
  T gamma, gm1, inv_gm1, Rgas, inv_Rgas;
  T mu_ref, inv_T_ref, S, TrefS;  // TrefS = T_ref + S
  T lam_fac;                      // lambda = mu * lam_fac, lam_fac = cp/Pr = gamma R/((gamma-1) Pr)
  T Pr;
  int sutherland, viscous;
  T g[3];
};

// Eq. 2: conservative -> (rho,u,v,w,p,T)
template <class T>
__device__ __forceinline__ void cons_to_prim(const Gas<T>& gas, T r, T mx, T my, T mz, T E, T W[6]) {
  T ri = Num<T>::rcp(r);
  T u = mx * ri, v = my * ri, w = mz * ri;
  T p = gas.gm1 * (E - T(0.5) * (mx * u + my * v + mz * w));
  W[0] = r; W[1] = u; W[2] = v; W[3] = w; W[4] = p;
  W[5] = p * ri * gas.inv_Rgas;
}

// Sutherland: mu = mu_ref r sqrt(r) (T_ref+S)/(T+S), r = T/T_ref
template <class T>
__device__ __forceinline__ T viscosity(const Gas<T>& gas, T Tf) {
  if (!gas.sutherland) return gas.mu_ref;
  T r = Tf * gas.inv_T_ref;
  return gas.mu_ref * (r * Num<T>::sqrt_(r)) * gas.TrefS * Num<T>::rcp(Tf + gas.S);
}

// WENO5-JS, per cell: from the five cells (a,b,c,d,e) = v_{i-2..i+2} form
//   vm = W^-_{i+1/2}: the left-biased value at face i+1/2  = weno(a,b,c,d,e) of the definition,
//   vp = W^+_{i-1/2}: the right-biased value at face i-1/2 = weno(e,d,c,b,a).
// Both use the same smoothness indicators beta_0(a,b,c), beta_1(b,c,d), beta_2(c,d,e): the
// mirrored stencil swaps beta_0 <-> beta_2 and the linear weights (1,6,3)/10 <-> (3,6,1)/10.
// Difference form: v = p1 + [w0 (p0-p1) + w2 (p2-p1)] / sum, with second differences A_k,
//   vm: p0-p1 = (A0-A1)/3, p2-p1 = (A1-A2)/6;   vp: p0'-p1' = -(A1-A2)/3, p2'-p1' = -(A0-A1)/6,
// weights as products of the other two e_k = (beta_k+eps)^2 (one reciprocal per value).
// Indicators are carried as 4*beta (eps scaled likewise), which leaves the weights unchanged.
template <class T>
__device__ __forceinline__ void weno5_cell(T a, T b, T c, T d, T e, T& vm, T& vp) {
  using N = Num<T>;
  const T eps4 = T(4e-6), c133 = T(13.0 / 3.0), sixth = T(1.0 / 6.0);
  const T c30 = T(1.0 / 30.0), c20 = T(1.0 / 20.0);
  T A0 = N::fma_(T(-2), b, a) + c, A1 = N::fma_(T(-2), c, b) + d, A2 = N::fma_(T(-2), d, c) + e;
  T b0 = N::fma_(T(3), c, N::fma_(T(-4), b, a)), b1 = b - d, b2 = N::fma_(T(3), c, N::fma_(T(-4), d, e));
  T e0 = N::fma_(c133 * A0, A0, N::fma_(b0, b0, eps4));
  T e1 = N::fma_(c133 * A1, A1, N::fma_(b1, b1, eps4));
  T e2 = N::fma_(c133 * A2, A2, N::fma_(b2, b2, eps4));
  e0 *= e0; e1 *= e1; e2 *= e2;
  T E12 = e1 * e2, E02 = e0 * e2, E01 = e0 * e1;
  T t1 = E12 * (A0 - A1), t2 = E01 * (A1 - A2);
  T mid = T(0.6) * E02;
  {  // face i+1/2: weights (0.1 E12, 0.6 E02, 0.3 E01)
    T den = N::fma_(T(0.3), E01, N::fma_(T(0.1), E12, mid));
    T num = N::fma_(c30, t1, c20 * t2);
    T p1 = sixth * N::fma_(T(5), c, N::fma_(T(2), d, -b));
    vm = N::fma_(num, N::rcp(den), p1);
  }
  {  // face i-1/2: weights (0.3 E12, 0.6 E02, 0.1 E01)
    T den = N::fma_(T(0.1), E01, N::fma_(T(0.3), E12, mid));
    T num = N::fma_(c20, t1, c30 * t2);
    T p1 = sixth * N::fma_(T(5), c, N::fma_(T(2), b, -d));
    vp = N::fma_(-num, N::rcp(den), p1);
  }
}

// HLLC flux in the rotated frame: states (rho, un, ut1, ut2, p) -> F = [mass, n, t1, t2, energy]
template <class T>
__device__ __forceinline__ void hllc_rot(const Gas<T>& gas, const T L[5], const T R[5], T F[5]) {
  using N = Num<T>;
  T tL = N::rsqrt_(L[0]), tR = N::rsqrt_(R[0]);        // 1/sqrt(rho)
  T sL = L[0] * tL, sR = R[0] * tR;                      // sqrt(rho)
  T riL = tL * tL, riR = tR * tR;                        // 1/rho
  T cL = N::sqrt_(gas.gamma * L[4]) * tL, cR = N::sqrt_(gas.gamma * R[4]) * tR;
  T qL = L[1] * L[1] + L[2] * L[2] + L[3] * L[3], qR = R[1] * R[1] + R[2] * R[2] + R[3] * R[3];
  T EL = L[4] * gas.inv_gm1 + T(0.5) * L[0] * qL, ER = R[4] * gas.inv_gm1 + T(0.5) * R[0] * qR;
  T HL = (EL + L[4]) * riL, HR = (ER + R[4]) * riR;
  T rs = N::rcp(sL + sR);
  T wL = sL * rs, wR = sR * rs;
  T un = wL * L[1] + wR * R[1], u1 = wL * L[2] + wR * R[2], u2 = wL * L[3] + wR * R[3];
  T Ht = wL * HL + wR * HR;
  T ct = N::sqrt_(gas.gm1 * (Ht - T(0.5) * (un * un + u1 * u1 + u2 * u2)));
  T SL = N::min_(L[1] - cL, un - ct), SR = N::max_(R[1] + cR, un + ct);
  T mL = L[0] * (SL - L[1]), mR = R[0] * (SR - R[1]);
  T Ss = (R[4] - L[4] + L[1] * mL - R[1] * mR) * N::rcp(mL - mR);
  // side selected by sign(S*)  (S* == 0: both star fluxes are mathematically equal)
  bool left = Ss >= T(0);
  T rho = left ? L[0] : R[0], vn = left ? L[1] : R[1], v1 = left ? L[2] : R[2], v2 = left ? L[3] : R[3];
  T p = left ? L[4] : R[4], E = left ? EL : ER, SK = left ? SL : SR, m = left ? mL : mR;
  T ri = left ? riL : riR;
  T Sc = left ? N::min_(SL, T(0)) : N::max_(SR, T(0));  // min(S_L,0) / max(S_R,0)
  T mn = rho * vn;
  T F0 = mn, F1 = mn * vn + p, F2 = mn * v1, F3 = mn * v2, F4 = vn * (E + p);
  T dinv = N::rcp(SK - Ss);
  T fac = m * dinv;
  T dS = Ss - vn;
  T Es = fac * (E * ri + dS * Ss) + dS * p * dinv;       // fac*(E/rho + dS*(S* + p/m))
  F[0] = F0 + Sc * (fac - rho);
  F[1] = F1 + Sc * (fac * Ss - mn);
  F[2] = F2 + Sc * (fac * v1 - rho * v1);
  F[3] = F3 + Sc * (fac * v2 - rho * v2);
  F[4] = F4 + Sc * (Es - E);
}

// Dissipative flux (Eq. 4-5, rotated frame) of the face between cells -1 | 0 along DIR, subtracted
// from Fr = [mass, n, t1, t2, energy].
//   w(m, q): primitive q in {rho,u,v,w,p,T} of the cell at offset m in -2..1 along DIR
//   g(m, c): transverse centre derivatives at offset m in -2..1:
//            c = 0: d_t1 u_n, 1: d_t1 u_t1, 2: d_t2 u_n, 3: d_t2 u_t2
//   i24Xf: 1/(24 X_xi^f) of this face.   (n,t1,t2) = (DIR, DIR+1, DIR+2) mod 3.
template <class T, int DIR, class WAcc, class GAcc>
__device__ __forceinline__ void viscous_sub(const Gas<T>& gas, const WAcc& w, const GAcc& g, T i24Xf, T Fr[5]) {
  constexpr int n = DIR, t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  T dn[4], fv[4];  // normal derivative and face value of u_n, u_t1, u_t2, T
  constexpr int qv[4] = {1 + n, 1 + t1, 1 + t2, 5};
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    T m1 = w(-2, qv[c]), c0 = w(-1, qv[c]), p1 = w(0, qv[c]), p2 = w(1, qv[c]);
    dn[c] = (T(27) * (p1 - c0) - (p2 - m1)) * i24Xf;
    fv[c] = (T(9) * (c0 + p1) - (m1 + p2)) * T(1.0 / 16.0);
  }
  T gt[4];
#pragma unroll
  for (int c = 0; c < 4; ++c)
    gt[c] = (T(9) * (g(-1, c) + g(0, c)) - (g(-2, c) + g(1, c))) * T(1.0 / 16.0);
  T mu = viscosity<T>(gas, fv[3]);
  T div = dn[0] + gt[1] + gt[3];
  T tnn = mu * (T(2) * dn[0] - T(2.0 / 3.0) * div);
  T tn1 = mu * (gt[0] + dn[1]);
  T tn2 = mu * (gt[2] + dn[2]);
  Fr[1] -= tnn; Fr[2] -= tn1; Fr[3] -= tn2;
  Fr[4] -= fv[0] * tnn + fv[1] * tn1 + fv[2] * tn2 + mu * gas.lam_fac * dn[3];
}

// Rotated-frame component order of direction DIR: slot c of (rho, u_n, u_t1, u_t2, p) is
// primitive / conservative index rot_q<DIR>(c).
template <int DIR>
__device__ __forceinline__ constexpr int rot_q(int c) {
  return c == 0 ? 0 : (c == 4 ? 4 : 1 + (DIR + c - 1) % 3);
}

// Per-cell WENO of the five primitives of the cell at offset 0 (window -2..2 through w), in
// rotated order: Wm = W^-_{+1/2}, Wp = W^+_{-1/2}.
template <class T, int DIR, class WAcc>
__device__ __forceinline__ void weno_cell_states(const WAcc& w, T Wm[5], T Wp[5]) {
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    const int q = rot_q<DIR>(c);
    weno5_cell<T>(w(-2, q), w(-1, q), w(0, q), w(1, q), w(2, q), Wm[c], Wp[c]);
  }
}

// Total face flux F = F^c - F^d (Eq. 6) of the face between cells -1 | 0 from its rotated
// left / right states; un-rotated into (rho, rho u, rho v, rho w, E) slots.
template <class T, int DIR, bool VISC, class WAcc, class GAcc>
__device__ __forceinline__ void face_flux(const Gas<T>& gas, const T WL[5], const T WR[5], const WAcc& w,
                                          const GAcc& g, T i24Xf, T F[5]) {
  T Fr[5];
  hllc_rot<T>(gas, WL, WR, Fr);
  if (VISC) viscous_sub<T, DIR>(gas, w, g, i24Xf, Fr);
#pragma unroll
  for (int c = 0; c < 5; ++c) F[rot_q<DIR>(c)] = Fr[c];
}

}  // namespace jf
