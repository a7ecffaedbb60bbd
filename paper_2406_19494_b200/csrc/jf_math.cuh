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

// Double constants whose low mantissa word is not zero cannot be instruction immediates; as literals
// they are re-materialised by pairs of uniform moves inside the loops.  Read from constant memory they
// are direct operands of the FP64 instructions.
enum { K_EPS4 = 0, K_13_3, K_SIXTH, K_THIRD, K_4_3, K_2_3, K_COUNT };
#define JF_KVALS {4e-6, 13.0 / 3.0, 1.0 / 6.0, 1.0 / 3.0, 4.0 / 3.0, 2.0 / 3.0}
static __constant__ double kConstD[K_COUNT] = JF_KVALS;

// ---- packed single precision: two floats per value, arithmetic by the FP32x2 instructions of sm_100 (FFMA2 / FADD2 /
// FMUL2: two results per issue slot).  The fp32 sweeps are issue-slot bound (ncu: 78-85 % of the issue slots busy, FMA
// pipe 52 %), so the marching sweeps can run TWO columns per thread on this type (jf_f32x2.cuh).  Every operation rounds
// exactly as its scalar counterpart: a column's result does not depend on which column it is paired with.
struct __align__(8) F2 {
  float x, y;
  __device__ __forceinline__ F2() {}
  __device__ __forceinline__ F2(float a, float b) : x(a), y(b) {}
  __device__ __forceinline__ F2(float v) : x(v), y(v) {}
  __device__ __forceinline__ F2(double v) : x((float)v), y((float)v) {}
  __device__ __forceinline__ F2(int v) : x((float)v), y((float)v) {}
};
__device__ __forceinline__ unsigned long long f2_pack(F2 a) { unsigned long long r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y)); return r; }
__device__ __forceinline__ F2 f2_unpack(unsigned long long r) { F2 a; asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r)); return a; }
__device__ __forceinline__ F2 f2_fma(F2 a, F2 b, F2 c) {
  unsigned long long r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(f2_pack(a)), "l"(f2_pack(b)), "l"(f2_pack(c)));
  return f2_unpack(r);
}
__device__ __forceinline__ F2 operator+(F2 a, F2 b) { unsigned long long r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(a)), "l"(f2_pack(b))); return f2_unpack(r); }
__device__ __forceinline__ F2 operator-(F2 a, F2 b) { unsigned long long r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(a)), "l"(f2_pack(b))); return f2_unpack(r); }
__device__ __forceinline__ F2 operator*(F2 a, F2 b) { unsigned long long r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(a)), "l"(f2_pack(b))); return f2_unpack(r); }
__device__ __forceinline__ F2 operator-(F2 a) { return F2(-a.x, -a.y); }     // folds into the operand modifiers of FFMA2 / FADD2
__device__ __forceinline__ F2& operator+=(F2& a, F2 b) { a = a + b; return a; }
__device__ __forceinline__ F2& operator-=(F2& a, F2 b) { a = a - b; return a; }
__device__ __forceinline__ F2& operator*=(F2& a, F2 b) { a = a * b; return a; }
struct Mask2 { bool x, y; };

template <class T> struct Num;
template <> struct Num<double> {
  static constexpr bool NARROW = false;      // fp32 exponent range: the WENO weights must not be formed from products of (beta+eps)^2
  using Mask = bool;
  static __device__ __forceinline__ bool ge0(double a) { return a >= 0.0; }
  static __device__ __forceinline__ double sel(bool m, double a, double b) { return m ? a : b; }
#ifdef JF_NO_KCONST
  template <int I> static __device__ __forceinline__ double K() { constexpr double k[K_COUNT] = JF_KVALS; return k[I]; }
#else
  template <int I> static __device__ __forceinline__ double K() { return kConstD[I]; }
#endif
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
  static constexpr bool NARROW = true;
  using Mask = bool;
  static __device__ __forceinline__ bool ge0(float a) { return a >= 0.0f; }
  static __device__ __forceinline__ float sel(bool m, float a, float b) { return m ? a : b; }
  template <int I> static __device__ __forceinline__ float K() { constexpr double k[K_COUNT] = JF_KVALS; return float(k[I]); }
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

template <> struct Num<F2> {
  static constexpr bool NARROW = true;
  using Mask = Mask2;
  template <int I> static __device__ __forceinline__ F2 K() { constexpr double k[K_COUNT] = JF_KVALS; return F2(float(k[I])); }
  static __device__ __forceinline__ F2 fma_(F2 a, F2 b, F2 c) { return f2_fma(a, b, c); }
  static __device__ __forceinline__ F2 rcp(F2 a) {        // as Num<float>::rcp, per component
    F2 x;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(x.x) : "f"(a.x));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(x.y) : "f"(a.y));
    return f2_fma(x, f2_fma(-a, x, F2(1.0f)), x);
  }
  static __device__ __forceinline__ F2 rsqrt_(F2 a) {
    F2 y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y.x) : "f"(a.x));
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y.y) : "f"(a.y));
    F2 e = f2_fma(-(a * y), y, F2(1.0f));
    return f2_fma(y, F2(0.5f) * e, y);
  }
  static __device__ __forceinline__ F2 sqrt_(F2 a) { return a * rsqrt_(a); }
  static __device__ __forceinline__ F2 min_(F2 a, F2 b) { return F2(fminf(a.x, b.x), fminf(a.y, b.y)); }
  static __device__ __forceinline__ F2 max_(F2 a, F2 b) { return F2(fmaxf(a.x, b.x), fmaxf(a.y, b.y)); }
  static __device__ __forceinline__ F2 abs_(F2 a) { return F2(fabsf(a.x), fabsf(a.y)); }
  static __device__ __forceinline__ Mask2 ge0(F2 a) { return Mask2{a.x >= 0.0f, a.y >= 0.0f}; }
  static __device__ __forceinline__ F2 sel(Mask2 m, F2 a, F2 b) { return F2(m.x ? a.x : b.x, m.y ? a.y : b.y); }
};

// tangent scalar: value part by the same formulas as Num<double>, tangent by the chain rule
template <> struct Num<Dual> {
  using D = Num<double>;
  static constexpr bool NARROW = false;
  using Mask = bool;
  static __device__ __forceinline__ bool ge0(Dual a) { return a.v >= 0.0; }
  static __device__ __forceinline__ Dual sel(bool m, Dual a, Dual b) { return m ? a : b; }
  template <int I> static __device__ __forceinline__ Dual K() { return Dual(kConstD[I]); }
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
template <class T> __device__ __forceinline__ T shfl_up(unsigned m, T a, int d) { return __shfl_up_sync(m, a, d); }
__device__ __forceinline__ Dual shfl_up(unsigned m, Dual a, int d) {
  return Dual(__shfl_up_sync(m, a.v, d), __shfl_up_sync(m, a.d, d));
}
template <class T> __device__ __forceinline__ T shfl_xor(unsigned m, T a, int lm) { return __shfl_xor_sync(m, a, lm); }
__device__ __forceinline__ Dual shfl_xor(unsigned m, Dual a, int lm) {
  return Dual(__shfl_xor_sync(m, a.v, lm), __shfl_xor_sync(m, a.d, lm));
}
template <class T> __device__ __forceinline__ bool finite_(T a) { return isfinite(a); }
__device__ __forceinline__ bool finite_(Dual a) { return isfinite(a.v) && isfinite(a.d); }
template <class T> __device__ __forceinline__ T with_tangent(double v, double) { return T(v); }
template <> __device__ __forceinline__ Dual with_tangent<Dual>(double v, double d) { return Dual(v, d); }

// Cache-hinted global accesses.  Every array of a 256^3 step is larger than the L2 and is touched once per
// kernel, except the stage input U_s of the fused z + RK sweep, which a thread reads again four march steps
// after it entered the window: the once-only traffic is marked streaming (evict-first) so that those lines
// survive in the L2 until their second use, which is marked last-use.
__device__ __forceinline__ void st_cs(double* p, double v) { __stcs(p, v); }
__device__ __forceinline__ void st_cs(float* p, float v) { __stcs(p, v); }
__device__ __forceinline__ void st_cs(Dual* p, Dual v) { __stcs(reinterpret_cast<double2*>(p), make_double2(v.v, v.d)); }
#ifdef JF_L2HINTS
__device__ __forceinline__ double ld_stream(const double* p) { return __ldcs(p); }
__device__ __forceinline__ float ld_stream(const float* p) { return __ldcs(p); }
__device__ __forceinline__ Dual ld_stream(const Dual* p) { const double2 v = __ldcs(reinterpret_cast<const double2*>(p)); return Dual(v.x, v.y); }
__device__ __forceinline__ double ld_last(const double* p) { return __ldlu(p); }
__device__ __forceinline__ float ld_last(const float* p) { return __ldlu(p); }
__device__ __forceinline__ Dual ld_last(const Dual* p) { const double2 v = __ldlu(reinterpret_cast<const double2*>(p)); return Dual(v.x, v.y); }
__device__ __forceinline__ void st_stream(double* p, double v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream(float* p, float v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream(Dual* p, Dual v) { __stcs(reinterpret_cast<double2*>(p), make_double2(v.v, v.d)); }
#else
template <class T> __device__ __forceinline__ T ld_stream(const T* p) { return *p; }
template <class T> __device__ __forceinline__ T ld_last(const T* p) { return *p; }
template <class T> __device__ __forceinline__ void st_stream(T* p, T v) { *p = v; }
#endif

// gas / transport constants handed to every kernel
template <class T>
struct Gas {
  T gamma, gm1, inv_gm1, Rgas, inv_Rgas;
  T mu_ref, inv_T_ref, S, TrefS;  // TrefS = T_ref + S
  T lam_fac;                      // lambda = mu * lam_fac, lam_fac = cp/Pr = gamma R/((gamma-1) Pr)
  T Pr;
  int sutherland, viscous;
  int has_g;                      // any non-zero body acceleration (Eq. 1 source)
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
// Everything is built from the first differences D1..D4 = b-a, c-b, d-c, e-d:
//   second differences A0 = D2-D1, A1 = D3-D2, A2 = D4-D3;
//   first-derivative parts of the indicators  a-4b+3c = A0+2 D2,  b-d = -(D2+D3),  3c-4d+e = A2-2 D3;
//   candidates  p1 = c + D3/3 + D2/6,  p0-p1 = (A0-A1)/3,  p2-p1 = (A1-A2)/6  (mirrored: p1' = c - D2/3 - D3/6).
// v = p1 + [w0 (p0-p1) + w2 (p2-p1)] / sum with the weights as products of the other two
// e_k = (beta_k+eps)^2 (one reciprocal per value; fp32 forms 1/e_k instead, see below); with t1 = E12 (A0-A1),
// t2 = E01 (A1-A2):
//   vm = c + D2/6 + [D3 + (t1 + 1.5 t2)/(E12 + 6 E02 + 3 E01)]/3,
//   vp = c - D3/6 - [D2 + (1.5 t1 + t2)/(3 E12 + 6 E02 + E01)]/3.
// Indicators are carried as 4*beta (eps scaled likewise), which leaves the weights unchanged.
// 47 arithmetic instructions per variable and cell.
template <class T>
__device__ __forceinline__ void weno5_cell(T a, T b, T c, T d, T e, T& vm, T& vp) {
  using N = Num<T>;
  const T eps4 = N::template K<K_EPS4>(), c133 = N::template K<K_13_3>(), sixth = N::template K<K_SIXTH>(), third = N::template K<K_THIRD>();
  T D1 = b - a, D2 = c - b, D3 = d - c, D4 = e - d;
  T A0 = D2 - D1, A1 = D3 - D2, A2 = D4 - D3;
  T b0 = N::fma_(T(2), D2, A0), b1 = D2 + D3, b2 = N::fma_(T(-2), D3, A2);
  T e0 = N::fma_(c133 * A0, A0, N::fma_(b0, b0, eps4));
  T e1 = N::fma_(c133 * A1, A1, N::fma_(b1, b1, eps4));
  T e2 = N::fma_(c133 * A2, A2, N::fma_(b2, b2, eps4));
  T E12, E02, E01;
  if (N::NARROW) {
    // fp32: the pair products e_k e_l ~ beta^4 ~ (jump)^8 leave the exponent range once a primitive jumps by ~1e4
    // (SI pressures with a mild shock).  Dividing all three products by e_0 e_1 e_2 leaves the weights unchanged
    // and gives (E12, E02, E01) = (1/e_0, 1/e_1, 1/e_2): three reciprocals, every factor within range.
    const T r0 = N::rcp(e0), r1 = N::rcp(e1), r2 = N::rcp(e2);
    E12 = r0 * r0; E02 = r1 * r1; E01 = r2 * r2;
  } else {
    e0 *= e0; e1 *= e1; e2 *= e2;
    E12 = e1 * e2; E02 = e0 * e2; E01 = e0 * e1;
  }
  T t1 = E12 * (A0 - A1), t2 = E01 * (A1 - A2);
  {  // face i+1/2: weights (0.1 E12, 0.6 E02, 0.3 E01)
    T den = N::fma_(T(3), E01, N::fma_(T(6), E02, E12));
    T num = N::fma_(T(1.5), t2, t1);
    vm = N::fma_(third, N::fma_(num, N::rcp(den), D3), N::fma_(sixth, D2, c));
  }
  {  // face i-1/2: weights (0.3 E12, 0.6 E02, 0.1 E01)
    T den = N::fma_(T(3), E12, N::fma_(T(6), E02, E01));
    T num = N::fma_(T(1.5), t1, t2);
    vp = N::fma_(-third, N::fma_(num, N::rcp(den), D2), N::fma_(-sixth, D3, c));
  }
}

// HLLC flux in the rotated frame: states (rho, un, ut1, ut2, p) -> F = [mass, n, t1, t2, energy].
// H_K = (E_K + p_K)/rho_K is formed as c_K^2/(gamma-1) + q_K/2 (the same quantity for an ideal gas), so
// that E is needed on the selected side only; the tangential momentum fluxes of the closed form,
// rho un ut + S (fac ut - rho ut), equal ut times the mass flux.
template <class T>
__device__ __forceinline__ void hllc_rot(const Gas<T>& gas, const T L[5], const T R[5], T F[5]) {
  using N = Num<T>;
  T tL = N::rsqrt_(L[0]), tR = N::rsqrt_(R[0]);        // 1/sqrt(rho)
  T sL = L[0] * tL, sR = R[0] * tR;                      // sqrt(rho)
  T riL = tL * tL, riR = tR * tR;                        // 1/rho
  T aL = gas.gamma * L[4] * riL, aR = gas.gamma * R[4] * riR;   // c^2
  T cL = aL * N::rsqrt_(aL), cR = aR * N::rsqrt_(aR);
  T hL = T(0.5) * (L[1] * L[1] + L[2] * L[2] + L[3] * L[3]), hR = T(0.5) * (R[1] * R[1] + R[2] * R[2] + R[3] * R[3]);
  T HL = N::fma_(aL, gas.inv_gm1, hL), HR = N::fma_(aR, gas.inv_gm1, hR);
  T rs = N::rcp(sL + sR);
  T wL = sL * rs, wR = sR * rs;
  T un = wL * L[1] + wR * R[1], u1 = wL * L[2] + wR * R[2], u2 = wL * L[3] + wR * R[3];
  T Ht = wL * HL + wR * HR;
  T ct = N::sqrt_(gas.gm1 * (Ht - T(0.5) * (un * un + u1 * u1 + u2 * u2)));
  T SL = N::min_(L[1] - cL, un - ct), SR = N::max_(R[1] + cR, un + ct);
  T mL = L[0] * (SL - L[1]), mR = R[0] * (SR - R[1]);
  T Ss = (R[4] - L[4] + L[1] * mL - R[1] * mR) * N::rcp(mL - mR);
  // side selected by sign(S*)  (S* == 0: both star fluxes are mathematically equal)
  const typename N::Mask left = N::ge0(Ss);
  T rho = N::sel(left, L[0], R[0]), vn = N::sel(left, L[1], R[1]), v1 = N::sel(left, L[2], R[2]), v2 = N::sel(left, L[3], R[3]);
  T p = N::sel(left, L[4], R[4]), hq = N::sel(left, hL, hR), SK = N::sel(left, SL, SR), m = N::sel(left, mL, mR);
  T ri = N::sel(left, riL, riR);
  T Sc = N::sel(left, N::min_(SL, T(0)), N::max_(SR, T(0)));  // min(S_L,0) / max(S_R,0)
  T E = N::fma_(rho, hq, p * gas.inv_gm1);
  T mn = rho * vn;
  T dinv = N::rcp(SK - Ss);
  T fac = m * dinv;
  T dS = Ss - vn;
  T Es = fac * (E * ri + dS * Ss) + dS * p * dinv;       // fac*(E/rho + dS*(S* + p/m))
  F[0] = N::fma_(Sc, fac - rho, mn);
  F[1] = N::fma_(Sc, N::fma_(fac, Ss, -mn), N::fma_(mn, vn, p));
  F[2] = v1 * F[0];
  F[3] = v2 * F[0];
  F[4] = N::fma_(Sc, Es - E, vn * (E + p));
}

// Dissipative flux (Eq. 4-5, rotated frame) of the face between cells -1 | 0 along DIR, subtracted
// from Fr = [mass, n, t1, t2, energy].
//   w(m, q): primitive q in {rho,u,v,w,p,T} of the cell at offset m in -2..1 along DIR
//   g(m, c): transverse centre derivatives at offset m in -2..1:
//            c = 0: d_t1 u_n, 1: d_t2 u_n, 2: d_t1 u_t1 + d_t2 u_t2 (tau_nn needs only the sum, and the
//            face interpolation is linear, so the gradient pass stores the sum: 3 arrays per sweep, not 4)
//   i24Xf: 1/(24 X_xi^f) of this face.   (n,t1,t2) = (DIR, DIR+1, DIR+2) mod 3.
template <class T, int DIR, int ORD, class WAcc, class GAcc>
__device__ __forceinline__ void viscous_sub(const Gas<T>& gas, const WAcc& w, const GAcc& g, T i24Xf, T Fr[5]) {
  constexpr int n = DIR, t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  // Unscaled stencil sums: dn = 24 X_xi^f * (normal derivative), fv = 16 * (face value), gt = 16 * (face
  // interpolation of the transverse centre derivative) of u_n, u_t1, u_t2, T; the scale factors are folded
  // into mX = mu/(24 X_xi^f) and mG = mu/16.
  // ORD == 6: the sixth-order members on cells -3..2 about the face,
  // dn = 1920 X_xi^f d_n = 2250 (0 - -1) - 125 (1 - -2) + 9 (2 - -3), fv = 256 I^f = 150 (-1 + 0) - 25 (-2 + 1) + 3 (-3 + 2);
  // the table then holds 1/(1920 X_xi^f) and the interpolation scale is 1/256.
  T dn[4], fv[4];
  constexpr int qv[4] = {1 + n, 1 + t1, 1 + t2, 5};
  constexpr double ISC = ORD == 6 ? 1.0 / 256.0 : 1.0 / 16.0;
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    T m1 = w(-2, qv[c]), c0 = w(-1, qv[c]), p1 = w(0, qv[c]), p2 = w(1, qv[c]);
    if (ORD == 6) {
      T m2 = w(-3, qv[c]), p3 = w(2, qv[c]);
      dn[c] = Num<T>::fma_(T(2250), p1 - c0, Num<T>::fma_(T(-125), p2 - m1, T(9) * (p3 - m2)));
      fv[c] = Num<T>::fma_(T(150), c0 + p1, Num<T>::fma_(T(-25), m1 + p2, T(3) * (m2 + p3)));
    } else {
      dn[c] = Num<T>::fma_(T(27), p1 - c0, m1 - p2);
      fv[c] = Num<T>::fma_(T(9), c0 + p1, -(m1 + p2));
    }
  }
  T gt[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    if (ORD == 6)
      gt[c] = Num<T>::fma_(T(150), g(-1, c) + g(0, c), Num<T>::fma_(T(-25), g(-2, c) + g(1, c), T(3) * (g(-3, c) + g(2, c))));
    else
      gt[c] = Num<T>::fma_(T(9), g(-1, c) + g(0, c), -(g(-2, c) + g(1, c)));
  }
  T mu = gas.sutherland ? viscosity<T>(gas, fv[3] * T(ISC)) : gas.mu_ref;
  T mX = mu * i24Xf, mG = mu * T(ISC);
  // tau_nn = mu (2 d_n u_n - 2/3 div) = mu (4/3 d_n u_n - 2/3 (d_t1 u_t1 + d_t2 u_t2))
  T tnn = Num<T>::fma_(mX * Num<T>::template K<K_4_3>(), dn[0], -(mG * Num<T>::template K<K_2_3>()) * gt[2]);
  T tn1 = Num<T>::fma_(mX, dn[1], mG * gt[0]);
  T tn2 = Num<T>::fma_(mX, dn[2], mG * gt[1]);
  Fr[1] -= tnn; Fr[2] -= tn1; Fr[3] -= tn2;
  T work = Num<T>::fma_(fv[2], tn2, Num<T>::fma_(fv[1], tn1, fv[0] * tnn));
  Fr[4] = Num<T>::fma_(-(mX * gas.lam_fac), dn[3], Num<T>::fma_(T(-ISC), work, Fr[4]));
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
template <class T, int DIR, bool VISC, int ORD = 4, class WAcc, class GAcc>
__device__ __forceinline__ void face_flux(const Gas<T>& gas, const T WL[5], const T WR[5], const WAcc& w,
                                          const GAcc& g, T i24Xf, T F[5]) {
  T Fr[5];
  hllc_rot<T>(gas, WL, WR, Fr);
  if (VISC) viscous_sub<T, DIR, ORD>(gas, w, g, i24Xf, Fr);
#pragma unroll
  for (int c = 0; c < 5; ++c) F[rot_q<DIR>(c)] = Fr[c];
}

}  // namespace jf
