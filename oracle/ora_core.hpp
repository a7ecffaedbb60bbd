// ora_core.hpp — scheme formulas of the CPU ORACLE (test infrastructure, not the product).
// One function per formula of SURVEY.md §8(c) O1, O4, O5, O6 (stencils); written out
// exactly as stated there, no blocking / fusion / reordering.  Templated on the scalar type
// so the same text serves double, float and the flop-counting type.
#pragma once
#include <cmath>
#include <algorithm>

namespace ora {

// ---------------------------------------------------------------- scalar helpers
inline double s_sqrt(double a) { return std::sqrt(a); }
inline float  s_sqrt(float a)  { return std::sqrt(a); }
inline double s_min(double a, double b) { return a < b ? a : b; }
inline float  s_min(float a, float b)   { return a < b ? a : b; }
inline double s_max(double a, double b) { return a > b ? a : b; }
inline float  s_max(float a, float b)   { return a > b ? a : b; }
inline double s_abs(double a) { return std::fabs(a); }
inline float  s_abs(float a)  { return std::fabs(a); }
inline double s_val(double a) { return a; }
inline double s_val(float a)  { return (double)a; }
// Extended precision (x87 long double, 64-bit mantissa): the ARBITER instantiation.  It gives the
// discrete scheme's own result ~2000 times more accurately than double, so that "GPU vs oracle"
// differences at the 1e-10 level can be judged by who is closer to it (tests/test_gpu_parity.py).
inline long double s_sqrt(long double a) { return std::sqrt(a); }
inline long double s_min(long double a, long double b) { return a < b ? a : b; }
inline long double s_max(long double a, long double b) { return a > b ? a : b; }
inline long double s_abs(long double a) { return std::fabs(a); }
inline double s_val(long double a) { return (double)a; }

// Rational constants num/den of the scheme (13/12, 1/6, 1/10, 2/3, eps = 1/10^6, ...).  double, float
// and the counting type take the double-rounded quotient exactly as before this helper existed;
// the arbiter forms the quotient in its own precision (a double-rounded 0.1 would cap it at 1e-17).
template <class R> inline R cst(double num, double den) { return R(num / den); }
template <> inline long double cst<long double>(double num, double den) { return (long double)num / (long double)den; }

// Flop-counting scalar: add/sub/mul/min/max = 1, div = 1, sqrt = 1 (each tallied apart);
// abs / sign / compare / select = 0 (SURVEY §8(d) convention).
struct Cnt {
  double v;
  static inline double n_basic = 0, n_div = 0, n_sqrt = 0;
  Cnt() : v(0) {}
  Cnt(double x) : v(x) {}
  explicit operator double() const { return v; }
};
inline Cnt operator+(Cnt a, Cnt b) { Cnt::n_basic += 1; return Cnt(a.v + b.v); }
inline Cnt operator-(Cnt a, Cnt b) { Cnt::n_basic += 1; return Cnt(a.v - b.v); }
inline Cnt operator*(Cnt a, Cnt b) { Cnt::n_basic += 1; return Cnt(a.v * b.v); }
inline Cnt operator/(Cnt a, Cnt b) { Cnt::n_div += 1; return Cnt(a.v / b.v); }
inline Cnt operator-(Cnt a) { return Cnt(-a.v); }
inline bool operator<(Cnt a, Cnt b) { return a.v < b.v; }
inline bool operator>(Cnt a, Cnt b) { return a.v > b.v; }
inline bool operator<=(Cnt a, Cnt b) { return a.v <= b.v; }
inline bool operator>=(Cnt a, Cnt b) { return a.v >= b.v; }
inline Cnt s_sqrt(Cnt a) { Cnt::n_sqrt += 1; return Cnt(std::sqrt(a.v)); }
inline Cnt s_min(Cnt a, Cnt b) { Cnt::n_basic += 1; return a.v < b.v ? a : b; }
inline Cnt s_max(Cnt a, Cnt b) { Cnt::n_basic += 1; return a.v > b.v ? a : b; }
inline Cnt s_abs(Cnt a) { return Cnt(std::fabs(a.v)); }
inline double s_val(Cnt a) { return a.v; }

// ---------------------------------------------------------------- O1 thermodynamics
// Eq. 2: E = rho*e + 1/2 rho u.u ; ideal gas.
template <class R>
inline void cons_to_prim(R gamma, const R U[5], R W[5]) {
  R rho = U[0];
  R u = U[1] / rho, v = U[2] / rho, w = U[3] / rho;
  R p = (gamma - R(1)) * (U[4] - R(0.5) * rho * (u * u + v * v + w * w));
  W[0] = rho; W[1] = u; W[2] = v; W[3] = w; W[4] = p;
}
template <class R>
inline void prim_to_cons(R gamma, const R W[5], R U[5]) {
  U[0] = W[0]; U[1] = W[0] * W[1]; U[2] = W[0] * W[2]; U[3] = W[0] * W[3];
  U[4] = W[4] / (gamma - R(1)) + R(0.5) * W[0] * (W[1] * W[1] + W[2] * W[2] + W[3] * W[3]);
}
// Sutherland (form = SURVEY O1): mu = mu_ref r sqrt(r) (T_ref+S)/(T+S), r=T/T_ref
template <class R>
inline R viscosity(int sutherland, R mu_ref, R T_ref, R S, R T) {
  if (!sutherland) return mu_ref;
  R r = T / T_ref;
  return mu_ref * (r * s_sqrt(r)) * (T_ref + S) / (T + S);
}

// ---------------------------------------------------------------- O4 WENO5-JS
// Jiang & Shu smoothness indicators, candidate parabolas, nonlinear weights; eps = 1e-6.
// Value at the face between v2 and v3 of the stencil (v0..v4).
template <class R>
inline R weno5(R v0, R v1, R v2, R v3, R v4, R* beta_out = nullptr, R* om_out = nullptr,
               R* p_out = nullptr) {
  const R eps = cst<R>(1, 1e6), c1312 = cst<R>(13, 12), sixth = cst<R>(1, 6);
  R a0 = v0 - R(2) * v1 + v2, b0 = v0 - R(4) * v1 + R(3) * v2;
  R a1 = v1 - R(2) * v2 + v3, b1 = v1 - v3;
  R a2 = v2 - R(2) * v3 + v4, b2 = R(3) * v2 - R(4) * v3 + v4;
  R beta0 = c1312 * (a0 * a0) + R(0.25) * (b0 * b0);
  R beta1 = c1312 * (a1 * a1) + R(0.25) * (b1 * b1);
  R beta2 = c1312 * (a2 * a2) + R(0.25) * (b2 * b2);
  R p0 = sixth * (R(2) * v0 - R(7) * v1 + R(11) * v2);
  R p1 = sixth * (-v1 + R(5) * v2 + R(2) * v3);
  R p2 = sixth * (R(2) * v2 + R(5) * v3 - v4);
  R e0 = beta0 + eps, e1 = beta1 + eps, e2 = beta2 + eps;
  R al0 = cst<R>(1, 10) / (e0 * e0);
  R al1 = cst<R>(6, 10) / (e1 * e1);
  R al2 = cst<R>(3, 10) / (e2 * e2);
  R sum = al0 + al1 + al2;
  if (beta_out) { beta_out[0] = beta0; beta_out[1] = beta1; beta_out[2] = beta2; }
  if (om_out) { om_out[0] = al0 / sum; om_out[1] = al1 / sum; om_out[2] = al2 / sum; }
  if (p_out) { p_out[0] = p0; p_out[1] = p1; p_out[2] = p2; }
  return (al0 * p0 + al1 * p1 + al2 * p2) / sum;
}

// ---------------------------------------------------------------- Eq. 3 physical flux
// Direction d: normal n = d, tangentials t1 = (d+1)%3, t2 = (d+2)%3 (cyclic).
template <class R>
inline void flux_phys(int d, R gamma, const R W[5], R F[5]) {
  int n = d, t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  R rho = W[0], un = W[1 + n], ut1 = W[1 + t1], ut2 = W[1 + t2], p = W[4];
  R E = p / (gamma - R(1)) + R(0.5) * rho * (un * un + ut1 * ut1 + ut2 * ut2);
  F[0] = rho * un;
  F[1 + n] = rho * un * un + p;
  F[1 + t1] = rho * un * ut1;
  F[1 + t2] = rho * un * ut2;
  F[4] = un * (E + p);
}

// ---------------------------------------------------------------- O5 HLLC
// Toro's HLLC with Roe-average (Einfeldt/Batten) wave speeds, branch-free sgn(S*) form.
template <class R>
inline void hllc(int d, R gamma, const R WL[5], const R WR[5], R F[5]) {
  int n = d, t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  R rho[2] = {WL[0], WR[0]};
  R un[2] = {WL[1 + n], WR[1 + n]};
  R ut1[2] = {WL[1 + t1], WR[1 + t1]};
  R ut2[2] = {WL[1 + t2], WR[1 + t2]};
  R p[2] = {WL[4], WR[4]};
  R E[2], c[2], H[2], s[2];
  for (int K = 0; K < 2; ++K) {
    E[K] = p[K] / (gamma - R(1)) +
           R(0.5) * rho[K] * (un[K] * un[K] + ut1[K] * ut1[K] + ut2[K] * ut2[K]);
    c[K] = s_sqrt(gamma * p[K] / rho[K]);
    H[K] = (E[K] + p[K]) / rho[K];
    s[K] = s_sqrt(rho[K]);
  }
  R ssum = s[0] + s[1];
  R un_t = (s[0] * un[0] + s[1] * un[1]) / ssum;
  R ut1_t = (s[0] * ut1[0] + s[1] * ut1[1]) / ssum;
  R ut2_t = (s[0] * ut2[0] + s[1] * ut2[1]) / ssum;
  R H_t = (s[0] * H[0] + s[1] * H[1]) / ssum;
  R c_t = s_sqrt((gamma - R(1)) * (H_t - R(0.5) * (un_t * un_t + ut1_t * ut1_t + ut2_t * ut2_t)));
  R SL = s_min(un[0] - c[0], un_t - c_t);
  R SR = s_max(un[1] + c[1], un_t + c_t);
  R SK[2] = {SL, SR};
  R m[2] = {rho[0] * (SL - un[0]), rho[1] * (SR - un[1])};
  R Sstar = (p[1] - p[0] + un[0] * m[0] - un[1] * m[1]) / (m[0] - m[1]);
  R FK[2][5], UK[2][5], UsK[2][5];
  for (int K = 0; K < 2; ++K) {
    // U_K and F_K in the rotated frame order [rho, n, t1, t2, E]
    UK[K][0] = rho[K]; UK[K][1] = rho[K] * un[K]; UK[K][2] = rho[K] * ut1[K];
    UK[K][3] = rho[K] * ut2[K]; UK[K][4] = E[K];
    FK[K][0] = rho[K] * un[K];
    FK[K][1] = rho[K] * un[K] * un[K] + p[K];
    FK[K][2] = rho[K] * un[K] * ut1[K];
    FK[K][3] = rho[K] * un[K] * ut2[K];
    FK[K][4] = un[K] * (E[K] + p[K]);
    R fac = m[K] / (SK[K] - Sstar);
    UsK[K][0] = fac;
    UsK[K][1] = fac * Sstar;
    UsK[K][2] = fac * ut1[K];
    UsK[K][3] = fac * ut2[K];
    UsK[K][4] = fac * (E[K] / rho[K] + (Sstar - un[K]) * (Sstar + p[K] / m[K]));
  }
  R sg = Sstar > R(0) ? R(1) : (Sstar < R(0) ? R(-1) : R(0));
  R wL = R(0.5) * (R(1) + sg), wR = R(0.5) * (R(1) - sg);
  R SLm = s_min(SL, R(0)), SRp = s_max(SR, R(0));
  R Frot[5];
  for (int q = 0; q < 5; ++q)
    Frot[q] = wL * (FK[0][q] + SLm * (UsK[0][q] - UK[0][q])) +
              wR * (FK[1][q] + SRp * (UsK[1][q] - UK[1][q]));
  F[0] = Frot[0]; F[1 + n] = Frot[1]; F[1 + t1] = Frot[2]; F[1 + t2] = Frot[3]; F[4] = Frot[4];
}

// ---------------------------------------------------------------- O6 central stencils
// Evaluated in difference form so a constant field gives an exactly zero derivative.
template <class R>
inline R d_centre(R m2, R m1, R p1, R p2, R Xc) {  // phi_{i-2}, phi_{i-1}, phi_{i+1}, phi_{i+2}
  return (R(8) * (p1 - m1) - (p2 - m2)) / (R(12) * Xc);
}
template <class R>
inline R d_face(R m1, R c0, R p1, R p2, R Xf) {  // phi_{i-1}, phi_i, phi_{i+1}, phi_{i+2}
  return (R(27) * (p1 - c0) - (p2 - m1)) / (R(24) * Xf);
}
template <class R>
inline R i_face(R m1, R c0, R p1, R p2) {
  return (R(9) * (c0 + p1) - (m1 + p2)) / R(16);
}

// Sixth-order members of the same family (the paper's DNS used "6th-order central" dissipative
// fluxes).  The coefficients are fixed by polynomial exactness on the symmetric 6- / 7-point
// stencils: centre derivative (-1, 9, -45, 0, 45, -9, 1)/60, face derivative from cell values
// (75/64, -25/384, 3/640) on the three symmetric pairs, face interpolation (150, -25, 3)/256; difference form.
template <class R>
inline R d_centre6(R m3, R m2, R m1, R p1, R p2, R p3, R Xc) {  // phi_{i-3..i-1}, phi_{i+1..i+3}
  return (R(45) * (p1 - m1) - R(9) * (p2 - m2) + (p3 - m3)) / (R(60) * Xc);
}
template <class R>
inline R d_face6(R m2, R m1, R c0, R p1, R p2, R p3, R Xf) {  // phi_{i-2} .. phi_{i+3}, face i+1/2
  return (R(2250) * (p1 - c0) - R(125) * (p2 - m1) + R(9) * (p3 - m2)) / (R(1920) * Xf);
}
template <class R>
inline R i_face6(R m2, R m1, R c0, R p1, R p2, R p3) {
  return (R(150) * (c0 + p1) - R(25) * (m1 + p2) + R(3) * (m2 + p3)) / R(256);
}

}  // namespace ora
