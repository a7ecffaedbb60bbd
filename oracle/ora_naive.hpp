// ora_naive.hpp — second, deliberately naive RHS path of the CPU ORACLE (test infrastructure).
// For every CELL it recomputes its six face fluxes from scratch (no flux sharing), straight
// from the conservative array with explicit index arithmetic, WENO5 in normalised-weight form
// and HLLC as Toro's four explicit cases.  It exists only to pin ora::rhs by redundancy on
// tiny grids (SURVEY §8(c) "brute force on 8^3").  double only.
#pragma once
#include "ora_solver.hpp"

namespace ora_naive {

using ora::Config;
using ora::NH;

struct Cell { double rho, vel[3], p, T; };

inline Cell load_cell(const Config& c, const double* U, int i, int j, int k) {
  size_t Px = c.P[0], Py = c.P[1], Pz = c.P[2], vol = Px * Py * Pz;
  size_t o = ((size_t)(k + NH) * Py + (j + NH)) * Px + (i + NH);
  double r = U[o], mx = U[vol + o], my = U[2 * vol + o], mz = U[3 * vol + o], E = U[4 * vol + o];
  Cell s;
  s.rho = r; s.vel[0] = mx / r; s.vel[1] = my / r; s.vel[2] = mz / r;
  s.p = (c.gamma - 1.0) * (E - 0.5 * (mx * mx + my * my + mz * mz) / r);
  s.T = s.p / (r * c.Rgas);
  return s;
}

inline double weno_js(const double v[5]) {
  double b[3], p[3], w[3], d[3] = {0.1, 0.6, 0.3};
  b[0] = 13.0 / 12.0 * std::pow(v[0] - 2 * v[1] + v[2], 2) + 0.25 * std::pow(v[0] - 4 * v[1] + 3 * v[2], 2);
  b[1] = 13.0 / 12.0 * std::pow(v[1] - 2 * v[2] + v[3], 2) + 0.25 * std::pow(v[1] - v[3], 2);
  b[2] = 13.0 / 12.0 * std::pow(v[2] - 2 * v[3] + v[4], 2) + 0.25 * std::pow(3 * v[2] - 4 * v[3] + v[4], 2);
  p[0] = (2 * v[0] - 7 * v[1] + 11 * v[2]) / 6.0;
  p[1] = (-v[1] + 5 * v[2] + 2 * v[3]) / 6.0;
  p[2] = (2 * v[2] + 5 * v[3] - v[4]) / 6.0;
  double sum = 0;
  for (int k = 0; k < 3; ++k) { w[k] = d[k] / ((b[k] + 1e-6) * (b[k] + 1e-6)); sum += w[k]; }
  double r = 0;
  for (int k = 0; k < 3; ++k) r += (w[k] / sum) * p[k];
  return r;
}

// Toro's HLLC, four cases; states given as (rho, un, ut1, ut2, p); flux in the same frame.
inline void hllc_toro(double gamma, const double L[5], const double Rr[5], double F[5]) {
  auto energy = [&](const double* s) { return s[4] / (gamma - 1) + 0.5 * s[0] * (s[1] * s[1] + s[2] * s[2] + s[3] * s[3]); };
  auto flux = [&](const double* s, double* f) {
    double E = energy(s);
    f[0] = s[0] * s[1]; f[1] = s[0] * s[1] * s[1] + s[4]; f[2] = s[0] * s[1] * s[2];
    f[3] = s[0] * s[1] * s[3]; f[4] = s[1] * (E + s[4]);
  };
  double EL = energy(L), ER = energy(Rr);
  double cL = std::sqrt(gamma * L[4] / L[0]), cR = std::sqrt(gamma * Rr[4] / Rr[0]);
  double HL = (EL + L[4]) / L[0], HR = (ER + Rr[4]) / Rr[0];
  double wl = std::sqrt(L[0]), wr = std::sqrt(Rr[0]);
  double ua = (wl * L[1] + wr * Rr[1]) / (wl + wr), va = (wl * L[2] + wr * Rr[2]) / (wl + wr);
  double wa = (wl * L[3] + wr * Rr[3]) / (wl + wr), Ha = (wl * HL + wr * HR) / (wl + wr);
  double ca = std::sqrt((gamma - 1) * (Ha - 0.5 * (ua * ua + va * va + wa * wa)));
  double SL = std::min(L[1] - cL, ua - ca), SR = std::max(Rr[1] + cR, ua + ca);
  double Ss = (Rr[4] - L[4] + L[0] * L[1] * (SL - L[1]) - Rr[0] * Rr[1] * (SR - Rr[1])) /
              (L[0] * (SL - L[1]) - Rr[0] * (SR - Rr[1]));
  auto star = [&](const double* s, double SK, double E, double* f) {
    double fk[5]; flux(s, fk);
    double fac = s[0] * (SK - s[1]) / (SK - Ss);
    double Us[5] = {fac, fac * Ss, fac * s[2], fac * s[3],
                    fac * (E / s[0] + (Ss - s[1]) * (Ss + s[4] / (s[0] * (SK - s[1]))))};
    double Uk[5] = {s[0], s[0] * s[1], s[0] * s[2], s[0] * s[3], E};
    for (int q = 0; q < 5; ++q) f[q] = fk[q] + SK * (Us[q] - Uk[q]);
  };
  if (SL >= 0) { flux(L, F); return; }
  if (SR <= 0) { flux(Rr, F); return; }
  if (Ss > 0) { star(L, SL, EL, F); return; }
  if (Ss < 0) { star(Rr, SR, ER, F); return; }
  double a[5], b[5]; star(L, SL, EL, a); star(Rr, SR, ER, b);
  for (int q = 0; q < 5; ++q) F[q] = 0.5 * (a[q] + b[q]);
}

// total flux (convective - dissipative) through the face on the high side of cell (i,j,k) along d
inline void face_flux(const Config& c, const double* U, int d, int i, int j, int k, bool inv, bool visc, double F[5]) {
  int n = d, t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  int e[3] = {0, 0, 0}; e[d] = 1;
  for (int q = 0; q < 5; ++q) F[q] = 0;
  if (inv) {
    double sL[5][5], sR[5][5];  // [var][stencil]
    for (int m = 0; m < 5; ++m) {
      Cell a = load_cell(c, U, i + (m - 2) * e[0], j + (m - 2) * e[1], k + (m - 2) * e[2]);
      Cell b = load_cell(c, U, i + (3 - m) * e[0], j + (3 - m) * e[1], k + (3 - m) * e[2]);
      double va[5] = {a.rho, a.vel[n], a.vel[t1], a.vel[t2], a.p};
      double vb[5] = {b.rho, b.vel[n], b.vel[t1], b.vel[t2], b.p};
      for (int q = 0; q < 5; ++q) { sL[q][m] = va[q]; sR[q][m] = vb[q]; }
    }
    double L[5], Rr[5], f[5];
    for (int q = 0; q < 5; ++q) { L[q] = weno_js(sL[q]); Rr[q] = weno_js(sR[q]); }
    hllc_toro(c.gamma, L, Rr, f);
    F[0] += f[0]; F[1 + n] += f[1]; F[1 + t1] += f[2]; F[1 + t2] += f[3]; F[4] += f[4];
  }
  if (visc && c.viscous) {
    // full velocity-gradient tensor G[a][b] = d u_a / d x_b and grad T at the face
    auto cellat = [&](int sn, int s1, int s2) {
      int id[3] = {i, j, k}; id[n] += sn; id[t1] += s1; id[t2] += s2;
      return load_cell(c, U, id[0], id[1], id[2]);
    };
    double Xf = c.Xf[n][(d == 0 ? i : d == 1 ? j : k) + NH];
    int it[3] = {i, j, k};
    double X1 = c.Xc[t1][it[t1] + NH], X2 = c.Xc[t2][it[t2] + NH];
    double G[3][3], gT, uf[3], Tf;
    Cell cm = cellat(-1, 0, 0), c0 = cellat(0, 0, 0), c1 = cellat(1, 0, 0), c2 = cellat(2, 0, 0);
    if (c.visc_order == 6) {
      // sixth order, weights written out: derivative (9, -125, 2250 | 2250, -125, 9)/1920 on the pairs about the
      // face, interpolation (3, -25, 150, 150, -25, 3)/256, centre derivative (-1, 9, -45, 0, 45, -9, 1)/60
      const double wd[6] = {-9.0 / 1920, 125.0 / 1920, -2250.0 / 1920, 2250.0 / 1920, -125.0 / 1920, 9.0 / 1920};
      const double wi[6] = {3.0 / 256, -25.0 / 256, 150.0 / 256, 150.0 / 256, -25.0 / 256, 3.0 / 256};
      const double wc[7] = {-1.0 / 60, 9.0 / 60, -45.0 / 60, 0.0, 45.0 / 60, -9.0 / 60, 1.0 / 60};
      for (int a = 0; a < 3; ++a) { G[a][n] = 0; uf[a] = 0; G[a][t1] = 0; G[a][t2] = 0; }
      gT = 0; Tf = 0;
      for (int m = -2; m <= 3; ++m) {
        Cell cc = cellat(m, 0, 0);
        for (int a = 0; a < 3; ++a) { G[a][n] += wd[m + 2] * cc.vel[a] / Xf; uf[a] += wi[m + 2] * cc.vel[a]; }
        gT += wd[m + 2] * cc.T / Xf; Tf += wi[m + 2] * cc.T;
        for (int a = 0; a < 3; ++a) {
          double g1 = 0, g2 = 0;
          for (int r = -3; r <= 3; ++r) {
            if (r == 0) continue;
            g1 += wc[r + 3] * cellat(m, r, 0).vel[a] / X1;
            g2 += wc[r + 3] * cellat(m, 0, r).vel[a] / X2;
          }
          G[a][t1] += wi[m + 2] * g1; G[a][t2] += wi[m + 2] * g2;
        }
      }
    } else {
    for (int a = 0; a < 3; ++a) {
      G[a][n] = (27 * (c1.vel[a] - c0.vel[a]) - (c2.vel[a] - cm.vel[a])) / (24 * Xf);
      uf[a] = (9 * (c0.vel[a] + c1.vel[a]) - (cm.vel[a] + c2.vel[a])) / 16;
    }
    gT = (27 * (c1.T - c0.T) - (c2.T - cm.T)) / (24 * Xf);
    Tf = (9 * (c0.T + c1.T) - (cm.T + c2.T)) / 16;
    for (int a = 0; a < 3; ++a) {
      double g1[4], g2[4];
      for (int m = -1; m <= 2; ++m) {
        g1[m + 1] = (8 * (cellat(m, 1, 0).vel[a] - cellat(m, -1, 0).vel[a]) - (cellat(m, 2, 0).vel[a] - cellat(m, -2, 0).vel[a])) / (12 * X1);
        g2[m + 1] = (8 * (cellat(m, 0, 1).vel[a] - cellat(m, 0, -1).vel[a]) - (cellat(m, 0, 2).vel[a] - cellat(m, 0, -2).vel[a])) / (12 * X2);
      }
      G[a][t1] = (9 * (g1[1] + g1[2]) - (g1[0] + g1[3])) / 16;
      G[a][t2] = (9 * (g2[1] + g2[2]) - (g2[0] + g2[3])) / 16;
    }
    }
    double mu = c.mu.mu_ref;
    if (c.mu.sutherland) mu = c.mu.mu_ref * std::pow(Tf / c.mu.T_ref, 1.5) * (c.mu.T_ref + c.mu.S) / (Tf + c.mu.S);
    double lam = mu * c.gamma * c.Rgas / (c.gamma - 1) / c.Pr;
    double div = G[0][0] + G[1][1] + G[2][2];
    double tau[3];  // tau_{a n}, Eq. 5
    for (int a = 0; a < 3; ++a) tau[a] = mu * (G[a][n] + G[n][a] - (a == n ? 2.0 / 3.0 * div : 0.0));
    // Eq. 4: F^d = [0, tau_{.n}, sum u_a tau_{a n} - q_n], q = -lambda grad T
    for (int a = 0; a < 3; ++a) F[1 + a] -= tau[a];
    F[4] -= uf[0] * tau[0] + uf[1] * tau[1] + uf[2] * tau[2] + lam * gT;
  }
}

inline void rhs(const Config& c, const double* U, double* R, bool inv, bool visc, bool src) {
  size_t Px = c.P[0], Py = c.P[1], Pz = c.P[2], vol = Px * Py * Pz;
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < c.n[0]; ++i) {
        size_t o = ((size_t)(k + NH) * Py + (j + NH)) * Px + (i + NH);
        double acc[5] = {0, 0, 0, 0, 0};
        int id[3] = {i, j, k};
        for (int d = 0; d < 3; ++d) {
          int e[3] = {0, 0, 0}; e[d] = 1;
          double Fp[5], Fm[5];
          face_flux(c, U, d, i, j, k, inv, visc, Fp);
          face_flux(c, U, d, i - e[0], j - e[1], k - e[2], inv, visc, Fm);
          double dl = c.xf[d][id[d] + 1] - c.xf[d][id[d]];
          for (int q = 0; q < 5; ++q) acc[q] -= (Fp[q] - Fm[q]) / dl;
        }
        if (src) {
          Cell s = load_cell(c, U, i, j, k);
          for (int a = 0; a < 3; ++a) acc[1 + a] += s.rho * c.g[a];
          acc[4] += s.rho * (s.vel[0] * c.g[0] + s.vel[1] * c.g[1] + s.vel[2] * c.g[2]);
        }
        for (int q = 0; q < 5; ++q) R[q * vol + o] = acc[q];
      }
}

}  // namespace ora_naive
