// jf_f32x2.cuh — the marching (y / z) sweeps of the fp32 solver, TWO columns per thread on packed FP32x2 arithmetic.
//
// The scalar fp32 sweeps are bound by issue slots (ncu at 256^3: 78-85 % of the issue slots busy, FMA pipe 52 %): the
// FP32 pipe would take twice the arithmetic if the scheduler could issue it.  sm_100 has packed single-precision
// instructions (FFMA2 / FADD2 / FMUL2: two IEEE results per issue slot).  Here a thread marches the two columns
// (ix, io) and (ix, io + 1) — io along the non-marching, non-x axis — with every value held as an F2 (jf_math.cuh):
// the same device functions as the scalar kernel (weno5_cell, hllc_rot, viscous_sub, ...) instantiated on F2, so each
// column's arithmetic is the scalar kernel's formula by formula (the compiler's multiply-add contractions may differ, so
// the two agree to fp32 round-off, not bit for bit).  Selects, min / max and the MUFU seeds stay per component; loads and
// stores are one coalesced warp access per column.
//   The window ring holds F2 values (8 bytes, as a double): 400 B per thread = 50 KB per block of 128 threads / 256
//   columns, 3 blocks per SM (the layout and the budgets of the fp64 kernel).
// Storage type float, state arrays and metric tables as for the scalar fp32 solver.
#pragma once
#include "jf_kernels.cuh"

namespace jf {

__device__ __forceinline__ Gas<F2> gas_pair(const Gas<float>& g) {
  Gas<F2> h;
  h.gamma = F2(g.gamma); h.gm1 = F2(g.gm1); h.inv_gm1 = F2(g.inv_gm1); h.Rgas = F2(g.Rgas); h.inv_Rgas = F2(g.inv_Rgas);
  h.mu_ref = F2(g.mu_ref); h.inv_T_ref = F2(g.inv_T_ref); h.S = F2(g.S); h.TrefS = F2(g.TrefS);
  h.lam_fac = F2(g.lam_fac); h.Pr = F2(g.Pr);
  h.sutherland = g.sutherland; h.viscous = g.viscous; h.has_g = g.has_g;
  h.g[0] = F2(g.g[0]); h.g[1] = F2(g.g[1]); h.g[2] = F2(g.g[2]);
  return h;
}

#ifndef JF_YZ2_MINB
#define JF_YZ2_MINB 3
#endif
template <bool VISC, int ORD>
constexpr size_t yz2_smem_bytes() { return (size_t)yz_ring(ORD) * YZ<VISC>::NP * YZ_TX * YZ_TY * sizeof(Pair2<F2>); }

template <int DIR, bool VISC, int MODE, int ORD>
__global__ void __launch_bounds__(YZ_TX * YZ_TY, JF_YZ2_MINB)
sweep_yz2_kernel(Params<float> P, const float* __restrict__ U, const float* __restrict__ G, float* R, RKArgs<float> rk, int L) {
  using T = F2;
  using P2 = Pair2<T>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int YZ_RING = yz_ring(ORD), LO = YZ_RING - 3;   // slots hold cells c-LO .. c+2
  constexpr int NT = YZ_TX * YZ_TY, NP = YZ<VISC>::NP;
  constexpr int OTH = (DIR == 1) ? 2 : 1;    // the non-marching, non-x axis
  const int tid = threadIdx.y * YZ_TX + threadIdx.x;
  const int ix = blockIdx.x * YZ_TX + threadIdx.x;
  const int ioa = (blockIdx.y * YZ_TY + threadIdx.y) * 2;   // this thread's columns: (ix, ioa) and (ix, ioa + 1)
  const int N = P.n[DIR];
  if (ix >= P.n[0] || ioa >= P.n[OTH]) return;
  const bool vb = ioa + 1 < P.n[OTH];        // odd extent: the last thread's second column repeats its first and is not stored
  const unsigned sm = (unsigned)((DIR == 1) ? P.sy : P.sz), so = (unsigned)((DIR == 1) ? P.sz : P.sy);
  const unsigned cola = (unsigned)(ioa + NH) * so + (unsigned)(ix + NH);
  const unsigned colb = vb ? cola + so : cola;
  const int c0 = blockIdx.z * L, c1 = min(c0 + L, N);
  const Gas<T> gas = gas_pair(P.gas);
  constexpr int n = DIR, t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  const float* gsrc[3] = {G + (long long)(3 * t1 + n) * P.vol, G + (long long)(3 * t2 + n) * P.vol, G + (long long)(4 * n) * P.vol};
#ifdef JF_YZ2_LDCG
  auto ld2 = [&](const float* a, unsigned off) -> T { return T(__ldcg(a + cola + off), __ldcg(a + colb + off)); };
#else
  auto ld2 = [&](const float* a, unsigned off) -> T { return T(a[cola + off], a[colb + off]); };
#endif
  auto st2 = [&](float* a, unsigned off, T v) {
    a[cola + off] = v.x;
    if (vb) a[colb + off] = v.y;
  };
  P2* mine = reinterpret_cast<P2*>(smem_raw) + tid;
  auto put = [&](int slot, const T raw[5], const T gn[3]) {
    T W[6];
    cons_to_prim<T>(gas, raw[0], raw[1], raw[2], raw[3], raw[4], W);
    P2* dst = mine + slot * (NP * NT);
    dst[0] = P2{W[0], W[1]};
    dst[NT] = P2{W[2], W[3]};
    if (VISC) {
      dst[2 * NT] = P2{W[4], W[5]};
      dst[3 * NT] = P2{gn[0], gn[1]};
      dst[4 * NT].a = gn[2];
    } else {
      dst[2 * NT].a = W[4];
    }
  };
  T raw[5], gn[3] = {T(0.0f), T(0.0f), T(0.0f)};
  {
    T raws[5][5], gns[5][3];
#pragma unroll
    for (int s = 0; s < 5; ++s) {
      const unsigned o = (unsigned)(c0 + s) * sm;
#pragma unroll
      for (int q = 0; q < 5; ++q) raws[s][q] = ld2(U + q * P.vol, o);
#pragma unroll
      for (int c = 0; c < 3; ++c) gns[s][c] = VISC ? ld2(gsrc[c], o) : T(0.0f);
    }
#pragma unroll
    for (int s = 0; s < 5; ++s) put(s + LO - 2, raws[s], gns[s]);
  }
  // W^-_{c+1/2} of the previous step travels through the unused tenth word of ring slot q (viscous layout) instead of ten
  // registers: at JF_YZ2_MINB = 4 (128 registers) the kernel then compiles without spills
#ifdef JF_YZ2_XCHG
  constexpr bool XCHG = VISC;
#else
  constexpr bool XCHG = false;
#endif
  auto xw = [&](int q) -> T* { return &(mine + q * (NP * NT) + (NP - 1) * NT)->b; };
  T WmPrev[5], Fprev[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    WmPrev[q] = T(1.0f); Fprev[q] = T(0.0f);
    if (XCHG) *xw(q) = T(1.0f);
  }
  int s0 = 0;                                // slot of cell c-LO
  float xf_n = VISC ? P.i24Xf[DIR][c0 - 1 + NH - 1] : 0.0f, idl_n = P.inv_dl[DIR][c0 - 1 + NH - 1];
  for (int c = c0 - 1; c <= c1; ++c) {
    const int pc = c + NH;
    const T xf_c = T(xf_n), idl_c = T(idl_n);   // 1/(24 X_xi^f) of face c-1/2, 1/Delta of cell c-1: the same for both columns
    xf_n = VISC ? P.i24Xf[DIR][pc] : 0.0f;
    idl_n = P.inv_dl[DIR][pc];
    int slot[YZ_RING];
    {
      int s = s0;
#pragma unroll
      for (int m = 0; m < YZ_RING; ++m) { slot[m] = s * (NP * NT); s = (s == YZ_RING - 1) ? 0 : s + 1; }
    }
    auto w = [&](int m, int q) -> T {
      const P2 v = mine[slot[m + LO] + (q >> 1) * NT];
      return (q & 1) ? v.b : v.a;
    };
    auto g = [&](int m, int cc) -> T {
      const P2 v = mine[slot[m + LO] + (3 + (cc >> 1)) * NT];
      return (cc & 1) ? v.b : v.a;
    };
    T Wm[5], Wp[5];
    weno_cell_states<T, DIR>(w, Wm, Wp);
    if (XCHG) {
#pragma unroll
      for (int q = 0; q < 5; ++q) { T* x = xw(q); WmPrev[q] = *x; *x = Wm[q]; }
    }
    const bool more = c < c1;                // another cell follows: its window needs padded pc+3
    const bool upd = c > c0;                 // cell c-1 is in [c0, c1): update it
    const unsigned o = (unsigned)(pc - 1) * sm;
    T Rold[5], un[5], us[5];
    if (more) {
      const unsigned on = (unsigned)(pc + 3) * sm;
#pragma unroll
      for (int q = 0; q < 5; ++q) raw[q] = ld2(U + q * P.vol, on);
      if (VISC) {
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) gn[cc] = ld2(gsrc[cc], on);
      }
    }
    if (upd) {
#pragma unroll
      for (int q = 0; q < 5; ++q) Rold[q] = ld2(R + q * P.vol, o);
      if (MODE == 2) {
#pragma unroll
        for (int q = 0; q < 5; ++q) un[q] = ld2(rk.Un + q * P.vol, o);
      }
    }
    if (c >= c0) {                           // face c-1/2
      T F[5];
      face_flux<T, DIR, VISC, ORD>(gas, WmPrev, Wp, w, g, xf_c, F);
      if (upd) {
        T Rv[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) Rv[q] = Rold[q] - (F[q] - Fprev[q]) * idl_c;
        if (MODE >= 1 && gas.has_g) {
          T rho = w(-1, 0), u = w(-1, 1), v = w(-1, 2), ww = w(-1, 3);
          Rv[1] += rho * gas.g[0]; Rv[2] += rho * gas.g[1]; Rv[3] += rho * gas.g[2];
          Rv[4] += rho * (u * gas.g[0] + v * gas.g[1] + ww * gas.g[2]);
        }
        if (MODE == 2) {
#pragma unroll
          for (int q = 0; q < 5; ++q) us[q] = ld2(U + q * P.vol, o);
          const T dtv = T(rk.dt_dev ? (float)(*rk.dt_dev) : rk.dt), ra = T(rk.a), rb = T(rk.b);
#pragma unroll
          for (int q = 0; q < 5; ++q) st2(rk.Uout + q * P.vol, o, ra * un[q] + rb * (us[q] + dtv * Rv[q]));
        } else {
#pragma unroll
          for (int q = 0; q < 5; ++q) st2(R + q * P.vol, o, Rv[q]);
        }
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) Fprev[q] = F[q];
    }
    if (!XCHG) {
#pragma unroll
      for (int q = 0; q < 5; ++q) WmPrev[q] = Wm[q];
    }
    if (more) put(s0, raw, gn);              // cell c+3 replaces cell c-LO
    s0 = (s0 == YZ_RING - 1) ? 0 : s0 + 1;
  }
}

}  // namespace jf
