// jf_pc.cuh — producer / consumer form of the marching (y / z) sweeps (fp64, viscous, fourth-order flux).
//
// A march step of sweep_yz_kernel is two phases of different character: the per-cell WENO (235 FP64 instructions in
// five independent chains, small state) and the face flux with the update (HLLC's long dependent chain, the loads
// and stores, the carried flux).  Here the two phases of one column run in TWO warps: warps 0-3 of a block are
// producers (window loads, cons -> prim, WENO), warps 4-7 consumers (HLLC + dissipative flux, divergence, source,
// RK stage), paired 1:1 over the same 32 columns and the same SM sub-partition (warp w and w + 4), with different
// register budgets (setmaxnreg per warp group: JF_PC_SETMAXNREG; off, because both roles compile spill-free inside the 128
// registers two blocks of 256 threads leave, and ptxas does not spend a larger budget it is offered on the consumer).  Per step the producer hands W^-_{c+1/2}, W^+_{c-1/2} to the consumer
// through 80 bytes of shared memory per column; the window ring (six slots, so that the producer can refill the
// oldest cell while the consumer still reads the four cells its face needs) is shared by the pair.  Two named
// barriers per pair (64 threads each): `full` (producer arrives, consumer waits) and `empty` (consumer arrives,
// producer waits): the producer's WENO of cell c + 1 overlaps the consumer's flux of face c - 1/2.
//   Shared memory: (6 x 5 + 5) x 16 B = 560 B per column, 70 KB per block of 128 columns, two blocks per SM: the
//   same 140-150 KB the plain kernel uses (the L1 it leaves matters: DESIGN.md section 6), 4 warps per
//   sub-partition instead of 3, 256 instead of 384 columns in flight per SM.
// Same device functions as sweep_yz_kernel (the compiler contracts a few operations differently: the two agree to 1e-15).
// MEASURED AND NOT ADOPTED (tgv256 fp64, ms per step, plain | producer/consumer): y 1.96 | 2.37, z + RK 2.22 | 2.53 — 20 % slower:
// a third fewer columns in flight, a single-buffered hand-over (only WENO(c+1) overlaps flux(c)), 20 extra shared-memory
// accesses and two barriers per step cost more than the fourth warp per sub-partition returns.  Selectable with JF_YZ_PC=1
// (fp64, viscous, fourth-order flux); the default stays sweep_yz_kernel.  profiles/r2_experiments.md.
#pragma once
#include "jf_kernels.cuh"

namespace jf {

__device__ __forceinline__ void nb_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void nb_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

#ifndef JF_PC_PROD_REGS
#define JF_PC_PROD_REGS 104
#endif
#ifndef JF_PC_CONS_REGS
#define JF_PC_CONS_REGS 152
#endif
constexpr int PC_COLS = 128, PC_RING = 6, PC_NP = 5;
constexpr size_t pc_smem_bytes() { return (size_t)(PC_RING * PC_NP + 5) * PC_COLS * sizeof(Pair2<double>); }

template <int DIR, int MODE>
__global__ void __launch_bounds__(256, 2)
sweep_yz_pc_kernel(Params<double> P, const double* __restrict__ U, const double* __restrict__ G, double* R, RKArgs<double> rk,
                   int L) {
  using T = double;
  using P2 = Pair2<T>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NT = PC_COLS, NP = PC_NP, RING = PC_RING, LO = 3;   // slots hold cells c-3 .. c+2
  constexpr int OTH = (DIR == 1) ? 2 : 1;
  const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int role = wid >> 2, pw = wid & 3;            // role 0: producer, 1: consumer; pair index
  const int colid = pw * 32 + lane;                   // column of the block (shared by the two roles)
  const int ix0 = blockIdx.x * 32 + lane, io0 = blockIdx.y * 4 + pw;
  // no thread leaves early (named barriers, setmaxnreg): out-of-range columns work on a clamped column and do not store
  const bool valid = ix0 < P.n[0] && io0 < P.n[OTH];
  const int ix = min(ix0, P.n[0] - 1), io = min(io0, P.n[OTH] - 1);
  const int N = P.n[DIR];
  const unsigned sm = (unsigned)((DIR == 1) ? P.sy : P.sz), so = (unsigned)((DIR == 1) ? P.sz : P.sy);
  const unsigned col = (unsigned)(io + NH) * so + (unsigned)(ix + NH);
  const int c0 = blockIdx.z * L, c1 = min(c0 + L, N);
  const Gas<T> gas = P.gas;
  constexpr int n = DIR, t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  P2* ring = reinterpret_cast<P2*>(smem_raw) + colid;                        // [RING][NP][NT]
  P2* xch = reinterpret_cast<P2*>(smem_raw) + (size_t)RING * NP * NT + colid;   // [5][NT]: (W^-_q, W^+_q)
  const int b_full = 1 + 2 * pw, b_empty = 2 + 2 * pw;

  if (role == 0) {
    // ------------------------------------------------------------ producer: window, WENO
#ifdef JF_PC_SETMAXNREG
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(JF_PC_PROD_REGS));
#endif
    const T* gsrc[3] = {G + (long long)(3 * t1 + n) * P.vol, G + (long long)(3 * t2 + n) * P.vol, G + (long long)(4 * n) * P.vol};
    auto put = [&](int slot, const T raw[5], const T gn[3]) {
      T W[6];
      cons_to_prim<T>(gas, raw[0], raw[1], raw[2], raw[3], raw[4], W);
      P2* dst = ring + slot * (NP * NT);
      dst[0] = P2{W[0], W[1]};
      dst[NT] = P2{W[2], W[3]};
      dst[2 * NT] = P2{W[4], W[5]};
      dst[3 * NT] = P2{gn[0], gn[1]};
      dst[4 * NT].a = gn[2];
    };
    T raw[5], gn[3];
    {
      T raws[5][5], gns[5][3];
#pragma unroll
      for (int s = 0; s < 5; ++s) {
        const unsigned o = col + (unsigned)(c0 + s) * sm;
#pragma unroll
        for (int q = 0; q < 5; ++q) raws[s][q] = (U + q * P.vol)[o];
#pragma unroll
        for (int c = 0; c < 3; ++c) gns[s][c] = gsrc[c][o];
      }
#pragma unroll
      for (int s = 0; s < 5; ++s) put(s + LO - 2, raws[s], gns[s]);
    }
    int s0 = 0;                                // slot of cell c-3
    for (int c = c0 - 1; c <= c1; ++c) {
      const int pc = c + NH;
      const bool more = c < c1;
      if (more) {                              // the cell that enters the window at the end of this step
        const unsigned on = col + (unsigned)(pc + 3) * sm;
#pragma unroll
        for (int q = 0; q < 5; ++q) raw[q] = (U + q * P.vol)[on];
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) gn[cc] = gsrc[cc][on];
      }
      int slot[RING];
      {
        int s = s0;
#pragma unroll
        for (int m = 0; m < RING; ++m) { slot[m] = s * (NP * NT); s = (s == RING - 1) ? 0 : s + 1; }
      }
      auto w = [&](int m, int q) -> T {
        const P2 v = ring[slot[m + LO] + (q >> 1) * NT];
        return (q & 1) ? v.b : v.a;
      };
      T Wm[5], Wp[5];
      weno_cell_states<T, DIR>(w, Wm, Wp);
      nb_sync(b_empty, 64);                    // the consumer is done with the exchange words and with cell c-3
#pragma unroll
      for (int q = 0; q < 5; ++q) xch[q * NT] = P2{Wm[q], Wp[q]};
      if (more) put(s0, raw, gn);              // cell c+3 replaces cell c-3
      __threadfence_block();
      nb_arrive(b_full, 64);
      s0 = (s0 == RING - 1) ? 0 : s0 + 1;
    }
  } else {
    // ------------------------------------------------------------ consumer: face flux, divergence, source, RK stage
#ifdef JF_PC_SETMAXNREG
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(JF_PC_CONS_REGS));
#endif
    T WmPrev[5], Fprev[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) { WmPrev[q] = T(1); Fprev[q] = T(0); }
    int s0 = 0;
    T xf_n = P.i24Xf[DIR][c0 - 1 + NH - 1], idl_n = P.inv_dl[DIR][c0 - 1 + NH - 1];
    nb_arrive(b_empty, 64);                    // prime: the exchange words are free
    for (int c = c0 - 1; c <= c1; ++c) {
      const int pc = c + NH;
      const T xf_c = xf_n, idl_c = idl_n;      // 1/(24 X_xi^f) of face c-1/2, 1/Delta of cell c-1
      xf_n = P.i24Xf[DIR][pc];
      idl_n = P.inv_dl[DIR][pc];
      const bool upd = c > c0;                 // cell c-1 is in [c0, c1): update it
      const unsigned o = col + (unsigned)(pc - 1) * sm;
      T Rold[5], un[5];
      if (upd) {                               // in flight while this warp waits for the producer
#pragma unroll
        for (int q = 0; q < 5; ++q) Rold[q] = (R + q * P.vol)[o];
        if (MODE == 2) {
#pragma unroll
          for (int q = 0; q < 5; ++q) un[q] = (rk.Un + q * P.vol)[o];
        }
      }
      int slot[RING];
      {
        int s = s0;
#pragma unroll
        for (int m = 0; m < RING; ++m) { slot[m] = s * (NP * NT); s = (s == RING - 1) ? 0 : s + 1; }
      }
      auto w = [&](int m, int q) -> T {
        const P2 v = ring[slot[m + LO] + (q >> 1) * NT];
        return (q & 1) ? v.b : v.a;
      };
      auto g = [&](int m, int cc) -> T {
        const P2 v = ring[slot[m + LO] + (3 + (cc >> 1)) * NT];
        return (cc & 1) ? v.b : v.a;
      };
      nb_sync(b_full, 64);                     // W^-(c), W^+(c) and the window up to cell c+2 are in place
      T Wm[5], Wp[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) { const P2 v = xch[q * NT]; Wm[q] = v.a; Wp[q] = v.b; }
      if (c >= c0) {                           // face c-1/2
        T F[5];
        face_flux<T, DIR, true, 4>(gas, WmPrev, Wp, w, g, xf_c, F);
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
            T us[5];
#pragma unroll
            for (int q = 0; q < 5; ++q) us[q] = (U + q * P.vol)[o];
            const T dtv = rk.dt_dev ? T(*rk.dt_dev) : rk.dt;
            if (valid) {
#pragma unroll
              for (int q = 0; q < 5; ++q) (rk.Uout + q * P.vol)[o] = rk.a * un[q] + rk.b * (us[q] + dtv * Rv[q]);
            }
          } else if (valid) {
#pragma unroll
            for (int q = 0; q < 5; ++q) (R + q * P.vol)[o] = Rv[q];
          }
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) Fprev[q] = F[q];
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) WmPrev[q] = Wm[q];
      if (c < c1) nb_arrive(b_empty, 64);      // done with the exchange words and with cell c-3 of the next step
      s0 = (s0 == RING - 1) ? 0 : s0 + 1;
    }
  }
}

}  // namespace jf
