// jf_tma.cuh — TMA (cp.async.bulk.tensor) + mbarrier primitives for sm_100a, and the TMA-staged kernels.
//
// north_star asks for tiles staged in shared memory via TMA.  The sweeps hold their windows per thread and are
// bound by the FP64 pipe and by shared-memory capacity, so TMA is used where a kernel is a
// pure tile mover: gradient_tma_kernel, the a5 centre-derivative pass.  One elected thread issues one 4-D box copy
// per (x,y) plane of the block's tile (all four variables it needs, halo rim included, out-of-range cells
// zero-filled by the hardware) into a ring of NS planes, two planes ahead of the arithmetic; the other threads
// never compute a global load address.
#pragma once
#include <cstdint>
#include <cuda.h>
#include "jf_kernels.cuh"

namespace jf {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
// generic-proxy accesses to shared memory made visible to / ordered before the async proxy (TMA)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// 4-D box global -> shared, completion counted in bytes on `bar`
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

// ------------------------------------------------------------------ a5 (part) centre gradients, TMA-staged
// Same outputs as gradient_kernel (G[3*axis+comp] = D^c_axis u_comp off the diagonal, the diagonal slots hold the
// sums of the other two diagonal derivatives; same arithmetic, same instruction sequences per value: the two
// kernels agree bit for bit).  Block = GM_TX x GM_TY threads owning that tile of the (x,y) plane, marching along z
// over [k0, k1).  Plane p of the tile with its 2-cell rim, variables rho, rho u, rho v, rho w, arrives by ONE TMA box
// {GM_SX, GM_SY, 1, 4} in slot (p - pstart) % NS.  Per plane: wait for the box; convert it in place to (u,v,w) (each
// cell once, 1.7 cells per thread); __syncthreads; the elected thread re-arms the slot the previous plane used and
// issues the box of plane p + NS - 1; every thread forms the x / y derivatives of its cell from the shared plane and
// the z derivative of the plane two steps back from a five-deep register queue of its own cell.
#ifndef JF_GT_NS
#define JF_GT_NS 3
#endif
constexpr int GT_NS = JF_GT_NS;
template <class T>
struct GradTmaSmem {
  alignas(128) T raw[GT_NS][4][GM_SY][GM_SX];
  T sd[2][2][GM_TX * GM_TY];
  alignas(8) uint64_t full[GT_NS];
};

template <class T>
__global__ void __launch_bounds__(GM_TX * GM_TY, 3)
gradient_tma_kernel(Params<T> P, const __grid_constant__ CUtensorMap mapU, T* __restrict__ G, int Lz) {
  extern __shared__ __align__(128) unsigned char smem_tma[];
  GradTmaSmem<T>& S = *reinterpret_cast<GradTmaSmem<T>*>(smem_tma);
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * GM_TX + tx;
  const int x0 = blockIdx.x * GM_TX, y0 = blockIdx.y * GM_TY;
  const int px = x0 + tx, py = y0 + ty;
  const int Px = P.P[0], Py = P.P[1], Pz = P.P[2];
  const int k0 = blockIdx.z * Lz, k1 = min(k0 + Lz, Pz);
  const bool own = px < Px && py < Py;
  const unsigned o_own = (unsigned)py * (unsigned)P.sy + (unsigned)px;
  const unsigned sz = (unsigned)P.sz;
  const bool dx_ok = own && px >= NH && px < P.n[0] + NH, dy_ok = own && py >= NH && py < P.n[1] + NH;
  const T scx = dx_ok ? P.i12Xc[0][px] : T(0), scy = dy_ok ? P.i12Xc[1][py] : T(0);
  const int pstart = max(k0 - 2, 0), pend = min(k1 + 1, Pz - 1);   // planes loaded: [pstart, pend]
  constexpr uint32_t BOX_BYTES = 4u * GM_SY * GM_SX * sizeof(T);
  constexpr int NCELL = GM_SY * GM_SX, NTHR = GM_TX * GM_TY;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < GT_NS; ++s) mbar_init(&S.full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
#pragma unroll
    for (int s = 0; s < GT_NS; ++s)
      if (pstart + s <= pend) {
        mbar_arrive_expect_tx(&S.full[s], BOX_BYTES);
        tma_load_4d(&S.raw[s][0][0][0], &mapU, &S.full[s], x0 - 2, y0 - 2, pstart + s, 0);
      }
  }
  __syncthreads();
  T q[5][3];                                   // (u,v,w) of the own cell at planes p-4 .. p
#pragma unroll
  for (int a = 0; a < 5; ++a) q[a][0] = q[a][1] = q[a][2] = T(0);
  int slot = 0;
  uint32_t parity = 0;
  for (int p = pstart; p <= pend; ++p) {
    mbar_wait(&S.full[slot], parity);
    T* rw = &S.raw[slot][0][0][0];
#pragma unroll
    for (int r = 0; r < (NCELL + NTHR - 1) / NTHR; ++r) {
      const int c = tid + r * NTHR;
      if (c < NCELL) {
        const int cy = c / GM_SX, cx = c - cy * GM_SX;
        const bool in = (unsigned)(x0 - 2 + cx) < (unsigned)Px && (unsigned)(y0 - 2 + cy) < (unsigned)Py;
        const T ri = Num<T>::rcp(in ? rw[c] : T(1));
        rw[NCELL + c] = in ? rw[NCELL + c] * ri : T(0);
        rw[2 * NCELL + c] = in ? rw[2 * NCELL + c] * ri : T(0);
        rw[3 * NCELL + c] = in ? rw[3 * NCELL + c] * ri : T(0);
      }
    }
    __syncthreads();
    // every thread is past the derivative pass of plane p-1: its slot can take plane p-1+NS
    if (tid == 0 && p > pstart && p - 1 + GT_NS <= pend) {
      const int ps = (slot == 0) ? GT_NS - 1 : slot - 1;
      fence_proxy_async();
      mbar_arrive_expect_tx(&S.full[ps], BOX_BYTES);
      tma_load_4d(&S.raw[ps][0][0][0], &mapU, &S.full[ps], x0 - 2, y0 - 2, p - 1 + GT_NS, 0);
    }
    const int b = p & 1;
    {
      const T u = S.raw[slot][1][ty + 2][tx + 2], v = S.raw[slot][2][ty + 2][tx + 2], w = S.raw[slot][3][ty + 2][tx + 2];
#pragma unroll
      for (int a = 0; a < 4; ++a) { q[a][0] = q[a + 1][0]; q[a][1] = q[a + 1][1]; q[a][2] = q[a + 1][2]; }
      q[4][0] = u; q[4][1] = v; q[4][2] = w;
    }
    const unsigned op = o_own + (unsigned)p * sz;
    T dxu = T(0), dyv = T(0);                  // the diagonal derivatives of plane p
    if (p >= k0 && p < k1) {
      if (dx_ok) {
        T d[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const T* r = &S.raw[slot][1 + c][ty + 2][tx + 2];
          d[c] = (T(8) * (r[1] - r[-1]) - (r[2] - r[-2])) * scx;
        }
        dxu = d[0];
        st_stream((G + (long long)1 * P.vol) + op, d[1]);
        st_stream((G + (long long)2 * P.vol) + op, d[2]);
      }
      if (dy_ok) {
        T d[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const T* r = &S.raw[slot][1 + c][ty + 2][tx + 2];
          d[c] = (T(8) * (r[GM_SX] - r[-GM_SX]) - (r[2 * GM_SX] - r[-2 * GM_SX])) * scy;
        }
        dyv = d[1];
        st_stream((G + (long long)3 * P.vol) + op, d[0]);
        st_stream((G + (long long)5 * P.vol) + op, d[2]);
      }
      if (dx_ok && dy_ok) st_stream((G + (long long)8 * P.vol) + op, dxu + dyv);
    }
    const int pzc = p - 2;                     // plane whose z derivative is complete now
    if (own && pzc >= k0 && pzc < k1 && pzc >= NH && pzc < P.n[2] + NH && p - 4 >= pstart) {
      const T scz = P.i12Xc[2][pzc];
      T d[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) d[c] = (T(8) * (q[3][c] - q[1][c]) - (q[4][c] - q[0][c])) * scz;
      const unsigned oz = op - 2u * sz;
      st_stream((G + (long long)6 * P.vol) + oz, d[0]);
      st_stream((G + (long long)7 * P.vol) + oz, d[1]);
      if (dy_ok) st_stream((G + (long long)0 * P.vol) + oz, S.sd[b][1][tid] + d[2]);
      if (dx_ok) st_stream((G + (long long)4 * P.vol) + oz, d[2] + S.sd[b][0][tid]);
    }
    S.sd[b][0][tid] = dxu; S.sd[b][1][tid] = dyv;   // slot p & 1 held plane p-2 until here
    if (++slot == GT_NS) { slot = 0; parity ^= 1u; }
  }
}

}  // namespace jf
