// jf_dual.cuh — forward-mode (tangent) scalar for libjf.
//
// The paper's point is that the Disturbance Wall makes the boundary parameters reachable by
// differentiation ("end-to-end optimization").  Every kernel of libjf is a
// template on its scalar type, so the tangent of the whole hot path with respect to the disturbance
// parameters (A, kappa) is obtained by instantiating the SAME kernels on a dual number
// (value, directional derivative): no separate differentiated code that could drift from the primal.
// Non-smooth points (min / max / sign selections in HLLC, the wall-temperature floor) take the
// derivative of the selected branch; WENO5-JS weights are smooth (eps > 0).
#pragma once
#include <cuda_runtime.h>
#include <cmath>

namespace jf {

struct Dual {
  double v, d;   // value, tangent
  __host__ __device__ Dual() {}
  __host__ __device__ Dual(double v_) : v(v_), d(0.0) {}
  __host__ __device__ Dual(float v_) : v((double)v_), d(0.0) {}
  __host__ __device__ Dual(int v_) : v((double)v_), d(0.0) {}
  __host__ __device__ Dual(unsigned v_) : v((double)v_), d(0.0) {}
  __host__ __device__ Dual(double v_, double d_) : v(v_), d(d_) {}
  __host__ __device__ explicit operator double() const { return v; }
};

__host__ __device__ __forceinline__ Dual operator+(Dual a, Dual b) { return Dual(a.v + b.v, a.d + b.d); }
__host__ __device__ __forceinline__ Dual operator-(Dual a, Dual b) { return Dual(a.v - b.v, a.d - b.d); }
__host__ __device__ __forceinline__ Dual operator-(Dual a) { return Dual(-a.v, -a.d); }
__host__ __device__ __forceinline__ Dual operator*(Dual a, Dual b) { return Dual(a.v * b.v, a.v * b.d + a.d * b.v); }
__host__ __device__ __forceinline__ Dual operator/(Dual a, Dual b) {
  const double q = a.v / b.v;
  return Dual(q, (a.d - q * b.d) / b.v);
}
__host__ __device__ __forceinline__ Dual& operator+=(Dual& a, Dual b) { a = a + b; return a; }
__host__ __device__ __forceinline__ Dual& operator-=(Dual& a, Dual b) { a = a - b; return a; }
__host__ __device__ __forceinline__ Dual& operator*=(Dual& a, Dual b) { a = a * b; return a; }
__host__ __device__ __forceinline__ bool operator<(Dual a, Dual b) { return a.v < b.v; }
__host__ __device__ __forceinline__ bool operator>(Dual a, Dual b) { return a.v > b.v; }
__host__ __device__ __forceinline__ bool operator<=(Dual a, Dual b) { return a.v <= b.v; }
__host__ __device__ __forceinline__ bool operator>=(Dual a, Dual b) { return a.v >= b.v; }
__host__ __device__ __forceinline__ bool operator==(Dual a, Dual b) { return a.v == b.v; }

}  // namespace jf
