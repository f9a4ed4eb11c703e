// tslb_pair.cuh -- two lattice nodes (x, x+1) processed by one thread.
//
// For fp32 the pair maps onto Blackwell's packed fp32 pipe (FADD2 / FMUL2 / FFMA2 on sm_100a:
// one issue slot, two IEEE-rounded results), which halves the issue pressure of this
// issue-bound stencil.  For fp64 it is two scalar operations.
#pragma once
#include <cuda_runtime.h>

namespace tslb {

template <typename T> struct Pair;

template <> struct __align__(8) Pair<float> {
  float x, y;
  __device__ __forceinline__ Pair() {}
  __device__ __forceinline__ explicit Pair(float s) : x(s), y(s) {}
  __device__ __forceinline__ Pair(float a, float b) : x(a), y(b) {}
};
template <> struct __align__(16) Pair<double> {
  double x, y;
  __device__ __forceinline__ Pair() {}
  __device__ __forceinline__ explicit Pair(double s) : x(s), y(s) {}
  __device__ __forceinline__ Pair(double a, double b) : x(a), y(b) {}
};

typedef Pair<float> F2;
typedef Pair<double> D2;

__device__ __forceinline__ F2 operator+(F2 a, F2 b) {
  float2 r = __fadd2_rn(make_float2(a.x, a.y), make_float2(b.x, b.y));
  return F2(r.x, r.y);
}
__device__ __forceinline__ F2 operator-(F2 a, F2 b) {
  float2 r = __fadd2_rn(make_float2(a.x, a.y), make_float2(-b.x, -b.y));
  return F2(r.x, r.y);
}
__device__ __forceinline__ F2 operator*(F2 a, F2 b) {
  float2 r = __fmul2_rn(make_float2(a.x, a.y), make_float2(b.x, b.y));
  return F2(r.x, r.y);
}
// a*b + c
__device__ __forceinline__ F2 pfma(F2 a, F2 b, F2 c) {
  float2 r = __ffma2_rn(make_float2(a.x, a.y), make_float2(b.x, b.y), make_float2(c.x, c.y));
  return F2(r.x, r.y);
}
// a*s + c with a broadcast scalar
__device__ __forceinline__ F2 pfma(F2 a, float s, F2 c) { return pfma(a, F2(s), c); }
__device__ __forceinline__ F2 operator*(F2 a, float s) { return a * F2(s); }

__device__ __forceinline__ D2 operator+(D2 a, D2 b) { return D2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ D2 operator-(D2 a, D2 b) { return D2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ D2 operator*(D2 a, D2 b) { return D2(a.x * b.x, a.y * b.y); }
__device__ __forceinline__ D2 pfma(D2 a, D2 b, D2 c) { return D2(fma(a.x, b.x, c.x), fma(a.y, b.y, c.y)); }
__device__ __forceinline__ D2 pfma(D2 a, double s, D2 c) { return D2(fma(a.x, s, c.x), fma(a.y, s, c.y)); }
__device__ __forceinline__ D2 operator*(D2 a, double s) { return D2(a.x * s, a.y * s); }

__device__ __forceinline__ F2 pneg(F2 a) { return F2(-a.x, -a.y); }
__device__ __forceinline__ D2 pneg(D2 a) { return D2(-a.x, -a.y); }
__device__ __forceinline__ float pneg(float a) { return -a; }
__device__ __forceinline__ double pneg(double a) { return -a; }
// scalar overloads so the same templates serve the one-node-per-thread kernels
__device__ __forceinline__ float pfma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double pfma(double a, double b, double c) { return fma(a, b, c); }

template <typename T>
__device__ __forceinline__ Pair<T> lds_pair(const T *p) {   // p must be 2*sizeof(T)-aligned
  return *reinterpret_cast<const Pair<T> *>(p);
}
template <typename T>
__device__ __forceinline__ void sts_pair(T *p, Pair<T> v) {
  *reinterpret_cast<Pair<T> *>(p) = v;
}

}  // namespace tslb
