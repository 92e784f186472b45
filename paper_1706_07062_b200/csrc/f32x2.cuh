// f32x2.cuh -- packed pair of floats as an arithmetic type for the templates of ks_geodesic.cuh.
//
// Blackwell (sm_100) has packed FP32x2 instructions (PTX add/mul/fma.f32x2, SASS FADD2/FMUL2/FFMA2): one
// issue slot performs the same IEEE operation on two independent floats held in an aligned register pair.
// The FP32 integrator is bound by issue slots, not by the FP32 pipe, so it runs TWO
// geodesics per thread, one in each half of every register pair: the right-hand side and the RK4 step
// are the very same templates instantiated with T = f32x2, and each geodesic's arithmetic is bit-for-bit
// the arithmetic of the scalar float instantiation (the library is compiled with --fmad=false, every
// fused multiply-add is explicit in the source).
#pragma once
#include <cuda_runtime.h>
#include "ks_geodesic.cuh"

namespace gray2 {

struct f32x2 {
  float2 v;
  __device__ __forceinline__ f32x2() {}
  __device__ __forceinline__ f32x2(float s) : v(make_float2(s, s)) {}
  __device__ __forceinline__ f32x2(double s) : v(make_float2((float)s, (float)s)) {}
  __device__ __forceinline__ f32x2(int s) : v(make_float2((float)s, (float)s)) {}
  __device__ __forceinline__ f32x2(float lo, float hi) : v(make_float2(lo, hi)) {}
  __device__ __forceinline__ explicit f32x2(float2 w) : v(w) {}
};

__device__ __forceinline__ f32x2 operator*(f32x2 a, f32x2 b) { return f32x2(__fmul2_rn(a.v, b.v)); }
__device__ __forceinline__ f32x2 operator+(f32x2 a, f32x2 b) { return f32x2(__fadd2_rn(a.v, b.v)); }
__device__ __forceinline__ f32x2 operator-(f32x2 a) { return f32x2(-a.v.x, -a.v.y); }
__device__ __forceinline__ f32x2 operator-(f32x2 a, f32x2 b) { return f32x2(__fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y))); }
__device__ __forceinline__ f32x2 &operator*=(f32x2 &a, f32x2 b) { a = a * b; return a; }

template <> __device__ __forceinline__ f32x2 fma_<f32x2>(f32x2 a, f32x2 b, f32x2 c) {
  return f32x2(__ffma2_rn(a.v, b.v, c.v));
}

// rsqrt / rcp have no packed form: two MUFU operations.
template <> struct fastmath<f32x2> {
  static __device__ __forceinline__ f32x2 rsqrt(f32x2 x) {
    return f32x2(fastmath<float>::rsqrt(x.v.x), fastmath<float>::rsqrt(x.v.y));
  }
  static __device__ __forceinline__ f32x2 rcp(f32x2 x) {
    return f32x2(fastmath<float>::rcp(x.v.x), fastmath<float>::rcp(x.v.y));
  }
};

// componentwise minimum (declared in bl_geodesic.cuh for the scalar types)
template <typename T> __device__ __forceinline__ T min_(T a, T b);
template <> __device__ __forceinline__ f32x2 min_<f32x2>(f32x2 a, f32x2 b) {
  return f32x2(fminf(a.v.x, b.v.x), fminf(a.v.y, b.v.y));
}

template <int C> __device__ __forceinline__ float half_of(f32x2 a) { return C == 0 ? a.v.x : a.v.y; }
template <int C> __device__ __forceinline__ void set_half(f32x2 &a, float s) {
  if (C == 0) a.v.x = s; else a.v.y = s;
}

// copy half C of every variable of a packed ray (or of its residuals)
template <int C, typename R> __device__ __forceinline__ void copy_half(R &d, const R &s) {
  set_half<C>(d.t, half_of<C>(s.t)); set_half<C>(d.x, half_of<C>(s.x)); set_half<C>(d.y, half_of<C>(s.y));
  set_half<C>(d.z, half_of<C>(s.z)); set_half<C>(d.u0, half_of<C>(s.u0)); set_half<C>(d.u1, half_of<C>(s.u1));
  set_half<C>(d.u2, half_of<C>(s.u2)); set_half<C>(d.u3, half_of<C>(s.u3));
}
template <int C> __device__ __forceinline__ void clear_half(Carry<f32x2> &c) {
  set_half<C>(c.t, 0.0f); set_half<C>(c.x, 0.0f); set_half<C>(c.y, 0.0f); set_half<C>(c.z, 0.0f);
  set_half<C>(c.u0, 0.0f); set_half<C>(c.u1, 0.0f); set_half<C>(c.u2, 0.0f); set_half<C>(c.u3, 0.0f);
}

}  // namespace gray2
