// bl_geodesic.cuh -- the geodesic right-hand side in Boyer-Lindquist coordinates (eq. 1), the
// second coordinate system of the paper's benchmark (Table 2 "BL" rows), behind
// the same RK4 stepper and the same persistent kernel as the Kerr-Schild form.
//
// The paper prints the BL metric only.  Right-hand side used here:
// eq. (1) is   ds^2 = -dt^2 + Sigma (dr^2/Delta + dtheta^2) + P sin^2 dphi^2 + A (dt - a sin^2 dphi)^2 ,
//   Sigma = r^2 + a^2 cos^2,  Delta = r^2 - 2r + a^2,  P = r^2 + a^2,  A = 2r/Sigma,
// and the Euler-Lagrange equations of L = (1/2) g_ab xdot^a xdot^b give, with (t', r', th', ph') = xdot,
//   omega = t' - a sin^2 ph' ,  W = A omega ,  B = 2 a^2 sin cos / Sigma   (d_theta Sigma = -B Sigma)
//   A_r = 2/Sigma - A^2 ,  A_theta = A B ,  A' = A_r r' + A B th'
//   t''  = W' = [ P A' omega - 2 a A (a sin cos th' W - sin^2 r r' ph') ] / Delta      (from p_t, p_phi const)
//   ph'' = [ a W' + 2 cot(theta) th' (a W - P ph') - 2 r r' ph' ] / P
//   r''  = (Delta/Sigma) [ r (sin^2 ph'^2 + th'^2) + A_r omega^2 / 2 ] - [ r/Sigma - (r-1)/Delta ] r'^2 + B th' r'
//   th'' = (1/Sigma) [ sin cos ph' (P ph' - 2 a W) + A B omega^2 / 2 - 2 r r' th' ] - (B/2) (r'^2/Delta - th'^2)
// Four reciprocals (Sigma, Delta, P, sin^2) and sin/cos of theta per evaluation: the trigonometric functions
// are what the paper names as the cost of this system in double precision.
//
// sin and cos.  Only sin^2 and sin cos enter (cos^2 = 1 - sin^2 inside Sigma), both of period pi, computed
// without table or slow path from the Taylor polynomials of sin y, cos y in y^2:
//   float / packed pair: y = theta - n pi, |y| <= pi/2 (two-constant Cody-Waite with FMA, n by the
//     add-and-subtract-1.5*2^23 trick), 6 / 6 terms (remainder < 1e-9), no quadrant logic;
//   double: y = theta - n pi/2, |y| <= pi/4, 8 / 8 terms (remainder < 2e-18) and a swap (sin, cos) ->
//     (cos, -sin) for odd n; the selects run on the integer pipe, which is idle in the FP64 kernel, and save
//     six FP64-pipe instructions per evaluation over the period-pi form (10 / 11 terms).
#pragma once
#include "ks_geodesic.cuh"

namespace gray2 {

template <typename T> struct TrigConst;
template <> struct TrigConst<double> {
  static constexpr int NS = 8, NC = 8;
  static constexpr bool quadrant = true;
  static constexpr double inv_period = 0.63661977236758134308, magic = 6755399441055744.0;   // 2/pi, 1.5 * 2^52
  static constexpr double p_hi = 1.57079632679489655800, p_lo = 6.123233995736766e-17;       // pi/2 = p_hi + p_lo
};
template <> struct TrigConst<float> {
  static constexpr int NS = 6, NC = 6;
  static constexpr bool quadrant = false;
  static constexpr double inv_period = 0.31830988618379067154, magic = 12582912.0;           // 1/pi, 1.5 * 2^23
  static constexpr double p_hi = 3.1415927410125732, p_lo = -8.742278000372485e-8;           // float(pi), pi - float(pi)
};

// S(z) = sum_{k>=1} (-1)^k z^(k-1) / (2k+1)!  so that  sin y = y + y^3 S(y^2)
template <typename T, int N> __device__ __forceinline__ T sin_series(T z) {
  constexpr double c[10] = {-1.0 / 6.0, 1.0 / 120.0, -1.0 / 5040.0, 1.0 / 362880.0, -1.0 / 39916800.0,
                            1.0 / 6227020800.0, -1.0 / 1307674368000.0, 1.0 / 355687428096000.0,
                            -1.0 / 121645100408832000.0, 1.0 / 51090942171709440000.0};
  T p = T(c[N - 1]);
#pragma unroll
  for (int i = N - 2; i >= 0; --i) p = fma_(p, z, T(c[i]));
  return p;
}

// C(z) = sum_{k>=1} (-1)^k z^(k-1) / (2k)!  so that  cos y = 1 + y^2 C(y^2)
template <typename T, int N> __device__ __forceinline__ T cos_series(T z) {
  constexpr double c[11] = {-1.0 / 2.0, 1.0 / 24.0, -1.0 / 720.0, 1.0 / 40320.0, -1.0 / 3628800.0,
                            1.0 / 479001600.0, -1.0 / 87178291200.0, 1.0 / 20922789888000.0,
                            -1.0 / 6402373705728000.0, 1.0 / 2432902008176640000.0,
                            -1.0 / 1124000727777607680000.0};
  T p = T(c[N - 1]);
#pragma unroll
  for (int i = N - 2; i >= 0; --i) p = fma_(p, z, T(c[i]));
  return p;
}

// sin^2(theta) and sin(theta) cos(theta).  K = TrigConst of the scalar type behind T (float for the pair).
template <typename T, typename K>
__device__ __forceinline__ void bl_trig(T th, T &s2, T &sc) {
  T t = th * T(K::inv_period) + T(K::magic);       // the integer nearest to theta / period, in the low bits
  T n = t + T(-K::magic);
  T y = fma_(n, T(-K::p_hi), th);
  y = fma_(n, T(-K::p_lo), y);
  T z = y * y;
  T s = fma_(y * z, sin_series<T, K::NS>(z), y);
  T c = fma_(z, cos_series<T, K::NC>(z), T(1));
  if constexpr (K::quadrant) {
    // period pi/2: odd n  ->  (sin, cos)(theta) = +-(cos y, -sin y)
    const bool odd = (__double2loint(t) & 1) != 0;
    const T ss = odd ? c : s;
    const T cc = odd ? -s : c;
    s = ss; c = cc;
  }
  s2 = s * s; sc = s * c;
}

// xddot^mu at (r, theta) for xdot = (u0, u1, u2, u3) = d(t, r, theta, phi)/dlambda.
template <typename T, typename K>
__device__ __forceinline__ void bl_accel(const SpinConst<T> &k, T r, T th, T u0, T u1, T u2, T u3,
                                         T &a0, T &a1, T &a2, T &a3) {
  T s2, sc;
  bl_trig<T, K>(th, s2, sc);
  const T r2 = r * r;
  const T P = r2 + k.a2;
  const T Sig = fma_(-k.a2, s2, P);               // r^2 + a^2 cos^2
  const T tr = r + r;
  const T Dl = P + (-tr);
  const T iS = fastmath<T>::rcp(Sig), iD = fastmath<T>::rcp(Dl), iP = fastmath<T>::rcp(P), is2 = fastmath<T>::rcp(s2);
  const T A = tr * iS;
  const T B = (k.two_a2 * sc) * iS;
  const T as2 = k.a * s2;
  const T om = fma_(-as2, u3, u0);
  const T W = A * om;
  const T Ar = fma_(-A, A, iS + iS);
  const T AB = A * B;
  const T Bu2 = B * u2;
  const T Ad = fma_(Ar, u1, A * Bu2);
  const T tru1 = tr * u1;
  const T tru1u3 = tru1 * u3;
  // 2aA (a sin cos th' W - sin^2 r r' ph') = (B th') (2r W) - (a sin^2 A) (2r r' ph')   since A Sigma = 2r
  const T Wd = fma_(as2 * A, tru1u3, fma_(-Bu2, tr * W, (P * Ad) * om)) * iD;
  a0 = Wd;
  const T cot2 = (sc + sc) * is2;
  const T Y = fma_(k.a, W, -(P * u3));
  a3 = iP * fma_(k.a, Wd, fma_(cot2 * u2, Y, -tru1u3));
  const T om2h = (T(0.5) * om) * om;
  const T u1s = u1 * u1, u2s = u2 * u2;
  const T Kk = fma_(s2 * u3, u3, u2s);
  const T M = fma_(r, Kk, Ar * om2h);
  const T G = fma_(r, iS, -((r + T(-1)) * iD));
  a1 = fma_(Dl * iS, M, fma_(-G, u1s, Bu2 * u1));
  const T N = fma_(sc * u3, fma_(P, u3, -(k.two_a * W)), fma_(AB, om2h, -tru1 * u2));
  a2 = fma_(iS, N, -((T(0.5) * B) * fma_(u1s, iD, -u2s)));
}

// Sum whose finiteness stands for the finiteness of all eight variables (stopping test, DESIGN R5).
template <typename T> __device__ __forceinline__ T bl_probe(const Ray<T> &s) {
  return ((s.t + s.y) + (s.z + s.u0)) + ((s.u1 + s.u2) + s.u3);
}

template <typename T> __device__ __forceinline__ T min_(T a, T b);
template <> __device__ __forceinline__ double min_<double>(double a, double b) { return fmin(a, b); }
template <> __device__ __forceinline__ float min_<float>(float a, float b) { return fminf(a, b); }

// Classic RK4; Ray<T> holds (t, r, theta, phi, t', r', theta', phi') in (t, x, y, z, u0..u3).
// The result goes to `o` (and the residuals of the FP32 sums to `oc`); the return value is the smallest radius among the positions of stages 2-4 and the
// result.  Eq. (1) is singular at Delta = 0 and a stage evaluated at or beyond the horizon is meaningless, so
// the caller accepts the step only if that radius is still outside the capture radius (DESIGN R20).
template <typename T, typename K>
__device__ __forceinline__ T rk4_step_bl(const SpinConst<T> &k, const Ray<T> &s, const Carry<T> &c, T h, Ray<T> &o, Carry<T> &oc) {
  const T hh = T(0.5) * h, h6 = h * T(1.0 / 6.0);
  T b0, b1, b2, b3, v0, v1, v2, v3, pr, pth, rmin;
  T St, Sr, Sth, Sph, S0, S1, S2, S3;
  // stage 1
  bl_accel<T, K>(k, s.x, s.y, s.u0, s.u1, s.u2, s.u3, b0, b1, b2, b3);
  St = s.u0; Sr = s.u1; Sth = s.u2; Sph = s.u3;
  S0 = b0; S1 = b1; S2 = b2; S3 = b3;
  pr = fma_(hh, s.u1, s.x); pth = fma_(hh, s.u2, s.y);
  v0 = fma_(hh, b0, s.u0); v1 = fma_(hh, b1, s.u1); v2 = fma_(hh, b2, s.u2); v3 = fma_(hh, b3, s.u3);
  rmin = pr;
  // stage 2
  bl_accel<T, K>(k, pr, pth, v0, v1, v2, v3, b0, b1, b2, b3);
  St = fma_(T(2), v0, St); Sr = fma_(T(2), v1, Sr); Sth = fma_(T(2), v2, Sth); Sph = fma_(T(2), v3, Sph);
  S0 = fma_(T(2), b0, S0); S1 = fma_(T(2), b1, S1); S2 = fma_(T(2), b2, S2); S3 = fma_(T(2), b3, S3);
  pr = fma_(hh, v1, s.x); pth = fma_(hh, v2, s.y);
  v0 = fma_(hh, b0, s.u0); v1 = fma_(hh, b1, s.u1); v2 = fma_(hh, b2, s.u2); v3 = fma_(hh, b3, s.u3);
  rmin = min_(rmin, pr);
  // stage 3
  bl_accel<T, K>(k, pr, pth, v0, v1, v2, v3, b0, b1, b2, b3);
  St = fma_(T(2), v0, St); Sr = fma_(T(2), v1, Sr); Sth = fma_(T(2), v2, Sth); Sph = fma_(T(2), v3, Sph);
  S0 = fma_(T(2), b0, S0); S1 = fma_(T(2), b1, S1); S2 = fma_(T(2), b2, S2); S3 = fma_(T(2), b3, S3);
  pr = fma_(h, v1, s.x); pth = fma_(h, v2, s.y);
  v0 = fma_(h, b0, s.u0); v1 = fma_(h, b1, s.u1); v2 = fma_(h, b2, s.u2); v3 = fma_(h, b3, s.u3);
  rmin = min_(rmin, pr);
  // stage 4
  bl_accel<T, K>(k, pr, pth, v0, v1, v2, v3, b0, b1, b2, b3);
  o = s;
  oc = c;
  if constexpr (!Carry<T>::compensated) {      // double: plain sums
    advance(o.t, h6, St + v0); advance(o.x, h6, Sr + v1); advance(o.y, h6, Sth + v2); advance(o.z, h6, Sph + v3);
    advance(o.u0, h6, S0 + b0); advance(o.u1, h6, S1 + b1); advance(o.u2, h6, S2 + b2); advance(o.u3, h6, S3 + b3);
  } else {                                                 // FP32: compensated sums (Carry, ks_geodesic.cuh)
    advance(o.t, oc.t, h6, St + v0); advance(o.x, oc.x, h6, Sr + v1); advance(o.y, oc.y, h6, Sth + v2);
    advance(o.z, oc.z, h6, Sph + v3); advance(o.u0, oc.u0, h6, S0 + b0); advance(o.u1, oc.u1, h6, S1 + b1);
    advance(o.u2, oc.u2, h6, S2 + b2); advance(o.u3, oc.u3, h6, S3 + b3);
  }
  return min_(rmin, o.x);
}

}  // namespace gray2
