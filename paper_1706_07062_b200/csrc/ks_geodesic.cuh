// ks_geodesic.cuh -- device arithmetic of the hot path: Kerr-Schild geodesic right-hand side in the
// regrouped form of PAPER.md:98-117 (eq. 10-14), and the classic RK4 step of PAPER.md:164.
//
// Everything here lives in registers; one thread owns one geodesic.  Template parameter T is the
// arithmetic type (double or float).  No table of Christoffel symbols is ever formed.
//
// Derivation (checked against the brute-force connection to 1e-41 in
// 40-digit arithmetic).  With M = 1, spin a, position (x,y,z), velocity (u0,u1,u2,u3) = dx^mu/dlambda:
//
//   w = x^2+y^2+z^2 - a^2,  D = sqrt(w^2 + 4 a^2 z^2),  r^2 = (w + D)/2                      (eq. 5)
//   D equals Sigma = r^2 + a^2 z^2/r^2, so  f = 2 r^3/(r^4 + a^2 z^2) = 2 r / D                (eq. 3)
//   P = r^2 + a^2,  l = ((r x + a y)/P, (r y - a x)/P, z/r)                                    (eq. 4)
//   grad r = (f/2) (x, y, z P / r^2)
//   grad f = f [ c1 grad r - c2 e_z ],  c1 = 3/r - 2 f,  c2 = 2 a^2 z / (D r^2)
//   d_j l_i = (grad r)_j A_i + B_ji,  A = ((x - 2 r l1)/P, (y - 2 r l2)/P, -l3/r),
//             B = [[r/P, -a/P, 0], [a/P, r/P, 0], [0, 0, 1/r]]
//
// The 12 elements xdot_{beta,alpha} = g_{beta gamma,alpha} xdot^gamma of PAPER.md:100 never need to be
// stored: with U = u0 + l.u they collapse to (ks_accel below uses a further regrouping of the same terms)
//   omega = curl l = grad r x A + (0, 0, -2a/P)                 (antisymmetric part of d_j l_i)
//   q     = u_i u_j d_j l_i = (u.grad r)(A.u) + (r/P)(u1^2+u2^2) + u3^2 / r   (symmetric part)
//   l.grad f = f (c1 - c2 l3)       because l.grad r = 1 and (l.grad) l = 0 (l is a geodesic null field)
//   F   = -(1/2) f U^2 (l.grad f)                                              (eq. 12)
//   xddot^0 = U (u.grad f) + f q - F                                          (eq. 13)
//   xddot^i = (1/2) U^2 d_i f + f U (u x omega)_i - l_i xddot^0               (eq. 14)
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace gray2 {

// ---- fast reciprocal square root / reciprocal ---------------------------------------------------
// FP64: hardware seed (MUFU.RSQ64H / MUFU.RCP64H, about 20 good bits) followed by ONE third-order
// correction, which leaves a relative error of a few 1e-16 -- ample for the 1e-9 parity bound, and
// 3-5 DFMA-pipe instructions instead of the ~12 plus a slow-path branch of IEEE division and sqrt.
// FP32: the MUFU approximation itself (max relative error 2^-22.4 for rsqrt, 1 ulp for rcp).
template <typename T> struct fastmath;

template <> struct fastmath<double> {
  static __device__ __forceinline__ double rsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x * y, y, 1.0);            // e = 1 - x y^2
    double c = fma(0.375, e, 0.5);             // y <- y (1 + e/2 + 3 e^2/8)
    return fma(y * e, c, y);
  }
  static __device__ __forceinline__ double rcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);                // e = 1 - x y
    double t = fma(e, e, e);                   // y <- y (1 + e + e^2)
    return fma(y, t, y);
  }
  // The stopping tests of the hot loop run on the integer pipe (the FP64 pipe is the one that is full):
  // finite <=> exponent field not all ones; and for a >= 0 or NaN, b > 0 finite, the IEEE order of a and b
  // is the order of their bit patterns -- a NaN compares above every finite b, so it fails the `le` test
  // that always accompanies the `ge` test (a NaN with the sign bit set fails `ge`).
  static __device__ __forceinline__ bool finite(double x) { return (__double2hiint(x) & 0x7ff00000) != 0x7ff00000; }
  static __device__ __forceinline__ bool ge_pos(double a, double b) { return __double_as_longlong(a) >= __double_as_longlong(b); }
  static __device__ __forceinline__ bool le_pos(double a, double b) { return __double_as_longlong(a) <= __double_as_longlong(b); }
};

template <> struct fastmath<float> {
  static __device__ __forceinline__ float rsqrt(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
  }
  static __device__ __forceinline__ float rcp(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
  }
  static __device__ __forceinline__ bool finite(float x) { return fabsf(x) <= 3.402823466e38f; }
  static __device__ __forceinline__ bool ge_pos(float a, float b) { return a >= b; }
  static __device__ __forceinline__ bool le_pos(float a, float b) { return a <= b; }
};

template <typename T> __device__ __forceinline__ T fma_(T a, T b, T c);
template <> __device__ __forceinline__ double fma_<double>(double a, double b, double c) { return fma(a, b, c); }
template <> __device__ __forceinline__ float fma_<float>(float a, float b, float c) { return fmaf(a, b, c); }

// Spin-dependent constants, computed once on the host.
template <typename T> struct SpinConst {
  T a, a2, two_a, two_a2, four_a2;
};

// Position-only part of the right-hand side (shared by the stopping test, the step rule and stage 1).
//
// Final regrouping: with n = (x, y, zeta), zeta = z P / r^2, one has
// grad r = (f/2) n and grad f = alpha n - beta e_z; the unit vector l and the vector A enter the spatial
// acceleration only through  -c_A A_i - l_i xddot^0 , and both are combinations of (x, y) and
// (r x + a y, r y - a x) / P, so that
//   xddot^1 = kappa x + mu y - c_B u2 ,  xddot^2 = kappa y - mu x + c_B u1 ,
//   xddot^3 = c_n zeta + l3 (c_A / r - xddot^0) - (U^2/2) beta
// with scalars kappa, mu, c_n, c_A, c_B built from the dot products below: l1, l2, A1, A2 and curl l are
// never formed.
template <typename T> struct Geometry {
  T r, rinv, Pinv, hf, f, l3, zeta;
  T fc1, beta, lf;          // grad f = f c1 (f/2) n - beta e_z ;  lf = l . grad f = f c1 - beta l3
  T trP, rP, taP;           // 2r/P, r/P, 2a/P
};

template <typename T>
__device__ __forceinline__ void ks_radius(const SpinConst<T> &k, T x, T y, T z, T &r, T &rinv, T &Dinv, T &r2) {
  T w = fma_(x, x, fma_(y, y, fma_(z, z, -k.a2)));
  T b = k.two_a * z;
  T D2 = fma_(b, b, w * w);
  Dinv = fastmath<T>::rsqrt(D2);
  r2 = T(0.5) * fma_(D2, Dinv, w);          // (w + D)/2 with D = D2 / sqrt(D2)
  rinv = fastmath<T>::rsqrt(r2);
  r = r2 * rinv;
}

template <typename T>
__device__ __forceinline__ void ks_geometry(const SpinConst<T> &k, T x, T y, T z, Geometry<T> &g) {
  T Dinv, r2;
  ks_radius(k, x, y, z, g.r, g.rinv, Dinv, r2);
  const T r = g.r, rinv = g.rinv;
  T P = r2 + k.a2;
  T Pinv = fastmath<T>::rcp(P);
  g.Pinv = Pinv;
  T hf = r * Dinv;                 // f / 2 = r / Sigma
  T f = hf + hf;
  g.hf = hf;
  g.f = f;
  g.l3 = z * rinv;
  g.zeta = (P * rinv) * g.l3;                      // z P / r^2
  T c1 = fma_(T(3), rinv, -(f + f));
  g.fc1 = f * c1;
  g.beta = (k.four_a2 * g.l3) * (Dinv * Dinv);     // f c2 = (2r/D) 2a^2 z/(D r^2) = 4 a^2 l3 / D^2
  g.lf = fma_(-g.beta, g.l3, g.fc1);
  g.rP = r * Pinv;
  g.trP = g.rP + g.rP;
  g.taP = k.two_a * Pinv;
}

// The first products of the velocity-dependent part.  U = l_alpha u^alpha also serves as the finiteness probe
// of the stopping test, so the kernels evaluate this once at the top of a step and hand it to stage 1.
template <typename T> struct Vel {
  T xu, Lu, U;              // x u1 + y u2 ;  P (l1 u1 + l2 u2) ;  l_alpha u^alpha
};

template <typename T>
__device__ __forceinline__ Vel<T> ks_vel(const SpinConst<T> &k, const Geometry<T> &g, T x, T y, T u0, T u1, T u2, T u3) {
  Vel<T> w;
  w.xu = fma_(x, u1, y * u2);
  T yu = fma_(y, u1, -x * u2);
  w.Lu = fma_(g.r, w.xu, k.a * yu);
  w.U = fma_(g.l3, u3, fma_(g.Pinv, w.Lu, u0));
  return w;
}

// Velocity-dependent part: xddot^mu from the geometry, the position and u (eq. 13-14).
template <typename T>
__device__ __forceinline__ void ks_accel(const SpinConst<T> &k, const Geometry<T> &g, const Vel<T> &w, T x, T y,
                                         T u1, T u2, T u3, T &a0, T &a1, T &a2, T &a3) {
  const T xu = w.xu, Lu = w.Lu, U = w.U;
  T w3 = u3 * g.rinv;
  T Au = fma_(g.Pinv, fma_(-g.trP, Lu, xu), -(g.l3 * w3));
  T unv = fma_(g.zeta, u3, xu);                    // n . u
  T ur = g.hf * unv;                               // u . grad r
  T s12 = fma_(u1, u1, u2 * u2);
  T q = fma_(ur, Au, fma_(g.rP, s12, u3 * w3));
  T uf = fma_(g.fc1, ur, -g.beta * u3);            // u . grad f   (alpha n.u = f c1 u.grad r)
  T hU2 = T(0.5) * (U * U);
  T fU = g.f * U;
  a0 = fma_(g.f, fma_(hU2, g.lf, q), U * uf);
  T cn = g.hf * fma_(fU, Au, hU2 * g.fc1);         // f U (f/2) A.u + (U^2/2) alpha
  T cA = fU * ur;
  T cB = fU * g.taP;
  T e2 = g.Pinv * fma_(cA, g.trP, -a0);
  T kap = fma_(e2, g.r, fma_(-cA, g.Pinv, cn));
  T mu = e2 * k.a;
  a1 = fma_(kap, x, fma_(mu, y, -cB * u2));
  a2 = fma_(kap, y, fma_(-mu, x, cB * u1));
  a3 = fma_(cn, g.zeta, fma_(g.l3, fma_(cA, g.rinv, -a0), -hU2 * g.beta));
}

template <typename T>
__device__ __forceinline__ void ks_accel(const SpinConst<T> &k, const Geometry<T> &g, T x, T y,
                                         T u0, T u1, T u2, T u3, T &a0, T &a1, T &a2, T &a3) {
  ks_accel(k, g, ks_vel(k, g, x, y, u0, u1, u2, u3), x, y, u1, u2, u3, a0, a1, a2, a3);
}

// One geodesic's 8 variables.
template <typename T> struct Ray {
  T t, x, y, z, u0, u1, u2, u3;
};

// FP32 only: the running residuals of the eight state sums (DESIGN R12).  A ray of cfg3 takes ~1000 steps
// whose increments h u, h xddot are 1e2...1e5 times smaller than the variables they are added to, so a plain
// float sum rounds away the low bits of every increment; the accumulated loss (an equivalent shift of the
// impact parameter by ~2e-4 M) is what limited the FP32 integrator, not the float right-hand side.  Each
// variable is therefore carried as an unevaluated sum hi + lo (compensated summation, Kahan 1965): the
// right-hand side sees hi, the increment is added as  inc = fma(h/6, S, lo); t = hi + inc; lo = inc - (t - hi).
// Three more instructions per variable and step.  The double kernels do not need it (Carry<double> is empty).
template <typename T> struct Carry {
  static constexpr bool compensated = true;
  T t, x, y, z, u0, u1, u2, u3;
  __device__ __forceinline__ void clear() { t = x = y = z = u0 = u1 = u2 = u3 = T(0); }
};
template <> struct Carry<double> {
  static constexpr bool compensated = false;
  __device__ __forceinline__ void clear() {}
};

// hi <- hi + w S  (w = h/6; S = k1 + 2 k2 + 2 k3 + k4), compensated when a residual is carried.
template <typename T>
__device__ __forceinline__ void advance(T &hi, T &lo, T w, T S) {
  const T inc = fma_(w, S, lo);
  const T t = hi + inc;
  lo = inc - (t - hi);
  hi = t;
}
__device__ __forceinline__ void advance(double &hi, double w, double S) { hi = fma(w, S, hi); }

// Classic RK4.  `g1` is the geometry at the current position (already needed by the
// stopping test and the step rule), so stage 1 costs only the velocity-dependent part.
template <typename T>
__device__ __forceinline__ void rk4_step(const SpinConst<T> &k, Ray<T> &s, Carry<T> &c, const Geometry<T> &g1, const Vel<T> &w1, T h) {
  const T hh = T(0.5) * h, h6 = h * T(1.0 / 6.0);
  T b0, b1, b2, b3;                      // stage acceleration
  T v0, v1, v2, v3;                      // stage velocity
  T px, py, pz;                          // stage position
  T St, Sx, Sy, Sz, S0, S1, S2, S3;      // k1 + 2 k2 + 2 k3 (+ k4)
  Geometry<T> g;
  // stage 1
  ks_accel(k, g1, w1, s.x, s.y, s.u1, s.u2, s.u3, b0, b1, b2, b3);
  St = s.u0; Sx = s.u1; Sy = s.u2; Sz = s.u3;
  S0 = b0; S1 = b1; S2 = b2; S3 = b3;
  px = fma_(hh, s.u1, s.x); py = fma_(hh, s.u2, s.y); pz = fma_(hh, s.u3, s.z);
  v0 = fma_(hh, b0, s.u0); v1 = fma_(hh, b1, s.u1); v2 = fma_(hh, b2, s.u2); v3 = fma_(hh, b3, s.u3);
  // stage 2
  ks_geometry(k, px, py, pz, g);
  ks_accel(k, g, px, py, v0, v1, v2, v3, b0, b1, b2, b3);
  St = fma_(T(2), v0, St); Sx = fma_(T(2), v1, Sx); Sy = fma_(T(2), v2, Sy); Sz = fma_(T(2), v3, Sz);
  S0 = fma_(T(2), b0, S0); S1 = fma_(T(2), b1, S1); S2 = fma_(T(2), b2, S2); S3 = fma_(T(2), b3, S3);
  px = fma_(hh, v1, s.x); py = fma_(hh, v2, s.y); pz = fma_(hh, v3, s.z);
  v0 = fma_(hh, b0, s.u0); v1 = fma_(hh, b1, s.u1); v2 = fma_(hh, b2, s.u2); v3 = fma_(hh, b3, s.u3);
  // stage 3
  ks_geometry(k, px, py, pz, g);
  ks_accel(k, g, px, py, v0, v1, v2, v3, b0, b1, b2, b3);
  St = fma_(T(2), v0, St); Sx = fma_(T(2), v1, Sx); Sy = fma_(T(2), v2, Sy); Sz = fma_(T(2), v3, Sz);
  S0 = fma_(T(2), b0, S0); S1 = fma_(T(2), b1, S1); S2 = fma_(T(2), b2, S2); S3 = fma_(T(2), b3, S3);
  px = fma_(h, v1, s.x); py = fma_(h, v2, s.y); pz = fma_(h, v3, s.z);
  v0 = fma_(h, b0, s.u0); v1 = fma_(h, b1, s.u1); v2 = fma_(h, b2, s.u2); v3 = fma_(h, b3, s.u3);
  // stage 4
  ks_geometry(k, px, py, pz, g);
  ks_accel(k, g, px, py, v0, v1, v2, v3, b0, b1, b2, b3);
  if constexpr (!Carry<T>::compensated) {      // double: plain sums
    (void)c;
    advance(s.t, h6, St + v0); advance(s.x, h6, Sx + v1); advance(s.y, h6, Sy + v2); advance(s.z, h6, Sz + v3);
    advance(s.u0, h6, S0 + b0); advance(s.u1, h6, S1 + b1); advance(s.u2, h6, S2 + b2); advance(s.u3, h6, S3 + b3);
  } else {
    advance(s.t, c.t, h6, St + v0); advance(s.x, c.x, h6, Sx + v1); advance(s.y, c.y, h6, Sy + v2);
    advance(s.z, c.z, h6, Sz + v3); advance(s.u0, c.u0, h6, S0 + b0); advance(s.u1, c.u1, h6, S1 + b1);
    advance(s.u2, c.u2, h6, S2 + b2); advance(s.u3, c.u3, h6, S3 + b3);
  }
}

// ---- coordinate-time form ------------------------------------------------------
// v^mu = dx^mu/dt, v^0 = 1.  PAPER.md:146 eq. (18): the right-hand side is the affine one evaluated with
// u = (1, v) and recombined,  dv^i/dt = xddot^i - xddot^0 v^i  -- "the same computational complexity".
template <typename T>
__device__ __forceinline__ void ks_accel_coordtime(const SpinConst<T> &k, const Geometry<T> &g, const Vel<T> &w, T x, T y,
                                                   T v1, T v2, T v3, T &d1, T &d2, T &d3) {
  T a0, a1, a2, a3;
  ks_accel(k, g, w, x, y, v1, v2, v3, a0, a1, a2, a3);
  d1 = fma_(-a0, v1, a1);
  d2 = fma_(-a0, v2, a2);
  d3 = fma_(-a0, v3, a3);
}

// Classic RK4 in t of the six variables (x, v); uses Ray<T> with u0 unused (v^0 = 1) and t advanced by
// the caller (t += h exactly).
// hi <- hi + h v + small, exactly: the product h v is split into its float value and its rounding error (one FMA),
// the error joins the small terms in the residual.  Used for the positions of the FP32 coordinate-time form.
template <typename T>
__device__ __forceinline__ void advance_exact(T &hi, T &lo, T h, T v, T small) {
  const T p = h * v;
  const T e = fma_(h, v, -p);               // p + e = h v exactly
  const T t = hi + p;
  const T l = (p - (t - hi)) + ((lo + e) + small);   // what t lacks of hi + lo + h v + small
  hi = t + l;
  lo = l - (hi - t);
}

template <typename T>
__device__ __forceinline__ void rk4_step_coordtime(const SpinConst<T> &k, Ray<T> &s, Carry<T> &c, const Geometry<T> &g1, const Vel<T> &w1, T h) {
  const T hh = T(0.5) * h, h6 = h * T(1.0 / 6.0);
  T b1, b2, b3, v1, v2, v3, px, py, pz;
  T Sx, Sy, Sz, S1, S2, S3;
  T B1, B2, B3;                          // FP32: b(stage 1) + b(stage 2) + b(stage 3), see below
  Geometry<T> g;
  ks_accel_coordtime(k, g1, w1, s.x, s.y, s.u1, s.u2, s.u3, b1, b2, b3);
  Sx = s.u1; Sy = s.u2; Sz = s.u3; S1 = b1; S2 = b2; S3 = b3;
  B1 = b1; B2 = b2; B3 = b3;
  px = fma_(hh, s.u1, s.x); py = fma_(hh, s.u2, s.y); pz = fma_(hh, s.u3, s.z);
  v1 = fma_(hh, b1, s.u1); v2 = fma_(hh, b2, s.u2); v3 = fma_(hh, b3, s.u3);
  ks_geometry(k, px, py, pz, g);
  ks_accel_coordtime(k, g, ks_vel(k, g, px, py, T(1), v1, v2, v3), px, py, v1, v2, v3, b1, b2, b3);
  Sx = fma_(T(2), v1, Sx); Sy = fma_(T(2), v2, Sy); Sz = fma_(T(2), v3, Sz);
  S1 = fma_(T(2), b1, S1); S2 = fma_(T(2), b2, S2); S3 = fma_(T(2), b3, S3);
  B1 = B1 + b1; B2 = B2 + b2; B3 = B3 + b3;
  px = fma_(hh, v1, s.x); py = fma_(hh, v2, s.y); pz = fma_(hh, v3, s.z);
  v1 = fma_(hh, b1, s.u1); v2 = fma_(hh, b2, s.u2); v3 = fma_(hh, b3, s.u3);
  ks_geometry(k, px, py, pz, g);
  ks_accel_coordtime(k, g, ks_vel(k, g, px, py, T(1), v1, v2, v3), px, py, v1, v2, v3, b1, b2, b3);
  Sx = fma_(T(2), v1, Sx); Sy = fma_(T(2), v2, Sy); Sz = fma_(T(2), v3, Sz);
  S1 = fma_(T(2), b1, S1); S2 = fma_(T(2), b2, S2); S3 = fma_(T(2), b3, S3);
  B1 = B1 + b1; B2 = B2 + b2; B3 = B3 + b3;
  px = fma_(h, v1, s.x); py = fma_(h, v2, s.y); pz = fma_(h, v3, s.z);
  v1 = fma_(h, b1, s.u1); v2 = fma_(h, b2, s.u2); v3 = fma_(h, b3, s.u3);
  ks_geometry(k, px, py, pz, g);
  ks_accel_coordtime(k, g, ks_vel(k, g, px, py, T(1), v1, v2, v3), px, py, v1, v2, v3, b1, b2, b3);
  if constexpr (!Carry<T>::compensated) {
    (void)c; (void)B1; (void)B2; (void)B3;
    advance(s.x, h6, Sx + v1); advance(s.y, h6, Sy + v2); advance(s.z, h6, Sz + v3);
    advance(s.u1, h6, S1 + b1); advance(s.u2, h6, S2 + b2); advance(s.u3, h6, S3 + b3);
  } else {
    // FP32 positions.  The RK4 sum (h/6)(v + 2 v_2 + 2 v_3 + v_4) with v_2 = v + (h/2) b_1, v_3 = v + (h/2) b_2,
    // v_4 = v + h b_3 is  h v + (h^2/6)(b_1 + b_2 + b_3), and it is formed that way: h v exactly (advance_exact), the
    // small second term and what the compensated sum holds of v beside its float (c.u, up to half an ulp) into the
    // residual.  Added up as floats the sum is rounded at the size of 6 v, a relative 1e-7, and on the way in, where
    // v hardly changes, the SAME rounding recurs at every step: measured 2.7e-5 M after 200 M, 7e-5 M on arrival at
    // the hole from 1841 M.  Under dt = eta r that offset is a fixed fraction of a step, i.e. it keeps its size
    // relative to r on the way out: 7e-5 M at r = 15 M leaves as 5e-6 r.  c.u matters for the
    // same reason -- v = u/u^t is not a float, so it is non-zero from the first step and constant while v is.
    (void)Sx; (void)Sy; (void)Sz;
    const T h26 = h * h6;
    advance_exact(s.x, c.x, h, s.u1, fma_(h, c.u1, h26 * B1));
    advance_exact(s.y, c.y, h, s.u2, fma_(h, c.u2, h26 * B2));
    advance_exact(s.z, c.z, h, s.u3, fma_(h, c.u3, h26 * B3));
    advance(s.u1, c.u1, h6, S1 + b1); advance(s.u2, c.u2, h6, S2 + b2); advance(s.u3, c.u3, h6, S3 + b3);
  }
}

}  // namespace gray2
