// gray2_kernels.cuh -- CUDA kernels of the hot path (sm_100a).  See include/gray2.h for the contract.
//
//   init_null_kernel       one thread per pixel, writes the SoA state
//   init_explicit_kernel   AoS staging buffer -> SoA state, optional u^t solve   (a2)
//   integrate_kernel       persistent lanes: each lane keeps ONE geodesic in registers and steps it
//                          with the fused right-hand side + RK4 until its stopping test fires, then
//                          stores it and takes the next geodesic from a global queue (warp-aggregated
//                          atomic: one atomicAdd per warp per refill, ballot + popc prefix)  (a3-a7, a9)
//   invariants_kernel      E, L_z, Q, u.u in double from the stored state          (a8)
//   count_status_kernel    final status histogram for gray2_stats
#pragma once
#include <stdint.h>
#include "../../include/gray2.h"
#include "ks_geodesic.cuh"
#include "f32x2.cuh"
#include "bl_geodesic.cuh"

namespace gray2 {

template <typename T> struct StateView {
  T *q[8];
  double *lambda;
  int32_t *status;
  int32_t *nsteps;
  const int32_t *order;     // gray2_state.order; read by the ORDERED instantiations of the integrators only
};

template <typename T> struct StepParams {
  SpinConst<T> k;
  T eta_or_h;          // eta (mode 1) or h_fixed (mode 0), already multiplied by dir
  T r_capture;         // capture_factor * r_plus
  T r_escape;
  T r_escape_fin;     // min(r_escape, largest finite value of T)
  double lambda_end;
  double dir;
  int32_t mode;
  int32_t max_steps;
  int32_t clip;        // 0 only when dir*lambda_end = +inf: the lambda_end test can never fire, skip it
};

// u^t from g_ab u^a u^b = -mu2 (future-directed root), DESIGN R3/R7:
//   (1-f) ut^2 - 2 f c ut - (|v|^2 + mu2 + f c^2) = 0 ,  c = l.v
__device__ __forceinline__ double solve_ut(double a, double x, double y, double z,
                                           double vx, double vy, double vz, double mu2) {
  double R2 = x * x + y * y + z * z, w = R2 - a * a;
  double r2 = 0.5 * (w + sqrt(w * w + 4.0 * a * a * z * z));
  double r = sqrt(r2);
  double f = 2.0 * r2 * r / (r2 * r2 + a * a * z * z);
  double P = r2 + a * a;
  double c = ((r * x + a * y) * vx + (r * y - a * x) * vy) / P + z * vz / r;
  double A = 1.0 - f, B = f * c, C = vx * vx + vy * vy + vz * vz + mu2 + f * c * c;
  return (B + sqrt(B * B + A * C)) / A;
}

// Shard of one image: ray indices are dealt out in tiles of `tile` consecutive indices, tile t
// to rank t mod world; the shard-local ray `idx` of rank `rank` is the image's ray
//   pix = ((idx / tile) * world + rank) * tile + idx % tile.
// The whole image is the case tile = nx*ny, rank = 0, world = 1 (pix = idx).
template <typename T>
__global__ void init_null_kernel(StateView<T> s, uint64_t n_local, double a_eff, double r_obs, double sin_i,
                                 double cos_i, double Wa, double Wb, int32_t nx, int32_t ny, uint64_t tile,
                                 uint32_t rank, uint32_t world) {
  uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_local) return;
  uint64_t pix = ((idx / tile) * world + rank) * tile + idx % tile;
  int32_t j = (int32_t)(pix % (uint64_t)nx), kk = (int32_t)(pix / (uint64_t)nx);
  double alpha = -Wa + ((double)j + 0.5) * (2.0 * Wa / (double)nx);
  double beta = -Wb + ((double)kk + 0.5) * (2.0 * Wb / (double)ny);
  // n = (sin i, 0, cos i), e_alpha = (0,1,0), e_beta = (-cos i, 0, sin i)
  double x = r_obs * sin_i - beta * cos_i;
  double y = alpha;
  double z = r_obs * cos_i + beta * sin_i;
  double vx = -sin_i, vy = 0.0, vz = -cos_i;
  double ut = solve_ut(a_eff, x, y, z, vx, vy, vz, 0.0);
  s.q[0][idx] = T(0); s.q[1][idx] = T(x); s.q[2][idx] = T(y); s.q[3][idx] = T(z);
  s.q[4][idx] = T(ut); s.q[5][idx] = T(vx); s.q[6][idx] = T(vy); s.q[7][idx] = T(vz);
  s.lambda[idx] = 0.0; s.status[idx] = GRAY2_ACTIVE; s.nsteps[idx] = 0;
}

template <typename T>
__global__ void init_explicit_kernel(StateView<T> s, const double *__restrict__ xu8, uint64_t n, double a,
                                     int32_t renorm, double mu2) {
  uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n) return;
  const double2 *row = reinterpret_cast<const double2 *>(xu8 + idx * 8);
  double2 v0 = row[0], v1 = row[1], v2 = row[2], v3 = row[3];
  double ut = v2.x;
  if (renorm) ut = solve_ut(a, v0.y, v1.x, v1.y, v2.y, v3.x, v3.y, mu2);
  s.q[0][idx] = T(v0.x); s.q[1][idx] = T(v0.y); s.q[2][idx] = T(v1.x); s.q[3][idx] = T(v1.y);
  s.q[4][idx] = T(ut); s.q[5][idx] = T(v2.y); s.q[6][idx] = T(v3.x); s.q[7][idx] = T(v3.y);
  s.lambda[idx] = 0.0; s.status[idx] = GRAY2_ACTIVE; s.nsteps[idx] = 0;
}

// ---- the fused integrator ------------------------------------------------------------------------
// MODE: 0 fixed step, 1 radius-scaled step.  CLIP: false only when dir*lambda_end = +inf, i.e. the
// lambda_end test can never fire and the last step never needs clipping.
//
// Loop structure.  The outer loop refills idle lanes from the global queue; the inner loop advances
// every lane of the warp by one RK4 step per pass and leaves as soon as ANY lane's stopping test fires
// (one vote per step).  In the hot path the stopping rule of gray2_step_control costs four compares:
// the tests are ordered only in the (rare) slow path that classifies and stores a finished ray.
//
// FORM: 0 affine parameter (eq. 13-14, eight variables); 1 coordinate time (eq. 18, six variables): the
// clock `lam` is then t itself, v^i = u^i/u^t on load, and (t, x, 1, v) is stored; `lambda` is untouched;
// 2 affine parameter in Boyer-Lindquist coordinates (bl_geodesic.cuh): the state is (t, r, theta, phi) and
// its derivatives, the radius of the step rule and of the stopping tests is the coordinate r itself.
//
// ORDERED: the queue position is mapped to a geodesic through the caller's schedule s.order (gray2_state.order);
// a separate instantiation, so that the code of the unordered kernel does not depend on the feature.
template <typename T, int THREADS, int MIN_BLOCKS, int MODE, bool CLIP, int FORM, bool ORDERED = false>
__global__ void __launch_bounds__(THREADS, MIN_BLOCKS)
integrate_kernel(StateView<T> s, uint64_t n, StepParams<T> p, unsigned long long *queue,
                 unsigned long long *steps_out) {
  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;
  const SpinConst<T> k = p.k;

  Ray<T> ray;
  ray.t = ray.x = ray.y = ray.u0 = ray.u1 = ray.u2 = ray.u3 = T(0);
  ray.z = T(3);                // idle lanes integrate a harmless dummy state (never stored)
  if constexpr (FORM == 2) { ray.x = T(3); ray.y = T(1); }
  Carry<T> car;                // FP32: residuals of the compensated state sums (empty in double)
  car.clear();
  double lam = 0.0;
  int32_t nst = 0, nst0 = 0;
  uint64_t idx = 0;
  bool have = false;           // this lane holds an ACTIVE geodesic
  bool cap = false;            // FORM 2: the last step was rejected, a stage reached the capture radius
  bool drained = false;        // warp-uniform: the queue has no more work
  unsigned long long my_steps = 0;

  for (;;) {
    // ---- refill idle lanes from the global queue (warp-aggregated) ------------------------------
    unsigned idle = __ballot_sync(0xffffffffu, !have);
    if (idle && !drained) {
      unsigned cnt = __popc(idle);
      int leader = __ffs(idle) - 1;
      unsigned long long base = 0;
      if ((int)lane == leader) base = atomicAdd(queue, (unsigned long long)cnt);
      base = __shfl_sync(0xffffffffu, base, leader);
      if (base + cnt >= n) drained = true;
      if (!have) {
        uint64_t mine = base + __popc(idle & lt_mask);      // position in the queue
        // ... and the geodesic the schedule puts there; an entry outside 0..n-1 (a negative one included: it
        // converts to a huge index) names no geodesic and is passed over like the end of the queue
        if constexpr (ORDERED) { if (mine < n) mine = (uint64_t)s.order[mine]; }
        if (mine < n) {
          // the status and the state are fetched together (one round trip to memory instead of two); an entry
          // that turns out not to be ACTIVE is dropped and its slot of the lane refilled at the next pass
          const int32_t st_in = s.status[mine];
          Ray<T> in;
          in.t = s.q[0][mine]; in.x = s.q[1][mine]; in.y = s.q[2][mine]; in.z = s.q[3][mine];
          in.u0 = s.q[4][mine]; in.u1 = s.q[5][mine]; in.u2 = s.q[6][mine]; in.u3 = s.q[7][mine];
          double lam_in = 0.0;
          if constexpr (FORM != 1) lam_in = s.lambda[mine];
          const int32_t nst_in = s.nsteps[mine];
          if (st_in == GRAY2_ACTIVE) {
            idx = mine;
            ray = in;
            car.clear();
            if constexpr (FORM == 1) {
              lam = (double)ray.t;
              if constexpr (Carry<T>::compensated) {
                // FP32: v = u / u^t in double, split into the float the right-hand side sees and the residual of
                // the compensated sum, so that the coordinate velocity starts without a rounding error of its own
                // (a float division here is 1.5 ulp of direction: 1e-4 M of impact parameter over 1000 M)
                const double inv = 1.0 / (double)ray.u0;
                const double v1 = (double)ray.u1 * inv, v2 = (double)ray.u2 * inv, v3 = (double)ray.u3 * inv;
                ray.u1 = (T)v1; ray.u2 = (T)v2; ray.u3 = (T)v3; ray.u0 = T(1);
                car.u1 = (T)(v1 - (double)ray.u1); car.u2 = (T)(v2 - (double)ray.u2); car.u3 = (T)(v3 - (double)ray.u3);
              } else {
                T w = fastmath<T>::rcp(ray.u0);
                ray.u1 *= w; ray.u2 *= w; ray.u3 *= w; ray.u0 = T(1);
              }
            } else {
              lam = lam_in;
            }
            nst = nst0 = nst_in;
            have = true;
          }
        }
      }
      continue;   // entries that were not ACTIVE leave the lane idle: ask again
    }
    if (idle == 0xffffffffu) break;   // nothing held and the queue is drained

    // ---- step all lanes until one of them has to stop ---------------------------------------------
    for (;;) {
      Geometry<T> g;
      Vel<T> w;
      T U;
      if constexpr (FORM == 2) {
        g.r = ray.x;
        U = bl_probe(ray);
      } else {
        ks_geometry(k, ray.x, ray.y, ray.z, g);
        w = ks_vel(k, g, ray.x, ray.y, ray.u0, ray.u1, ray.u2, ray.u3);     // reused by stage 1 of the step
        U = w.U;
      }
      // NaN fails every compare; r_escape_fin = min(r_escape, largest finite) so that r = inf fails too
      bool go = fastmath<T>::ge_pos(g.r, p.r_capture) && fastmath<T>::le_pos(g.r, p.r_escape_fin) &&
                fastmath<T>::finite(U) && fastmath<T>::finite(ray.t) && (nst < p.max_steps);
      if (CLIP) go = go && (p.dir * (p.lambda_end - lam) > 0.0);
      if constexpr (FORM == 2) go = go && !cap;
      if (__any_sync(0xffffffffu, have && !go)) {
        if (have && !go) {
          // classify in the order of gray2_step_control and store the state where the test fired
          int32_t st = GRAY2_ACTIVE;    // lambda_end reached: stays ACTIVE (resumable)
          if (!(fastmath<T>::finite(g.r) && fastmath<T>::finite(U) && fastmath<T>::finite(ray.t))) st = GRAY2_INVALID;
          else if (g.r < p.r_capture || cap) st = GRAY2_CAPTURED;
          else if (g.r > p.r_escape) st = GRAY2_ESCAPED;
          else if (nst >= p.max_steps) st = GRAY2_MAXSTEPS;
          cap = false;
          if constexpr (FORM == 1) ray.t = (T)lam;
          s.q[0][idx] = ray.t; s.q[1][idx] = ray.x; s.q[2][idx] = ray.y; s.q[3][idx] = ray.z;
          s.q[4][idx] = ray.u0; s.q[5][idx] = ray.u1; s.q[6][idx] = ray.u2; s.q[7][idx] = ray.u3;
          if constexpr (FORM != 1) s.lambda[idx] = lam;
          s.status[idx] = st; s.nsteps[idx] = nst;
          my_steps += (unsigned long long)(nst - nst0);
          have = false;
        }
        break;
      }
      T h = (MODE == 1) ? p.eta_or_h * g.r : p.eta_or_h;
      double lam_next = lam + (double)h;
      if (CLIP) {
        // the clipped last step lands on lambda_end itself (DESIGN R22)
        double rem = p.lambda_end - lam;
        if (fabs((double)h) > fabs(rem)) { h = (T)rem; lam_next = p.lambda_end; }
      }
      if constexpr (FORM == 2) {
        // the step is accepted only if no stage position, and not its result, is inside the capture radius;
        // otherwise the geodesic ends as CAPTURED at the state it has now (DESIGN R20)
        Ray<T> nxt;
        Carry<T> ncar;
        T rmin = rk4_step_bl<T, TrigConst<T>>(k, ray, car, h, nxt, ncar);
        if (rmin < p.r_capture) cap = true;
        else { ray = nxt; car = ncar; lam = lam_next; nst += 1; }
      } else {
        if constexpr (FORM == 1) rk4_step_coordtime(k, ray, car, g, w, h);
        else rk4_step(k, ray, car, g, w, h);
        lam = lam_next;
        nst += 1;
      }
    }
  }

  // ---- per-warp reduction of the step count -----------------------------------------------------
  for (int off = 16; off > 0; off >>= 1) my_steps += __shfl_down_sync(0xffffffffu, my_steps, off);
  if (lane == 0 && my_steps) atomicAdd(steps_out, my_steps);
}

// ---- FP32, two geodesics per thread (packed FP32x2 arithmetic, see f32x2.cuh) -----------------------
// Same loop structure as integrate_kernel.  Each thread owns two slots (the halves of every register
// pair); a warp therefore holds 64 geodesics, refilled slot by slot from the same queue.
struct PairSlot {
  uint64_t idx;
  double lam;
  int32_t nst, nst0;
  bool have;
  bool cap;     // FORM 2: the last step was rejected, a stage reached the capture radius
};

template <int C, int FORM, bool ORDERED>
__device__ __forceinline__ void load_slot(const StateView<float> &s, uint64_t n, uint64_t mine, Ray<f32x2> &ray,
                                          Carry<f32x2> &car, PairSlot &sl) {
  if (mine >= n) return;
  if constexpr (ORDERED) {
    mine = (uint64_t)s.order[mine];
    if (mine >= n) return;       // an entry outside 0..n-1 names no geodesic
  }
  // the status and the state are fetched together (one round trip to memory instead of two)
  const int32_t st_in = s.status[mine];
  float t = s.q[0][mine], x = s.q[1][mine], y = s.q[2][mine], z = s.q[3][mine];
  float u0 = s.q[4][mine], u1 = s.q[5][mine], u2 = s.q[6][mine], u3 = s.q[7][mine];
  double lam_in = 0.0;
  if (FORM != 1) lam_in = s.lambda[mine];
  const int32_t nst_in = s.nsteps[mine];
  if (st_in == GRAY2_ACTIVE) {
    sl.idx = mine;
    clear_half<C>(car);
    if (FORM == 1) {
      // v = u / u^t in double, split into the float the right-hand side sees and the residual of the compensated
      // sum (see integrate_kernel)
      sl.lam = (double)t;
      const double inv = 1.0 / (double)u0;
      const double v1 = (double)u1 * inv, v2 = (double)u2 * inv, v3 = (double)u3 * inv;
      u1 = (float)v1; u2 = (float)v2; u3 = (float)v3; u0 = 1.0f;
      set_half<C>(car.u1, (float)(v1 - (double)u1)); set_half<C>(car.u2, (float)(v2 - (double)u2));
      set_half<C>(car.u3, (float)(v3 - (double)u3));
    } else {
      sl.lam = lam_in;
    }
    set_half<C>(ray.t, t); set_half<C>(ray.x, x); set_half<C>(ray.y, y);
    set_half<C>(ray.z, z); set_half<C>(ray.u0, u0); set_half<C>(ray.u1, u1);
    set_half<C>(ray.u2, u2); set_half<C>(ray.u3, u3);
    sl.nst = sl.nst0 = nst_in;
    sl.have = true;
    sl.cap = false;
  }
}

template <int C, bool CLIP>
__device__ __forceinline__ bool slot_may_step(const StepParams<float> &p, const Geometry<f32x2> &g, f32x2 U,
                                              const Ray<f32x2> &ray, const PairSlot &sl) {
  float r = half_of<C>(g.r);
  bool go = (r >= p.r_capture) && (r <= p.r_escape_fin) && fastmath<float>::finite(half_of<C>(U)) &&
            fastmath<float>::finite(half_of<C>(ray.t)) && (sl.nst < p.max_steps);
  if (CLIP) go = go && (p.dir * (p.lambda_end - sl.lam) > 0.0);
  return go && !sl.cap;
}

template <int C, int FORM>
__device__ __forceinline__ void store_slot(const StateView<float> &s, const StepParams<float> &p,
                                           const Geometry<f32x2> &g, f32x2 U, const Ray<f32x2> &ray, PairSlot &sl,
                                           unsigned long long &my_steps) {
  float r = half_of<C>(g.r), t = half_of<C>(ray.t);
  int32_t st = GRAY2_ACTIVE;
  if (!(fastmath<float>::finite(r) && fastmath<float>::finite(half_of<C>(U)) && fastmath<float>::finite(t))) st = GRAY2_INVALID;
  else if (r < p.r_capture || sl.cap) st = GRAY2_CAPTURED;
  else if (r > p.r_escape) st = GRAY2_ESCAPED;
  else if (sl.nst >= p.max_steps) st = GRAY2_MAXSTEPS;
  const uint64_t i = sl.idx;
  s.q[0][i] = FORM == 1 ? (float)sl.lam : t;
  s.q[1][i] = half_of<C>(ray.x); s.q[2][i] = half_of<C>(ray.y); s.q[3][i] = half_of<C>(ray.z);
  s.q[4][i] = half_of<C>(ray.u0); s.q[5][i] = half_of<C>(ray.u1); s.q[6][i] = half_of<C>(ray.u2);
  s.q[7][i] = half_of<C>(ray.u3);
  if (FORM != 1) s.lambda[i] = sl.lam;
  s.status[i] = st; s.nsteps[i] = sl.nst;
  my_steps += (unsigned long long)(sl.nst - sl.nst0);
  sl.have = false;
}

template <int THREADS, int MIN_BLOCKS, int MODE, bool CLIP, int FORM, bool ORDERED = false>
__global__ void __launch_bounds__(THREADS, MIN_BLOCKS)
integrate_kernel_f32x2(StateView<float> s, uint64_t n, StepParams<float> p, unsigned long long *queue,
                       unsigned long long *steps_out) {
  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;
  const SpinConst<f32x2> k{f32x2(p.k.a), f32x2(p.k.a2), f32x2(p.k.two_a), f32x2(p.k.two_a2), f32x2(p.k.four_a2)};

  Ray<f32x2> ray;
  ray.t = ray.x = ray.y = ray.u0 = ray.u1 = ray.u2 = ray.u3 = f32x2(0.0f);
  ray.z = f32x2(3.0f);         // idle slots integrate a harmless dummy state (never stored)
  if constexpr (FORM == 2) { ray.x = f32x2(3.0f); ray.y = f32x2(1.0f); }
  Carry<f32x2> car;            // residuals of the compensated state sums (ks_geodesic.cuh)
  car.clear();
  PairSlot A{0, 0.0, 0, 0, false, false}, B{0, 0.0, 0, 0, false, false};
  bool drained = false;
  unsigned long long my_steps = 0;

  for (;;) {
    unsigned idleA = __ballot_sync(0xffffffffu, !A.have), idleB = __ballot_sync(0xffffffffu, !B.have);
    if ((idleA | idleB) && !drained) {
      unsigned cntA = __popc(idleA), cnt = cntA + __popc(idleB);
      unsigned long long base = 0;
      if (lane == 0) base = atomicAdd(queue, (unsigned long long)cnt);
      base = __shfl_sync(0xffffffffu, base, 0);
      if (base + cnt >= n) drained = true;
      if (!A.have) load_slot<0, FORM, ORDERED>(s, n, base + __popc(idleA & lt_mask), ray, car, A);
      if (!B.have) load_slot<1, FORM, ORDERED>(s, n, base + cntA + __popc(idleB & lt_mask), ray, car, B);
      continue;
    }
    if ((idleA & idleB) == 0xffffffffu) break;

    for (;;) {
      Geometry<f32x2> g;
      Vel<f32x2> w;
      f32x2 U;
      if constexpr (FORM == 2) {
        g.r = ray.x;
        U = bl_probe(ray);
      } else {
        ks_geometry(k, ray.x, ray.y, ray.z, g);
        w = ks_vel(k, g, ray.x, ray.y, ray.u0, ray.u1, ray.u2, ray.u3);
        U = w.U;
      }
      bool stopA = A.have && !slot_may_step<0, CLIP>(p, g, U, ray, A);
      bool stopB = B.have && !slot_may_step<1, CLIP>(p, g, U, ray, B);
      if (__any_sync(0xffffffffu, stopA || stopB)) {
        if (stopA) store_slot<0, FORM>(s, p, g, U, ray, A, my_steps);
        if (stopB) store_slot<1, FORM>(s, p, g, U, ray, B, my_steps);
        break;
      }
      f32x2 h = (MODE == 1) ? f32x2(p.eta_or_h) * g.r : f32x2(p.eta_or_h);
      double nextA = A.lam + (double)h.v.x, nextB = B.lam + (double)h.v.y;
      if (CLIP) {
        // the clipped last step lands on lambda_end itself (DESIGN R22)
        double remA = p.lambda_end - A.lam, remB = p.lambda_end - B.lam;
        if (fabs((double)h.v.x) > fabs(remA)) { h.v.x = (float)remA; nextA = p.lambda_end; }
        if (fabs((double)h.v.y) > fabs(remB)) { h.v.y = (float)remB; nextB = p.lambda_end; }
      }
      if constexpr (FORM == 2) {
        Ray<f32x2> nxt;
        Carry<f32x2> ncar;
        f32x2 rmin = rk4_step_bl<f32x2, TrigConst<float>>(k, ray, car, h, nxt, ncar);
        if (rmin.v.x < p.r_capture) A.cap = true;
        else { copy_half<0>(ray, nxt); copy_half<0>(car, ncar); A.lam = nextA; A.nst += 1; }
        if (rmin.v.y < p.r_capture) B.cap = true;
        else { copy_half<1>(ray, nxt); copy_half<1>(car, ncar); B.lam = nextB; B.nst += 1; }
      } else {
        if constexpr (FORM == 1) rk4_step_coordtime(k, ray, car, g, w, h);
        else rk4_step(k, ray, car, g, w, h);
        A.lam = nextA; B.lam = nextB;
        A.nst += 1; B.nst += 1;
      }
    }
  }

  for (int off = 16; off > 0; off >>= 1) my_steps += __shfl_down_sync(0xffffffffu, my_steps, off);
  if (lane == 0 && my_steps) atomicAdd(steps_out, my_steps);
}

// ---- integration with the paper's convergence diagnostics (section 3, Fig. 4-9) ----------------------
// One thread per geodesic (these runs are small: thousands of orbits x a few step sizes).  The samples are
// the states at the step boundaries, the initial state included; see gray2_diagnostics in gray2.h.
struct DiagView {
  double *max_abs_u2, *cos_peak, *dphi_cycle, *t_zmax1, *t_zmax2;
};

__device__ __forceinline__ double wrap_pi(double d) {
  const double pi = 3.14159265358979323846;
  while (d > pi) d -= 2.0 * pi;
  while (d <= -pi) d += 2.0 * pi;
  return d;
}

template <typename T, int MODE>
__global__ void integrate_diag_kernel(StateView<T> s, uint64_t n, StepParams<T> p, double mu2, DiagView out,
                                      unsigned long long *steps_out) {
  uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n) return;
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  if (s.status[idx] != GRAY2_ACTIVE) {   // not touched: no samples, every diagnostic is NaN
    out.max_abs_u2[idx] = nan; out.cos_peak[idx] = nan; out.dphi_cycle[idx] = nan;
    out.t_zmax1[idx] = nan; out.t_zmax2[idx] = nan;
    return;
  }
  const SpinConst<T> k = p.k;
  Ray<T> ray;
  ray.t = s.q[0][idx]; ray.x = s.q[1][idx]; ray.y = s.q[2][idx]; ray.z = s.q[3][idx];
  ray.u0 = s.q[4][idx]; ray.u1 = s.q[5][idx]; ray.u2 = s.q[6][idx]; ray.u3 = s.q[7][idx];
  Carry<T> car;
  car.clear();
  double lam = s.lambda[idx];
  int32_t nst = s.nsteps[idx], nst0 = nst, st = GRAY2_ACTIVE;
  // accumulators
  double u2max = nan, c2 = 0.0, c1 = 0.0, peak = nan, phi0 = 0.0, phiprev = 0.0, phiunf = 0.0;
  double zprev = 0.0, uzprev = 0.0, tprev = 0.0, dphi = nan, tz0 = nan, tz1 = nan;
  long long ks = 0;
  int ntz = 0;
  bool have_peak = false, have_dphi = false;
  for (;;) {
    Geometry<T> g;
    ks_geometry(k, ray.x, ray.y, ray.z, g);
    const Vel<T> w = ks_vel(k, g, ray.x, ray.y, ray.u0, ray.u1, ray.u2, ray.u3);
    const T U = w.U;
    if (!(fastmath<T>::finite(g.r) && fastmath<T>::finite(U) && fastmath<T>::finite(ray.t))) { st = GRAY2_INVALID; break; }
    {   // ---- sample k ----
      double u0 = (double)ray.u0, u1 = (double)ray.u1, u2 = (double)ray.u2, u3 = (double)ray.u3;
      double Ud = (double)U, fd = (double)g.f, r = (double)g.r, z = (double)ray.z, t = (double)ray.t;
      double nrm = fabs(-u0 * u0 + u1 * u1 + u2 * u2 + u3 * u3 + fd * Ud * Ud + mu2);
      double c = fabs(z) / r;
      double phi = atan2((double)ray.y, (double)ray.x) - atan2((double)k.a, r);
      if (ks == 0) {
        u2max = nrm; phi0 = phi; phiunf = phi;
      } else {
        if (nrm > u2max) u2max = nrm;
        double unf = phiunf + wrap_pi(phi - phiprev);
        if (ks >= 2 && !have_peak && c1 >= c2 && c1 > c) {
          peak = c1 - (c - c2) * (c - c2) / (8.0 * (c2 - 2.0 * c1 + c));
          have_peak = true;
        }
        if (!have_dphi && zprev < 0.0 && z >= 0.0) {         // ks >= 1 here: the pair (z_0, z_1) counts
          double w = -zprev / (z - zprev);
          dphi = phiunf + w * (unf - phiunf) - phi0;
          have_dphi = true;
        }
        if (ntz < 2 && uzprev > 0.0 && u3 <= 0.0) {
          double tt = tprev + (t - tprev) * uzprev / (uzprev - u3);
          if (ntz == 0) tz0 = tt; else tz1 = tt;
          ntz += 1;
        }
        phiunf = unf;
      }
      c2 = c1; c1 = c; phiprev = phi; zprev = z; uzprev = u3; tprev = t;
      ks += 1;
    }
    if (g.r < p.r_capture) { st = GRAY2_CAPTURED; break; }
    if (g.r > p.r_escape) { st = GRAY2_ESCAPED; break; }
    if (nst >= p.max_steps) { st = GRAY2_MAXSTEPS; break; }
    if (p.dir * (p.lambda_end - lam) <= 0.0) break;
    T h = (MODE == 1) ? p.eta_or_h * g.r : p.eta_or_h;
    double lam_next = lam + (double)h, rem = p.lambda_end - lam;
    if (fabs((double)h) > fabs(rem)) { h = (T)rem; lam_next = p.lambda_end; }     // DESIGN R22
    rk4_step(k, ray, car, g, w, h);
    lam = lam_next;
    nst += 1;
  }
  s.q[0][idx] = ray.t; s.q[1][idx] = ray.x; s.q[2][idx] = ray.y; s.q[3][idx] = ray.z;
  s.q[4][idx] = ray.u0; s.q[5][idx] = ray.u1; s.q[6][idx] = ray.u2; s.q[7][idx] = ray.u3;
  s.lambda[idx] = lam; s.status[idx] = st; s.nsteps[idx] = nst;
  out.max_abs_u2[idx] = u2max; out.cos_peak[idx] = peak; out.dphi_cycle[idx] = dphi;
  out.t_zmax1[idx] = tz0; out.t_zmax2[idx] = tz1;
  if (nst > nst0) atomicAdd(steps_out, (unsigned long long)(nst - nst0));
}

// ---- invariants (always double) ------------------------------------------------------------------
template <typename T>
__global__ void invariants_kernel(StateView<T> s, uint64_t n, double a, double mu2, double *__restrict__ E,
                                  double *__restrict__ Lz, double *__restrict__ Q, double *__restrict__ norm) {
  uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n) return;
  double x = (double)s.q[1][idx], y = (double)s.q[2][idx], z = (double)s.q[3][idx];
  double u0 = (double)s.q[4][idx], u1 = (double)s.q[5][idx], u2 = (double)s.q[6][idx], u3 = (double)s.q[7][idx];
  double R2 = x * x + y * y + z * z, w = R2 - a * a;
  double r2 = 0.5 * (w + sqrt(w * w + 4.0 * a * a * z * z));
  double r = sqrt(r2), P = r2 + a * a;
  double f = 2.0 * r2 * r / (r2 * r2 + a * a * z * z);
  double l1 = (r * x + a * y) / P, l2 = (r * y - a * x) / P, l3 = z / r;
  double U = u0 + l1 * u1 + l2 * u2 + l3 * u3;
  // lower the index with g = eta + f l l :  u_0 = -u^0 + f U ,  u_i = u^i + f l_i U
  double c0 = -u0 + f * U, cx = u1 + f * l1 * U, cy = u2 + f * l2 * U, cz = u3 + f * l3 * U;
  double nn = c0 * u0 + cx * u1 + cy * u2 + cz * u3;
  double e = -c0;
  double lz = x * cy - y * cx;
  double c = l3, s2 = 1.0 - c * c;
  double q = P * c * c * (cx * cx + cy * cy) - 2.0 * r * c * (x * cx + y * cy) * cz + r2 * s2 * cz * cz +
             a * a * c * c * (mu2 - e * e);
  E[idx] = e; Lz[idx] = lz; Q[idx] = q; norm[idx] = nn;
}

// Boyer-Lindquist state: E = -u_t, L_z = u_phi, u_theta = Sigma theta', with eq. (1) in the form
// ds^2 = -dt^2 + Sigma (dr^2/Delta + dtheta^2) + P sin^2 dphi^2 + A (dt - a sin^2 dphi)^2.
template <typename T>
__global__ void invariants_bl_kernel(StateView<T> s, uint64_t n, double a, double mu2, double *__restrict__ E,
                                     double *__restrict__ Lz, double *__restrict__ Q, double *__restrict__ norm) {
  uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n) return;
  double r = (double)s.q[1][idx], th = (double)s.q[2][idx];
  double u0 = (double)s.q[4][idx], u1 = (double)s.q[5][idx], u2 = (double)s.q[6][idx], u3 = (double)s.q[7][idx];
  double sn, cs;
  sincos(th, &sn, &cs);
  double s2 = sn * sn, c2 = cs * cs, a2 = a * a;
  double Sig = r * r + a2 * c2, P = r * r + a2, Dl = P - 2.0 * r, A = 2.0 * r / Sig;
  double om = u0 - a * s2 * u3, W = A * om;
  double e = u0 - W;
  double lz = s2 * (P * u3 - a * W);
  double pth = Sig * u2;
  E[idx] = e; Lz[idx] = lz;
  Q[idx] = pth * pth + c2 * (a2 * (mu2 - e * e) + lz * lz / s2);
  norm[idx] = -u0 * u0 + Sig * (u1 * u1 / Dl + u2 * u2) + P * s2 * u3 * u3 + W * om;
}

// ---- the coordinate map Kerr-Schild <-> Boyer-Lindquist (DESIGN R18; the paper's Appendix is missing,
// PAPER.md:207).  x + i y = (r + i a) sin(theta) e^{i phi_KS}, z = r cos(theta), t_KS = t_BL + T(r),
// phi_KS = phi_BL + Phi(r), dT/dr = 2r/Delta, dPhi/dr = a/Delta.  Always evaluated in double.
__device__ __forceinline__ void bl_shift(double a, double r, double &T, double &Phi) {
  double d2 = 1.0 - a * a;
  if (d2 > 0.0) {
    double sq = sqrt(d2), rp = 1.0 + sq, rm = 1.0 - sq, w = 0.5 / sq;       // 1/(r_+ - r_-)
    double lp = log(fabs(r - rp)), lm = log(fabs(r - rm));
    T = 2.0 * w * (rp * lp - rm * lm);
    Phi = a * w * (lp - lm);
  } else {                                                                   // double root r_+ = r_- = 1
    T = 2.0 * log(fabs(r - 1.0)) - 2.0 / (r - 1.0);
    Phi = -a / (r - 1.0);
  }
}

template <typename T>
__global__ void ks_to_bl_kernel(StateView<T> src, StateView<T> dst, uint64_t n, double a) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double t = (double)src.q[0][i], x = (double)src.q[1][i], y = (double)src.q[2][i], z = (double)src.q[3][i];
  double u0 = (double)src.q[4][i], u1 = (double)src.q[5][i], u2 = (double)src.q[6][i], u3 = (double)src.q[7][i];
  double a2 = a * a, rho2 = x * x + y * y;
  double w = rho2 + z * z - a2, D = sqrt(w * w + 4.0 * a2 * z * z);
  double r2 = 0.5 * (w + D), r = sqrt(r2), P = r2 + a2, Dl = P - 2.0 * r;
  double cs = z / r, sn = sqrt(rho2 / P);
  // implicit differentiation of eq. (5): r' = [r^2 (x.u) + a^2 z u^z] / (r D)
  double rd = (r2 * (x * u1 + y * u2 + z * u3) + a2 * z * u3) / (r * D);
  double thd = (cs * rd - u3) / (r * sn);
  double phd = (x * u2 - y * u1) / rho2 + a * rd / P;       // d/dlambda of arg(x + i y) - arg(r + i a)
  double Tr, Phr;
  bl_shift(a, r, Tr, Phr);
  dst.q[0][i] = (T)(t - Tr);
  dst.q[1][i] = (T)r;
  dst.q[2][i] = (T)atan2(sn, cs);
  dst.q[3][i] = (T)(atan2(y, x) - atan2(a, r) - Phr);
  dst.q[4][i] = (T)(u0 - 2.0 * r / Dl * rd);
  dst.q[5][i] = (T)rd;
  dst.q[6][i] = (T)thd;
  dst.q[7][i] = (T)(phd - a / Dl * rd);
  dst.lambda[i] = src.lambda[i]; dst.status[i] = src.status[i]; dst.nsteps[i] = src.nsteps[i];
}

template <typename T>
__global__ void bl_to_ks_kernel(StateView<T> src, StateView<T> dst, uint64_t n, double a) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double t = (double)src.q[0][i], r = (double)src.q[1][i], th = (double)src.q[2][i], ph = (double)src.q[3][i];
  double u0 = (double)src.q[4][i], rd = (double)src.q[5][i], thd = (double)src.q[6][i], phd = (double)src.q[7][i];
  double Dl = r * r - 2.0 * r + a * a, Tr, Phr;
  bl_shift(a, r, Tr, Phr);
  double sn, cs, sp, cp;
  sincos(th, &sn, &cs);
  sincos(ph + Phr, &sp, &cp);
  double ex = r * cp - a * sp, ey = r * sp + a * cp;         // (x, y) = (ex, ey) sin(theta)
  double x = ex * sn, y = ey * sn;
  double phk = phd + a / Dl * rd;                            // d phi_KS / dlambda
  dst.q[0][i] = (T)(t + Tr);
  dst.q[1][i] = (T)x;
  dst.q[2][i] = (T)y;
  dst.q[3][i] = (T)(r * cs);
  dst.q[4][i] = (T)(u0 + 2.0 * r / Dl * rd);
  dst.q[5][i] = (T)(rd * cp * sn - y * phk + ex * cs * thd);
  dst.q[6][i] = (T)(rd * sp * sn + x * phk + ey * cs * thd);
  dst.q[7][i] = (T)(rd * cs - r * sn * thd);
  dst.lambda[i] = src.lambda[i]; dst.status[i] = src.status[i]; dst.nsteps[i] = src.nsteps[i];
}

// Diagnostic: the Boyer-Lindquist right-hand side alone.  pos: 2 arrays of n (r, theta), u and out: 4 arrays.
template <typename T>
__global__ void rhs_bl_kernel(SpinConst<T> k, uint64_t n, const T *__restrict__ pos, const T *__restrict__ u,
                              T *__restrict__ out) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  T a0, a1, a2, a3;
  bl_accel<T, TrigConst<T>>(k, pos[i], pos[n + i], u[i], u[n + i], u[2 * n + i], u[3 * n + i], a0, a1, a2, a3);
  out[i] = a0; out[n + i] = a1; out[2 * n + i] = a2; out[3 * n + i] = a3;
}

// Diagnostic: the right-hand side alone, for element-wise parity tests against the oracle.
// pos: 3 arrays of n (x,y,z), u: 4 arrays of n, out: 4 arrays of n, all of type T, SoA.
template <typename T>
__global__ void rhs_kernel(SpinConst<T> k, uint64_t n, const T *__restrict__ pos, const T *__restrict__ u,
                           T *__restrict__ out) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  Geometry<T> g;
  ks_geometry(k, pos[i], pos[n + i], pos[2 * n + i], g);
  T a0, a1, a2, a3;
  ks_accel(k, g, pos[i], pos[n + i], u[i], u[n + i], u[2 * n + i], u[3 * n + i], a0, a1, a2, a3);
  out[i] = a0; out[n + i] = a1; out[2 * n + i] = a2; out[3 * n + i] = a3;
}

// ---- longest-first schedule (gray2_order_longest_first): counting sort of the indices by decreasing key ----
constexpr int kOrderBins = 4096;

__global__ void order_max_kernel(const int32_t *__restrict__ key, uint64_t n, unsigned *kmax) {
  unsigned m = 0;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
    m = max(m, (unsigned)max(key[i], 0));
  for (int off = 16; off > 0; off >>= 1) m = max(m, __shfl_down_sync(0xffffffffu, m, off));
  if ((threadIdx.x & 31) == 0 && m) atomicMax(kmax, m);
}

__device__ __forceinline__ unsigned order_bin(int32_t key, unsigned kmax) {
  // bin 0 holds the largest keys; width = ceil((kmax + 1) / bins)
  const unsigned width = kmax / kOrderBins + 1;
  return (kmax - min((unsigned)max(key, 0), kmax)) / width;
}

__global__ void order_hist_kernel(const int32_t *__restrict__ key, uint64_t n, const unsigned *kmax, unsigned *hist) {
  const unsigned km = *kmax;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
    atomicAdd(&hist[order_bin(key[i], km)], 1u);
}

// one block of kOrderBins / 4 threads: exclusive prefix sum of the histogram -> the cursor of every bin
__global__ void order_scan_kernel(const unsigned *__restrict__ hist, unsigned *cursor) {
  __shared__ unsigned part[kOrderBins / 4];
  const unsigned t = threadIdx.x;
  unsigned v[4], sum = 0;
#pragma unroll
  for (int j = 0; j < 4; ++j) { v[j] = hist[4 * t + j]; sum += v[j]; }
  part[t] = sum;
  __syncthreads();
  for (unsigned off = 1; off < kOrderBins / 4; off <<= 1) {
    unsigned add = t >= off ? part[t - off] : 0u;
    __syncthreads();
    part[t] += add;
    __syncthreads();
  }
  unsigned run = part[t] - sum;
#pragma unroll
  for (int j = 0; j < 4; ++j) { cursor[4 * t + j] = run; run += v[j]; }
}

__global__ void order_scatter_kernel(const int32_t *__restrict__ key, uint64_t n, const unsigned *kmax, unsigned *cursor,
                                     int32_t *__restrict__ order) {
  const unsigned km = *kmax;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
    order[atomicAdd(&cursor[order_bin(key[i], km)], 1u)] = (int32_t)i;
}

__global__ void count_status_kernel(const int32_t *__restrict__ status, uint64_t n, gray2_stats *stats) {
  unsigned long long c[5] = {0, 0, 0, 0, 0};
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
    int32_t st = status[i];
#pragma unroll
    for (int v = 0; v < 5; ++v) c[v] += (st == v);
  }
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    for (int off = 16; off > 0; off >>= 1) c[v] += __shfl_down_sync(0xffffffffu, c[v], off);
  }
  if ((threadIdx.x & 31) == 0) {
    if (c[0]) atomicAdd((unsigned long long *)&stats->n_active, c[0]);
    if (c[1]) atomicAdd((unsigned long long *)&stats->n_captured, c[1]);
    if (c[2]) atomicAdd((unsigned long long *)&stats->n_escaped, c[2]);
    if (c[3]) atomicAdd((unsigned long long *)&stats->n_maxsteps, c[3]);
    if (c[4]) atomicAdd((unsigned long long *)&stats->n_invalid, c[4]);
  }
}

}  // namespace gray2
