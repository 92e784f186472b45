/*
 * gray2_oracle.h -- CPU ORACLE for the GRay2 hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * This library is the slow, plain, double-precision statement of what the CUDA path
 * (include/gray2.h) must compute.  It shares no code with the CUDA path and is never
 * called by it.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * It follows the paper (arXiv:1706.07062, /root/reference/PAPER.md) literally:
 *   metric      g = eta + f l l               PAPER.md:55-66  (eq. 2-5)
 *   derivatives analytic d_c g_ab             implicit differentiation of eq. (5)
 *   connection  Gamma = 1/2 g^-1 (dg+dg-dg)   PAPER.md:91     (eq. 8)
 *   geodesic    xdd = -Gamma xd xd            PAPER.md:87     (eq. 7), full 4x4x4 loop
 *   stepper     classic 4th-order Runge-Kutta PAPER.md:164
 * It does NOT use the regrouped eq. (10)-(14) form; that is the CUDA side's formula.
 *
 * Units G = c = M = 1.  All arrays are HOST memory owned by the caller.
 * Parity pins: see DESIGN.md "Oracle pins"; no function here is "parity unpinned".
 */
#ifndef GRAY2_ORACLE_H
#define GRAY2_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_ACTIVE = 0, ORACLE_CAPTURED = 1, ORACLE_ESCAPED = 2, ORACLE_MAXSTEPS = 3, ORACLE_INVALID = 4 };
enum { ORACLE_NULL = 0, ORACLE_TIMELIKE = 1 };
enum { ORACLE_KS = 0, ORACLE_BL = 1 };   /* coordinates of a state: Cartesian Kerr-Schild / Boyer-Lindquist */

typedef struct {
  double  *q[8];      /* t,x,y,z,u^t,u^x,u^y,u^z : n doubles each (SoA)             */
  double  *lambda;    /* n : affine parameter reached                               */
  int32_t *status;    /* n : ORACLE_ACTIVE ...                                      */
  int32_t *nsteps;    /* n : RK4 steps taken so far                                 */
  uint64_t n;
  double   a_eff;     /* spin used by the integrator (= -a for reversed rays)       */
  int32_t  kind;      /* ORACLE_NULL / ORACLE_TIMELIKE (nominal mu^2 for Carter Q)  */
  int32_t  reversed;  /* 1: time-reversed ray of a backward trace                   */
  int32_t  coords;    /* ORACLE_KS: q = t,x,y,z,u^t,u^x,u^y,u^z ; ORACLE_BL: q = t,r,theta,phi,u^t,u^r,u^theta,u^phi.
                         oracle_integrate and oracle_invariants follow it; the coordinate-time and
                         diagnostics drivers accept ORACLE_KS only                   */
} oracle_state;

typedef struct {
  int32_t mode;            /* 0: h = dir*h_fixed ; 1: h = dir*eta*r (KS r at step start) */
  double  h_fixed, eta;
  int32_t dir;             /* +1 or -1                                                   */
  double  capture_factor;  /* CAPTURED when r < capture_factor * r_plus                  */
  double  r_escape;        /* ESCAPED  when r > r_escape (+inf allowed)                  */
  int32_t max_steps;       /* per-ray total                                              */
} oracle_step_control;

typedef struct { uint64_t steps, n_captured, n_escaped, n_maxsteps, n_invalid, n_active; } oracle_stats;

/* ---- the four operations of the boundary, on host arrays ---- */
int oracle_init_null(oracle_state *s, double a, double r_obs, double inclination_rad,
                     double fov_half_alpha, double fov_half_beta, int32_t nx, int32_t ny);
int oracle_init_explicit(oracle_state *s, double a, const double *xu8, uint64_t n, int32_t kind, int32_t renormalise_ut);
int oracle_init_timelike(oracle_state *s, double a, const double *xu8, uint64_t n, int32_t renormalise_ut);  /* kind = TIMELIKE */
int oracle_integrate(oracle_state *s, uint64_t n, double lambda_end,
                     const oracle_step_control *sc, oracle_stats *stats /* may be NULL */);
int oracle_invariants(const oracle_state *s, uint64_t n, double *E, double *Lz, double *Q, double *norm);

/* ---- building blocks, exported so that the tests can pin each of them ---- */
double oracle_ks_r(double a, double x, double y, double z);                         /* eq. (5)            */
void   oracle_ks_metric(double a, const double pos[3], double g[16]);               /* eq. (2)-(4)        */
void   oracle_ks_metric_inverse(double a, const double pos[3], double gi[16]);      /* eta - f l^a l^b    */
void   oracle_ks_dmetric(double a, const double pos[3], double dg[64]);             /* dg[c*16+a*4+b]     */
void   oracle_ks_dmetric_fd(double a, const double pos[3], double step, double dg[64]); /* central diffs  */
void   oracle_ks_christoffel(double a, const double pos[3], double Gam[64]);        /* Gam[m*16+a*4+b]    */
void   oracle_ks_accel(double a, const double pos[3], const double u[4], double acc[4]);        /* eq. (7) */
void   oracle_ks_accel_fd(double a, const double pos[3], const double u[4], double step, double acc[4]);
void   oracle_rk4_step(double a, double y[8], double h);                            /* one RK4 step       */
void   oracle_invariants_one(double a, int32_t kind, const double y[8], double out[4]); /* E,Lz,Q,norm   */
/* fixed-step trajectory: writes y after every `stride` steps (and the initial state first):
   out has (nsteps/stride + 1) * 8 doubles. */
void   oracle_trajectory(double a, const double y0[8], double h, int64_t nsteps, int64_t stride, double *out);

/* ---- coordinate-time form (eq. 15): six variables, v^mu = dx^mu/dt, v^0 = 1 ---- */
void   oracle_ks_coordtime_accel(double a, const double pos[3], const double v[3], double dv[3]);  /* eq. (15) */
void   oracle_rk4_step_coordtime(double a, double y[6], double h);                 /* y = x,y,z,vx,vy,vz */
void   oracle_trajectory_coordtime(double a, const double y0[7], double h, int64_t nsteps, int64_t stride,
                                   double *out);                                    /* rows t,x,y,z,vx,vy,vz */
/* same driver loop as oracle_integrate with t in the role of lambda: stops at t_end (stays ACTIVE).
   On entry v^i = q[5+i]/q[4]; on exit q[4] = 1, q[5..7] = v^i; `lambda` is not touched. */
int    oracle_integrate_coordtime(oracle_state *s, uint64_t n, double t_end,
                                  const oracle_step_control *sc, oracle_stats *stats);

/* ---- diagnostics of the paper's convergence experiments (section 3; Fig. 4-9), see gray2_oracle.c ----
   out5n: 5 arrays of n doubles: max|u.u + mu^2|, first fitted peak of |cos theta|, Delta phi of the first
   complete polar cycle, times of the first two maxima of z.  NaN where the event never occurs. */
int    oracle_integrate_diagnostics(oracle_state *s, uint64_t n, double lambda_end,
                                    const oracle_step_control *sc, double *out5n, oracle_stats *stats);

/* ---- Boyer-Lindquist coordinates (eq. 1): the second coordinate system of the paper's
   benchmark (Table 2 "BL" rows) and an independent check of the KS integrator ---- */
void   oracle_bl_metric(double a, const double X[4], double g[16]);                 /* X = t,r,theta,phi  */
void   oracle_bl_dmetric(double a, const double X[4], double dg[64]);               /* analytic, dg[c*16+a*4+b] */
void   oracle_bl_dmetric_fd(double a, const double X[4], double dg[64]);            /* 4th-order central diffs  */
void   oracle_bl_accel(double a, const double X[4], const double u[4], double acc[4]);    /* eq. (7)-(8), analytic dg */
void   oracle_bl_accel_fd(double a, const double X[4], const double u[4], double acc[4]); /* same from dmetric_fd   */
void   oracle_bl_rk4_step(double a, double y[8], double h);
/* the step of oracle_integrate on BL states: returns 1 and leaves y untouched when the position of a
   stage, or the result of the step, has r < r_capture (the ray then ends as CAPTURED, DESIGN R20) */
int    oracle_bl_rk4_step_guarded(double a, double y[8], double h, double r_capture);
void   oracle_bl_trajectory(double a, const double y0[8], double h, int64_t nsteps, int64_t stride, double *out);
void   oracle_bl_invariants_one(double a, int32_t kind, const double y[8], double out[4]); /* E,Lz,Q,norm */
/* the coordinate map between the two systems (the paper's Appendix is missing; DESIGN R18):
     x + i y = (r + i a) sin(theta) e^{i phi_KS},  z = r cos(theta),
     t_KS = t_BL + T(r),  phi_KS = phi_BL + Phi(r),  dT/dr = 2r/Delta,  dPhi/dr = a/Delta.
   y_out and y_in are 8-vectors (position, then contravariant velocity). */
void   oracle_bl_to_ks_one(double a, const double y_bl[8], double y_ks[8]);
void   oracle_ks_to_bl_one(double a, const double y_ks[8], double y_bl[8]);
/* whole states: dst arrays are caller-owned, dst->coords = to_coords on return; lambda, status, nsteps,
   a_eff, kind, reversed are copied.  Returns 1 on bad arguments (src->coords == to_coords included). */
int    oracle_convert(const oracle_state *src, oracle_state *dst, uint64_t n, int32_t to_coords);

int    oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
