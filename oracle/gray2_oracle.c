/*
 * gray2_oracle.c -- CPU ORACLE for the GRay2 hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double precision.  Shares nothing with the CUDA path.  See gray2_oracle.h.
 * Every function cites the passage of /root/reference/PAPER.md (arXiv:1706.07062) it follows;
 * "DESIGN Rn" refers to the numbered readings in DESIGN.md where the paper is silent.
 *
 * Parity pins (tests/test_oracle_*.py): eq.(5) residual, l.l=1, g g^-1 = 1, Schwarzschild limit,
 * central differences of the metric, Gamma symmetry, Newtonian limit, conservation rates,
 * Table 1 of the paper, 4th-order convergence, photon sphere,
 * circular-orbit period, ISCO, epicyclic frequency, Bardeen shadow, Carter radial potential,
 * independent Boyer-Lindquist integration.  No function is "parity unpinned".
 */
#define _GNU_SOURCE
#include "gray2_oracle.h"
#include <math.h>
#include <stddef.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------
 * C1.  Kerr-Schild radius r(x,y,z), eq. (5):
 *        x^2 + y^2 + z^2 = r^2 + a^2 (1 - z^2/r^2)
 *      multiplied by r^2:  r^4 - (R^2 - a^2) r^2 - a^2 z^2 = 0,  positive root for r^2.
 * ---------------------------------------------------------------------------------------- */
double oracle_ks_r(double a, double x, double y, double z)
{
  double R2 = x * x + y * y + z * z;
  double w = R2 - a * a;
  double r2 = 0.5 * (w + sqrt(w * w + 4.0 * a * a * z * z));
  return sqrt(r2);
}

/* f and l_alpha of PAPER.md:59-61, eq. (3)-(4) (M = 1). */
static void ks_f_l(double a, const double pos[3], double *r_out, double *f_out, double l[4])
{
  double x = pos[0], y = pos[1], z = pos[2];
  double r = oracle_ks_r(a, x, y, z);
  double r2 = r * r;
  *r_out = r;
  *f_out = 2.0 * r2 * r / (r2 * r2 + a * a * z * z);
  l[0] = 1.0;
  l[1] = (r * x + a * y) / (r2 + a * a);
  l[2] = (r * y - a * x) / (r2 + a * a);
  l[3] = z / r;
}

static const double ETA[4] = { -1.0, 1.0, 1.0, 1.0 };

/* PAPER.md:55 eq. (2): g_ab = eta_ab + f l_a l_b. */
void oracle_ks_metric(double a, const double pos[3], double g[16])
{
  double r, f, l[4];
  ks_f_l(a, pos, &r, &f, l);
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j)
      g[i * 4 + j] = (i == j ? ETA[i] : 0.0) + f * l[i] * l[j];
}

/* Inverse of a Kerr-Schild metric: g^ab = eta^ab - f l^a l^b, l^a = eta^ab l_b (l is null).
 * Not printed in the paper; pinned in tests by g * g^-1 = 1. */
void oracle_ks_metric_inverse(double a, const double pos[3], double gi[16])
{
  double r, f, l[4], lu[4];
  ks_f_l(a, pos, &r, &f, l);
  for (int i = 0; i < 4; ++i) lu[i] = ETA[i] * l[i];
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j)
      gi[i * 4 + j] = (i == j ? ETA[i] : 0.0) - f * lu[i] * lu[j];
}

/* C2.  Analytic first derivatives of the metric, d_c g_ab, by implicit differentiation of eq. (5):
 *   d_i r = f x_i / 2 (i = x,y),  d_z r = f z (r^2+a^2) / (2 r^2)
 *   d_i f = f [ (3/r - 2 f) d_i r - delta_iz 2 a^2 z / (r^4 + a^2 z^2) ]
 *   d_j l_x = [ d_j r (x - 2 r l_x) + r delta_jx + a delta_jy ] / (r^2+a^2)
 *   d_j l_y = [ d_j r (y - 2 r l_y) + r delta_jy - a delta_jx ] / (r^2+a^2)
 *   d_j l_z = ( delta_jz - l_z d_j r ) / r ,  d_j l_0 = 0 ,  d_t (anything) = 0.
 * Then d_c g_ab = (d_c f) l_a l_b + f (d_c l_a) l_b + f l_a (d_c l_b)   (64 numbers).
 * Layout: dg[c*16 + a*4 + b], c = derivative index (0 = t). */
void oracle_ks_dmetric(double a, const double pos[3], double dg[64])
{
  double x = pos[0], y = pos[1], z = pos[2];
  double r, f, l[4];
  ks_f_l(a, pos, &r, &f, l);
  double r2 = r * r, P = r2 + a * a, S = r2 * r2 + a * a * z * z;
  double dr[4], df[4], dl[4][4]; /* dr[c], df[c], dl[c][alpha] ; index 0 = t */
  dr[0] = 0.0;
  dr[1] = 0.5 * f * x;
  dr[2] = 0.5 * f * y;
  dr[3] = 0.5 * f * z * P / r2;
  for (int c = 0; c < 4; ++c) {
    double dcz = (c == 3) ? 1.0 : 0.0, dcx = (c == 1) ? 1.0 : 0.0, dcy = (c == 2) ? 1.0 : 0.0;
    df[c] = f * ((3.0 / r - 2.0 * f) * dr[c] - dcz * 2.0 * a * a * z / S);
    dl[c][0] = 0.0;
    dl[c][1] = (dr[c] * (x - 2.0 * r * l[1]) + r * dcx + a * dcy) / P;
    dl[c][2] = (dr[c] * (y - 2.0 * r * l[2]) + r * dcy - a * dcx) / P;
    dl[c][3] = (dcz - l[3] * dr[c]) / r;
  }
  df[0] = 0.0;
  for (int al = 0; al < 4; ++al) dl[0][al] = 0.0;
  for (int c = 0; c < 4; ++c)
    for (int i = 0; i < 4; ++i)
      for (int j = 0; j < 4; ++j)
        dg[c * 16 + i * 4 + j] = df[c] * l[i] * l[j] + f * dl[c][i] * l[j] + f * l[i] * dl[c][j];
}

/* Plainer variant: central differences of the metric itself (no analytic derivative at all). */
void oracle_ks_dmetric_fd(double a, const double pos[3], double step, double dg[64])
{
  double gp[16], gm[16], p[3];
  for (int k = 0; k < 16; ++k) dg[k] = 0.0; /* d_t g = 0 : metric is stationary */
  for (int c = 1; c < 4; ++c) {
    memcpy(p, pos, sizeof p);
    p[c - 1] = pos[c - 1] + step; oracle_ks_metric(a, p, gp);
    p[c - 1] = pos[c - 1] - step; oracle_ks_metric(a, p, gm);
    for (int k = 0; k < 16; ++k) dg[c * 16 + k] = (gp[k] - gm[k]) / (2.0 * step);
  }
}

/* PAPER.md:91 eq. (8): Gamma^m_ab = 1/2 g^{m nu} ( g_{nu a,b} + g_{nu b,a} - g_{ab,nu} ). */
static void christoffel_from(const double gi[16], const double dg[64], double Gam[64])
{
  for (int m = 0; m < 4; ++m)
    for (int al = 0; al < 4; ++al)
      for (int be = 0; be < 4; ++be) {
        double s = 0.0;
        for (int nu = 0; nu < 4; ++nu)
          s += gi[m * 4 + nu] * (dg[be * 16 + nu * 4 + al] + dg[al * 16 + nu * 4 + be] - dg[nu * 16 + al * 4 + be]);
        Gam[m * 16 + al * 4 + be] = 0.5 * s;
      }
}

void oracle_ks_christoffel(double a, const double pos[3], double Gam[64])
{
  double gi[16], dg[64];
  oracle_ks_metric_inverse(a, pos, gi);
  oracle_ks_dmetric(a, pos, dg);
  christoffel_from(gi, dg, Gam);
}

/* PAPER.md:87 eq. (7): xdd^m = - Gamma^m_ab xd^a xd^b, full triple loop, no regrouping. */
static void accel_from(const double Gam[64], const double u[4], double acc[4])
{
  for (int m = 0; m < 4; ++m) {
    double s = 0.0;
    for (int al = 0; al < 4; ++al)
      for (int be = 0; be < 4; ++be)
        s += Gam[m * 16 + al * 4 + be] * u[al] * u[be];
    acc[m] = -s;
  }
}

void oracle_ks_accel(double a, const double pos[3], const double u[4], double acc[4])
{
  double Gam[64];
  oracle_ks_christoffel(a, pos, Gam);
  accel_from(Gam, u, acc);
}

void oracle_ks_accel_fd(double a, const double pos[3], const double u[4], double step, double acc[4])
{
  double gi[16], dg[64], Gam[64];
  oracle_ks_metric_inverse(a, pos, gi);
  oracle_ks_dmetric_fd(a, pos, step, dg);
  christoffel_from(gi, dg, Gam);
  accel_from(Gam, u, acc);
}

/* C4.  y = (t,x,y,z,u^t,u^x,u^y,u^z);  y' = (u^mu, xdd^mu(x^i,u^mu)).  Autonomous. */
static void ks_deriv(double a, const double y[8], double dy[8])
{
  for (int m = 0; m < 4; ++m) dy[m] = y[4 + m];
  oracle_ks_accel(a, &y[1], &y[4], &dy[4]);
}

/* "classic 4th-order Runge-Kutta".
 *   k1 = y'(y), k2 = y'(y + h/2 k1), k3 = y'(y + h/2 k2), k4 = y'(y + h k3),
 *   y <- y + h/6 (k1 + 2 k2 + 2 k3 + k4). */
typedef void (*deriv_fn)(double a, const double y[8], double dy[8]);

static void rk4_generic(deriv_fn F, double a, double y[8], double h)
{
  double k1[8], k2[8], k3[8], k4[8], w[8];
  F(a, y, k1);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + 0.5 * h * k1[i];
  F(a, w, k2);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + 0.5 * h * k2[i];
  F(a, w, k3);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + h * k3[i];
  F(a, w, k4);
  for (int i = 0; i < 8; ++i) y[i] = y[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
}

void oracle_rk4_step(double a, double y[8], double h) { rk4_generic(ks_deriv, a, y, h); }

void oracle_trajectory(double a, const double y0[8], double h, int64_t nsteps, int64_t stride, double *out)
{
  double y[8];
  memcpy(y, y0, sizeof y);
  memcpy(out, y, sizeof y);
  int64_t rec = 1;
  for (int64_t s = 1; s <= nsteps; ++s) {
    oracle_rk4_step(a, y, h);
    if (s % stride == 0) { memcpy(out + 8 * rec, y, sizeof y); ++rec; }
  }
}

/* ------------------------------------------------------------------------------------------
 * C7.  Invariants.  u_0 = -u^0 + f U,  u_i = u^i + f l_i U,  U = l_a u^a  (index lowered with eq. 2).
 *   norm = u_a u^a                       (the paper's error indicator u^2)
 *   E    = -u_0                          (d_t is Killing)
 *   L_z  = x u_y - y u_x                 (x d_y - y d_x is Killing: rotating phi_KS rotates x+iy)
 *   Q    = u_theta^2 + cos^2(theta) [ a^2 (mu^2 - E^2) + L_z^2 / sin^2(theta) ]   (Carter; Table 1 "Q")
 * written without 1/sin(theta) (DESIGN R8), c = z/r, s^2 = 1 - c^2, P = r^2 + a^2:
 *   Q = P c^2 (u_x^2+u_y^2) - 2 r c (x u_x + y u_y) u_z + r^2 s^2 u_z^2 + a^2 c^2 (mu^2 - E^2)
 * mu^2 is the NOMINAL value from `kind` (0 null, 1 time-like).
 * ---------------------------------------------------------------------------------------- */
void oracle_invariants_one(double a, int32_t kind, const double y[8], double out[4])
{
  double r, f, l[4], g[16], ulow[4];
  const double *u = &y[4];
  ks_f_l(a, &y[1], &r, &f, l);
  oracle_ks_metric(a, &y[1], g);
  for (int i = 0; i < 4; ++i) {
    double s = 0.0;
    for (int j = 0; j < 4; ++j) s += g[i * 4 + j] * u[j];
    ulow[i] = s;
  }
  double norm = 0.0;
  for (int i = 0; i < 4; ++i) norm += ulow[i] * u[i];
  double E = -ulow[0];
  double x = y[1], yy = y[2], z = y[3];
  double Lz = x * ulow[2] - yy * ulow[1];
  double c = z / r, s2 = 1.0 - c * c, P = r * r + a * a;
  double mu2 = (kind == ORACLE_TIMELIKE) ? 1.0 : 0.0;
  double Q = P * c * c * (ulow[1] * ulow[1] + ulow[2] * ulow[2])
           - 2.0 * r * c * (x * ulow[1] + yy * ulow[2]) * ulow[3]
           + r * r * s2 * ulow[3] * ulow[3]
           + a * a * c * c * (mu2 - E * E);
  out[0] = E; out[1] = Lz; out[2] = Q; out[3] = norm;
}

int oracle_invariants(const oracle_state *s, uint64_t n, double *E, double *Lz, double *Q, double *norm)
{
  if (!s || n == 0 || n > s->n || !E || !Lz || !Q || !norm) return 1;
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < (int64_t)n; ++k) {
    double y[8], o[4];
    for (int m = 0; m < 8; ++m) y[m] = s->q[m][k];
    if (s->coords == ORACLE_BL) oracle_bl_invariants_one(s->a_eff, s->kind, y, o);
    else oracle_invariants_one(s->a_eff, s->kind, y, o);
    E[k] = o[0]; Lz[k] = o[1]; Q[k] = o[2]; norm[k] = o[3];
  }
  return 0;
}

/* u^t from g_ab u^a u^b = -mu^2 given the spatial components (future-directed root), DESIGN R3:
 *   -(u^t)^2 + |u|^2 + f (u^t + c)^2 = -mu^2 ,  c = l_i u^i
 *   (1-f) (u^t)^2 - 2 f c u^t - (|u|^2 + mu^2 + f c^2) = 0
 *   u^t = [ f c + sqrt( f^2 c^2 + (1-f)(|u|^2 + mu^2 + f c^2) ) ] / (1-f)      (needs f < 1) */
static double solve_ut(double a, const double pos[3], const double v[3], double mu2)
{
  double r, f, l[4];
  ks_f_l(a, pos, &r, &f, l);
  double c = l[1] * v[0] + l[2] * v[1] + l[3] * v[2];
  double A = 1.0 - f, B = f * c, C = v[0] * v[0] + v[1] * v[1] + v[2] * v[2] + mu2 + f * c * c;
  return (B + sqrt(B * B + A * C)) / A;
}

/* ------------------------------------------------------------------------------------------
 * Image-plane initial conditions ("integrate backwards null geodesics from an image
 * at an initial radius"; the construction itself is not in the paper: DESIGN R1-R3).
 *  R1 pixel centres: alpha_j = -Wa + (j+1/2) 2Wa/nx ; beta_k likewise ; index = k*nx + j.
 *  R2 observer direction n = (sin i, 0, cos i), e_alpha = (0,1,0), e_beta = (-cos i, 0, sin i);
 *     position = r_obs n + alpha e_alpha + beta e_beta in Cartesian KS ; t = 0 ; parallel rays.
 *  R3 the backward trace is run as the time-reversed forward problem: spin a_eff = -a,
 *     spatial tangent -n (unit Euclidean length), u^t = future-directed null root, dir = +1.
 * ---------------------------------------------------------------------------------------- */
int oracle_init_null(oracle_state *s, double a, double r_obs, double inc,
                     double Wa, double Wb, int32_t nx, int32_t ny)
{
  if (!s || nx <= 0 || ny <= 0 || (uint64_t)nx * (uint64_t)ny != s->n) return 1;
  if (!(fabs(a) <= 1.0) || !(r_obs > 1.0 + sqrt(1.0 - a * a))) return 1;
  double ae = -a;
  s->a_eff = ae; s->kind = ORACLE_NULL; s->reversed = 1; s->coords = ORACLE_KS;
  double si = sin(inc), ci = cos(inc);
  double nvec[3] = { si, 0.0, ci }, ea[3] = { 0.0, 1.0, 0.0 }, eb[3] = { -ci, 0.0, si };
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < ny; ++k)
    for (int64_t j = 0; j < nx; ++j) {
      double alpha = -Wa + ((double)j + 0.5) * (2.0 * Wa / (double)nx);
      double beta  = -Wb + ((double)k + 0.5) * (2.0 * Wb / (double)ny);
      double pos[3], v[3];
      for (int c = 0; c < 3; ++c) {
        pos[c] = r_obs * nvec[c] + alpha * ea[c] + beta * eb[c];
        v[c] = -nvec[c];
      }
      int64_t idx = k * nx + j;
      s->q[0][idx] = 0.0;
      s->q[1][idx] = pos[0]; s->q[2][idx] = pos[1]; s->q[3][idx] = pos[2];
      s->q[4][idx] = solve_ut(ae, pos, v, 0.0);
      s->q[5][idx] = v[0]; s->q[6][idx] = v[1]; s->q[7][idx] = v[2];
      s->lambda[idx] = 0.0; s->status[idx] = ORACLE_ACTIVE; s->nsteps[idx] = 0;
    }
  return 0;
}

/* Explicit 8-vectors ("8 variables") of either kind: the paper's convergence experiments start
 * from explicit data for photons (the spherical photon orbits of Table 1) and
 * for particles (the circular orbits with the v_z kick).  xu8 is AoS n x 8.
 * kind: ORACLE_NULL (mu^2 = 0) or ORACLE_TIMELIKE (mu^2 = 1); it is recorded in the state (Carter's Q uses
 * it, DESIGN R8) and renormalise_ut != 0 re-solves u^t from g u u = -mu^2 (DESIGN R7). */
int oracle_init_explicit(oracle_state *s, double a, const double *xu8, uint64_t n, int32_t kind, int32_t renorm)
{
  if (!s || !xu8 || n == 0 || n > s->n || !(fabs(a) <= 1.0)) return 1;
  if (kind != ORACLE_NULL && kind != ORACLE_TIMELIKE) return 1;
  s->a_eff = a; s->kind = kind; s->reversed = 0; s->coords = ORACLE_KS;
  for (uint64_t k = 0; k < n; ++k) {
    for (int m = 0; m < 8; ++m) s->q[m][k] = xu8[k * 8 + m];
    if (renorm) s->q[4][k] = solve_ut(a, &xu8[k * 8 + 1], &xu8[k * 8 + 5], kind == ORACLE_TIMELIKE ? 1.0 : 0.0);
    s->lambda[k] = 0.0; s->status[k] = ORACLE_ACTIVE; s->nsteps[k] = 0;
  }
  return 0;
}

int oracle_init_timelike(oracle_state *s, double a, const double *xu8, uint64_t n, int32_t renorm)
{
  return oracle_init_explicit(s, a, xu8, n, ORACLE_TIMELIKE, renorm);
}

/* ------------------------------------------------------------------------------------------
 * C5.  Driver loop for one geodesic (stopping rule PAPER.md:296-302: "pass by or are close enough
 * to the event horizon, or escape"; step rule and order of tests: DESIGN R4-R6).
 * ---------------------------------------------------------------------------------------- */
static int all_finite(const double y[8])
{
  for (int i = 0; i < 8; ++i) if (!isfinite(y[i])) return 0;
  return 1;
}

static void integrate_one(double a, int32_t coords, double y[8], double *lambda, int32_t *status,
                          int32_t *nsteps, double lambda_end, const oracle_step_control *sc)
{
  double r_plus = 1.0 + sqrt(1.0 - a * a);
  double dir = (double)sc->dir;
  while (*status == ORACLE_ACTIVE) {
    /* the radius of the stopping tests and of the step rule is the same scalar in both systems: the
       KS r of eq. (5) "is identical to" the BL r, which is a coordinate there */
    double r = (coords == ORACLE_BL) ? y[1] : oracle_ks_r(a, y[1], y[2], y[3]);
    if (!isfinite(r) || !all_finite(y)) { *status = ORACLE_INVALID; break; }
    if (r < sc->capture_factor * r_plus) { *status = ORACLE_CAPTURED; break; }
    if (r > sc->r_escape)                { *status = ORACLE_ESCAPED;  break; }
    if (*nsteps >= sc->max_steps)        { *status = ORACLE_MAXSTEPS; break; }
    if (dir * (lambda_end - *lambda) <= 0.0) break; /* stays ACTIVE: resumable */
    double h = dir * (sc->mode == 1 ? sc->eta * r : sc->h_fixed);
    /* clip the last step; the clock then lands on lambda_end itself, not on lambda + (lambda_end - lambda),
       which may differ from it by an ulp and would cost one more, ulp-sized, step (DESIGN R22) */
    int clipped = fabs(h) > fabs(lambda_end - *lambda);
    if (clipped) h = lambda_end - *lambda;
    if (coords == ORACLE_BL) {
      /* a stage at r < capture radius: CAPTURED at the state before this step (DESIGN R20) */
      if (oracle_bl_rk4_step_guarded(a, y, h, sc->capture_factor * r_plus)) { *status = ORACLE_CAPTURED; break; }
    } else oracle_rk4_step(a, y, h);
    *lambda = clipped ? lambda_end : *lambda + h;
    *nsteps += 1;
  }
}

int oracle_integrate(oracle_state *s, uint64_t n, double lambda_end,
                     const oracle_step_control *sc, oracle_stats *stats)
{
  if (!s || !sc || n == 0 || n > s->n) return 1;
  if (sc->mode == 1 ? !(sc->eta > 0.0) : !(sc->h_fixed > 0.0)) return 1;
  if (sc->dir != 1 && sc->dir != -1) return 1;
  uint64_t steps = 0, nc = 0, ne = 0, nm = 0, ni = 0, na = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : steps, nc, ne, nm, ni, na)
  for (int64_t k = 0; k < (int64_t)n; ++k) {
    double y[8];
    for (int m = 0; m < 8; ++m) y[m] = s->q[m][k];
    int32_t st = s->status[k], ns = s->nsteps[k], ns0 = ns;
    double lam = s->lambda[k];
    integrate_one(s->a_eff, s->coords, y, &lam, &st, &ns, lambda_end, sc);
    for (int m = 0; m < 8; ++m) s->q[m][k] = y[m];
    s->status[k] = st; s->nsteps[k] = ns; s->lambda[k] = lam;
    steps += (uint64_t)(ns - ns0);
    nc += (st == ORACLE_CAPTURED); ne += (st == ORACLE_ESCAPED); nm += (st == ORACLE_MAXSTEPS);
    ni += (st == ORACLE_INVALID);  na += (st == ORACLE_ACTIVE);
  }
  if (stats) {
    stats->steps = steps; stats->n_captured = nc; stats->n_escaped = ne;
    stats->n_maxsteps = nm; stats->n_invalid = ni; stats->n_active = na;
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * Coordinate-time integration (section 2.2).  v^mu = dx^mu/dt, v^0 = 1.
 * PAPER.md:131 eq. (15), literally, with the full connection:
 *   dv^i/dt = -Gamma^i_ab v^a v^b + Gamma^0_ab v^a v^b v^i
 * Six variables (x^i, v^i); t advances by exactly h per step.  The 8-array state is reused:
 * on entry v^i = u^i / u^t, on exit q[4] = 1 and q[5..7] = v^i (DESIGN R19).
 * ---------------------------------------------------------------------------------------- */
void oracle_ks_coordtime_accel(double a, const double pos[3], const double v[3], double dv[3])
{
  double Gam[64], u[4] = { 1.0, v[0], v[1], v[2] }, acc[4];
  oracle_ks_christoffel(a, pos, Gam);
  accel_from(Gam, u, acc);               /* acc^mu = -Gamma^mu_ab v^a v^b */
  for (int i = 0; i < 3; ++i) dv[i] = acc[1 + i] - acc[0] * v[i];
}

/* y = (x,y,z,vx,vy,vz); classic RK4 in t. */
static void ct_deriv(double a, const double y[6], double dy[6])
{
  for (int i = 0; i < 3; ++i) dy[i] = y[3 + i];
  oracle_ks_coordtime_accel(a, &y[0], &y[3], &dy[3]);
}

void oracle_rk4_step_coordtime(double a, double y[6], double h)
{
  double k1[6], k2[6], k3[6], k4[6], w[6];
  ct_deriv(a, y, k1);
  for (int i = 0; i < 6; ++i) w[i] = y[i] + 0.5 * h * k1[i];
  ct_deriv(a, w, k2);
  for (int i = 0; i < 6; ++i) w[i] = y[i] + 0.5 * h * k2[i];
  ct_deriv(a, w, k3);
  for (int i = 0; i < 6; ++i) w[i] = y[i] + h * k3[i];
  ct_deriv(a, w, k4);
  for (int i = 0; i < 6; ++i) y[i] = y[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
}

/* fixed-step trajectory in t: out rows are (t,x,y,z,vx,vy,vz), initial row first. */
void oracle_trajectory_coordtime(double a, const double y0[7], double h, int64_t nsteps, int64_t stride, double *out)
{
  double t = y0[0], y[6];
  memcpy(y, y0 + 1, sizeof y);
  out[0] = t; memcpy(out + 1, y, sizeof y);
  int64_t rec = 1;
  for (int64_t s = 1; s <= nsteps; ++s) {
    oracle_rk4_step_coordtime(a, y, h);
    t = y0[0] + (double)s * h;
    if (s % stride == 0) { out[7 * rec] = t; memcpy(out + 7 * rec + 1, y, sizeof y); ++rec; }
  }
}

int oracle_integrate_coordtime(oracle_state *s, uint64_t n, double t_end,
                               const oracle_step_control *sc, oracle_stats *stats)
{
  if (!s || !sc || n == 0 || n > s->n || s->coords != ORACLE_KS) return 1;
  if (sc->mode == 1 ? !(sc->eta > 0.0) : !(sc->h_fixed > 0.0)) return 1;
  if (sc->dir != 1 && sc->dir != -1) return 1;
  uint64_t steps = 0, nc = 0, ne = 0, nm = 0, ni = 0, na = 0;
  const double a = s->a_eff, r_plus = 1.0 + sqrt(1.0 - a * a), dir = (double)sc->dir;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : steps, nc, ne, nm, ni, na)
  for (int64_t k = 0; k < (int64_t)n; ++k) {
    int32_t st = s->status[k], ns = s->nsteps[k], ns0 = ns;
    if (st == ORACLE_ACTIVE) {
      double t = s->q[0][k], y[6];
      for (int i = 0; i < 3; ++i) { y[i] = s->q[1 + i][k]; y[3 + i] = s->q[5 + i][k] / s->q[4][k]; }
      for (;;) {
        double r = oracle_ks_r(a, y[0], y[1], y[2]);
        int fin = isfinite(r) && isfinite(t);
        for (int i = 0; i < 6; ++i) fin = fin && isfinite(y[i]);
        if (!fin) { st = ORACLE_INVALID; break; }
        if (r < sc->capture_factor * r_plus) { st = ORACLE_CAPTURED; break; }
        if (r > sc->r_escape) { st = ORACLE_ESCAPED; break; }
        if (ns >= sc->max_steps) { st = ORACLE_MAXSTEPS; break; }
        if (dir * (t_end - t) <= 0.0) break;
        double h = dir * (sc->mode == 1 ? sc->eta * r : sc->h_fixed);
        int clipped = fabs(h) > fabs(t_end - t);            /* DESIGN R22: land on t_end itself */
        if (clipped) h = t_end - t;
        oracle_rk4_step_coordtime(a, y, h);
        t = clipped ? t_end : t + h;
        ns += 1;
      }
      s->q[0][k] = t;
      for (int i = 0; i < 3; ++i) { s->q[1 + i][k] = y[i]; s->q[5 + i][k] = y[3 + i]; }
      s->q[4][k] = 1.0;
      s->status[k] = st; s->nsteps[k] = ns;
    }
    steps += (uint64_t)(ns - ns0);
    nc += (st == ORACLE_CAPTURED); ne += (st == ORACLE_ESCAPED); nm += (st == ORACLE_MAXSTEPS);
    ni += (st == ORACLE_INVALID);  na += (st == ORACLE_ACTIVE);
  }
  if (stats) {
    stats->steps = steps; stats->n_captured = nc; stats->n_escaped = ne;
    stats->n_maxsteps = nm; stats->n_invalid = ni; stats->n_active = na;
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * Diagnostics of the paper's convergence experiments, accumulated over the samples k = 0,1,2,...
 * (the states at the step boundaries of the driver loop above, the initial state included):
 *   max_abs_u2  max_k | g u u + mu^2 |                          PAPER.md:217, :231 (Fig. 4-5)
 *   cos_peak    first local maximum of c_k = |z_k| / r_k, refined by the quadratic through the three
 *               samples around it: c_i - (c_{i+1}-c_{i-1})^2 / (8 (c_{i-1} - 2 c_i + c_{i+1}))
 *                                                                PAPER.md:247 (Fig. 6-7)
 *   dphi_cycle  unfolded KS azimuth phi = atan2(y,x) - atan2(a,r) advanced up to the first upward zero
 *               of z (z_k < 0 <= z_{k+1}), located by linear interpolation, minus phi_0
 *                                                                PAPER.md:249 (Fig. 8)
 *   t_zmax1,2   KS times of the first two maxima of z, i.e. downward zeros of u^z (u^z_k > 0 >= u^z_{k+1}),
 *               linear interpolation in t                        PAPER.md:263 (Fig. 9)
 * Quantities that never occur are NaN.  out: 5 arrays of n doubles.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
  double u2max, cprev2, cprev1, peak, phi0, phiprev, phiunf, zprev, uzprev, tprev, dphi, tz[2];
  int64_t k;
  int have_peak, have_dphi, ntz;
} diag_acc;

static double wrap_pi(double d)
{
  while (d > M_PI) d -= 2.0 * M_PI;
  while (d <= -M_PI) d += 2.0 * M_PI;
  return d;
}

static void diag_sample(diag_acc *D, double a, int32_t kind, const double y[8])
{
  double inv[4];
  oracle_invariants_one(a, kind, y, inv);
  double u2 = fabs(inv[3] + (kind == ORACLE_TIMELIKE ? 1.0 : 0.0));
  double r = oracle_ks_r(a, y[1], y[2], y[3]);
  double c = fabs(y[3]) / r;
  double phi = atan2(y[2], y[1]) - atan2(a, r);
  if (D->k == 0) {
    D->u2max = u2; D->phi0 = phi; D->phiunf = phi;
  } else {
    if (u2 > D->u2max) D->u2max = u2;
    double phiunf = D->phiunf + wrap_pi(phi - D->phiprev);
    if (D->k >= 2 && !D->have_peak && D->cprev1 >= D->cprev2 && D->cprev1 > c) {
      double y0 = D->cprev2, y1 = D->cprev1, y2 = c;
      D->peak = y1 - (y2 - y0) * (y2 - y0) / (8.0 * (y0 - 2.0 * y1 + y2));
      D->have_peak = 1;
    }
    if (!D->have_dphi && D->zprev < 0.0 && y[3] >= 0.0) {     /* k >= 1 here: the pair (z_0, z_1) counts */
      double w = -D->zprev / (y[3] - D->zprev);
      D->dphi = D->phiunf + w * (phiunf - D->phiunf) - D->phi0;
      D->have_dphi = 1;
    }
    if (D->ntz < 2 && D->uzprev > 0.0 && y[7] <= 0.0) {
      D->tz[D->ntz] = D->tprev + (y[0] - D->tprev) * D->uzprev / (D->uzprev - y[7]);
      D->ntz += 1;
    }
    D->phiunf = phiunf;
  }
  D->cprev2 = D->cprev1; D->cprev1 = c;
  D->phiprev = phi; D->zprev = y[3]; D->uzprev = y[7]; D->tprev = y[0];
  D->k += 1;
}

int oracle_integrate_diagnostics(oracle_state *s, uint64_t n, double lambda_end,
                                 const oracle_step_control *sc, double *out5n, oracle_stats *stats)
{
  if (!s || !sc || !out5n || n == 0 || n > s->n || s->coords != ORACLE_KS) return 1;
  if (sc->mode == 1 ? !(sc->eta > 0.0) : !(sc->h_fixed > 0.0)) return 1;
  if (sc->dir != 1 && sc->dir != -1) return 1;
  uint64_t steps = 0, nc = 0, ne = 0, nm = 0, ni = 0, na = 0;
  const double a = s->a_eff, r_plus = 1.0 + sqrt(1.0 - a * a), dir = (double)sc->dir;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : steps, nc, ne, nm, ni, na)
  for (int64_t k = 0; k < (int64_t)n; ++k) {
    double y[8];
    for (int m = 0; m < 8; ++m) y[m] = s->q[m][k];
    int32_t st = s->status[k], ns = s->nsteps[k], ns0 = ns;
    double lam = s->lambda[k];
    diag_acc D;
    memset(&D, 0, sizeof D);
    D.peak = D.dphi = D.tz[0] = D.tz[1] = NAN;
    while (st == ORACLE_ACTIVE) {
      double r = oracle_ks_r(a, y[1], y[2], y[3]);
      if (!isfinite(r) || !all_finite(y)) { st = ORACLE_INVALID; break; }
      diag_sample(&D, a, s->kind, y);
      if (r < sc->capture_factor * r_plus) { st = ORACLE_CAPTURED; break; }
      if (r > sc->r_escape) { st = ORACLE_ESCAPED; break; }
      if (ns >= sc->max_steps) { st = ORACLE_MAXSTEPS; break; }
      if (dir * (lambda_end - lam) <= 0.0) break;
      double h = dir * (sc->mode == 1 ? sc->eta * r : sc->h_fixed);
      int clipped = fabs(h) > fabs(lambda_end - lam);     /* DESIGN R22: land on lambda_end itself */
      if (clipped) h = lambda_end - lam;
      oracle_rk4_step(a, y, h);
      lam = clipped ? lambda_end : lam + h;
      ns += 1;
    }
    for (int m = 0; m < 8; ++m) s->q[m][k] = y[m];
    s->status[k] = st; s->nsteps[k] = ns; s->lambda[k] = lam;
    out5n[0 * n + k] = D.k ? D.u2max : NAN;
    out5n[1 * n + k] = D.peak; out5n[2 * n + k] = D.dphi;
    out5n[3 * n + k] = D.tz[0]; out5n[4 * n + k] = D.tz[1];
    steps += (uint64_t)(ns - ns0);
    nc += (st == ORACLE_CAPTURED); ne += (st == ORACLE_ESCAPED); nm += (st == ORACLE_MAXSTEPS);
    ni += (st == ORACLE_INVALID);  na += (st == ORACLE_ACTIVE);
  }
  if (stats) {
    stats->steps = steps; stats->n_captured = nc; stats->n_escaped = ne;
    stats->n_maxsteps = nm; stats->n_invalid = ni; stats->n_active = na;
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * C8.  Boyer-Lindquist coordinates.
 * PAPER.md:47 eq. (1), M = 1, coordinates X = (t, r, theta, phi):
 *   ds^2 = -(1 - 2r/rho^2) dt^2 - (4 r a sin^2/rho^2) dphi dt + (rho^2/Delta) dr^2 + rho^2 dtheta^2
 *          + (r^2 + a^2 + 2 r a^2 sin^2/rho^2) sin^2 dphi^2 ,
 *   rho^2 = r^2 + a^2 cos^2(theta),  Delta = r^2 - 2 r + a^2.
 * The paper prints the metric only (5 elements, 10 derivatives, 20 Christoffel symbols);
 * here the derivatives are eq. (1) differentiated element by element (quotient rule, nothing regrouped),
 * the inverse comes from Gauss-Jordan elimination, and eq. (8), eq. (7) are the same generic routines
 * as for Kerr-Schild.  Nothing Kerr-Schild specific is used.  A second derivative routine takes 4th-order
 * central differences of the metric, so that the analytic one is pinned by something other than itself.
 * ---------------------------------------------------------------------------------------- */
void oracle_bl_metric(double a, const double X[4], double g[16])
{
  double r = X[1], th = X[2];
  double st = sin(th), ct = cos(th), s2 = st * st;
  double rho2 = r * r + a * a * ct * ct, Delta = r * r - 2.0 * r + a * a;
  for (int k = 0; k < 16; ++k) g[k] = 0.0;
  g[0 * 4 + 0] = -(1.0 - 2.0 * r / rho2);
  g[0 * 4 + 3] = g[3 * 4 + 0] = -2.0 * r * a * s2 / rho2;
  g[1 * 4 + 1] = rho2 / Delta;
  g[2 * 4 + 2] = rho2;
  g[3 * 4 + 3] = (r * r + a * a + 2.0 * r * a * a * s2 / rho2) * s2;
}

void oracle_bl_dmetric(double a, const double X[4], double dg[64])
{
  double r = X[1], th = X[2];
  double s = sin(th), c = cos(th), s2 = s * s, s4 = s2 * s2, a2 = a * a;
  double rho2 = r * r + a2 * c * c, rho4 = rho2 * rho2, Delta = r * r - 2.0 * r + a2;
  double rho2_r = 2.0 * r, rho2_th = -2.0 * a2 * s * c, Delta_r = 2.0 * r - 2.0;
  for (int k = 0; k < 64; ++k) dg[k] = 0.0;
  double *dr = &dg[1 * 16], *dt = &dg[2 * 16];          /* d/dr and d/dtheta; d/dt = d/dphi = 0 */
  /* g_tt = -1 + 2r/rho2 */
  dr[0 * 4 + 0] = 2.0 / rho2 - 2.0 * r * rho2_r / rho4;
  dt[0 * 4 + 0] = -2.0 * r * rho2_th / rho4;
  /* g_tphi = -2 r a s2 / rho2 */
  dr[0 * 4 + 3] = dr[3 * 4 + 0] = -2.0 * a * s2 / rho2 + 2.0 * r * a * s2 * rho2_r / rho4;
  dt[0 * 4 + 3] = dt[3 * 4 + 0] = -4.0 * r * a * s * c / rho2 + 2.0 * r * a * s2 * rho2_th / rho4;
  /* g_rr = rho2 / Delta */
  dr[1 * 4 + 1] = rho2_r / Delta - rho2 * Delta_r / (Delta * Delta);
  dt[1 * 4 + 1] = rho2_th / Delta;
  /* g_thth = rho2 */
  dr[2 * 4 + 2] = rho2_r;
  dt[2 * 4 + 2] = rho2_th;
  /* g_phiphi = (r^2 + a^2) s2 + 2 r a^2 s4 / rho2 */
  dr[3 * 4 + 3] = 2.0 * r * s2 + 2.0 * a2 * s4 / rho2 - 2.0 * r * a2 * s4 * rho2_r / rho4;
  dt[3 * 4 + 3] = 2.0 * (r * r + a2) * s * c + 8.0 * r * a2 * s2 * s * c / rho2 - 2.0 * r * a2 * s4 * rho2_th / rho4;
}

void oracle_bl_dmetric_fd(double a, const double X[4], double dg[64])
{
  for (int k = 0; k < 64; ++k) dg[k] = 0.0;
  for (int c = 1; c <= 2; ++c) { /* metric depends on r and theta only */
    double step = 1e-3 * (c == 1 ? fmax(1.0, fabs(X[1])) : 1.0);
    double Y[4], g1p[16], g1m[16], g2p[16], g2m[16];
    memcpy(Y, X, sizeof Y);
    Y[c] = X[c] + step;       oracle_bl_metric(a, Y, g1p);
    Y[c] = X[c] - step;       oracle_bl_metric(a, Y, g1m);
    Y[c] = X[c] + 2.0 * step; oracle_bl_metric(a, Y, g2p);
    Y[c] = X[c] - 2.0 * step; oracle_bl_metric(a, Y, g2m);
    for (int k = 0; k < 16; ++k)
      dg[c * 16 + k] = (8.0 * (g1p[k] - g1m[k]) - (g2p[k] - g2m[k])) / (12.0 * step);
  }
}

static void invert4(const double m[16], double inv[16])
{
  double A[4][8];
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j) { A[i][j] = m[i * 4 + j]; A[i][4 + j] = (i == j) ? 1.0 : 0.0; }
  for (int c = 0; c < 4; ++c) {
    int p = c;
    for (int i = c + 1; i < 4; ++i) if (fabs(A[i][c]) > fabs(A[p][c])) p = i;
    if (p != c) for (int j = 0; j < 8; ++j) { double t = A[c][j]; A[c][j] = A[p][j]; A[p][j] = t; }
    double d = A[c][c];
    for (int j = 0; j < 8; ++j) A[c][j] /= d;
    for (int i = 0; i < 4; ++i) if (i != c) {
      double fct = A[i][c];
      for (int j = 0; j < 8; ++j) A[i][j] -= fct * A[c][j];
    }
  }
  for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) inv[i * 4 + j] = A[i][4 + j];
}

void oracle_bl_accel(double a, const double X[4], const double u[4], double acc[4])
{
  double g[16], gi[16], dg[64], Gam[64];
  oracle_bl_metric(a, X, g);
  invert4(g, gi);
  oracle_bl_dmetric(a, X, dg);
  christoffel_from(gi, dg, Gam);
  accel_from(Gam, u, acc);
}

void oracle_bl_accel_fd(double a, const double X[4], const double u[4], double acc[4])
{
  double g[16], gi[16], dg[64], Gam[64];
  oracle_bl_metric(a, X, g);
  invert4(g, gi);
  oracle_bl_dmetric_fd(a, X, dg);
  christoffel_from(gi, dg, Gam);
  accel_from(Gam, u, acc);
}

static void bl_deriv(double a, const double y[8], double dy[8])
{
  for (int m = 0; m < 4; ++m) dy[m] = y[4 + m];
  oracle_bl_accel(a, &y[0], &y[4], &dy[4]);
}

void oracle_bl_rk4_step(double a, double y[8], double h) { rk4_generic(bl_deriv, a, y, h); }

/* The same classic RK4 step with the capture test applied to the positions at which stages 2-4 are
 * evaluated (DESIGN R20): eq. (1) is singular at Delta = 0, so a stage evaluated at or beyond
 * the horizon is meaningless, and with h = eta r a geodesic that falls in reaches it within one step of
 * r = capture_factor r_+.  Returns 1 and leaves y untouched if the radius of a stage position, or of the
 * result of the step, is below r_capture: the last stored state of a captured ray is then one that only
 * well-defined evaluations have produced. */
int oracle_bl_rk4_step_guarded(double a, double y[8], double h, double r_capture)
{
  double k1[8], k2[8], k3[8], k4[8], w[8];
  bl_deriv(a, y, k1);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + 0.5 * h * k1[i];
  if (w[1] < r_capture) return 1;
  bl_deriv(a, w, k2);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + 0.5 * h * k2[i];
  if (w[1] < r_capture) return 1;
  bl_deriv(a, w, k3);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + h * k3[i];
  if (w[1] < r_capture) return 1;
  bl_deriv(a, w, k4);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
  if (w[1] < r_capture) return 1;       /* the result of the step is held to the same test */
  memcpy(y, w, sizeof w);
  return 0;
}

void oracle_bl_trajectory(double a, const double y0[8], double h, int64_t nsteps, int64_t stride, double *out)
{
  double y[8];
  memcpy(y, y0, sizeof y);
  memcpy(out, y, sizeof y);
  int64_t rec = 1;
  for (int64_t s = 1; s <= nsteps; ++s) {
    rk4_generic(bl_deriv, a, y, h);
    if (s % stride == 0) { memcpy(out + 8 * rec, y, sizeof y); ++rec; }
  }
}

/* E = -u_t, L_z = u_phi, Carter's Q = u_theta^2 + cos^2(theta) [a^2 (mu^2 - E^2) + L_z^2 / sin^2(theta)]
   (Carter 1968; the paper's Table 1 lists Phi = L_z/E and Q/E^2), u.u = g_ab u^a u^b;
   indices lowered with eq. (1). */
void oracle_bl_invariants_one(double a, int32_t kind, const double y[8], double out[4])
{
  double g[16], ulow[4];
  const double *u = &y[4];
  oracle_bl_metric(a, &y[0], g);
  for (int i = 0; i < 4; ++i) {
    double s = 0.0;
    for (int j = 0; j < 4; ++j) s += g[i * 4 + j] * u[j];
    ulow[i] = s;
  }
  double norm = 0.0;
  for (int i = 0; i < 4; ++i) norm += ulow[i] * u[i];
  double E = -ulow[0], Lz = ulow[3];
  double st = sin(y[2]), ct = cos(y[2]);
  double mu2 = (kind == ORACLE_TIMELIKE) ? 1.0 : 0.0;
  double Q = ulow[2] * ulow[2] + ct * ct * (a * a * (mu2 - E * E) + Lz * Lz / (st * st));
  out[0] = E; out[1] = Lz; out[2] = Q; out[3] = norm;
}

/* T(r) and Phi(r) with dT/dr = 2r/Delta, dPhi/dr = a/Delta (partial fractions over the roots r_+- of Delta;
   the double root of the extremal case integrates to a pole instead of a logarithm). */
static void bl_shift(double a, double r, double *T, double *Phi)
{
  double d2 = 1.0 - a * a;
  if (d2 > 0.0) {
    double rp = 1.0 + sqrt(d2), rm = 1.0 - sqrt(d2);
    *T = 2.0 / (rp - rm) * (rp * log(fabs(r - rp)) - rm * log(fabs(r - rm)));
    *Phi = a / (rp - rm) * log(fabs((r - rp) / (r - rm)));
  } else {
    *T = 2.0 * log(fabs(r - 1.0)) - 2.0 / (r - 1.0);
    *Phi = -a / (r - 1.0);
  }
}

/* J[i][j] = d(t_KS, x, y, z)_i / d(t_BL, r, theta, phi_BL)_j at the point (r, theta, phi_KS). */
static void bl_jacobian(double a, double r, double th, double ph_ks, double J[16])
{
  double Delta = r * r - 2.0 * r + a * a;
  double st = sin(th), ct = cos(th), cp = cos(ph_ks), sp = sin(ph_ks);
  double x = (r * cp - a * sp) * st, y = (r * sp + a * cp) * st;
  double dph_dr = a / Delta;                    /* d phi_KS / d r at fixed phi_BL */
  for (int k = 0; k < 16; ++k) J[k] = 0.0;
  J[0 * 4 + 0] = 1.0;
  J[0 * 4 + 1] = 2.0 * r / Delta;
  J[1 * 4 + 1] = cp * st - y * dph_dr;
  J[2 * 4 + 1] = sp * st + x * dph_dr;
  J[3 * 4 + 1] = ct;
  J[1 * 4 + 2] = (r * cp - a * sp) * ct;
  J[2 * 4 + 2] = (r * sp + a * cp) * ct;
  J[3 * 4 + 2] = -r * st;
  J[1 * 4 + 3] = -y;
  J[2 * 4 + 3] = x;
}

void oracle_bl_to_ks_one(double a, const double yb[8], double yk[8])
{
  double r = yb[1], th = yb[2], T, Phi, J[16];
  bl_shift(a, r, &T, &Phi);
  double ph_ks = yb[3] + Phi;
  yk[0] = yb[0] + T;
  yk[1] = (r * cos(ph_ks) - a * sin(ph_ks)) * sin(th);
  yk[2] = (r * sin(ph_ks) + a * cos(ph_ks)) * sin(th);
  yk[3] = r * cos(th);
  bl_jacobian(a, r, th, ph_ks, J);
  for (int i = 0; i < 4; ++i) {
    double s = 0.0;
    for (int j = 0; j < 4; ++j) s += J[i * 4 + j] * yb[4 + j];
    yk[4 + i] = s;
  }
}

/* The inverse map: r from eq. (5), theta = arccos(z/r) in [0, pi], phi_KS = arg(x + i y) - arg(r + i a);
   the velocity solves J u_BL = u_KS (Gauss-Jordan).  On the axis J is singular and the result is not
   finite: that is the coordinate singularity of the BL system, reported as data. */
void oracle_ks_to_bl_one(double a, const double yk[8], double yb[8])
{
  double r = oracle_ks_r(a, yk[1], yk[2], yk[3]);
  double c = yk[3] / r;
  if (c > 1.0) c = 1.0;
  if (c < -1.0) c = -1.0;
  double th = acos(c);
  double ph_ks = atan2(yk[2], yk[1]) - atan2(a, r);
  double T, Phi, J[16], Ji[16];
  bl_shift(a, r, &T, &Phi);
  yb[0] = yk[0] - T; yb[1] = r; yb[2] = th; yb[3] = ph_ks - Phi;
  bl_jacobian(a, r, th, ph_ks, J);
  invert4(J, Ji);
  for (int i = 0; i < 4; ++i) {
    double s = 0.0;
    for (int j = 0; j < 4; ++j) s += Ji[i * 4 + j] * yk[4 + j];
    yb[4 + i] = s;
  }
}

int oracle_convert(const oracle_state *src, oracle_state *dst, uint64_t n, int32_t to_coords)
{
  if (!src || !dst || n == 0 || n > src->n || n > dst->n) return 1;
  if (to_coords != ORACLE_KS && to_coords != ORACLE_BL) return 1;
  if (src->coords == to_coords) return 1;
  dst->a_eff = src->a_eff; dst->kind = src->kind; dst->reversed = src->reversed; dst->coords = to_coords;
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < (int64_t)n; ++k) {
    double yi[8], yo[8];
    for (int m = 0; m < 8; ++m) yi[m] = src->q[m][k];
    if (to_coords == ORACLE_BL) oracle_ks_to_bl_one(src->a_eff, yi, yo);
    else oracle_bl_to_ks_one(src->a_eff, yi, yo);
    for (int m = 0; m < 8; ++m) dst->q[m][k] = yo[m];
    dst->lambda[k] = src->lambda[k]; dst->status[k] = src->status[k]; dst->nsteps[k] = src->nsteps[k];
  }
  return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
