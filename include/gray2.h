/*
 * gray2.h -- C-ABI of the B200-native batched Kerr-Schild geodesic integrator
 *            (data-parallel hot path of GRay2, Chan et al. 2017, arXiv:1706.07062).
 *
 * "PAPER.md:N" cites line N of the paper text; "DESIGN Rn" the numbered readings in DESIGN.md that
 * fill the points the paper leaves open.  Units G = c = M = 1.
 *
 * What is computed (all of it in CUDA kernels for sm_100a; there is no CPU fallback):
 *   gray2_init_null      image-plane initial conditions of null geodesics      PAPER.md:296; DESIGN R1-R3
 *   gray2_init_explicit  explicit 8-vectors (t,x,y,z,u^t,u^x,u^y,u^z) of photons or particles
 *   (gray2_init_timelike: its time-like case)
 *   gray2_integrate      classic RK4 of the geodesic equation in Cartesian Kerr-Schild
 *                        coordinates, metric g = eta + f l l (eq. 2-5), right-hand side in
 *                        the regrouped form of eq. (10)-(14), each geodesic advanced
 *                        until it is close to the horizon, escapes, or exhausts its step budget
 *
 *   gray2_invariants     E, L_z, Carter Q and u.u ("u^2"; Table 1 "Phi", "Q")
 * and, around these four: gray2_integrate_coordtime (the coordinate-time form),
 * gray2_integrate_diagnostics (the convergence measurements of section 3), gray2_convert plus
 * gray2_state.coords (the Boyer-Lindquist system of the paper's Table 2, behind the same gray2_integrate),
 * gray2_init_null_shard (one image shared by several GPUs), gray2_state.order plus
 * gray2_order_longest_first (an optional schedule of the integrators), gray2_init_explicit_noalloc (explicit
 * initial data for programs that must not allocate GPU memory).
 *
 * Memory and ownership.  Every pointer inside gray2_state, and every output array, is a DEVICE pointer
 * owned by the caller (e.g. a torch tensor) and only borrowed while the enqueued work runs.  The
 * library allocates no device memory of its own except a 4 KiB work-queue scratch per device (64 slots
 * handed out round-robin; a call that gets a slot whose previous user is still running waits for it on
 * the device, so any number of integrations may be in flight), the 32 KiB histogram of
 * gray2_order_longest_first (per device, allocated at its first call) and the staging buffers
 * of gray2_init_explicit (per device; n x 64 bytes each, one per calling stream up to eight, grown on demand,
 * reused, released at process exit).  Not allocated but part of the library's device code, and so held by every
 * GPU that loads it: the fixed 4 MiB staging array of gray2_init_explicit_noalloc.  `host_xu8` is a HOST pointer.
 * gray2_state and gray2_step_control themselves are HOST structs, read during the call.
 *
 * Threads.  Any number of host threads may call into the library at once (the scratch pools are locked, the
 * launch choice of gray2_set_launch is one atomic word per precision); two calls that write the same
 * gray2_state must be ordered by the caller.
 *
 * Devices.  Work runs on the CUDA device that is current in the calling thread; all pointers and the
 * stream must belong to it.  Every call may be used on several devices of one process: the library's own
 * scratch (work queues, staging buffers, copy stream) is kept per device.
 *
 * Asynchrony.  Every call enqueues on `cuda_stream` (a cudaStream_t passed as void*, NULL = default
 * stream) and returns; results are valid after the caller synchronises that stream.
 *
 * Errors.  Every call returns a gray2_err; nothing throws or aborts.  GRAY2_EINVAL: bad argument
 * (NULL pointer, n == 0, |a| > 1, r_obs <= r_plus, nx*ny != s->n, eta <= 0, prec mismatch, ...).
 * GRAY2_ESTATE: n larger than s->n.  GRAY2_ECUDA: a CUDA runtime error (text via gray2_last_error()).
 * Numerical trouble of a single geodesic is data (status GRAY2_INVALID), never an error.
 *
 * Determinism.  No arithmetic crosses geodesics: every output element depends only on that geodesic's
 * input, not on scheduling, so results are bit-reproducible run to run.
 */
#ifndef GRAY2_H
#define GRAY2_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { GRAY2_F64 = 0, GRAY2_F32 = 1 } gray2_precision;
typedef enum { GRAY2_NULL = 0, GRAY2_TIMELIKE = 1 } gray2_kind;        /* nominal mu^2 = 0 or 1 */
typedef enum { GRAY2_ACTIVE = 0, GRAY2_CAPTURED = 1, GRAY2_ESCAPED = 2,
               GRAY2_MAXSTEPS = 3, GRAY2_INVALID = 4 } gray2_ray_status;
typedef enum { GRAY2_OK = 0, GRAY2_EINVAL = 1, GRAY2_ESTATE = 2, GRAY2_ECUDA = 3 } gray2_err;
/* Coordinates of a state.  GRAY2_KS: Cartesian Kerr-Schild, the system of the method.
 * GRAY2_BL: Boyer-Lindquist (eq. 1), the second system of the paper's benchmark (Table 2 "BL"
 * rows): q = t,r,theta,phi,u^t,u^r,u^theta,u^phi. */
typedef enum { GRAY2_KS = 0, GRAY2_BL = 1 } gray2_coords;

/* State of n geodesics, structure of arrays (8 variables per geodesic; SoA: PAPER.md:316). */
typedef struct {
  void    *q[8];        /* t,x,y,z,u^t,u^x,u^y,u^z : n elements each, double (F64) or float (F32)      */
  double  *lambda;      /* n : affine parameter reached (always double)                                 */
  int32_t *status;      /* n : gray2_ray_status                                                         */
  int32_t *nsteps;      /* n : RK4 steps taken so far                                                   */
  uint64_t n;
  double   a_eff;       /* spin used by the integrator; = -a for states made by gray2_init_null (R3)    */
  int32_t  prec;        /* gray2_precision of q[]                                                       */
  int32_t  kind;        /* gray2_kind: mu^2 inside Carter's Q (gray2_invariants) and |u.u + mu^2| (diagnostics) */
  int32_t  reversed;    /* 1: time-reversed ray of a backward trace (physical t = -t, L_z = -L_z)       */
  int32_t  coords;      /* gray2_coords of q[]; set to GRAY2_KS by gray2_init_*, to the target by         */
                        /* gray2_convert; gray2_integrate and gray2_invariants follow it                  */
  const int32_t *order; /* optional (NULL = none): DEVICE array of n int32, a permutation of 0..n-1.  The   */
                        /* integrators hand geodesic order[k] to the k-th lane that asks for work (SURVEY   */
                        /* 8(a) a6, 8(b): "optional order array").  It changes the schedule only -- no       */
                        /* output bit depends on it -- and is used only by calls that cover all n geodesics.  */
                        /* Longest first shortens the tail of a launch (gray2_order_longest_first).           */
                        /* A wrong array is data, not an error: an entry outside 0..n-1 is passed over; a       */
                        /* geodesic listed twice is integrated by two lanes that store the same bits (its steps  */
                        /* are counted twice in gray2_stats.steps); a geodesic listed nowhere is not touched      */
                        /* and stays ACTIVE (gray2_stats.n_active tells).                                         */
} gray2_state;
/* Fill a gray2_state from zero (memset or = {0}): fields added by later versions of this header (`order` so far)
 * mean "not used" when zero, and the library reads every field. */

/* Step and stopping rule (DESIGN R4-R6).  For every geodesic with status ACTIVE, repeat:
 *   r = Kerr-Schild radius of the current position (eq. 5);
 *   not finite -> INVALID;  r < capture_factor * r_plus -> CAPTURED;  r > r_escape -> ESCAPED;
 *   nsteps >= max_steps -> MAXSTEPS;  dir*(lambda_end - lambda) <= 0 -> return, still ACTIVE;
 *   h = dir * (mode == 1 ? eta * r : h_fixed), clipped so that lambda does not pass lambda_end;
 *   one RK4 step of size h;  lambda += h;  nsteps += 1.
 * The stored state is the state at which a test fired (no interpolation).  r_plus = 1 + sqrt(1 - a^2). */
typedef struct {
  int32_t mode;            /* 0: fixed step ; 1: radius-scaled step                                     */
  double  h_fixed, eta;
  int32_t dir;             /* +1 or -1 (states from gray2_init_null are run with +1)                    */
  double  capture_factor;  /* e.g. 1.01                                                                 */
  double  r_escape;        /* +inf allowed                                                              */
  int32_t max_steps;       /* per-geodesic total, counted from the state's nsteps                       */
} gray2_step_control;

typedef struct { uint64_t steps, n_captured, n_escaped, n_maxsteps, n_invalid, n_active; } gray2_stats;

/* Image-plane initial conditions.  Pixel (j,k), j = 0..nx-1 fastest, index k*nx + j,
 * has impact parameters alpha_j = -fov_half_alpha + (j+1/2) 2 fov_half_alpha / nx, beta_k likewise (R1).
 * Observer direction n = (sin i, 0, cos i), e_alpha = (0,1,0), e_beta = (-cos i, 0, sin i); the ray
 * starts at r_obs n + alpha e_alpha + beta e_beta, t = 0 (R2).  The backward trace is set up as the
 * time-reversed forward problem (R3): s->a_eff = -a, s->reversed = 1, spatial tangent -n, u^t the
 * future-directed root of g u u = 0.  Also sets s->kind = GRAY2_NULL, lambda = 0, status = ACTIVE,
 * nsteps = 0.  s->q, s->lambda, s->status, s->nsteps, s->n and s->prec must be filled by the caller. */
int gray2_init_null(gray2_state *s, double a, double r_obs, double inclination_rad,
                    double fov_half_alpha, double fov_half_beta, int32_t nx, int32_t ny,
                    void *cuda_stream);
/* One image shared by `world` GPUs (geodesics are independent, "trivially parallelizable";
 * SURVEY 8(e)): the nx*ny ray indices are dealt out in tiles of tile_rays consecutive indices, tile t to rank
 * t mod world, so that the long near-critical rays spread evenly over the GPUs.  Fills the rays of rank
 * `rank`, compactly: shard-local ray j is the image's ray ((j / tile_rays) * world + rank) * tile_rays +
 * j % tile_rays, with the same initial data, bit for bit, as gray2_init_null gives that ray.  s->n must equal
 * gray2_shard_count(nx*ny, tile_rays, rank, world).  No data moves between GPUs during integration; the
 * caller gathers the shards afterwards if it wants the image in one place. */
int gray2_init_null_shard(gray2_state *s, double a, double r_obs, double inclination_rad,
                          double fov_half_alpha, double fov_half_beta, int32_t nx, int32_t ny,
                          uint64_t tile_rays, int32_t rank, int32_t world, void *cuda_stream);
uint64_t gray2_shard_count(uint64_t n, uint64_t tile_rays, int32_t rank, int32_t world);   /* 0 on bad arguments */

/* Explicit initial conditions of either kind.  The paper's convergence experiments start from explicit data
 * for PHOTONS (the six spherical photon orbits of Table 1) and for PARTICLES
 * (circular orbits with a v_z kick); the state has 8 variables per geodesic.
 * host_xu8: HOST array of n x 8 doubles (AoS: t,x,y,z,u^t,u^x,u^y,u^z).  Copies them into the first n slots
 * of the SoA state (converted to float for F32).  kind: GRAY2_NULL (mu^2 = 0) or GRAY2_TIMELIKE (mu^2 = 1);
 * with renormalise_ut != 0 u^t is replaced by the future-directed root of g u u = -mu^2 (R7).  Sets
 * s->a_eff = a, s->kind = kind (Carter's Q in gray2_invariants follows it, R8), s->reversed = 0,
 * lambda = 0, status = ACTIVE, nsteps = 0.  The host array may be reused as soon as the call returns: the
 * call waits for its own host-to-device copy (made on an internal stream of the current device, so that it
 * does not queue behind earlier work on cuda_stream) and for nothing else; the state is filled in stream
 * order on cuda_stream like the output of every other call.  GRAY2_EINVAL for an unknown kind. */
int gray2_init_explicit(gray2_state *s, double a, const double *host_xu8, uint64_t n, int32_t kind,
                        int32_t renormalise_ut, void *cuda_stream);
/* The call north_star names: gray2_init_explicit with kind = GRAY2_TIMELIKE. */
int gray2_init_timelike(gray2_state *s, double a, const double *host_xu8, uint64_t n,
                        int32_t renormalise_ut, void *cuda_stream);

/* gray2_init_explicit for programs that must not allocate GPU memory: same arguments, same kernel, same state
 * bit for bit, but the call allocates and frees nothing, on its first use or ever.
 *
 * Who needs it.  gray2_init_explicit parks the host array in a device buffer that the library owns and replaces
 * (cudaFree, then cudaMalloc) whenever a call brings more geodesics than the slot of its stream has held so far.
 * Which call does that depends on n and on the stream, so one warm-up call does not get it out of the way.  That
 * is no good for
 *   - a program that has handed nearly all of the GPU's memory to an allocator of its own (torch's caching
 *     allocator after a large reservation, a renderer's arena, a job held to a fixed budget beside other tenants):
 *     a cudaMalloc from inside this library fails there with out-of-memory, or takes memory the program counted on;
 *   - a frame or control loop (the paper's interactive mode integrates and draws every frame):
 *     cudaMalloc and cudaFree make the whole device wait, so the one call that grows the buffer stalls every other
 *     stream for that frame;
 *   - a program whose memory is checked once at start-up and locked down afterwards.
 *
 * What it uses instead.  A fixed staging array of GRAY2_NOALLOC_MAX_GEODESICS x 64 bytes = 4 MiB that is part
 * of the library's device code: every GPU on which the library's kernels are loaded holds those 4 MiB from then
 * until the process exits, whether this call is ever made or not.  n > GRAY2_NOALLOC_MAX_GEODESICS is refused
 * with GRAY2_EINVAL (the error text names the limit) and nothing is enqueued: feed a larger batch in pieces,
 * each piece into its own part of the state (a gray2_state whose pointers are offset), one after the other on
 * one stream.
 *
 * First call on a device.  It looks up where the array lives on the current device (cudaGetSymbolAddress, which
 * makes the CUDA runtime load the library's device code there if it has not yet) and keeps the answer; later
 * calls on that device only enqueue.  Make that first call on each device while the program starts up, before
 * any stream capture begins.
 *
 * One array for everybody.  All calls on a device, from any stream or host thread, stage through the same
 * array, and it keeps what the last call left in it.  Nothing in it has to start at zero: the call overwrites
 * the first 64 n bytes and its kernel reads exactly those, so old contents are never seen.  But two calls whose
 * GPU work can overlap -- different streams with nothing ordering them -- write and read the array at the same
 * time and both come out wrong; the library does not detect this.  Calls on one stream are safe (stream order),
 * and so are calls on different devices (each device has its own copy of the array).
 *
 * The host array.  The copy is enqueued on cuda_stream itself (there is no internal stream and no event on this
 * path), so unlike gray2_init_explicit the call does not wait for it: host_xu8 must stay valid and unchanged
 * until cuda_stream has got past this call (pageable memory is read before the call returns, pinned memory when
 * the stream reaches the copy).  Everything else -- kind, renormalise_ut, the fields set in s, the errors -- is
 * as for gray2_init_explicit. */
#define GRAY2_NOALLOC_MAX_GEODESICS 65536
int gray2_init_explicit_noalloc(gray2_state *s, double a, const double *host_xu8, uint64_t n, int32_t kind,
                                int32_t renormalise_ut, void *cuda_stream);

/* Integrate the first n geodesics of s (see gray2_step_control).  Only ACTIVE geodesics are touched, so
 * the call is resumable and a second identical call is a no-op.  prec must equal s->prec.
 * FP32 states: the right-hand side is evaluated in float, the eight state sums y <- y + (h/6)(k1+2k2+2k3+k4)
 * are carried with a float residual each (compensated summation) while a geodesic lives in registers, so
 * that the low bits of the ~1000 small increments of a ray are not rounded away one by one (DESIGN R12); the
 * residual is dropped when the geodesic is stored, i.e. at every call boundary the state is plain float.
 * The clipped last step lands on lambda_end itself (R22).
 * device_stats: DEVICE pointer to one gray2_stats, or NULL; it is OVERWRITTEN with the RK4 steps taken
 * by this call and the final status counts over the first n geodesics.
 *
 * Boyer-Lindquist states (s->coords = GRAY2_BL, made by gray2_convert): the same classic RK4, the same step
 * and stopping rule with r = q[1] (the BL radius "is identical to" the KS r of eq. 5), the
 * right-hand side being the Euler-Lagrange equations of eq. (1) (the paper prints the metric only; form
 * and derivation: csrc/bl_geodesic.cuh).  Eq. (1) is singular on the horizon and on the axis
 * (PAPER.md:49-51).  Horizon (DESIGN R20): the capture test is applied to the positions of RK4 stages 2-4 and
 * to the result of the step as well; if one of them has r < capture_factor * r_plus the step is rejected
 * and the geodesic ends as CAPTURED at the state it had before that step, so no evaluation ever takes place
 * at Delta <= 0.  Axis (DESIGN R21): nothing is done; with h = eta r a passage closer to the axis than about
 * 2 eta radians is not resolved and such geodesics come out wrong (the paper's reason for Kerr-Schild
 * coordinates); a state exactly on the axis has no finite BL velocity and ends as GRAY2_INVALID. */
int gray2_integrate(gray2_state *s, uint64_t n, double lambda_end, const gray2_step_control *sc,
                    int32_t prec, gray2_stats *device_stats, void *cuda_stream);
/* The coordinate map between the two systems for the first n geodesics (the paper's Appendix is missing,
 * PAPER.md:207; DESIGN R18):  x + i y = (r + i a) sin(theta) e^{i phi_KS},  z = r cos(theta),
 * t_KS = t_BL + T(r),  phi_KS = phi_BL + Phi(r),  dT/dr = 2r/Delta,  dPhi/dr = a/Delta,  a = src->a_eff,
 * T and Phi being the partial-fraction logarithms over the roots of Delta (the pole of the double root when
 * a^2 = 1); velocities are mapped with the Jacobian.  theta in [0, pi], phi in the principal range on output.
 * Evaluated in double whatever the precision of the state.  dst: caller-owned arrays of the same precision
 * as src (dst->q.., lambda, status, nsteps, n, prec filled by the caller); on return dst->coords = to_coords
 * and a_eff, kind, reversed, lambda, status, nsteps are copied.  dst may be src itself (each geodesic is read
 * completely before it is written); partial overlap is not allowed.  On the axis
 * the BL velocity is not finite (data, not an error).  GRAY2_EINVAL if src is already in to_coords. */
int gray2_convert(const gray2_state *src, gray2_state *dst, uint64_t n, int32_t to_coords, void *cuda_stream);

/* Coordinate-time form (section 2.2; eq. 18): integrates dv^i/dt = xddot^i - xddot^0 v^i,
 * v^mu = dx^mu/dt with v^0 = 1, six variables, with the same classic RK4 and the same step and stopping
 * rule as gray2_integrate, the KS coordinate time t = q[0] playing the role of lambda: the step is
 * dt = dir * (mode == 1 ? eta * r : h_fixed), clipped so that t does not pass t_end, and a geodesic that
 * reaches t_end stays ACTIVE ("integrate to a target KS coordinate time", method i).
 * On entry v^i = q[5+i] / q[4]; on exit q[0] = t, q[4] = 1 and q[5..7] = v^i (DESIGN R19): a tangent
 * vector of the same curve with another normalisation, so ratios such as L_z/E and Q/E^2 from
 * gray2_invariants keep their meaning.  s->lambda is not touched.  device_stats as for gray2_integrate.
 * FP32 states: the clock is q[0], a float, so t_end is rounded to float too: a geodesic that has reached the target
 * holds exactly float(t_end), and a second identical call is a no-op as in double.  float(t_end) is the NEAREST
 * float: the time reached may lie on either side of the t_end asked for, by up to half a float ulp of it (3e-5 M at
 * t ~ 1000 M); pass a t_end that is a float already if the geodesics must not pass it.  Accuracy in FP32: as for
 * gray2_integrate, 1e-4 of max(|component|, r) on every geodesic that is not critical for FP32 (DESIGN R12); on 30
 * random images (spin, inclination, field of view, 100 M <= r_obs <= 2000 M, eta = 0.005 ... 0.02) the largest error
 * of such a geodesic is 1.4e-5, the median 3e-7 (tests/test_gpu_sweep.py).  The positions are advanced as
 * x + h v + (h^2/6)(b_1 + b_2 + b_3) with the product h v carried exactly and the residual of v included: with
 * dt = eta r a position error on arrival at the hole leaves multiplied by r_escape / r_periapsis, so a relative 1e-7
 * per step on the way in is not affordable. */
int gray2_integrate_coordtime(gray2_state *s, uint64_t n, double t_end, const gray2_step_control *sc,
                              int32_t prec, gray2_stats *device_stats, void *cuda_stream);

/* Diagnostics of the paper's convergence experiments (section 3), accumulated over the
 * samples k = 0, 1, 2, ... = the states at the step boundaries of this call, the initial state included.
 * Five DEVICE arrays of n doubles, always evaluated in double; NaN where the event never occurs:
 *   max_abs_u2  max_k |g u u + mu^2|, mu^2 nominal from s->kind                     (Fig. 4-5)
 *   cos_peak    first local maximum of c_k = |z_k|/r_k refined by the quadratic through the three samples
 *               around it: c_i - (c_{i+1}-c_{i-1})^2 / (8 (c_{i-1} - 2 c_i + c_{i+1}))  (Fig. 6-7)
 *   dphi_cycle  unfolded KS azimuth phi = atan2(y,x) - atan2(a,r) at the first upward zero of z
 *               (z_k < 0 <= z_{k+1}, linear interpolation) minus phi_0                  (Fig. 8)
 *   t_zmax1,2   KS times of the first two maxima of z: downward zeros of u^z, linear interpolation in t
 *                                                                                       (Fig. 9) */
typedef struct {
  double *max_abs_u2, *cos_peak, *dphi_cycle, *t_zmax1, *t_zmax2;
} gray2_diagnostics;

/* gray2_integrate (affine form, same step and stopping rule, same final state bit for bit) plus the
 * diagnostics above.  One thread per geodesic: meant for the convergence studies (thousands of orbits),
 * not for images.  The accumulators start afresh at every call. */
int gray2_integrate_diagnostics(gray2_state *s, uint64_t n, double lambda_end, const gray2_step_control *sc,
                                int32_t prec, const gray2_diagnostics *diag, gray2_stats *device_stats,
                                void *cuda_stream);

/* Constants of the RUN geodesic, always evaluated in double from the stored state (DESIGN R8):
 *   norm = g_ab u^a u^b ;  E = -u_t ;  L_z = x u_y - y u_x ;
 *   Q = u_theta^2 + cos^2(theta) [ a^2 (mu^2 - E^2) + L_z^2 / sin^2(theta) ], mu^2 nominal from s->kind.
 * For s->reversed = 1 the physical photon has L_z = -L_z(run) in the spacetime of spin -a_eff; E, Q equal.
 * E, Lz, Q, norm: DEVICE arrays of n doubles each. */
int gray2_invariants(const gray2_state *s, uint64_t n, double *E, double *Lz, double *Q, double *norm,
                     void *cuda_stream);

/* Longest-first schedule from a previous trace of the same (or a similar) batch: order <- the indices 0..n-1
 * sorted by decreasing steps_hint[k] (e.g. the nsteps array an earlier gray2_integrate left for the same image:
 * movie frames, parameter scans).  Counting sort on the device, 4096 bins over [0, max hint]; the order inside a
 * bin is unspecified (it cannot change a result).  The paper's kernel pays the whole tail -- every ray runs until
 * the slowest one of the image is done; with per-ray termination the tail is the last ray of
 * every lane, and it is shortest when the short rays come last.  steps_hint, order: DEVICE arrays of n int32. */
int gray2_order_longest_first(const int32_t *steps_hint, uint64_t n, int32_t *order, void *cuda_stream);

/* Optional tuning of gray2_integrate's launch (0 = library default).  Results never depend on it.  Calls that
 * follow a schedule (gray2_state.order) always run in the default shape: the ordered kernels exist for it only. */
int gray2_set_launch(int32_t prec, int32_t threads_per_block, int32_t blocks_per_sm);

/* Exact floating-point operation counts of one RK4 step of one geodesic in this library's code path
 * (FMA = 2 flops, add/mul = 1, each rsqrt/rcp = 1), used for the roofline figure; see DESIGN.md.  The FP32
 * counts include the three extra additions per state variable of the compensated sums (530 + 24 = 554). */
int gray2_flops_per_step(int32_t prec);
int gray2_flops_per_step_coordtime(int32_t prec);
int gray2_flops_per_step_bl(int32_t prec);

/* Diagnostic entry, not one of the four calls of the path: the geodesic right-hand side of eq. (13)-(14)
 * alone, at n points, so that tests can compare it element by element with the oracle's eq. (7).
 * pos (3 n: x.., y.., z..), u (4 n: u^t.., u^x.., u^y.., u^z..), out (4 n): DEVICE arrays, SoA, of
 * double (GRAY2_F64) or float (GRAY2_F32). */
int gray2_rhs(int32_t prec, double a, uint64_t n, const void *pos, const void *u, void *out, void *cuda_stream);
/* The same for the Boyer-Lindquist right-hand side: pos (2 n: r.., theta..), u (4 n: u^t.., u^r.., u^theta..,
 * u^phi..), out (4 n). */
int gray2_rhs_bl(int32_t prec, double a, uint64_t n, const void *pos, const void *u, void *out, void *cuda_stream);

const char *gray2_last_error(void);   /* thread-local text of the last error of the calling thread */
const char *gray2_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GRAY2_H */
