// gray2_abi.cu -- the C-ABI of include/gray2.h: argument checks, launch configuration, launches.
// Every step of the path runs in the kernels of gray2_kernels.cuh; nothing here computes on the host
// beyond a handful of scalars (r_plus, sin/cos of the inclination, spin constants).
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <atomic>
#include <mutex>

#include "../../include/gray2.h"
#include "gray2_kernels.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}

#define CUDA_TRY(expr)                                                                         \
  do {                                                                                         \
    cudaError_t e_ = (expr);                                                                   \
    if (e_ != cudaSuccess) return fail(GRAY2_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

// ---- work-queue scratch: per device, 64 slots of one 64-byte line each, handed out round-robin ---------
// Slot i holds the queue counter at word 8 i and the step counter at word 8 i + 1.  A slot is handed out
// again only after 63 later calls; should the work that last used it still be running then (more than 64
// integrations in flight on different streams), the new user's stream waits for it: every slot carries an
// event recorded behind its last user.
constexpr int kQueueSlots = 64;
constexpr int kMaxDevices = 64;
struct Scratch {
  unsigned *order_bins = nullptr;            // device, 2 * kOrderBins + 1 words (gray2_order_longest_first)
  cudaEvent_t order_done = nullptr;          // recorded behind its last user
  unsigned long long *queue = nullptr;       // device, kQueueSlots * 8 words
  cudaEvent_t done[kQueueSlots] = {};        // recorded behind the last work that used the slot
  unsigned next = 0;
  int num_sms = 0;
  bool ready = false;
};
Scratch g_scratch[kMaxDevices];
std::mutex g_scratch_lock;   // queue, done, next, num_sms, ready
std::mutex g_order_lock;     // order_bins, order_done (gray2_order_longest_first only)

struct QueueSlot {
  unsigned long long *queue, *steps;
  cudaEvent_t done;
  int num_sms;
};

// Takes the next slot of the current device and makes `st` wait for the slot's previous user.
int acquire_slot(cudaStream_t st, QueueSlot *out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(GRAY2_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices) return fail(GRAY2_ECUDA, "device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> guard(g_scratch_lock);
  Scratch &sc = g_scratch[dev];
  if (!sc.ready) {
    e = cudaDeviceGetAttribute(&sc.num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess && !sc.queue) e = cudaMalloc(&sc.queue, kQueueSlots * 8 * sizeof(unsigned long long));
    for (int i = 0; i < kQueueSlots && e == cudaSuccess; ++i)
      if (!sc.done[i]) e = cudaEventCreateWithFlags(&sc.done[i], cudaEventDisableTiming);
    if (e != cudaSuccess) return fail(GRAY2_ECUDA, "scratch allocation: %s", cudaGetErrorString(e));
    sc.ready = true;
  }
  const unsigned slot = sc.next++ % kQueueSlots;
  out->queue = sc.queue + 8 * slot;
  out->steps = out->queue + 1;
  out->done = sc.done[slot];
  out->num_sms = sc.num_sms;
  e = cudaStreamWaitEvent(st, out->done, 0);   // a never-recorded event is complete: no wait
  if (e != cudaSuccess) return fail(GRAY2_ECUDA, "cudaStreamWaitEvent: %s", cudaGetErrorString(e));
  return GRAY2_OK;
}

// ---- staging buffers of gray2_init_explicit: per device, one slot per calling stream -----------------
constexpr int kStages = 8;
struct Stage {
  cudaStream_t key; bool made; double *buf; size_t bytes; cudaEvent_t copied, consumed;
  std::mutex mu;       // buf, bytes and the order of the work enqueued through this slot; key and made: g_stage_lock
};
struct StagePool { Stage slot[kStages] = {}; cudaStream_t copy_stream = nullptr; unsigned next = 0; };
StagePool g_stages[kMaxDevices];
std::mutex g_stage_lock;     // which stream owns which slot, and the copy stream; never held across a wait

// ---- launch configuration of the integrator (gray2_set_launch) ------------------------------------
// (threads << 16) | blocks_per_sm in ONE atomic word per precision, 0 = default, so that an integration that
// races with gray2_set_launch sees either the old pair or the new one, never a mixture.
std::atomic<uint32_t> g_launch[2] = {{0u}, {0u}};

template <typename T> gray2::StateView<T> view_of(const gray2_state *s) {
  gray2::StateView<T> v;
  for (int m = 0; m < 8; ++m) v.q[m] = static_cast<T *>(s->q[m]);
  v.lambda = s->lambda; v.status = s->status; v.nsteps = s->nsteps;
  v.order = s->order;
  return v;
}

int check_state(const gray2_state *s, const char *who) {
  if (!s) return fail(GRAY2_EINVAL, "%s: state is NULL", who);
  if (s->n == 0) return fail(GRAY2_EINVAL, "%s: state has n == 0", who);
  for (int m = 0; m < 8; ++m)
    if (!s->q[m]) return fail(GRAY2_EINVAL, "%s: state q[%d] is NULL", who, m);
  if (!s->lambda || !s->status || !s->nsteps) return fail(GRAY2_EINVAL, "%s: lambda/status/nsteps is NULL", who);
  if (s->prec != GRAY2_F64 && s->prec != GRAY2_F32) return fail(GRAY2_EINVAL, "%s: unknown precision %d", who, s->prec);
  if (s->coords != GRAY2_KS && s->coords != GRAY2_BL) return fail(GRAY2_EINVAL, "%s: unknown coordinates %d", who, s->coords);
  return GRAY2_OK;
}

}  // namespace

// ---- integrator dispatch ----------------------------------------------------------------------------
namespace {

template <typename T, int THREADS, int MIN_BLOCKS, int FORM, bool ORDERED = false>
cudaError_t launch_integrate(const gray2_state *s, uint64_t n, const gray2::StepParams<T> &p,
                             unsigned long long *queue, unsigned long long *steps, int num_sms, cudaStream_t st) {
  uint64_t want = (n + THREADS - 1) / THREADS;
  uint64_t cap = (uint64_t)num_sms * MIN_BLOCKS;
  unsigned grid = (unsigned)(want < cap ? want : cap);
  auto v = view_of<T>(s);
  if (p.mode == 1) {
    if (p.clip) gray2::integrate_kernel<T, THREADS, MIN_BLOCKS, 1, true, FORM, ORDERED><<<grid, THREADS, 0, st>>>(v, n, p, queue, steps);
    else        gray2::integrate_kernel<T, THREADS, MIN_BLOCKS, 1, false, FORM, ORDERED><<<grid, THREADS, 0, st>>>(v, n, p, queue, steps);
  } else {
    if (p.clip) gray2::integrate_kernel<T, THREADS, MIN_BLOCKS, 0, true, FORM, ORDERED><<<grid, THREADS, 0, st>>>(v, n, p, queue, steps);
    else        gray2::integrate_kernel<T, THREADS, MIN_BLOCKS, 0, false, FORM, ORDERED><<<grid, THREADS, 0, st>>>(v, n, p, queue, steps);
  }
  return cudaGetLastError();
}

// FP32 with two geodesics per thread (packed FP32x2 arithmetic)
template <int THREADS, int MIN_BLOCKS, int FORM, bool ORDERED = false>
cudaError_t launch_integrate_x2(const gray2_state *s, uint64_t n, const gray2::StepParams<float> &p,
                                unsigned long long *queue, unsigned long long *steps, int num_sms, cudaStream_t st) {
  uint64_t want = (n + 2 * THREADS - 1) / (2 * THREADS);
  uint64_t cap = (uint64_t)num_sms * MIN_BLOCKS;
  unsigned grid = (unsigned)(want < cap ? want : cap);
  auto v = view_of<float>(s);
  if (p.mode == 1) {
    if (p.clip) gray2::integrate_kernel_f32x2<THREADS, MIN_BLOCKS, 1, true, FORM, ORDERED><<<grid, THREADS, 0, st>>>(v, n, p, queue, steps);
    else        gray2::integrate_kernel_f32x2<THREADS, MIN_BLOCKS, 1, false, FORM, ORDERED><<<grid, THREADS, 0, st>>>(v, n, p, queue, steps);
  } else {
    if (p.clip) gray2::integrate_kernel_f32x2<THREADS, MIN_BLOCKS, 0, true, FORM, ORDERED><<<grid, THREADS, 0, st>>>(v, n, p, queue, steps);
    else        gray2::integrate_kernel_f32x2<THREADS, MIN_BLOCKS, 0, false, FORM, ORDERED><<<grid, THREADS, 0, st>>>(v, n, p, queue, steps);
  }
  return cudaGetLastError();
}

struct LaunchChoice { int threads, blocks; };

// Compiled variants of the affine-parameter integrator; the first entry of each list is the default
// and the only one compiled for the coordinate-time form and for the Boyer-Lindquist form.  FP32: the entries
// 256x2, 128x3, 128x4 and 256x1 run two geodesics per thread (integrate_kernel_f32x2), 128x8 and 128x6 one per
// thread (integrate_kernel<float>); every variant gives bit-identical results.  FP64 128x2 + FP32 256x1 are the
// pair that fits one SM's register file side by side (both precisions of one image at once, bench.py "both").
constexpr int kNumVariants = 6;
constexpr LaunchChoice kF64Variants[kNumVariants] = {{128, 3}, {128, 4}, {64, 6}, {256, 1}, {128, 2}, {128, 1}};
constexpr LaunchChoice kF32Variants[kNumVariants] = {{256, 2}, {128, 3}, {128, 4}, {128, 8}, {128, 6}, {256, 1}};

template <typename T>
cudaError_t dispatch_integrate(int form, int threads, int blocks, const gray2_state *s, uint64_t n,
                               const gray2::StepParams<T> &p, unsigned long long *q, unsigned long long *steps,
                               int sms, cudaStream_t st, bool *found) {
  *found = true;
  // A schedule (gray2_state.order) is used only by a call that covers the whole state, and runs in the default
  // launch shape of its form (the ordered kernels are compiled for that shape only).
  if (s->order && n == s->n) {
    if constexpr (sizeof(T) == 8) {
      if (form == 1) return launch_integrate<T, 128, 3, 1, true>(s, n, p, q, steps, sms, st);
      if (form == 2) return launch_integrate<T, 128, 3, 2, true>(s, n, p, q, steps, sms, st);
      return launch_integrate<T, 128, 3, 0, true>(s, n, p, q, steps, sms, st);
    } else {
      if (form == 1) return launch_integrate_x2<256, 2, 1, true>(s, n, p, q, steps, sms, st);
      if (form == 2) return launch_integrate_x2<256, 2, 2, true>(s, n, p, q, steps, sms, st);
      return launch_integrate_x2<256, 2, 0, true>(s, n, p, q, steps, sms, st);
    }
  }
  if constexpr (sizeof(T) == 8) {
    if (form == 1) return launch_integrate<T, 128, 3, 1>(s, n, p, q, steps, sms, st);
    if (form == 2) {
      if (threads == 128 && blocks == 4) return launch_integrate<T, 128, 4, 2>(s, n, p, q, steps, sms, st);
      if (threads == 64 && blocks == 6) return launch_integrate<T, 64, 6, 2>(s, n, p, q, steps, sms, st);
      return launch_integrate<T, 128, 3, 2>(s, n, p, q, steps, sms, st);
    }
#define GRAY2_VARIANT(TH, BL) \
  if (threads == TH && blocks == BL) return launch_integrate<T, TH, BL, 0>(s, n, p, q, steps, sms, st);
    GRAY2_VARIANT(128, 3) GRAY2_VARIANT(128, 4) GRAY2_VARIANT(64, 6) GRAY2_VARIANT(256, 1) GRAY2_VARIANT(128, 2)
    GRAY2_VARIANT(128, 1)
#undef GRAY2_VARIANT
  } else {
    if (form == 1) return launch_integrate_x2<256, 2, 1>(s, n, p, q, steps, sms, st);
    if (form == 2) {
      if (threads == 128 && blocks == 4) return launch_integrate_x2<128, 4, 2>(s, n, p, q, steps, sms, st);
      if (threads == 128 && blocks == 3) return launch_integrate_x2<128, 3, 2>(s, n, p, q, steps, sms, st);
      return launch_integrate_x2<256, 2, 2>(s, n, p, q, steps, sms, st);
    }
#define GRAY2_VARIANT_X2(TH, BL) \
  if (threads == TH && blocks == BL) return launch_integrate_x2<TH, BL, 0>(s, n, p, q, steps, sms, st);
#define GRAY2_VARIANT(TH, BL) \
  if (threads == TH && blocks == BL) return launch_integrate<T, TH, BL, 0>(s, n, p, q, steps, sms, st);
    GRAY2_VARIANT_X2(128, 4) GRAY2_VARIANT_X2(128, 3) GRAY2_VARIANT_X2(256, 2) GRAY2_VARIANT_X2(256, 1)
    GRAY2_VARIANT(128, 8) GRAY2_VARIANT(128, 6)
#undef GRAY2_VARIANT
#undef GRAY2_VARIANT_X2
  }
  *found = false;
  return cudaSuccess;
}

// Step parameters of the kernels from the caller's step control (`end` = lambda_end or t_end).
template <typename T>
gray2::StepParams<T> make_params(double a, double end, const gray2_step_control *sc, bool always_clip) {
  gray2::StepParams<T> p;
  p.k.a = (T)a; p.k.a2 = (T)(a * a); p.k.two_a = (T)(2.0 * a); p.k.two_a2 = (T)(2.0 * a * a); p.k.four_a2 = (T)(4.0 * a * a);
  p.eta_or_h = (T)((double)sc->dir * (sc->mode == 1 ? sc->eta : sc->h_fixed));
  p.r_capture = (T)(sc->capture_factor * (1.0 + sqrt(1.0 - a * a)));
  p.r_escape = (T)sc->r_escape;
  // the hot loop tests r <= r_escape_fin with r_escape_fin finite, so that r = inf fails the test too
  const double big = sizeof(T) == 8 ? 1.7976931348623157e308 : 3.402823466e38;
  p.r_escape_fin = always_clip ? p.r_escape : (T)(sc->r_escape < big ? sc->r_escape : big);
  p.lambda_end = end;
  p.dir = (double)sc->dir;
  p.mode = sc->mode;
  p.max_steps = sc->max_steps;
  // clip = 0 only when dir * end = +inf: the end test can never fire and the last step never needs clipping
  p.clip = always_clip || !(isinf(end) && (double)sc->dir * end > 0.0);
  return p;
}

template <typename T>
int integrate_impl(int form, gray2_state *s, uint64_t n, double end, const gray2_step_control *sc,
                   gray2_stats *device_stats, cudaStream_t st) {
  // Coordinate-time form in FP32: the clock is q[0] itself, a float.  The target is rounded to float as well, so that
  // a geodesic that has reached it holds exactly the target and a second identical call is a no-op (with the double
  // target a stored float(t_end) < t_end would ask for one more, rounding-sized, step at every call).
  if (form == 1 && sizeof(T) == 4 && isfinite(end)) end = (double)(float)end;
  const gray2::StepParams<T> p = make_params<T>(s->a_eff, end, sc, /*always_clip=*/false);

  QueueSlot qs;
  int rc = acquire_slot(st, &qs);
  if (rc) return rc;
  unsigned long long *queue = qs.queue, *steps = qs.steps;
  CUDA_TRY(cudaMemsetAsync(queue, 0, 2 * sizeof(unsigned long long), st));

  const int pi = sizeof(T) == 8 ? 0 : 1;
  const LaunchChoice def = sizeof(T) == 8 ? kF64Variants[0] : kF32Variants[0];
  const uint32_t chosen = g_launch[pi].load(std::memory_order_relaxed);
  int threads = chosen ? (int)(chosen >> 16) : def.threads;
  int blocks = chosen ? (int)(chosen & 0xffffu) : def.blocks;
  // Small batches: a geodesic is ~1000 sequential steps, so a batch that cannot fill the GPU is bound by the
  // latency of one step, and what matters is to spread it over the SMs.  The packed FP32 kernel (512 geodesics per
  // block) would put cfg1's 4,096 rays on 8 SMs; the one-per-thread float kernel (128 per block) gives the same
  // bits from 32.  Only the affine Kerr-Schild form has that variant compiled, and only an unset launch choice
  // is overridden.
  // (Below 128 geodesics per SM only: larger batches are often one chunk of several in flight on other streams,
  // which fill the GPU together, and there the packed kernel's 15 % higher throughput counts.)
  if (sizeof(T) == 4 && !chosen && form == 0 && n < (uint64_t)qs.num_sms * 128) { threads = 128; blocks = 8; }
  bool found = false;
  cudaError_t e = dispatch_integrate<T>(form, threads, blocks, s, n, p, queue, steps, qs.num_sms, st, &found);
  if (!found) return fail(GRAY2_EINVAL, "gray2_integrate: no compiled variant for %d threads x %d blocks/SM", threads, blocks);
  if (e != cudaSuccess) return fail(GRAY2_ECUDA, "integrate_kernel launch: %s", cudaGetErrorString(e));

  if (device_stats) {
    CUDA_TRY(cudaMemsetAsync(device_stats, 0, sizeof(gray2_stats), st));
    CUDA_TRY(cudaMemcpyAsync(&device_stats->steps, steps, sizeof(unsigned long long), cudaMemcpyDeviceToDevice, st));
    unsigned grid = (unsigned)((n + 255) / 256);
    if (grid > (unsigned)(qs.num_sms * 8)) grid = (unsigned)(qs.num_sms * 8);
    gray2::count_status_kernel<<<grid, 256, 0, st>>>(s->status, n, device_stats);
    CUDA_TRY(cudaGetLastError());
  }
  CUDA_TRY(cudaEventRecord(qs.done, st));      // the slot is free again once this point of `st` is reached
  return GRAY2_OK;
}

}  // namespace

namespace {

template <typename T>
int diag_impl(gray2_state *s, uint64_t n, double lambda_end, const gray2_step_control *sc,
                     const gray2_diagnostics *d, gray2_stats *device_stats, cudaStream_t st) {
  // the diagnostics kernel always tests lambda_end and compares r with r_escape itself
  const gray2::StepParams<T> p = make_params<T>(s->a_eff, lambda_end, sc, /*always_clip=*/true);
  QueueSlot qs;
  int rc = acquire_slot(st, &qs);
  if (rc) return rc;
  unsigned long long *steps = qs.steps;
  CUDA_TRY(cudaMemsetAsync(steps, 0, sizeof(unsigned long long), st));
  gray2::DiagView out{d->max_abs_u2, d->cos_peak, d->dphi_cycle, d->t_zmax1, d->t_zmax2};
  double mu2 = s->kind == GRAY2_TIMELIKE ? 1.0 : 0.0;
  unsigned grid = (unsigned)((n + 63) / 64);
  if (sc->mode == 1) gray2::integrate_diag_kernel<T, 1><<<grid, 64, 0, st>>>(view_of<T>(s), n, p, mu2, out, steps);
  else gray2::integrate_diag_kernel<T, 0><<<grid, 64, 0, st>>>(view_of<T>(s), n, p, mu2, out, steps);
  CUDA_TRY(cudaGetLastError());
  if (device_stats) {
    CUDA_TRY(cudaMemsetAsync(device_stats, 0, sizeof(gray2_stats), st));
    CUDA_TRY(cudaMemcpyAsync(&device_stats->steps, steps, sizeof(unsigned long long), cudaMemcpyDeviceToDevice, st));
    unsigned g2 = (unsigned)((n + 255) / 256);
    if (g2 > (unsigned)(qs.num_sms * 8)) g2 = (unsigned)(qs.num_sms * 8);
    gray2::count_status_kernel<<<g2, 256, 0, st>>>(s->status, n, device_stats);
    CUDA_TRY(cudaGetLastError());
  }
  CUDA_TRY(cudaEventRecord(qs.done, st));
  return GRAY2_OK;
}

}  // namespace

// ---- the exported calls ------------------------------------------------------------------------------
extern "C" {

const char *gray2_last_error(void) { return g_err; }
const char *gray2_version(void) { return "gray2-b200 0.2 (sm_100a)"; }

/* Number of rays of rank `rank` when n rays are dealt out in tiles of tile_rays, tile t to rank t mod world. */
uint64_t gray2_shard_count(uint64_t n, uint64_t tile_rays, int32_t rank, int32_t world) {
  if (tile_rays == 0 || world <= 0 || rank < 0 || rank >= world) return 0;
  const uint64_t tiles = (n + tile_rays - 1) / tile_rays;                 // the last one may be ragged
  const uint64_t mine = tiles / (uint64_t)world + ((uint64_t)rank < tiles % (uint64_t)world ? 1 : 0);
  if (mine == 0) return 0;
  const uint64_t last_tile = tiles - 1, last_size = n - last_tile * tile_rays;
  const bool own_last = last_tile % (uint64_t)world == (uint64_t)rank;
  return own_last ? (mine - 1) * tile_rays + last_size : mine * tile_rays;
}

int gray2_init_null_shard(gray2_state *s, double a, double r_obs, double inc, double Wa, double Wb,
                          int32_t nx, int32_t ny, uint64_t tile_rays, int32_t rank, int32_t world,
                          void *cuda_stream) {
  if (s) s->coords = GRAY2_KS;
  int rc = check_state(s, "gray2_init_null");
  if (rc) return rc;
  if (!(fabs(a) <= 1.0)) return fail(GRAY2_EINVAL, "gray2_init_null: |a| must be <= 1 (got %g)", a);
  if (nx <= 0 || ny <= 0) return fail(GRAY2_EINVAL, "gray2_init_null: nx and ny must be positive");
  if (tile_rays == 0 || world <= 0 || rank < 0 || rank >= world)
    return fail(GRAY2_EINVAL, "gray2_init_null_shard: need tile_rays > 0 and 0 <= rank < world");
  const uint64_t n_local = gray2_shard_count((uint64_t)nx * (uint64_t)ny, tile_rays, rank, world);
  if (n_local != s->n)
    return fail(GRAY2_EINVAL, "gray2_init_null: s->n (%llu) must equal the number of rays of this call (%llu of %d x %d)",
                (unsigned long long)s->n, (unsigned long long)n_local, nx, ny);
  if (!(r_obs > 1.0 + sqrt(1.0 - a * a))) return fail(GRAY2_EINVAL, "gray2_init_null: r_obs must exceed r_plus");
  if (!(Wa > 0.0) || !(Wb > 0.0) || !isfinite(inc)) return fail(GRAY2_EINVAL, "gray2_init_null: bad field of view or inclination");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  s->a_eff = -a; s->kind = GRAY2_NULL; s->reversed = 1; s->coords = GRAY2_KS;
  unsigned grid = (unsigned)((s->n + 255) / 256);
  if (s->prec == GRAY2_F64)
    gray2::init_null_kernel<double><<<grid, 256, 0, st>>>(view_of<double>(s), n_local, -a, r_obs, sin(inc), cos(inc), Wa, Wb,
                                                          nx, ny, tile_rays, (uint32_t)rank, (uint32_t)world);
  else
    gray2::init_null_kernel<float><<<grid, 256, 0, st>>>(view_of<float>(s), n_local, -a, r_obs, sin(inc), cos(inc), Wa, Wb,
                                                         nx, ny, tile_rays, (uint32_t)rank, (uint32_t)world);
  CUDA_TRY(cudaGetLastError());
  return GRAY2_OK;
}

int gray2_init_null(gray2_state *s, double a, double r_obs, double inc, double Wa, double Wb,
                    int32_t nx, int32_t ny, void *cuda_stream) {
  if (nx <= 0 || ny <= 0) return fail(GRAY2_EINVAL, "gray2_init_null: nx and ny must be positive");
  return gray2_init_null_shard(s, a, r_obs, inc, Wa, Wb, nx, ny, (uint64_t)nx * (uint64_t)ny, 0, 1, cuda_stream);
}

int gray2_init_explicit(gray2_state *s, double a, const double *host_xu8, uint64_t n, int32_t kind, int32_t renorm,
                        void *cuda_stream) {
  const char *who = "gray2_init_explicit";
  if (s) s->coords = GRAY2_KS;
  int rc = check_state(s, who);
  if (rc) return rc;
  if (!host_xu8 || n == 0) return fail(GRAY2_EINVAL, "%s: host_xu8 is NULL or n == 0", who);
  if (n > s->n) return fail(GRAY2_ESTATE, "%s: n (%llu) exceeds s->n (%llu)", who, (unsigned long long)n, (unsigned long long)s->n);
  if (!(fabs(a) <= 1.0)) return fail(GRAY2_EINVAL, "%s: |a| must be <= 1 (got %g)", who, a);
  if (kind != GRAY2_NULL && kind != GRAY2_TIMELIKE) return fail(GRAY2_EINVAL, "%s: kind must be GRAY2_NULL or GRAY2_TIMELIKE", who);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return fail(GRAY2_ECUDA, "device ordinal %d out of range", dev);
  // Staging buffers for the AoS input: owned by the library, per device (like the work-queue scratch), grown
  // on demand and reused (a fresh stream-ordered allocation per call costs up to 100 ms when the pool has to
  // grow again).  A small pool, one slot per calling stream (round robin beyond kStages streams).  The
  // host-to-device copy runs on an internal stream of that device, so that it does not queue behind the
  // caller's earlier work on `st` (a caller that pipelines chunks over a few streams gets its inputs
  // prefetched while earlier chunks integrate); the caller's stream waits for the copy, the next copy into a
  // slot waits for the kernel that consumed it, and the host waits only for its own copy, after which
  // host_xu8 may be reused.
  const size_t bytes = (size_t)n * 8 * sizeof(double);
  const double mu2 = kind == GRAY2_TIMELIKE ? 1.0 : 0.0;
  cudaEvent_t copied;
  Stage *sl = nullptr;
  cudaStream_t copy_stream = nullptr;
  {
    // the pool-wide lock only while the slot is picked: growing a buffer (cudaFree, cudaMalloc, a wait for the kernel
    // that last read it) and enqueueing happen under the slot's own lock, so that one thread's larger batch does not
    // hold up the host-to-device copies of every other thread on every device
    std::lock_guard<std::mutex> guard(g_stage_lock);
    StagePool &pool = g_stages[dev];
    if (!pool.copy_stream) CUDA_TRY(cudaStreamCreateWithFlags(&pool.copy_stream, cudaStreamNonBlocking));
    copy_stream = pool.copy_stream;
    for (int i = 0; i < kStages && !sl; ++i)
      if (pool.slot[i].made && pool.slot[i].key == st) sl = &pool.slot[i];
    if (!sl) {
      Stage *cand = &pool.slot[pool.next % kStages];
      if (!cand->made) {
        cudaEvent_t e1 = nullptr, e2 = nullptr;
        CUDA_TRY(cudaEventCreateWithFlags(&e1, cudaEventDisableTiming));
        cudaError_t e = cudaEventCreateWithFlags(&e2, cudaEventDisableTiming);
        if (e != cudaSuccess) { cudaEventDestroy(e1); return fail(GRAY2_ECUDA, "%s: cudaEventCreate: %s", who, cudaGetErrorString(e)); }
        cand->copied = e1; cand->consumed = e2;
        cand->made = true;
      }
      pool.next++;
      cand->key = st;
      sl = cand;
    }
  }
  {
    std::lock_guard<std::mutex> guard(sl->mu);
    if (bytes > sl->bytes) {
      if (sl->buf) { CUDA_TRY(cudaEventSynchronize(sl->consumed)); cudaFree(sl->buf); sl->buf = nullptr; sl->bytes = 0; }
      CUDA_TRY(cudaMalloc(&sl->buf, bytes));
      sl->bytes = bytes;
    }
    CUDA_TRY(cudaStreamWaitEvent(copy_stream, sl->consumed, 0));      // the kernel that last read this slot
    CUDA_TRY(cudaMemcpyAsync(sl->buf, host_xu8, bytes, cudaMemcpyHostToDevice, copy_stream));
    CUDA_TRY(cudaEventRecord(sl->copied, copy_stream));
    CUDA_TRY(cudaStreamWaitEvent(st, sl->copied, 0));
    unsigned grid = (unsigned)((n + 255) / 256);
    if (s->prec == GRAY2_F64)
      gray2::init_explicit_kernel<double><<<grid, 256, 0, st>>>(view_of<double>(s), sl->buf, n, a, renorm, mu2);
    else
      gray2::init_explicit_kernel<float><<<grid, 256, 0, st>>>(view_of<float>(s), sl->buf, n, a, renorm, mu2);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaEventRecord(sl->consumed, st));
    copied = sl->copied;
  }
  CUDA_TRY(cudaEventSynchronize(copied));   // host_xu8 may be reused on return
  s->a_eff = a; s->kind = kind; s->reversed = 0; s->coords = GRAY2_KS;
  return GRAY2_OK;
}

int gray2_init_timelike(gray2_state *s, double a, const double *host_xu8, uint64_t n, int32_t renorm,
                        void *cuda_stream) {
  return gray2_init_explicit(s, a, host_xu8, n, GRAY2_TIMELIKE, renorm, cuda_stream);
}

// Arguments common to gray2_integrate, gray2_integrate_coordtime and gray2_integrate_diagnostics.
static int check_integrate_args(const char *who, const gray2_state *s, uint64_t n, double end,
                                const gray2_step_control *sc, int32_t prec) {
  if (!sc) return fail(GRAY2_EINVAL, "%s: step control is NULL", who);
  if (n == 0) return fail(GRAY2_EINVAL, "%s: n == 0", who);
  if (n > s->n) return fail(GRAY2_ESTATE, "%s: n (%llu) exceeds s->n (%llu)", who, (unsigned long long)n, (unsigned long long)s->n);
  if (prec != s->prec) return fail(GRAY2_EINVAL, "%s: prec (%d) differs from s->prec (%d)", who, prec, s->prec);
  if (sc->mode != 0 && sc->mode != 1) return fail(GRAY2_EINVAL, "%s: mode must be 0 or 1", who);
  if (sc->mode == 1 ? !(sc->eta > 0.0) : !(sc->h_fixed > 0.0)) return fail(GRAY2_EINVAL, "%s: step size must be > 0", who);
  if (sc->dir != 1 && sc->dir != -1) return fail(GRAY2_EINVAL, "%s: dir must be +1 or -1", who);
  if (!(sc->capture_factor > 0.0) || isnan(sc->r_escape) || isnan(end) || sc->max_steps < 0)
    return fail(GRAY2_EINVAL, "%s: bad capture_factor / r_escape / end value / max_steps", who);
  if (!(fabs(s->a_eff) <= 1.0)) return fail(GRAY2_EINVAL, "%s: |a_eff| must be <= 1", who);
  return GRAY2_OK;
}

static int integrate_common(int form, const char *who, gray2_state *s, uint64_t n, double end,
                            const gray2_step_control *sc, int32_t prec, gray2_stats *device_stats, void *cuda_stream) {
  int rc = check_state(s, who);
  if (rc) return rc;
  rc = check_integrate_args(who, s, n, end, sc, prec);
  if (rc) return rc;
  if (s->coords == GRAY2_BL) {
    if (form != 0) return fail(GRAY2_EINVAL, "%s: needs a Kerr-Schild state (s->coords = GRAY2_KS)", who);
    form = 2;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  return prec == GRAY2_F64 ? integrate_impl<double>(form, s, n, end, sc, device_stats, st)
                           : integrate_impl<float>(form, s, n, end, sc, device_stats, st);
}

int gray2_integrate(gray2_state *s, uint64_t n, double lambda_end, const gray2_step_control *sc,
                    int32_t prec, gray2_stats *device_stats, void *cuda_stream) {
  return integrate_common(0, "gray2_integrate", s, n, lambda_end, sc, prec, device_stats, cuda_stream);
}

int gray2_integrate_coordtime(gray2_state *s, uint64_t n, double t_end, const gray2_step_control *sc,
                              int32_t prec, gray2_stats *device_stats, void *cuda_stream) {
  return integrate_common(1, "gray2_integrate_coordtime", s, n, t_end, sc, prec, device_stats, cuda_stream);
}

int gray2_integrate_diagnostics(gray2_state *s, uint64_t n, double lambda_end, const gray2_step_control *sc,
                                int32_t prec, const gray2_diagnostics *diag, gray2_stats *device_stats,
                                void *cuda_stream) {
  const char *who = "gray2_integrate_diagnostics";
  int rc = check_state(s, who);
  if (rc) return rc;
  if (!sc || !diag) return fail(GRAY2_EINVAL, "%s: step control or diagnostics is NULL", who);
  if (s->coords != GRAY2_KS) return fail(GRAY2_EINVAL, "%s: needs a Kerr-Schild state (s->coords = GRAY2_KS)", who);
  if (!diag->max_abs_u2 || !diag->cos_peak || !diag->dphi_cycle || !diag->t_zmax1 || !diag->t_zmax2)
    return fail(GRAY2_EINVAL, "%s: a diagnostics array is NULL", who);
  rc = check_integrate_args(who, s, n, lambda_end, sc, prec);
  if (rc) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  return prec == GRAY2_F64 ? diag_impl<double>(s, n, lambda_end, sc, diag, device_stats, st)
                           : diag_impl<float>(s, n, lambda_end, sc, diag, device_stats, st);
}

int gray2_invariants(const gray2_state *s, uint64_t n, double *E, double *Lz, double *Q, double *norm,
                     void *cuda_stream) {
  int rc = check_state(s, "gray2_invariants");
  if (rc) return rc;
  if (n == 0 || !E || !Lz || !Q || !norm) return fail(GRAY2_EINVAL, "gray2_invariants: n == 0 or NULL output");
  if (n > s->n) return fail(GRAY2_ESTATE, "gray2_invariants: n exceeds s->n");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double mu2 = s->kind == GRAY2_TIMELIKE ? 1.0 : 0.0;
  unsigned grid = (unsigned)((n + 255) / 256);
  if (s->coords == GRAY2_BL) {
    if (s->prec == GRAY2_F64)
      gray2::invariants_bl_kernel<double><<<grid, 256, 0, st>>>(view_of<double>(s), n, s->a_eff, mu2, E, Lz, Q, norm);
    else
      gray2::invariants_bl_kernel<float><<<grid, 256, 0, st>>>(view_of<float>(s), n, s->a_eff, mu2, E, Lz, Q, norm);
  } else if (s->prec == GRAY2_F64)
    gray2::invariants_kernel<double><<<grid, 256, 0, st>>>(view_of<double>(s), n, s->a_eff, mu2, E, Lz, Q, norm);
  else
    gray2::invariants_kernel<float><<<grid, 256, 0, st>>>(view_of<float>(s), n, s->a_eff, mu2, E, Lz, Q, norm);
  CUDA_TRY(cudaGetLastError());
  return GRAY2_OK;
}

int gray2_convert(const gray2_state *src, gray2_state *dst, uint64_t n, int32_t to_coords, void *cuda_stream) {
  int rc = check_state(src, "gray2_convert");
  if (rc) return rc;
  if (to_coords != GRAY2_KS && to_coords != GRAY2_BL) return fail(GRAY2_EINVAL, "gray2_convert: unknown coordinates %d", to_coords);
  if (src->coords == to_coords) return fail(GRAY2_EINVAL, "gray2_convert: the state is already in those coordinates");
  if (!dst) return fail(GRAY2_EINVAL, "gray2_convert: dst is NULL");
  {
    gray2_state probe = *dst;              // dst->coords is an output: validate the rest (dst may be src itself)
    probe.coords = to_coords;
    rc = check_state(&probe, "gray2_convert");
    if (rc) return rc;
  }
  if (src->prec != dst->prec) return fail(GRAY2_EINVAL, "gray2_convert: src and dst differ in precision");
  if (n == 0) return fail(GRAY2_EINVAL, "gray2_convert: n == 0");
  if (n > src->n || n > dst->n) return fail(GRAY2_ESTATE, "gray2_convert: n exceeds the size of src or dst");
  if (!(fabs(src->a_eff) <= 1.0)) return fail(GRAY2_EINVAL, "gray2_convert: |a_eff| must be <= 1");
  const double a = src->a_eff;
  const int32_t prec = src->prec;
  const auto vs64 = view_of<double>(src), vd64 = view_of<double>(dst);
  const auto vs32 = view_of<float>(src), vd32 = view_of<float>(dst);
  dst->a_eff = src->a_eff; dst->kind = src->kind; dst->reversed = src->reversed; dst->coords = to_coords;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  unsigned grid = (unsigned)((n + 255) / 256);
  if (to_coords == GRAY2_BL) {
    if (prec == GRAY2_F64) gray2::ks_to_bl_kernel<double><<<grid, 256, 0, st>>>(vs64, vd64, n, a);
    else gray2::ks_to_bl_kernel<float><<<grid, 256, 0, st>>>(vs32, vd32, n, a);
  } else {
    if (prec == GRAY2_F64) gray2::bl_to_ks_kernel<double><<<grid, 256, 0, st>>>(vs64, vd64, n, a);
    else gray2::bl_to_ks_kernel<float><<<grid, 256, 0, st>>>(vs32, vd32, n, a);
  }
  CUDA_TRY(cudaGetLastError());
  return GRAY2_OK;
}

/* Diagnostic entry (not one of the four calls of the path): evaluates the geodesic right-hand side of
 * eq. (13)-(14) at n points.  pos (3 n), u (4 n), out (4 n): DEVICE arrays, SoA, double or float per prec. */
int gray2_rhs(int32_t prec, double a, uint64_t n, const void *pos, const void *u, void *out, void *cuda_stream) {
  if (!pos || !u || !out || n == 0) return fail(GRAY2_EINVAL, "gray2_rhs: NULL pointer or n == 0");
  if (prec != GRAY2_F64 && prec != GRAY2_F32) return fail(GRAY2_EINVAL, "gray2_rhs: unknown precision");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  unsigned grid = (unsigned)((n + 127) / 128);
  if (prec == GRAY2_F64) {
    gray2::SpinConst<double> k{a, a * a, 2.0 * a, 2.0 * a * a, 4.0 * a * a};
    gray2::rhs_kernel<double><<<grid, 128, 0, st>>>(k, n, (const double *)pos, (const double *)u, (double *)out);
  } else {
    gray2::SpinConst<float> k{(float)a, (float)(a * a), (float)(2.0 * a), (float)(2.0 * a * a), (float)(4.0 * a * a)};
    gray2::rhs_kernel<float><<<grid, 128, 0, st>>>(k, n, (const float *)pos, (const float *)u, (float *)out);
  }
  CUDA_TRY(cudaGetLastError());
  return GRAY2_OK;
}

int gray2_rhs_bl(int32_t prec, double a, uint64_t n, const void *pos, const void *u, void *out, void *cuda_stream) {
  if (!pos || !u || !out || n == 0) return fail(GRAY2_EINVAL, "gray2_rhs_bl: NULL pointer or n == 0");
  if (prec != GRAY2_F64 && prec != GRAY2_F32) return fail(GRAY2_EINVAL, "gray2_rhs_bl: unknown precision");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  unsigned grid = (unsigned)((n + 127) / 128);
  if (prec == GRAY2_F64) {
    gray2::SpinConst<double> k{a, a * a, 2.0 * a, 2.0 * a * a, 4.0 * a * a};
    gray2::rhs_bl_kernel<double><<<grid, 128, 0, st>>>(k, n, (const double *)pos, (const double *)u, (double *)out);
  } else {
    gray2::SpinConst<float> k{(float)a, (float)(a * a), (float)(2.0 * a), (float)(2.0 * a * a), (float)(4.0 * a * a)};
    gray2::rhs_bl_kernel<float><<<grid, 128, 0, st>>>(k, n, (const float *)pos, (const float *)u, (float *)out);
  }
  CUDA_TRY(cudaGetLastError());
  return GRAY2_OK;
}

/* Source-level count of ks_geodesic.cuh (FMA = 2, add/mul = 1, rsqrt/rcp = 1; negations and compares free):
 *   radius 16, rest of geometry 19, velocity part 72  ->  107 per right-hand side
 *   4 x 107 + RK4 combination 100 + step rule and lambda update 2 = 530 per step in double.
 * FP32 carries the eight state sums compensated (Carry<T>, ks_geodesic.cuh): each y <- y + w S costs an FMA and
 * three additions instead of one FMA, + 3 per variable = + 24 per step: 554. */
int gray2_flops_per_step(int32_t prec) { return prec == GRAY2_F32 ? 554 : 530; }

/* Coordinate-time form: 4 x (107 + 6) + RK4 combination of six variables 80 + step rule and t update 2 = 534;
 * FP32: three compensated velocity sums, + 9, and the three positions advanced as x + h v + (h^2/6)(b_1 + b_2 + b_3)
 * with the product h v carried exactly (advance_exact, ks_geodesic.cuh): 23 instead of 13 each, + 30, and h^2/6, + 1. */
int gray2_flops_per_step_coordtime(int32_t prec) { return prec == GRAY2_F32 ? 574 : 534; }

/* Boyer-Lindquist form, source-level count of bl_geodesic.cuh (same conventions):
 *   sin^2 and sin cos of theta: reduction 8, series 17 + 16, products 2 -> 43 (double: 8 / 8 terms, period pi/2),
 *                               reduction 8, series 13 + 12, products 2 -> 35 (float: 6 / 6 terms, period pi)
 *   rest of the right-hand side 81 (4 of them reciprocals)  ->  124 / 116 per right-hand side
 *   4 x RHS + RK4 combination 94 + finiteness probe 6 + step rule and lambda update 2 = 598 / 566 per step;
 *   FP32: eight compensated sums, + 24 = 590. */
int gray2_flops_per_step_bl(int32_t prec) { return prec == GRAY2_F32 ? 590 : 598; }

int gray2_order_longest_first(const int32_t *steps_hint, uint64_t n, int32_t *order, void *cuda_stream) {
  if (!steps_hint || !order || n == 0) return fail(GRAY2_EINVAL, "gray2_order_longest_first: NULL pointer or n == 0");
  if (n > 0x7fffffffull) return fail(GRAY2_EINVAL, "gray2_order_longest_first: n exceeds the range of an int32 index");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return fail(GRAY2_ECUDA, "device ordinal %d out of range", dev);
  constexpr int bins = gray2::kOrderBins;
  // One histogram per device: calls are serialised, under a lock of their own (the first call allocates, and
  // acquire_slot -- every integration of the process -- must not queue behind that).
  std::lock_guard<std::mutex> guard(g_order_lock);
  Scratch &sc = g_scratch[dev];
  if (!sc.order_bins) {
    // the event first, and both published together: a failure leaves nothing half made for the next call
    cudaEvent_t ev = nullptr;
    unsigned *mem = nullptr;
    CUDA_TRY(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    cudaError_t e = cudaMalloc(&mem, (2 * bins + 1) * sizeof(unsigned));
    if (e != cudaSuccess) {
      cudaEventDestroy(ev);
      return fail(GRAY2_ECUDA, "gray2_order_longest_first: cudaMalloc of the histogram: %s", cudaGetErrorString(e));
    }
    sc.order_done = ev;
    sc.order_bins = mem;
  }
  int sms = 0;
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  unsigned *hist = sc.order_bins, *cursor = hist + bins, *kmax = hist + 2 * bins;
  unsigned grid = (unsigned)((n + 255) / 256);
  if (grid > (unsigned)(sms * 8)) grid = (unsigned)(sms * 8);
  CUDA_TRY(cudaStreamWaitEvent(st, sc.order_done, 0));       // the previous user of the histogram, on any stream
  CUDA_TRY(cudaMemsetAsync(hist, 0, (2 * bins + 1) * sizeof(unsigned), st));
  gray2::order_max_kernel<<<grid, 256, 0, st>>>(steps_hint, n, kmax);
  gray2::order_hist_kernel<<<grid, 256, 0, st>>>(steps_hint, n, kmax, hist);
  gray2::order_scan_kernel<<<1, bins / 4, 0, st>>>(hist, cursor);
  gray2::order_scatter_kernel<<<grid, 256, 0, st>>>(steps_hint, n, kmax, cursor, order);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaEventRecord(sc.order_done, st));
  return GRAY2_OK;
}

int gray2_set_launch(int32_t prec, int32_t threads_per_block, int32_t blocks_per_sm) {
  if (prec != GRAY2_F64 && prec != GRAY2_F32) return fail(GRAY2_EINVAL, "gray2_set_launch: unknown precision");
  const LaunchChoice *list = prec == GRAY2_F64 ? kF64Variants : kF32Variants;
  bool ok = threads_per_block == 0 && blocks_per_sm == 0;
  for (int i = 0; i < kNumVariants && !ok; ++i) ok = list[i].threads == threads_per_block && list[i].blocks == blocks_per_sm;
  if (!ok) return fail(GRAY2_EINVAL, "gray2_set_launch: %d x %d is not a compiled variant", threads_per_block, blocks_per_sm);
  g_launch[prec].store(((uint32_t)threads_per_block << 16) | (uint32_t)blocks_per_sm, std::memory_order_relaxed);
  return GRAY2_OK;
}

}  // extern "C"

// ---- gray2_init_explicit_noalloc: explicit initial data without any allocation -----------------------
// gray2_init_explicit parks the caller's host array in a device buffer that the library cudaMallocs and, when a
// later call brings more geodesics, cudaFrees and cudaMallocs again.  Programs that have given the GPU's memory to
// an allocator of their own, that run a frame loop which a device-wide synchronisation would stall, or that lock
// allocation down after start-up cannot have that (the full account is beside the declaration in gray2.h).  For
// them the same kernel, init_explicit_kernel, reads its staging data from the array below instead: it is part of
// the library's device image, so it costs its 4 MiB on every GPU that loads the library, from the load until the
// process exits, called or not, and nobody ever allocates or frees it.
//
// g_noalloc_stage as written here in HOST code is only the host-side handle of the array, not a device address;
// handing it to a kernel or to cudaMemcpy as a pointer would make the GPU fault (or, where the GPU can reach host
// memory, quietly read the wrong bytes).  The device address is asked for once per device with
// cudaGetSymbolAddress, that device being current, and every later call uses the address kept here.
static __device__ __align__(256) double g_noalloc_stage[(size_t)GRAY2_NOALLOC_MAX_GEODESICS * 8];

namespace {

double *g_noalloc_addr[kMaxDevices] = {};   // device address of g_noalloc_stage on each device, NULL = not asked yet
std::mutex g_noalloc_lock;

// Device address of the staging array on the current device `dev`.  The first call per device does the look-up
// (the runtime loads the library's device code on that device first if it has not yet); no memory is allocated.
int noalloc_stage_of(int dev, double **out) {
  std::lock_guard<std::mutex> guard(g_noalloc_lock);
  if (!g_noalloc_addr[dev]) {
    void *addr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&addr, g_noalloc_stage);
    if (e != cudaSuccess || !addr)
      return fail(GRAY2_ECUDA, "gray2_init_explicit_noalloc: cudaGetSymbolAddress of the staging array on device %d: %s",
                  dev, cudaGetErrorString(e));
    g_noalloc_addr[dev] = static_cast<double *>(addr);
  }
  *out = g_noalloc_addr[dev];
  return GRAY2_OK;
}

}  // namespace

extern "C" int gray2_init_explicit_noalloc(gray2_state *s, double a, const double *host_xu8, uint64_t n, int32_t kind,
                                           int32_t renorm, void *cuda_stream) {
  const char *who = "gray2_init_explicit_noalloc";
  if (s) s->coords = GRAY2_KS;
  int rc = check_state(s, who);
  if (rc) return rc;
  if (!host_xu8 || n == 0) return fail(GRAY2_EINVAL, "%s: host_xu8 is NULL or n == 0", who);
  if (n > (uint64_t)GRAY2_NOALLOC_MAX_GEODESICS)
    return fail(GRAY2_EINVAL, "%s: n = %llu is more than the %d geodesics (GRAY2_NOALLOC_MAX_GEODESICS) the fixed staging "
                "array holds; split the batch, or use gray2_init_explicit if the program may allocate",
                who, (unsigned long long)n, (int)GRAY2_NOALLOC_MAX_GEODESICS);
  if (n > s->n) return fail(GRAY2_ESTATE, "%s: n (%llu) exceeds s->n (%llu)", who, (unsigned long long)n, (unsigned long long)s->n);
  if (!(fabs(a) <= 1.0)) return fail(GRAY2_EINVAL, "%s: |a| must be <= 1 (got %g)", who, a);
  if (kind != GRAY2_NULL && kind != GRAY2_TIMELIKE) return fail(GRAY2_EINVAL, "%s: kind must be GRAY2_NULL or GRAY2_TIMELIKE", who);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return fail(GRAY2_ECUDA, "device ordinal %d out of range", dev);
  double *stage = nullptr;
  rc = noalloc_stage_of(dev, &stage);
  if (rc) return rc;
  // Copy and kernel both go on the caller's stream: no internal stream and no events exist on this path.  The copy
  // overwrites the first 64 n bytes of the array and the kernel reads exactly those, so whatever an earlier call
  // left behind is never seen and nothing has to be cleared first.
  const double mu2 = kind == GRAY2_TIMELIKE ? 1.0 : 0.0;
  CUDA_TRY(cudaMemcpyAsync(stage, host_xu8, (size_t)n * 8 * sizeof(double), cudaMemcpyHostToDevice, st));
  unsigned grid = (unsigned)((n + 255) / 256);
  if (s->prec == GRAY2_F64)
    gray2::init_explicit_kernel<double><<<grid, 256, 0, st>>>(view_of<double>(s), stage, n, a, renorm, mu2);
  else
    gray2::init_explicit_kernel<float><<<grid, 256, 0, st>>>(view_of<float>(s), stage, n, a, renorm, mu2);
  CUDA_TRY(cudaGetLastError());
  s->a_eff = a; s->kind = kind; s->reversed = 0; s->coords = GRAY2_KS;
  return GRAY2_OK;
}
