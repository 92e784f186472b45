// bench_probe.cu -- FMA-only probe kernels for bench.py (NOT part of the product library).
//
// bench.py builds this file into libbench_probe.so and loads it itself, to measure the attainable FMA rate
// of the FP64 / FP32 pipe at the clocks of the moment, next to the nominal peak the roofline fraction is
// quoted against.  It uses the packed-pair type of the product's headers so that
// the packed probe issues the very FFMA2 instruction the FP32 integrator is made of.
//
//   int bench_fma_probe(int prec, int register_operands, int blocks, int threads, int iters,
//                       void *scratch /* device, >= 1 element */, void *cuda_stream)
//   prec: 0 double, 1 float.  register_operands: 0 multiplier and addend are immediates (best case of the
//   pipe); 1 three per-thread register operands, multiplier and addend shared by the eight chains; 2 every
//   chain has its own multiplier and addend (three fresh register reads per FMA: what real code issues);
//   3 (float only) as 2 with the packed FFMA2 instruction.  Flops = 16*iters*blocks*threads (32* for 3).
//   Returns 0, or 1 on a bad argument / launch error.
#include <cuda_runtime.h>
#include "paper_1706_07062_b200/csrc/f32x2.cuh"

using gray2::f32x2;
using gray2::fma_;

template <typename T, int REGS>
__global__ void fma_probe_kernel(int iters, T seed, T *__restrict__ out) {
  T a0 = seed + T(threadIdx.x), a1 = a0 + T(1), a2 = a0 + T(2), a3 = a0 + T(3);
  T a4 = a0 + T(4), a5 = a0 + T(5), a6 = a0 + T(6), a7 = a0 + T(7);
  if constexpr (REGS == 2) {
    const T d = T(threadIdx.x) * T(1e-9);
    const T m0 = T(0.999999) + d, m1 = T(0.999998) + d, m2 = T(0.999997) + d, m3 = T(0.999996) + d;
    const T m4 = T(0.999995) + d, m5 = T(0.999994) + d, m6 = T(0.999993) + d, m7 = T(0.999992) + d;
    const T c0 = T(1e-6) + d, c1 = T(2e-6) + d, c2 = T(3e-6) + d, c3 = T(4e-6) + d;
    const T c4 = T(5e-6) + d, c5 = T(6e-6) + d, c6 = T(7e-6) + d, c7 = T(8e-6) + d;
#pragma unroll 8
    for (int i = 0; i < iters; ++i) {
      a0 = fma_(a0, m0, c0); a1 = fma_(a1, m1, c1); a2 = fma_(a2, m2, c2); a3 = fma_(a3, m3, c3);
      a4 = fma_(a4, m4, c4); a5 = fma_(a5, m5, c5); a6 = fma_(a6, m6, c6); a7 = fma_(a7, m7, c7);
    }
  } else {
    const T m = REGS ? T(0.999999) + T(threadIdx.x) * T(1e-9) : T(0.999999);
    const T c = REGS ? T(1e-6) + T(threadIdx.x) * T(1e-9) : T(1e-6);
#pragma unroll 8
    for (int i = 0; i < iters; ++i) {
      a0 = fma_(a0, m, c); a1 = fma_(a1, m, c); a2 = fma_(a2, m, c); a3 = fma_(a3, m, c);
      a4 = fma_(a4, m, c); a5 = fma_(a5, m, c); a6 = fma_(a6, m, c); a7 = fma_(a7, m, c);
    }
  }
  T s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (s == T(-12345.678)) out[0] = s;   // never true; keeps the chains alive
}

__global__ void fma2_probe_kernel(int iters, float seed, float *__restrict__ out) {
  const float b = seed + (float)threadIdx.x, d = (float)threadIdx.x * 1e-9f;
  f32x2 a[8], m[8], c[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    a[j] = f32x2(b + (float)j, b + (float)j + 0.5f);
    m[j] = f32x2(0.999999f - (float)j * 1e-6f + d, 0.999991f - (float)j * 1e-6f + d);
    c[j] = f32x2((float)(j + 1) * 1e-6f + d, (float)(j + 1) * 1.5e-6f + d);
  }
#pragma unroll 8
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = fma_(a[j], m[j], c[j]);
  }
  f32x2 s = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
  if (s.v.x + s.v.y == -12345.678f) out[0] = s.v.x;   // never true; keeps the chains alive
}

extern "C" int bench_fma_probe(int prec, int register_operands, int blocks, int threads, int iters, void *scratch,
                               void *cuda_stream) {
  if (!scratch || blocks <= 0 || threads <= 0 || threads > 1024 || iters <= 0) return 1;
  if (register_operands < 0 || register_operands > 3 || (register_operands == 3 && prec != 1)) return 1;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (register_operands == 3) fma2_probe_kernel<<<blocks, threads, 0, st>>>(iters, 1.0f, (float *)scratch);
  else if (prec == 0) {
    if (register_operands == 2) fma_probe_kernel<double, 2><<<blocks, threads, 0, st>>>(iters, 1.0, (double *)scratch);
    else if (register_operands) fma_probe_kernel<double, 1><<<blocks, threads, 0, st>>>(iters, 1.0, (double *)scratch);
    else fma_probe_kernel<double, 0><<<blocks, threads, 0, st>>>(iters, 1.0, (double *)scratch);
  } else if (prec == 1) {
    if (register_operands == 2) fma_probe_kernel<float, 2><<<blocks, threads, 0, st>>>(iters, 1.0f, (float *)scratch);
    else if (register_operands) fma_probe_kernel<float, 1><<<blocks, threads, 0, st>>>(iters, 1.0f, (float *)scratch);
    else fma_probe_kernel<float, 0><<<blocks, threads, 0, st>>>(iters, 1.0f, (float *)scratch);
  } else return 1;
  return cudaGetLastError() == cudaSuccess ? 0 : 1;
}
