// peaks.cuh -- issue-rate micro-benchmarks behind brmppi_measure_peaks(): the denominators of the
// "alu"-bound roofline.  MEASURED_PEAKS.json carries only HBM GB/s and bf16
// TFLOP/s, neither of which bounds this path, so the per-SM instruction rates the roofline uses
// (issue 128, FMA pipe 128, ALU pipe 64, XU pipe 16 thread-instr/clk/SM) are confirmed here.
//
// Every kernel runs kIters x kUnroll independent instructions per thread on 8 independent
// register chains, 1024 threads per SM in one wave, and reports per-block clock64() spans.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace brmppi {

constexpr int kPeakIters = 2048;
constexpr int kPeakReps = 8;       // inner repetitions per loop trip: 64 instructions per branch
constexpr int kPeakChains = 8;

enum PeakKind { PEAK_FFMA = 0, PEAK_ALU = 1, PEAK_MUFU = 2, PEAK_MIX = 3, PEAK_IMAD_WIDE = 4 };

template <int KIND>
__global__ void __launch_bounds__(256) peak_kernel(float seed, long long* spans, float* sink) {
  float f[kPeakChains];
  uint32_t u[kPeakChains];
  unsigned long long w[kPeakChains];
#pragma unroll
  for (int i = 0; i < kPeakChains; ++i) {
    f[i] = seed + (float)(threadIdx.x + i);
    u[i] = (uint32_t)(threadIdx.x * 2654435761u + i);
    w[i] = u[i];
  }
  const float a = 0.999f + seed * 1e-9f, b = seed * 1e-3f;
  const uint32_t ua = __float_as_uint(a), ub = __float_as_uint(b) | 1u;
  __syncthreads();
  unsigned long long g0, g1;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
    for (int rep = 0; rep < kPeakReps; ++rep)
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) {
      if (KIND == PEAK_FFMA) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(a), "f"(b));
      } else if (KIND == PEAK_ALU) {
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[i]) : "r"(ua), "r"(ub));
      } else if (KIND == PEAK_MUFU) {
        asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
      } else if (KIND == PEAK_MIX) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(a), "f"(b));
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[i]) : "r"(ua), "r"(ub));
      } else {
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[i]) : "r"((uint32_t)w[i]), "r"(ua));
      }
    }
  }
  const long long t1 = clock64();
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
  float acc = 0.0f;
#pragma unroll
  for (int i = 0; i < kPeakChains; ++i) acc += f[i] + (float)u[i] + (float)(uint32_t)(w[i] >> 32);
  if (acc == 123.456f) sink[0] = acc;   // keep the chains alive
  if (threadIdx.x == 0) {
    spans[3 * blockIdx.x] = t1 - t0;
    spans[3 * blockIdx.x + 1] = (long long)g0;
    spans[3 * blockIdx.x + 2] = (long long)g1;
  }
}

// SM clock in MHz from clock64() against the nanosecond globaltimer.
__global__ void clock_rate_kernel(float* mhz_out) {
  unsigned long long g0, g1;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
  const long long c0 = clock64();
  float x = 1.0f;
  for (int i = 0; i < 200000; ++i) asm volatile("fma.rn.f32 %0, %0, %0, %0;" : "+f"(x));
  const long long c1 = clock64();
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
  if (x == 123.0f) mhz_out[1] = x;
  mhz_out[0] = (float)((double)(c1 - c0) * 1e3 / (double)(g1 - g0));
}

}  // namespace brmppi
