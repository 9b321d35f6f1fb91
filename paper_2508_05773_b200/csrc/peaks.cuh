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

enum PeakKind { PEAK_FFMA = 0, PEAK_ALU = 1, PEAK_MUFU = 2, PEAK_MIX = 3, PEAK_IMAD_WIDE = 4,
                PEAK_FMNMX = 5, PEAK_FFMA2 = 6, PEAK_FFMA2_DISTINCT = 7, PEAK_FADD2 = 8, PEAK_FFMA_FMNMX = 9,
                PEAK_FFMA2_FMNMX = 10, PEAK_IMAD_LO = 11, PEAK_IMAD_HI = 12, PEAK_KINDS = 13 };

__host__ __device__ constexpr int peak_instr_per_slot(int kind) {
  return (kind == PEAK_MIX || kind == PEAK_FFMA_FMNMX || kind == PEAK_FFMA2_FMNMX) ? 2 : 1;
}

template <int KIND>
__global__ void __launch_bounds__(256) peak_kernel(float seed, long long* spans, float* sink) {
  float f[kPeakChains], g[kPeakChains], h[kPeakChains];
  uint32_t u[kPeakChains];
  unsigned long long w[kPeakChains], q[kPeakChains], r[kPeakChains];
#pragma unroll
  for (int i = 0; i < kPeakChains; ++i) {
    f[i] = seed + (float)(threadIdx.x + i);
    g[i] = seed * 0.5f + (float)i;
    h[i] = seed * 0.25f - (float)i;
    u[i] = (uint32_t)(threadIdx.x * 2654435761u + i);
    w[i] = u[i];
    q[i] = ((unsigned long long)__float_as_uint(g[i]) << 32) | __float_as_uint(h[i]);
    r[i] = q[i] ^ 0x0000200000002000ull;
  }
  const float a = 0.999f + seed * 1e-9f, b = seed * 1e-3f;
  const uint32_t ua = __float_as_uint(a), ub = __float_as_uint(b) | 1u;
  const unsigned long long pa = ((unsigned long long)ua << 32) | ua, pb = ((unsigned long long)ub << 32) | ub;
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
      } else if (KIND == PEAK_IMAD_WIDE) {
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[i]) : "r"((uint32_t)w[i]), "r"(ua));
      } else if (KIND == PEAK_FMNMX) {          // alternate min / max so that pairs cannot fuse into FMNMX3
        if (rep & 1) asm volatile("min.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(g[i]));
        else asm volatile("max.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(h[i]));
      } else if (KIND == PEAK_FFMA2) {          // two operands shared by every instruction
        asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(w[i]) : "l"(pa), "l"(pb));
      } else if (KIND == PEAK_FFMA2_DISTINCT) { // three distinct 64-bit register operands
        asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(w[i]) : "l"(q[i]), "l"(r[i]));
      } else if (KIND == PEAK_FADD2) {
        asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(w[i]) : "l"(pa));
      } else if (KIND == PEAK_FFMA_FMNMX) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(a), "f"(b));
        if (rep & 1) asm volatile("min.f32 %0, %0, %1;" : "+f"(g[i]) : "f"(h[i]));
        else asm volatile("max.f32 %0, %0, %1;" : "+f"(g[i]) : "f"(a));
      } else if (KIND == PEAK_FFMA2_FMNMX) {
        asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(w[i]) : "l"(pa), "l"(pb));
        if (rep & 1) asm volatile("min.f32 %0, %0, %1;" : "+f"(g[i]) : "f"(h[i]));
        else asm volatile("max.f32 %0, %0, %1;" : "+f"(g[i]) : "f"(a));
      } else if (KIND == PEAK_IMAD_LO) {
        asm volatile("mul.lo.u32 %0, %0, %1;" : "+r"(u[i]) : "r"(ua));
      } else {
        asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(u[i]) : "r"(ua));
      }
    }
  }
  const long long t1 = clock64();
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
  float acc = 0.0f;
#pragma unroll
  for (int i = 0; i < kPeakChains; ++i) acc += f[i] + g[i] + h[i] + (float)u[i] + (float)(uint32_t)(w[i] >> 32) + (float)(uint32_t)q[i] + (float)(uint32_t)r[i];
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
