// Closed-form projection of BR-MPPI, eq. (11)-(12), PAPER.md:183-192:
//   z* = M^-1 [ p - A^T (A M^-1 A^T)^-1 (A M^-1 p - b) ],  M = W + rho I,  p = W z_des + rho/2 (z_hi + z_lo),
// z = [u_proj (2), u_proj^alpha (N_o)], A is N_o x d with d = 2 + N_o, W diagonal.  One thread per problem
// with everything in registers (N_o is a template parameter, all loops unroll): y = M^-1 p, r = A y - b,
// S = A M^-1 A^T by its lower triangle, Cholesky S = L L^T in place, two triangular solves, z = y - M^-1 A^T nu.
// A 128-thread CTA takes 128 consecutive problems; their A, b, z_des blocks are contiguous in HBM and are
// staged through shared memory with coalesced 16-byte loads, rows padded to an odd stride so that thread
// i reading word j of its own row hits bank (i * stride + j) mod 32 without conflict; z goes back the same
// way.  432 B and ~1.5 kflop per problem at N_o = 8: HBM-bound.
#pragma once
#include <cuda_runtime.h>

namespace brmppi {

constexpr int kProjMaxNo = 8;
constexpr int kProjBlock = 128;

struct ProjConst {
  float w[kProjMaxNo + 2], lo[kProjMaxNo + 2], hi[kProjMaxNo + 2];
  float rho;
};

__host__ __device__ constexpr int proj_odd(int x) { return x | 1; }

template <int NO>
struct ProjSmem {
  static constexpr int D = NO + 2;
  static constexpr int strideA = proj_odd(NO * D), strideB = proj_odd(NO), strideZ = proj_odd(D);
  static constexpr int words = kProjBlock * (strideA + strideB + strideZ);
};

// Copy `rows` rows of `len` contiguous words from global (rows back to back) to shared rows of `stride`.
__device__ __forceinline__ void proj_stage_in(float* dst, const float* __restrict__ src, int rows, int len, int stride) {
  const int total = rows * len;
  for (int i = threadIdx.x; i < total; i += kProjBlock) {
    const int r = i / len, c = i - r * len;
    dst[r * stride + c] = __ldg(src + i);
  }
}

template <int NO>
__global__ void __launch_bounds__(kProjBlock) project_batch(int n, const float* __restrict__ A, const float* __restrict__ b,
                                                            const float* __restrict__ z_des,
                                                            const __grid_constant__ ProjConst C, float* __restrict__ z_out) {
  using SM = ProjSmem<NO>;
  constexpr int D = SM::D;
  extern __shared__ float smem[];
  float* sA = smem;
  float* sB = sA + kProjBlock * SM::strideA;
  float* sZ = sB + kProjBlock * SM::strideB;
  const int first = blockIdx.x * kProjBlock;
  const int rows = min(kProjBlock, n - first);
  proj_stage_in(sA, A + (size_t)first * (NO * D), rows, NO * D, SM::strideA);
  proj_stage_in(sB, b + (size_t)first * NO, rows, NO, SM::strideB);
  proj_stage_in(sZ, z_des + (size_t)first * D, rows, D, SM::strideZ);
  __syncthreads();
  const int t = threadIdx.x;
  if (t < rows) {
    float minv[D], y[D], a[NO][D];
#pragma unroll
    for (int j = 0; j < D; ++j) {
      minv[j] = 1.0f / (C.w[j] + C.rho);
      y[j] = fmaf(C.w[j], sZ[t * SM::strideZ + j], 0.5f * C.rho * (C.hi[j] + C.lo[j])) * minv[j];
    }
#pragma unroll
    for (int i = 0; i < NO; ++i)
#pragma unroll
      for (int j = 0; j < D; ++j) a[i][j] = sA[t * SM::strideA + i * D + j];
    float nu[NO];
#pragma unroll
    for (int i = 0; i < NO; ++i) {          // r = A M^-1 p - b
      float acc = -sB[t * SM::strideB + i];
#pragma unroll
      for (int j = 0; j < D; ++j) acc = fmaf(a[i][j], y[j], acc);
      nu[i] = acc;
    }
    float S[NO][NO];                         // lower triangle of A M^-1 A^T
#pragma unroll
    for (int i = 0; i < NO; ++i)
#pragma unroll
      for (int k = 0; k <= i; ++k) {
        float acc = 0.0f;
#pragma unroll
        for (int j = 0; j < D; ++j) acc = fmaf(a[i][j] * minv[j], a[k][j], acc);
        S[i][k] = acc;
      }
#pragma unroll
    for (int k = 0; k < NO; ++k) {           // Cholesky, L overwrites S; 1/L_kk kept on the diagonal
      float dkk = S[k][k];
#pragma unroll
      for (int m = 0; m < k; ++m) dkk = fmaf(-S[k][m], S[k][m], dkk);
      const float inv = rsqrtf(dkk);
      S[k][k] = inv;
#pragma unroll
      for (int i = k + 1; i < NO; ++i) {
        float v = S[i][k];
#pragma unroll
        for (int m = 0; m < k; ++m) v = fmaf(-S[i][m], S[k][m], v);
        S[i][k] = v * inv;
      }
    }
#pragma unroll
    for (int i = 0; i < NO; ++i) {           // L w = r
      float v = nu[i];
#pragma unroll
      for (int m = 0; m < i; ++m) v = fmaf(-S[i][m], nu[m], v);
      nu[i] = v * S[i][i];
    }
#pragma unroll
    for (int i = NO - 1; i >= 0; --i) {      // L^T nu = w
      float v = nu[i];
#pragma unroll
      for (int m = i + 1; m < NO; ++m) v = fmaf(-S[m][i], nu[m], v);
      nu[i] = v * S[i][i];
    }
#pragma unroll
    for (int j = 0; j < D; ++j) {            // z = y - M^-1 A^T nu
      float acc = 0.0f;
#pragma unroll
      for (int i = 0; i < NO; ++i) acc = fmaf(a[i][j], nu[i], acc);
      sZ[t * SM::strideZ + j] = fmaf(-minv[j], acc, y[j]);
    }
  }
  __syncthreads();
  const int total = rows * D;
  float* out = z_out + (size_t)first * D;
  for (int i = threadIdx.x; i < total; i += kProjBlock) {
    const int r = i / D, c = i - r * D;
    out[i] = sZ[r * SM::strideZ + c];
  }
}

template <int NO>
inline cudaError_t launch_project(int n, const float* A, const float* b, const float* z_des, const ProjConst& C,
                                  float* z_out, cudaStream_t s) {
  const size_t bytes = sizeof(float) * ProjSmem<NO>::words;
  cudaError_t e = cudaFuncSetAttribute(project_batch<NO>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e != cudaSuccess) return e;
  project_batch<NO><<<(unsigned)((n + kProjBlock - 1) / kProjBlock), kProjBlock, bytes, s>>>(n, A, b, z_des, C, z_out);
  return cudaGetLastError();
}

inline cudaError_t launch_project_dyn(int n_o, int n, const float* A, const float* b, const float* z_des,
                                      const ProjConst& C, float* z_out, cudaStream_t s) {
  switch (n_o) {
    case 1: return launch_project<1>(n, A, b, z_des, C, z_out, s);
    case 2: return launch_project<2>(n, A, b, z_des, C, z_out, s);
    case 3: return launch_project<3>(n, A, b, z_des, C, z_out, s);
    case 4: return launch_project<4>(n, A, b, z_des, C, z_out, s);
    case 5: return launch_project<5>(n, A, b, z_des, C, z_out, s);
    case 6: return launch_project<6>(n, A, b, z_des, C, z_out, s);
    case 7: return launch_project<7>(n, A, b, z_des, C, z_out, s);
    case 8: return launch_project<8>(n, A, b, z_des, C, z_out, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace brmppi
