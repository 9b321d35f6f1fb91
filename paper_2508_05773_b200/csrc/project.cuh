// Closed-form projection of BR-MPPI, eq. (11)-(12), PAPER.md:183-192:
//   z* = M^-1 [ p - A^T (A M^-1 A^T)^-1 (A M^-1 p - b) ],  M = W + rho I,  p = W z_des + rho/2 (z_hi + z_lo),
// z = [u_proj (2), u_proj^alpha (N_o)], A is N_o x d with d = 2 + N_o, W diagonal.  One thread per problem
// with everything in registers (N_o is a template parameter, all loops unroll): y = M^-1 p, r = A y - b,
// S = A M^-1 A^T by its lower triangle, Cholesky S = L L^T in place, two triangular solves, z = y - M^-1 A^T nu.
// A 128-thread CTA takes 128 consecutive problems, whose A, b, z_des blocks are contiguous in HBM.  Two paths:
// project_batch_bulk (below; persistent CTAs, TMA bulk copies, every full block of a 16-byte aligned call)
// and project_block_generic (coalesced LDG into odd-stride shared rows; the ragged tail and unaligned
// pointers).  Both run the same arithmetic in the same order, so a problem's result does not depend on the
// path or on its position.  432 B and ~1 k instructions per problem at N_o = 8: HBM-bound on paper
// (DESIGN.md 6.9).
#pragma once

#include <atomic>
#include <cuda_runtime.h>
#include <cstdint>

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
#pragma unroll 8
  for (int i = threadIdx.x; i < total; i += kProjBlock) {
    const int r = i / len, c = i - r * len;
    dst[r * stride + c] = __ldg(src + i);
  }
}

// `rows` (<= 128) problems starting at problem `first`, by the whole CTA, through `smem` (ProjSmem<NO>::words).
template <int NO>
__device__ __forceinline__ void project_block_generic(float* smem, size_t first, int rows, const float* __restrict__ A,
                                                      const float* __restrict__ b, const float* __restrict__ z_des,
                                                      const ProjConst& C, float* __restrict__ z_out) {
  using SM = ProjSmem<NO>;
  constexpr int D = SM::D;
  float* sA = smem;
  float* sB = sA + kProjBlock * SM::strideA;
  float* sZ = sB + kProjBlock * SM::strideB;
  proj_stage_in(sA, A + first * (NO * D), rows, NO * D, SM::strideA);
  proj_stage_in(sB, b + first * NO, rows, NO, SM::strideB);
  proj_stage_in(sZ, z_des + first * D, rows, D, SM::strideZ);
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
  float* out = z_out + first * D;
#pragma unroll 4
  for (int i = threadIdx.x; i < total; i += kProjBlock) {
    const int r = i / D, c = i - r * D;
    out[i] = sZ[r * SM::strideZ + c];
  }
}

template <int NO>
__global__ void __launch_bounds__(kProjBlock) project_batch(int n, const float* __restrict__ A, const float* __restrict__ b,
                                                            const float* __restrict__ z_des,
                                                            const __grid_constant__ ProjConst C, float* __restrict__ z_out) {
  extern __shared__ float smem[];
  const size_t first = (size_t)blockIdx.x * kProjBlock;
  project_block_generic<NO>(smem, first, min(kProjBlock, n - (int)first), A, b, z_des, C, z_out);
}


// ---- bulk-copy (TMA 1-D) kernel -----------------------------------------------------------------------
// Full 128-problem blocks only.  The CTA's A, b and z_des blocks are contiguous in HBM and arrive by three
// cp.async.bulk copies issued by one thread, all completing on one mbarrier: no load passes through
// registers and no index arithmetic is issued for staging.  The A block lands unpadded.  For odd N_o a row is
// an odd number of words, so thread t reading word j of row t is conflict-free with scalar LDS.  For even
// N_o a row is a multiple of 16 bytes and is read with LDS.128; a quarter-warp's eight accesses then fall on
// two to four distinct 16-byte slots mod 8 (2- to 4-way conflicts), which costs the same shared-memory
// cycles as conflict-free scalar loads and is cheaper than what avoids it: one bulk copy per row into
// padded rows ran 2-45 % slower (profiles/r1d_project.md), the TMA unit being the limit then.
// z returns through one bulk store of the CTA's contiguous z block.
__device__ __forceinline__ uint32_t proj_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int NO>
struct ProjBulkSmem {
  static constexpr int D = NO + 2;
  static constexpr int rowA = NO * D;                       // words, a multiple of 4 for even NO
  static constexpr int strideA = rowA;                      // the block lands unpadded, as it lies in HBM
  static constexpr int offB = kProjBlock * strideA;         // words
  static constexpr int offZ = offB + kProjBlock * NO;
  static constexpr int offOut = (offZ + kProjBlock * D + 31) & ~31;   // two z-out buffers, 128-byte aligned
  static constexpr int outWords = (kProjBlock * D + 31) & ~31;
  static constexpr int offBar = offOut + 2 * outWords;      // one mbarrier
  static constexpr int bulk_words = offBar + 2;
  static constexpr int words = bulk_words > ProjSmem<NO>::words ? bulk_words : ProjSmem<NO>::words;
  static constexpr int bytes = words * 4;
  static constexpr unsigned tx = kProjBlock * (rowA + NO + D) * 4;
};

// Loads of one full block into the stage: three bulk copies (the CTA's A, b and z_des blocks are contiguous).
template <int NO>
__device__ __forceinline__ void proj_issue_loads(float* st, uint32_t bar, size_t first, const float* __restrict__ A,
                                                 const float* __restrict__ b, const float* __restrict__ z_des) {
  using SM = ProjBulkSmem<NO>;
  const int t = threadIdx.x;
  if (t == 0)
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(SM::tx) : "memory");
  if (t == 0) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(proj_smem_u32(st)), "l"(A + first * SM::rowA), "r"(kProjBlock * SM::rowA * 4), "r"(bar) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(proj_smem_u32(st + SM::offB)), "l"(b + first * NO), "r"(kProjBlock * NO * 4), "r"(bar) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(proj_smem_u32(st + SM::offZ)), "l"(z_des + first * SM::D), "r"(kProjBlock * SM::D * 4), "r"(bar)
                 : "memory");
  }
}

// Persistent: CTA c of the first gridDim.x - 1 takes the full blocks c, c + P, c + 2P, ... (P = gridDim.x - 1).
// A thread keeps its whole problem in registers, so the load stage is free again as soon as every thread has
// read its rows: the loads of the CTA's next block are issued right then and are in flight during the whole
// computation of the current one (one stage of 52 KB instead of two -> three CTAs per SM at N_o = 8).  z goes
// out through two small buffers so that a bulk store may still be reading one while the next is written.
// The last CTA takes the ragged tail (n_tail < 128 problems) through the generic path.
template <int NO>
__global__ void __launch_bounds__(kProjBlock) project_batch_bulk(int full_blocks, int n_tail, const float* __restrict__ A,
                                                                 const float* __restrict__ b,
                                                                 const float* __restrict__ z_des,
                                                                 const __grid_constant__ ProjConst C,
                                                                 float* __restrict__ z_out) {
  using SM = ProjBulkSmem<NO>;
  constexpr int D = SM::D;
  extern __shared__ __align__(128) float smem[];
  const int t = threadIdx.x;
  const int P = (int)gridDim.x - 1;
  if ((int)blockIdx.x == P) {
    if (n_tail > 0)
      project_block_generic<NO>(smem, (size_t)full_blocks * kProjBlock, n_tail, A, b, z_des, C, z_out);
    return;
  }
  const uint32_t bar0 = proj_smem_u32(smem + SM::offBar);
  if (t == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar0));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  int blk = blockIdx.x;
  if (blk < full_blocks) proj_issue_loads<NO>(smem, bar0, (size_t)blk * kProjBlock, A, b, z_des);
  float* const st = smem;
  for (int it = 0; blk < full_blocks; ++it, blk += P) {
    {
      const uint32_t parity = (uint32_t)it & 1u;
      uint32_t done = 0;
      while (!done)
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(bar0), "r"(parity) : "memory");
    }
    float minv[D], y[D], a[NO][D];
    const float* zrow = st + SM::offZ + t * D;
    float* const orow = smem + SM::offOut + (it & 1) * SM::outWords + t * D;
    if constexpr (NO % 2 == 0) {
#pragma unroll
      for (int j = 0; j < D; j += 2) {
        const float2 zd = *reinterpret_cast<const float2*>(zrow + j);
        minv[j] = 1.0f / (C.w[j] + C.rho);
        minv[j + 1] = 1.0f / (C.w[j + 1] + C.rho);
        y[j] = fmaf(C.w[j], zd.x, 0.5f * C.rho * (C.hi[j] + C.lo[j])) * minv[j];
        y[j + 1] = fmaf(C.w[j + 1], zd.y, 0.5f * C.rho * (C.hi[j + 1] + C.lo[j + 1])) * minv[j + 1];
      }
#pragma unroll
      for (int q = 0; q < SM::rowA / 4; ++q) {
        const float4 v = *reinterpret_cast<const float4*>(st + t * SM::strideA + 4 * q);
        a[(4 * q) / D][(4 * q) % D] = v.x;
        a[(4 * q + 1) / D][(4 * q + 1) % D] = v.y;
        a[(4 * q + 2) / D][(4 * q + 2) % D] = v.z;
        a[(4 * q + 3) / D][(4 * q + 3) % D] = v.w;
      }
    } else {
#pragma unroll
      for (int j = 0; j < D; ++j) {
        minv[j] = 1.0f / (C.w[j] + C.rho);
        y[j] = fmaf(C.w[j], zrow[j], 0.5f * C.rho * (C.hi[j] + C.lo[j])) * minv[j];
      }
#pragma unroll
      for (int i = 0; i < NO; ++i)
#pragma unroll
        for (int j = 0; j < D; ++j) a[i][j] = st[t * SM::strideA + i * D + j];
    }
    float nu[NO];
    if constexpr (NO % 2 == 0) {
#pragma unroll
      for (int i = 0; i < NO; i += 2) {
        const float2 bb = *reinterpret_cast<const float2*>(st + SM::offB + t * NO + i);
        nu[i] = -bb.x; nu[i + 1] = -bb.y;
      }
    } else {
#pragma unroll
      for (int i = 0; i < NO; ++i) nu[i] = -st[SM::offB + t * NO + i];
    }
    // every thread holds its problem in registers: hand the stage back and start the next block's loads; the
    // z-out buffer written below was last read by the bulk store of iteration it - 2
    // (the refill is an async-proxy write issued by another thread: bar.sync alone does not order this
    // thread's shared loads, possibly still in flight, before it -- the proxy fence does)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (t == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
    __syncthreads();
    if (blk + P < full_blocks) proj_issue_loads<NO>(smem, bar0, (size_t)(blk + P) * kProjBlock, A, b, z_des);
#pragma unroll
    for (int i = 0; i < NO; ++i)
#pragma unroll
      for (int j = 0; j < D; ++j) nu[i] = fmaf(a[i][j], y[j], nu[i]);
    float S[NO][NO];
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
    for (int k = 0; k < NO; ++k) {
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
    for (int i = 0; i < NO; ++i) {
      float v = nu[i];
#pragma unroll
      for (int m = 0; m < i; ++m) v = fmaf(-S[i][m], nu[m], v);
      nu[i] = v * S[i][i];
    }
#pragma unroll
    for (int i = NO - 1; i >= 0; --i) {
      float v = nu[i];
#pragma unroll
      for (int m = i + 1; m < NO; ++m) v = fmaf(-S[m][i], nu[m], v);
      nu[i] = v * S[i][i];
    }
    if constexpr (NO % 2 == 0) {
#pragma unroll
      for (int j = 0; j < D; j += 2) {
        float c0 = 0.0f, c1 = 0.0f;
#pragma unroll
        for (int i = 0; i < NO; ++i) { c0 = fmaf(a[i][j], nu[i], c0); c1 = fmaf(a[i][j + 1], nu[i], c1); }
        *reinterpret_cast<float2*>(orow + j) = make_float2(fmaf(-minv[j], c0, y[j]), fmaf(-minv[j + 1], c1, y[j + 1]));
      }
    } else {
#pragma unroll
      for (int j = 0; j < D; ++j) {
        float c0 = 0.0f;
#pragma unroll
        for (int i = 0; i < NO; ++i) c0 = fmaf(a[i][j], nu[i], c0);
        orow[j] = fmaf(-minv[j], c0, y[j]);
      }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the bulk store
    __syncthreads();
    if (t == 0) {
      asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                   ::"l"(z_out + (size_t)blk * kProjBlock * D),
                     "r"(proj_smem_u32(smem + SM::offOut + (it & 1) * SM::outWords)), "r"(kProjBlock * D * 4)
                   : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
  }
  if (t == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // smem must outlive the last store's read
}

constexpr int kProjMaxDevices = 64;

template <int NO>
inline cudaError_t launch_project(int n, const float* A, const float* b, const float* z_des, const ProjConst& C,
                                  float* z_out, cudaStream_t s) {
  [[maybe_unused]] constexpr int D = NO + 2;
  cudaError_t e;
  {
    // full 128-problem blocks through the bulk-copy kernel (needs 16-byte aligned arrays), the tail through
    // the generic one
    const int full = n / kProjBlock;
    const bool aligned = (((uintptr_t)A | (uintptr_t)b | (uintptr_t)z_des | (uintptr_t)z_out) & 15u) == 0;   // bulk copies
    if (full > 0 && aligned) {
      using SMB = ProjBulkSmem<NO>;
      // resident CTAs of this kernel per device: one atomic word per device, written once (the
      // function attribute is per device too); two threads racing compute the same value
      static std::atomic<int> resident[kProjMaxDevices];
      int dev = 0;
      if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
      int persistent_ctas = (dev >= 0 && dev < kProjMaxDevices) ? resident[dev].load(std::memory_order_acquire) : 0;
      if (persistent_ctas == 0) {
        e = cudaFuncSetAttribute(project_batch_bulk<NO>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMB::bytes);
        if (e != cudaSuccess) return e;
        int sms = 0, per_sm = 0;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, project_batch_bulk<NO>, kProjBlock, SMB::bytes);
        if (e != cudaSuccess) return e;
        persistent_ctas = sms * (per_sm > 0 ? per_sm : 1);
        if (persistent_ctas < 2) persistent_ctas = 2;     // one CTA for the full blocks, one for the tail
        if (dev >= 0 && dev < kProjMaxDevices) resident[dev].store(persistent_ctas, std::memory_order_release);
      }
      // P persistent CTAs for the full blocks + one CTA for the ragged tail, all resident in one wave
      const int P = full < persistent_ctas - 1 ? full : persistent_ctas - 1;
      project_batch_bulk<NO><<<(unsigned)(P + 1), kProjBlock, SMB::bytes, s>>>(full, n - full * kProjBlock, A, b, z_des, C, z_out);
      return cudaGetLastError();
    }
  }
  const size_t bytes = sizeof(float) * ProjSmem<NO>::words;
  {
    static std::atomic<int> configured[kProjMaxDevices];
    int dev = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if (dev < 0 || dev >= kProjMaxDevices || configured[dev].load(std::memory_order_acquire) == 0) {
      e = cudaFuncSetAttribute(project_batch<NO>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
      if (e != cudaSuccess) return e;
      if (dev >= 0 && dev < kProjMaxDevices) configured[dev].store(1, std::memory_order_release);
    }
  }
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
