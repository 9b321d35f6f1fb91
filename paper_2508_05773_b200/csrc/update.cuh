// update.cuh -- grid-level merge of the per-block online-softmax partials and the nominal update
// (DESIGN.md §2 rows a7/a8), warm-start shift and plant step (a9), and the debug kernels behind
// brmppi_debug_*.
//
// Merge of partials (m_p, eta_p, A_p[2T]) in partial-index order (deterministic, SURVEY §7 hard
// part 6):   m = min_p m_p;  c_p = exp(-(m_p - m)/lambda);  eta = sum_p c_p eta_p;
//            U[o] = sum_p c_p A_p[o] / eta                          (eq. 5)
#pragma once

#include <curand_philox4x32_x.h>   // library pin only: brmppi_debug_philox_raw(use_curand = 1)

#include "brmppi_device.cuh"
#include "hitch_filter.cuh"

namespace brmppi {

constexpr int kUpdateBlock = 256;
constexpr int kUpdateOutputsPerBlock = 1;   // one CTA per output channel o = 2 t + c

// One CTA per (output channel, scene): every thread takes partials p = tid, tid + 256, ...
// (coalesced rows, all loads of a thread independent and the first partial's issued together: one L2 round trip),
// then a fixed-order block reduction.  Every CTA recomputes the global minimum itself -- P * 12
// bytes from L2 -- rather than paying a third kernel or a grid-wide sync for it.
//
// MODE (K-sharded solves): the online-softmax state (m, eta, A[2T]) is associative, so a
// solve can be split over contexts / GPUs that each own a range of the samples.
//   kMergeLocal   this context's partials -> U, diagnostics, counter + 1            (the single-GPU path)
//   kMergeExport  this context's partials -> ONE shard record (m, argmin, eta, w2, nonfinite, A[2T]) in
//                 `shard`, nothing else touched
//   kMergeImport  n_shards shard records in `shard` ([n_shards][n_scenes][kShardHeader + 2T] floats, in
//                 shard order) -> U, diagnostics, counter + 1
// Shard record: words 0-1 = m (fp64), 2 = argmin (int), 3 = eta, 4 = sum w^2, 5 = nonfinite (int), 6-7 unused,
// 8 + o = A[o] (o = 2t + channel).
enum MergeMode { kMergeLocal = 0, kMergeExport = 1, kMergeImport = 2 };
constexpr int kShardHeader = 8;

template <int MODE>
__global__ void __launch_bounds__(kUpdateBlock)
merge_update(const __grid_constant__ DeviceParams P, float* shard, int n_shards) {
  __shared__ double sM[kUpdateBlock / 32];
  __shared__ int sI[kUpdateBlock / 32];
  __shared__ float sRed[4][kUpdateBlock / 32];
  const int scene = blockIdx.y, o = blockIdx.x;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int words = kShardHeader + 2 * P.T;
  // partial slots in use: the persistent kernel writes one per CTA whose tile range touches this
  // scene (CTA b owns the flat tiles [b Q, (b+1) Q)); the thread-per-sample kernels fill them all
  const int Pstride = P.n_partials;
  int Pn = Pstride;
  if (MODE == kMergeImport) {
    Pn = n_shards;
  } else if (P.tiles_per_cta > 0) {
    const int first = (scene * P.tiles_per_scene) / P.tiles_per_cta;
    const int last = ((scene + 1) * P.tiles_per_scene - 1) / P.tiles_per_cta;
    Pn = last - first + 1;
  }
  const double* pm = P.part_m + (size_t)scene * Pstride;
  const int* pi = P.part_argmin + (size_t)scene * Pstride;
  const float* peta = P.part_eta + (size_t)scene * Pstride;
  const float* pa = P.part_A + ((size_t)scene * 2 * P.T + o) * Pstride;
  const float* pw2 = P.part_w2 + (size_t)scene * Pstride;
  const int* pnf = P.part_nonfinite + (size_t)scene * Pstride;
  auto rec = [&](int p) { return shard + ((size_t)p * P.n_scenes + scene) * words; };
  auto part_m = [&](int p) { return MODE == kMergeImport ? *reinterpret_cast<const double*>(rec(p)) : pm[p]; };
  auto part_i = [&](int p) { return MODE == kMergeImport ? __float_as_int(rec(p)[2]) : pi[p]; };

  // A thread's first partial (its only one while there are no more partials than threads: one per SM) is
  // loaded whole before the minimum is known, so that the kernel is ONE L2 round trip deep, not two.
  const bool diag_cta = (o == 0);
  const bool have = tid < Pn;
  double m0 = CUDART_INF;
  int i0 = 0x7fffffff;
  float eta0 = 0.0f, acc0 = 0.0f, w20 = 0.0f, nf0 = 0.0f;
  if (have) {
    m0 = part_m(tid); i0 = part_i(tid);
    if (MODE == kMergeImport) {
      const float* r = rec(tid);
      eta0 = r[3]; acc0 = r[kShardHeader + o];
      if (diag_cta) { w20 = r[4]; nf0 = (float)__float_as_int(r[5]); }
    } else {
      eta0 = peta[tid]; acc0 = pa[tid];
      if (diag_cta) { w20 = pw2[tid]; nf0 = (float)pnf[tid]; }
    }
  }
  // global minimum and its sample index (lowest index on ties)
  double m = m0;
  int idx = i0;
  for (int p = tid + kUpdateBlock; p < Pn; p += kUpdateBlock) {
    const double om = part_m(p);
    const int oi = part_i(p);
    if (om < m || (om == m && oi < idx)) { m = om; idx = oi; }
  }
  warp_argmin(m, idx);
  if (lane == 0) { sM[warp] = m; sI[warp] = idx; }
  __syncthreads();
  m = sM[0]; idx = sI[0];
#pragma unroll
  for (int w = 1; w < kUpdateBlock / 32; ++w)
    if (sM[w] < m || (sM[w] == m && sI[w] < idx)) { m = sM[w]; idx = sI[w]; }
  const bool any_finite = m < CUDART_INF;

  float eta = 0.0f, acc = 0.0f, w2 = 0.0f, nf = 0.0f;
  if (have) {
    const float c = (any_finite && m0 < CUDART_INF) ? expf((float)(-(m0 - m) * (double)P.inv_lambda)) : 0.0f;
    eta = c * eta0; acc = c * acc0;
    if (diag_cta) { w2 = (c * c) * w20; nf = nf0; }
  }
  for (int p = tid + kUpdateBlock; p < Pn; p += kUpdateBlock) {
    const double mp = part_m(p);
    const float c = (any_finite && mp < CUDART_INF) ? expf((float)(-(mp - m) * (double)P.inv_lambda)) : 0.0f;
    if (MODE == kMergeImport) {
      const float* r = rec(p);
      eta = fmaf(c, r[3], eta);
      acc = fmaf(c, r[kShardHeader + o], acc);
      if (diag_cta) { w2 = fmaf(c * c, r[4], w2); nf += (float)__float_as_int(r[5]); }
    } else {
      eta = fmaf(c, peta[p], eta);
      acc = fmaf(c, pa[p], acc);
      if (diag_cta) { w2 = fmaf(c * c, pw2[p], w2); nf += (float)pnf[p]; }
    }
  }
  eta = warp_sum(eta); acc = warp_sum(acc); w2 = warp_sum(w2); nf = warp_sum(nf);
  if (lane == 0) { sRed[0][warp] = eta; sRed[1][warp] = acc; sRed[2][warp] = w2; sRed[3][warp] = nf; }
  __syncthreads();
  if (tid == 0) {
    eta = 0.0f; acc = 0.0f; w2 = 0.0f; nf = 0.0f;
#pragma unroll
    for (int w = 0; w < kUpdateBlock / 32; ++w) { eta += sRed[0][w]; acc += sRed[1][w]; w2 += sRed[2][w]; nf += sRed[3][w]; }
    if (MODE == kMergeExport) {
      float* r = shard + (size_t)scene * words;
      r[kShardHeader + o] = acc;
      if (diag_cta) {
        *reinterpret_cast<double*>(r) = m;
        r[2] = __int_as_float(any_finite ? idx : 0x7fffffff);
        r[3] = eta; r[4] = w2; r[5] = __int_as_float((int)nf); r[6] = 0.0f; r[7] = 0.0f;
      }
      return;
    }
    {
      // the new nominal also goes straight to its page-locked host mirror (zero-copy: brmppi_get_controls after a
      // solve then needs no copy node behind the graph); an update that is skipped mirrors the value that stays
      float* u = P.U + (size_t)scene * 2 * P.T + o;
      const bool upd = any_finite && eta > 0.0f;
      const float u_new = upd ? acc / eta : *u;
      if (upd) *u = u_new;
      if (P.U_host != nullptr) P.U_host[(size_t)scene * 2 * P.T + o] = u_new;
    }
    if (diag_cta) {
      brmppi_diag d;
      d.S_min = any_finite ? (float)m : CUDART_INF_F;
      d.argmin = any_finite ? idx : -1;
      d.eta = eta;
      d.ess = w2 > 0.0f ? eta * eta / w2 : 0.0f;
      d.n = 0ull;                       // filled in by the host, which tracks the counter
      d.nonfinite = (int)nf;
      P.diag[scene] = d;
      // the rollout kernels of this iteration have all finished (kernel boundary); the next
      // iteration draws fresh noise (reading 7).  Only this one thread touches the counter.
      if (scene == 0) *P.counter = *P.counter + 1u;
    }
  }
}

// Warm-start shift (reading 4) and, when PLANT, the kinematic plant step with the
// first control and constant-velocity obstacle advance (DESIGN.md §2 row a9).  One block per
// scene.  The plant step always uses libdevice sincosf/tanf: it runs once per control step.
constexpr int kShiftBlock = 128;
constexpr int kShiftMaxPerThread = (BRMPPI_MAX_T + kShiftBlock - 1) / kShiftBlock;

template <bool PLANT>
__global__ void __launch_bounds__(kShiftBlock) shift_plant(const __grid_constant__ DeviceParams P) {
  const int scene = blockIdx.x, tid = threadIdx.x, T = P.T;
  float2* U = reinterpret_cast<float2*>(P.U) + (size_t)scene * T;
  if (PLANT) {
    if (tid == 0 && (P.flags & BRMPPI_FLAG_MPCC)) {
      // eq. (6) under u = (j, omega) = U[0], the path parameter by the projection velocity (reading 31)
      const float2 u0 = U[0];
      float* x = P.state7 + 8 * scene;
      const float v = x[2], a = x[3], t1 = x[4], t2 = x[5], de = x[6], psi = x[7];
      const int M = P.path_M[scene];
      const float dpsi = P.path_dpsi[scene];
      int m = (int)floorf(psi / dpsi);
      m = m > M - 1 ? M - 1 : (m < 0 ? 0 : m);
      const float s = psi - (float)m * dpsi;
      const float* q = P.path_coef + ((size_t)scene * P.max_path_segments + m) * 16 + 8;   // theta^{1,r}
      const float th1r = fmaf(s, fmaf(s, fmaf(s, q[3], q[2]), q[1]), q[0]);
      float s1, c1;
      sincosf(t1, &s1, &c1);
      const float td = tanf(de), b = t1 - t2;
      x[0] = fmaf(P.dt * v, c1, x[0]);
      x[1] = fmaf(P.dt * v, s1, x[1]);
      x[2] = fmaf(P.dt, a, v);
      x[3] = fmaf(P.dt, u0.x, a);
      x[4] = wrap_angle(fmaf(P.dt * v * P.inv_L1, td, t1));
      x[5] = wrap_angle(fmaf(P.dt * v * P.inv_L2, fmaf(-P.Lh_over_L1 * td, cosf(b), sinf(b)), t2));
      x[6] = fminf(fmaxf(fmaf(P.dt, u0.y, de), P.dstate_lo), P.dstate_hi);
      x[7] = fminf(fmaxf(fmaf(P.dt, v * cosf(t1 - th1r), psi), 0.0f), (float)M * dpsi);
      reinterpret_cast<float2*>(P.u0_applied)[scene] = u0;
      if (P.u0_host != nullptr) reinterpret_cast<float2*>(P.u0_host)[scene] = u0;
    } else if (tid == 0) {
      const float2 u_ref = U[0];
      float4 x = reinterpret_cast<float4*>(P.state)[scene];
      float2 u0 = u_ref;
      int status = 0;
      if (P.hitch_filter) u0 = hitch_filter(P, x.z, x.w, u_ref, &status);   // Sec. V-D
      reinterpret_cast<float4*>(P.hitch_ref)[scene] = make_float4(u_ref.x, u_ref.y, __int_as_float(status), 0.0f);
      float s1, c1, s2, c2;
      sincosf(x.z, &s1, &c1);
      sincosf(x.w, &s2, &c2);
      const State N = kinematic_step(P, State{x.x, x.y, x.z, x.w}, s1, c1, s2, c2, u0.x, tanf(u0.y));
      reinterpret_cast<float4*>(P.state)[scene] = make_float4(N.x, N.y, wrap_angle(N.psi1), wrap_angle(N.psi2));
      reinterpret_cast<float2*>(P.u0_applied)[scene] = u0;
      if (P.u0_host != nullptr) reinterpret_cast<float2*>(P.u0_host)[scene] = u0;   // zero-copy: no D2H node in the step graph
    }
    const int n_obs = P.n_obs[scene];
    for (int i = tid; i < n_obs; i += kShiftBlock) {
      float* ob = P.obstacles + ((size_t)scene * P.max_obstacles + i) * 5;
      ob[0] = fmaf(P.dt, ob[3], ob[0]);
      ob[1] = fmaf(P.dt, ob[4], ob[1]);
    }
    const int n_se = P.max_superellipses > 0 ? P.n_se[scene] : 0;
    for (int i = tid; i < n_se; i += kShiftBlock) {
      float* q = P.se + ((size_t)scene * P.max_superellipses + i) * 8;
      q[0] = fmaf(P.dt, q[5], q[0]);
      q[1] = fmaf(P.dt, q[6], q[1]);
    }
  }
  float2 next[kShiftMaxPerThread];
#pragma unroll
  for (int r = 0; r < kShiftMaxPerThread; ++r) {
    const int t = tid + r * kShiftBlock;
    if (t + 1 < T) next[r] = U[t + 1];
  }
  __syncthreads();
#pragma unroll
  for (int r = 0; r < kShiftMaxPerThread; ++r) {
    const int t = tid + r * kShiftBlock;
    if (t + 1 < T) U[t] = next[r];
  }
}

// ---- debug kernels (brmppi_debug_*) ----------------------------------------------------------
__global__ void debug_philox(uint32_t key0, uint32_t key1, uint32_t n, int K, int T, uint32_t tag,
                             uint4* out) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)K * T) return;
  const uint32_t k = (uint32_t)(i / T), t = (uint32_t)(i % T);
  out[i] = philox4x32_10(t, n, k, tag, key0, key1);
}

// Arbitrary (counter, key) blocks through this library's generator, or through the toolkit's raw
// curand_Philox4x32_10(uint4, uint2) device function (the library pin of SURVEY §8(c)).
template <bool CURAND>
__global__ void debug_philox_raw(int n, const uint4* ctr, const uint2* key, uint4* out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 c = ctr[i];
  const uint2 k = key[i];
  out[i] = CURAND ? curand_Philox4x32_10(c, k) : philox4x32_10(c.x, c.y, c.z, c.w, k.x, k.y);
}

template <bool PRECISE>
__global__ void debug_sample_controls(const __grid_constant__ DeviceParams P, uint32_t n,
                                      const float2* U_nom, float2* u_out, float* alpha_out) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)P.K * P.T) return;
  const uint32_t k = (uint32_t)(i / P.T), t = (uint32_t)(i % P.T);
  if (u_out) u_out[i] = sample_control<PRECISE>(P, U_nom[t], t, n, k, P.key0, P.key1);
  if (alpha_out && t == 0) alpha_out[k] = sample_alpha(P, n, k, P.key0, P.key1);
}

}  // namespace brmppi
