// rollout_thread.cuh -- baseline rollout kernel: ONE THREAD PER SAMPLE, all steps a1-a7 of
// DESIGN.md §2 fused (north_star item 2, first form).  Kept as the simple kernel the phase-split
// tile kernel (rollout_tile.cuh) is compared against, and selected by
// BRMPPI_FLAG_KERNEL_THREAD_PER_SAMPLE.
//
//   per thread k:  alpha_k;  for t: Philox -> Box-Muller -> clamp -> Euler step (eq. 6) ->
//   disc centres -> for every (obstacle, disc): h_t, h_{t+1}, hinge -> stage cost;  S_k.
//   per block:     m_b = min S, w_k = exp(-(S_k - m_b)/lambda), eta_b, A_b[t] = sum_k w_k u_k[t]
//                  (controls regenerated from Philox -- nothing per-sample is kept in memory).
//
// State stays in registers; h_t is recomputed from the previous step's disc centres, so the
// register count does not depend on the obstacle count (SURVEY §7 hard part 4).
#pragma once

#include "brmppi_device.cuh"

namespace brmppi {

constexpr int kThreadBlock = 128;

// Block partial of the online softmax (a7) for the one-thread-per-sample kernels: block minimum,
// weights, eta, and the weighted control sums with the sampled controls regenerated from the
// counter-based generator (nothing per sample is kept in memory).  All kThreadBlock threads call it.
template <bool PRECISE>
__device__ __forceinline__ void thread_kernel_epilogue(const DeviceParams& P, const float2* sU, double* sRedM,
                                                       int* sRedI, float* sRedF, float* sA, double S, bool valid,
                                                       int k, int scene, uint32_t n, uint32_t key0, uint32_t key1) {
  const int T = P.T;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool finite = valid && (S == S) && (S < CUDART_INF) && (S > -CUDART_INF);
  double m = finite ? S : CUDART_INF;
  int idx = finite ? k + P.k_offset : 0x7fffffff;       // global sample index (K-sharded solves)
  warp_argmin(m, idx);
  if (lane == 0) { sRedM[warp] = m; sRedI[warp] = idx; }
  __syncthreads();
  m = sRedM[0]; idx = sRedI[0];
#pragma unroll
  for (int w = 1; w < 4; ++w)
    if (sRedM[w] < m || (sRedM[w] == m && sRedI[w] < idx)) { m = sRedM[w]; idx = sRedI[w]; }
  // S - m in fp64, then fp32 exp (SURVEY §7 hard part 2)
  const float wk = finite ? expf((float)(-(S - m) * (double)P.inv_lambda)) : 0.0f;
  float eta = warp_sum(wk), w2 = warp_sum(wk * wk);
  float nf = warp_sum((valid && !finite) ? 1.0f : 0.0f);
  if (lane == 0) { sRedF[warp] = eta; sRedF[4 + warp] = w2; sRedF[8 + warp] = nf; }

  // weighted control sums: regenerate u_k[t] from the counter-based generator, two Philox blocks = four steps =
  // eight outputs at a time; the eight per-lane products are reduced together by a transposing butterfly (4 + 2 + 1
  // exchanges leave each lane with one output's sum over its 4-lane class, two more finish it: 9 shuffles for 8
  // outputs)
  for (int t0 = 0; t0 < T; t0 += 4) {
    float a[8];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      float2 u0 = make_float2(0.0f, 0.0f), u1 = u0;
      const int t = t0 + 2 * h;
      if (finite && t < T)
        sample_control_pair<PRECISE>(P, sU[t], sU[min(t + 1, T - 1)], (uint32_t)(t >> 1), n, (uint32_t)(k + P.k_offset),
                                     key0, key1, &u0, &u1);
      a[4 * h + 0] = wk * u0.x; a[4 * h + 1] = wk * u0.y; a[4 * h + 2] = wk * u1.x; a[4 * h + 3] = wk * u1.y;
    }
    float b4[4], b2[2], b1;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const bool hi = (lane & 16) != 0;
      const float send = hi ? a[q] : a[q + 4], keep = hi ? a[q + 4] : a[q];
      b4[q] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const bool hi = (lane & 8) != 0;
      const float send = hi ? b4[q] : b4[q + 2], keep = hi ? b4[q + 2] : b4[q];
      b2[q] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
    {
      const bool hi = (lane & 4) != 0;
      const float send = hi ? b2[0] : b2[1], keep = hi ? b2[1] : b2[0];
      b1 = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    b1 += __shfl_xor_sync(0xffffffffu, b1, 2);
    b1 += __shfl_xor_sync(0xffffffffu, b1, 1);
    const int o = 2 * t0 + ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);   // lane bits -> output
    if ((lane & 3) == 0 && o < 2 * T) sA[warp * 2 * T + o] = b1;
  }
  __syncthreads();

  const int P_n = P.n_partials;
  const size_t pbase = (size_t)scene * P_n + blockIdx.x;
  if (tid == 0) {
    P.part_m[pbase] = m;
    P.part_argmin[pbase] = idx;
    P.part_eta[pbase] = (sRedF[0] + sRedF[1]) + (sRedF[2] + sRedF[3]);
    P.part_w2[pbase] = (sRedF[4] + sRedF[5]) + (sRedF[6] + sRedF[7]);
    P.part_nonfinite[pbase] = (int)((sRedF[8] + sRedF[9]) + (sRedF[10] + sRedF[11]));
  }
  for (int o = tid; o < 2 * T; o += kThreadBlock) {
    const float a = (sA[o] + sA[2 * T + o]) + (sA[4 * T + o] + sA[6 * T + o]);   // fixed order
    P.part_A[((size_t)scene * 2 * T + o) * P_n + blockIdx.x] = a;
  }
}

template <bool PRECISE>
__global__ void __launch_bounds__(kThreadBlock)
rollout_thread_per_sample(const __grid_constant__ DeviceParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // layout (16-byte aligned first): obs[max_obs] float4 (ox, oy, 1/rho^2, -) | vel[max_obs] float2
  // (dt vx, dt vy) | U_nom[T] float2 | red (4 double, 4 int, 12 float) | A_w[4][2T] float
  const int T = P.T;
  float4* sObs = reinterpret_cast<float4*>(smem_raw);
  float2* sVel = reinterpret_cast<float2*>(sObs + P.max_obstacles);
  float2* sU = sVel + P.max_obstacles;
  double* sRedM = reinterpret_cast<double*>(sU + T);
  int* sRedI = reinterpret_cast<int*>(sRedM + 4);
  float* sRedF = reinterpret_cast<float*>(sRedI + 4);                  // [3][4]
  float* sA = sRedF + 12;                                              // [4][2T]

  const int scene = blockIdx.y;
  const int tid = threadIdx.x;
  const int k = blockIdx.x * kThreadBlock + tid;
  const bool valid = k < P.K;
  const uint32_t n = *P.counter;
  // scene s uses seed + s (64-bit add on the key pair)
  const uint32_t key0 = P.key0 + (uint32_t)scene;
  const uint32_t key1 = P.key1 + (key0 < P.key0 ? 1u : 0u);

  const float4 x0 = reinterpret_cast<const float4*>(P.state)[scene];
  float4 g = reinterpret_cast<const float4*>(P.goal)[scene];
  g.x -= x0.x; g.y -= x0.y;                     // vehicle-centred frame
  const int n_obs = P.n_obs[scene];
  for (int i = tid; i < T; i += kThreadBlock)
    sU[i] = reinterpret_cast<const float2*>(P.U)[scene * T + i];
  for (int i = tid; i < n_obs; i += kThreadBlock) {
    const float* ob = P.obstacles + ((size_t)scene * P.max_obstacles + i) * 5;
    const float rho = ob[2] + P.disc_radius;
    sObs[i] = make_float4(ob[0] - x0.x, ob[1] - x0.y, 1.0f / (rho * rho), 0.0f);
    sVel[i] = make_float2(P.dt * ob[3], P.dt * ob[4]);
  }
  __syncthreads();

  // ---- rollout -------------------------------------------------------------------------
  double S = CUDART_INF;
  State X{0.0f, 0.0f, x0.z, x0.w};
  float alpha = 0.0f;
  if (valid) {
    alpha = sample_alpha(P, n, (uint32_t)(k + P.k_offset), key0, key1);
    const float one_minus_alpha = 1.0f - alpha;
    float s1, c1, s2, c2;
    sincos_t<PRECISE>(X.psi1, &s1, &c1);
    sincos_t<PRECISE>(X.psi2, &s2, &c2);
    float pcx[kMaxDiscs], pcy[kMaxDiscs];
    disc_centres(P, X, s1, c1, s2, c2, pcx, pcy);
    double track = 0.0, bar = 0.0;
    for (int t = 0; t < T; ++t) {
      const float2 u = sample_control<PRECISE>(P, sU[t], (uint32_t)t, n, (uint32_t)(k + P.k_offset), key0, key1);
      const float tan_d = tan_t<PRECISE>(u.y);
      const State Xn = kinematic_step(P, X, s1, c1, s2, c2, u.x, tan_d);
      sincos_t<PRECISE>(Xn.psi1, &s1, &c1);
      sincos_t<PRECISE>(Xn.psi2, &s2, &c2);
      float ncx[kMaxDiscs], ncy[kMaxDiscs];
      disc_centres(P, Xn, s1, c1, s2, c2, ncx, ncy);
      float pen = 0.0f;
      const float tf = (float)t;
      for (int i = 0; i < n_obs; ++i) {
        const float4 o = sObs[i];
        const float2 w = sVel[i];
        const float opx = fmaf(tf, w.x, o.x), opy = fmaf(tf, w.y, o.y);                 // o(t)
        const float onx = fmaf(tf + 1.0f, w.x, o.x), ony = fmaf(tf + 1.0f, w.y, o.y);   // o(t+1)
#pragma unroll
        for (int j = 0; j < kMaxDiscs; ++j) {
          if (j < P.n_discs) {
            const float dxp = pcx[j] - opx, dyp = pcy[j] - opy;
            const float dxn = ncx[j] - onx, dyn = ncy[j] - ony;
            const float hp = fmaf(fmaf(dxp, dxp, dyp * dyp), o.z, -1.0f);
            const float hn = fmaf(fmaf(dxn, dxn, dyn * dyn), o.z, -1.0f);
            pen += fmaxf(fmaf(one_minus_alpha, hp, -hn), 0.0f);   // barrier-rate hinge (a5)
          }
        }
      }
      const float stage = goal_cost(P, Xn, g) + fmaf(P.w_v * u.x, u.x, P.w_delta * u.y * u.y) +
                          hitch_cost(P, Xn, u.x);
      track += (double)stage;
      bar += (double)pen;
      X = Xn;
#pragma unroll
      for (int j = 0; j < kMaxDiscs; ++j) { pcx[j] = ncx[j]; pcy[j] = ncy[j]; }
    }
    S = track + (double)P.w_bar * bar + (double)(P.w_term * goal_cost(P, X, g));
    if (P.flags & BRMPPI_FLAG_WRITE_SAMPLES) {
      P.S[(size_t)scene * P.K + k] = (float)S;
      reinterpret_cast<float4*>(P.XT)[(size_t)scene * P.K + k] =
          make_float4(X.x + x0.x, X.y + x0.y, X.psi1, X.psi2);
    }
  }

  thread_kernel_epilogue<PRECISE>(P, sU, sRedM, sRedI, sRedF, sA, S, valid, k, scene, n, key0, key1);
}

inline size_t rollout_thread_smem_bytes(const DeviceParams& P) {
  return sizeof(float4) * P.max_obstacles + sizeof(float2) * P.max_obstacles + sizeof(float2) * P.T +
         sizeof(double) * 4 + sizeof(int) * 4 + sizeof(float) * 12 + sizeof(float) * 4 * 2 * P.T;
}

}  // namespace brmppi
