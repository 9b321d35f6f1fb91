// rollout_tile_kernel.cuh -- the phase-split tile kernel itself (design notes, plan and the
// phase-C inner loop are in rollout_tile.cuh).
//
// Register discipline: everything that lives for the whole kernel but is touched once per phase
// (start state, goal, obstacle counts) sits in the TileMisc block of shared memory, and every
// shared-memory section pointer is smem_raw + a constant-bank offset, so the long phase-C loop
// does not have to share the register file with values it never uses.
#pragma once

#include "rollout_tile.cuh"

namespace brmppi {

// resident CTAs per SM the register allocation is sized for (256-thread CTAs; 128-thread CTAs
// fit twice as many)
#ifndef BRMPPI_TILE_MIN_BLOCKS
#define BRMPPI_TILE_MIN_BLOCKS 2
#endif

#define BRMPPI_SMEM(type, off) reinterpret_cast<type*>(smem_raw + (off))

template <bool PRECISE, int ND>
__global__ void __launch_bounds__(kTileMaxThreads, BRMPPI_TILE_MIN_BLOCKS)
rollout_tile(const __grid_constant__ DeviceParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x;
  const int s = tid & (kTileSamples - 1), c = tid / kTileSamples;

  // ---- CTA prologue: scene data in the vehicle-centred frame ---------------
  {
    const int scene = blockIdx.y, T = P.T, nthreads = blockDim.x;
    float4* sObs = BRMPPI_SMEM(float4, P.off_obs);
    float2* sVel = BRMPPI_SMEM(float2, P.off_vel);
    float2* sUnom = BRMPPI_SMEM(float2, P.off_unom);
    float* sA = BRMPPI_SMEM(float, P.off_A);
    TileMisc* sM = BRMPPI_SMEM(TileMisc, P.off_misc);
    for (int i = tid; i < T; i += nthreads) sUnom[i] = reinterpret_cast<const float2*>(P.U)[(size_t)scene * T + i];
    for (int i = tid; i < 2 * T; i += nthreads) sA[i] = 0.0f;
    for (int i = tid; i < P.obs_padded; i += nthreads) {   // null obstacles: h == 0, hinge == 0
      sObs[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
      sVel[i] = make_float2(0.0f, 0.0f);
    }
    __syncthreads();
    {
      // every thread i < n_obs places obstacle i: moving obstacles first, static ones after
      // (groups without a moving one skip the o(t) update); ranks by counting, no serial pass
      const float4 x0 = reinterpret_cast<const float4*>(P.state)[scene];
      const int n_obs = P.n_obs[scene];
      const float* ob = P.obstacles + (size_t)scene * P.max_obstacles * 5;
      if (tid < n_obs) {
        int nm = 0, before_m = 0, before_s = 0;
        for (int j = 0; j < n_obs; ++j) {
          const bool mj = (ob[5 * j + 3] != 0.0f || ob[5 * j + 4] != 0.0f);
          nm += mj ? 1 : 0;
          if (j < tid) { before_m += mj ? 1 : 0; before_s += mj ? 0 : 1; }
        }
        const bool moving = (ob[5 * tid + 3] != 0.0f || ob[5 * tid + 4] != 0.0f);
        const int dst = moving ? before_m : nm + before_s;
        const float rho = ob[5 * tid + 2] + P.disc_radius;
        sObs[dst] = make_float4(ob[5 * tid + 0] - x0.x, ob[5 * tid + 1] - x0.y, 1.0f / (rho * rho), -1.0f);
        sVel[dst] = make_float2(P.dt * ob[5 * tid + 3], P.dt * ob[5 * tid + 4]);
        if (tid == 0) sM->n_moving = nm;
      }
      if (tid == 0) {
        float4 g = reinterpret_cast<const float4*>(P.goal)[scene];
        g.x -= x0.x; g.y -= x0.y;
        sM->x0 = x0;
        sM->g = g;
        sM->m = CUDART_INF; sM->argmin = 0x7fffffff; sM->eta = 0.0f; sM->w2 = 0.0f; sM->nonfinite = 0;
        if (n_obs == 0) sM->n_moving = 0;
        sM->n_groups = n_obs > 0 ? (n_obs + kObsGroup - 1) / kObsGroup : 1;
      }
    }
    __syncthreads();
  }

  for (int tile = blockIdx.x; tile < P.tiles_per_scene; tile += gridDim.x) {
    const int k = tile * kTileSamples + s;
    float effort = 0.0f;

    // ---- phase A: noise, perturb + clamp, effort (a1, a2) ------------------------------
    {
      const int TS = P.t_stride, T = P.T;
      const int t0 = c * P.chunk_len, t1 = min(t0 + P.chunk_len, T);
      const uint32_t n = *P.counter;
      const uint32_t key0 = P.key0 + blockIdx.y;
      const uint32_t key1 = P.key1 + (key0 < P.key0 ? 1u : 0u);
      const float2* sUnom = BRMPPI_SMEM(float2, P.off_unom);
      float* pV = BRMPPI_SMEM(float, P.off_planes) + s * TS;
      float* pD = pV + kTileSamples * TS;
      float* pP1 = pD + kTileSamples * TS;
      for (int t = t0; t < t1; ++t) {
        const float2 u = sample_control<PRECISE>(P, sUnom[t], (uint32_t)t, n, (uint32_t)k, key0, key1);
        const float tan_d = tan_t<PRECISE>(u.y);
        pV[t] = u.x;
        pD[t] = u.y;
        pP1[t + 1] = (P.dt * u.x) * P.inv_L1 * tan_d;          // dpsi1 of step t, parked at t+1
        effort = fmaf(P.w_v * u.x, u.x, fmaf(P.w_delta * u.y, u.y, effort));
      }
      if (c == 0) BRMPPI_SMEM(TileMisc, P.off_misc)->alpha[s] = sample_alpha(P, n, (uint32_t)k, key0, key1);
    }
    __syncthreads();

    // ---- phase B: serial Euler chain of eq. (6), one sample per thread (a3) -------------
    if (tid < kTileSamples) {
      const int TS = P.t_stride, T = P.T, L = P.chunk_len;
      const float* pV = BRMPPI_SMEM(float, P.off_planes) + s * TS;
      float* pP1 = BRMPPI_SMEM(float, P.off_planes) + (2 * kTileSamples + s) * TS;
      float* pP2 = pP1 + kTileSamples * TS;
      float2* sXY = BRMPPI_SMEM(float2, P.off_xy);        // [C+1][16] chunk-boundary (x, y)
      const float4 x0 = BRMPPI_SMEM(TileMisc, P.off_misc)->x0;
      float x = 0.0f, y = 0.0f, psi1 = x0.z, psi2 = x0.w;
      pP1[0] = psi1;
      pP2[0] = psi2;
      for (int cc = 0, t = 0; t < T; ++cc) {
        sXY[cc * kTileSamples + s] = make_float2(x, y);      // chunk-boundary position
        const int te = min(t + L, T);
        for (; t < te; ++t) {
          const float v = pV[t], b = pP1[t + 1];
          float s1, c1, s2, c2;
          sincos_t<PRECISE>(psi1, &s1, &c1);
          sincos_t<PRECISE>(psi2, &s2, &c2);
          const float a = P.dt * v;
          const float sb = s1 * c2 - c1 * s2;            // sin(psi1 - psi2)
          const float cb = fmaf(c1, c2, s1 * s2);        // cos(psi1 - psi2)
          x = fmaf(a, c1, x);
          y = fmaf(a, s1, y);
          psi1 += b;
          psi2 = fmaf(a * P.inv_L2, sb, fmaf(-(b * P.Lh_over_L2), cb, psi2));
          pP1[t + 1] = psi1;
          pP2[t + 1] = psi2;
        }
      }
      sXY[P.chunks * kTileSamples + s] = make_float2(x, y);   // x_T
    }
    __syncthreads();

    // ---- phase C: barrier, barrier-rate hinge, goal / heading / hitch cost (a4-a6) ------
    {
      const int TS = P.t_stride, T = P.T;
      const int t0 = c * P.chunk_len, t1 = min(t0 + P.chunk_len, T);
      const TileMisc* sM = BRMPPI_SMEM(TileMisc, P.off_misc);
      double track = 0.0, bar = 0.0;
      if (t0 < T) {
        const float* pV = BRMPPI_SMEM(float, P.off_planes) + s * TS;
        const float* pP1 = pV + 2 * kTileSamples * TS;
        const float* pP2 = pP1 + kTileSamples * TS;
        const float4* sObs = BRMPPI_SMEM(float4, P.off_obs);
        const float2* sVel = BRMPPI_SMEM(float2, P.off_vel);
        const float one_minus_alpha = 1.0f - sM->alpha[s];
        const float4 g = sM->g;
        const int n_moving = sM->n_moving, n_groups = sM->n_groups;
        const float2 xy = BRMPPI_SMEM(float2, P.off_xy)[c * kTileSamples + s];
        for (int grp = 0; grp < n_groups; ++grp) {
          const int ib = grp * kObsGroup;
          GroupCost gc;
          if (ib < n_moving)
            gc = cost_group<PRECISE, ND, true>(P, pV, pP1, pP2, sObs + ib, sVel + ib, xy.x, xy.y, t0, t1, one_minus_alpha, g, grp == 0);
          else
            gc = cost_group<PRECISE, ND, false>(P, pV, pP1, pP2, sObs + ib, sVel + ib, xy.x, xy.y, t0, t1, one_minus_alpha, g, grp == 0);
          track += gc.track; bar += gc.bar;
        }
        if (t1 == T) {   // terminal cost r_N(x_N), eq. (7); final state out
          const float2 xT = BRMPPI_SMEM(float2, P.off_xy)[P.chunks * kTileSamples + s];
          const State X{xT.x, xT.y, pP1[T], pP2[T]};
          track += (double)(P.w_term * goal_cost(P, X, g));
          if ((P.flags & BRMPPI_FLAG_WRITE_SAMPLES) && k < P.K) {
            const float4 x0 = sM->x0;
            reinterpret_cast<float4*>(P.XT)[(size_t)blockIdx.y * P.K + k] =
                make_float4(X.x + x0.x, X.y + x0.y, X.psi1, X.psi2);
          }
        }
      }
      BRMPPI_SMEM(double, P.off_cost)[c * kTileSamples + s] = track + (double)effort + (double)P.w_bar * bar;
    }
    __syncthreads();

    // ---- phase D: tile reduction, fold into the running online-softmax state (a7) -------
    if (tid < 32) {
      TileMisc* sM = BRMPPI_SMEM(TileMisc, P.off_misc);
      const double* sCost = BRMPPI_SMEM(double, P.off_cost);
      double S = CUDART_INF;
      const bool valid = (tid < kTileSamples) && (k < P.K);
      if (valid) {
        S = 0.0;
        for (int cc = 0; cc < P.chunks; ++cc) S += sCost[cc * kTileSamples + s];
        if (P.flags & BRMPPI_FLAG_WRITE_SAMPLES) P.S[(size_t)blockIdx.y * P.K + k] = (float)S;
      }
      const bool finite = valid && (S == S) && (S < CUDART_INF) && (S > -CUDART_INF);
      double m = finite ? S : CUDART_INF;
      int idx = finite ? k : 0x7fffffff;
      warp_argmin(m, idx);
      const double m_old = sM->m;
      const int idx_old = sM->argmin;
      const bool take_new = (m < m_old) || (m == m_old && idx < idx_old);
      const double m_new = take_new ? m : m_old;
      const float scale_old = (m_old < CUDART_INF) ? expf((float)(-(m_old - m_new) * (double)P.inv_lambda)) : 0.0f;
      const float w = finite ? expf((float)(-(S - m_new) * (double)P.inv_lambda)) : 0.0f;
      const float eta_t = warp_sum(w), w2_t = warp_sum(w * w);
      const float nf_t = warp_sum((valid && !finite) ? 1.0f : 0.0f);
      __syncwarp();
      if (tid < kTileSamples) sM->w[tid] = w;
      if (tid == 0) {
        sM->m = m_new;
        sM->argmin = take_new ? idx : idx_old;
        sM->eta = fmaf(sM->eta, scale_old, eta_t);
        sM->w2 = fmaf(sM->w2, scale_old * scale_old, w2_t);
        sM->nonfinite += (int)nf_t;
        sM->scale_old = scale_old;
      }
    }
    __syncthreads();

    // ---- phase E: running weighted control sums A[t] (a7) ------------------------------
    {
      const int TS = P.t_stride, T = P.T, nthreads = blockDim.x;
      const TileMisc* sM = BRMPPI_SMEM(TileMisc, P.off_misc);
      float* sA = BRMPPI_SMEM(float, P.off_A);
      const float* sV = BRMPPI_SMEM(float, P.off_planes);
      const float scale_old = sM->scale_old;
      for (int o = tid; o < 2 * T; o += nthreads) {
        const int ch = o >= T ? 1 : 0, t = o - ch * T;
        const float* plane = sV + ch * kTileSamples * TS;
        float acc = 0.0f;
#pragma unroll
        for (int ss = 0; ss < kTileSamples; ++ss) acc = fmaf(sM->w[ss], plane[ss * TS + t], acc);
        sA[o] = fmaf(sA[o], scale_old, acc);
      }
    }
    __syncthreads();
  }

  // ---- CTA partial -> HBM ---------------------------------------------------------------
  {
    const int Pn = P.n_partials, T = P.T, scene = blockIdx.y;
    const TileMisc* sM = BRMPPI_SMEM(TileMisc, P.off_misc);
    const float* sA = BRMPPI_SMEM(float, P.off_A);
    const size_t pbase = (size_t)scene * Pn + blockIdx.x;
    if (tid == 0) {
      P.part_m[pbase] = sM->m;
      P.part_argmin[pbase] = sM->argmin;
      P.part_eta[pbase] = sM->eta;
      P.part_w2[pbase] = sM->w2;
      P.part_nonfinite[pbase] = sM->nonfinite;
    }
    for (int o = tid; o < 2 * T; o += blockDim.x) {
      const int ch = o >= T ? 1 : 0, t = o - ch * T;
      P.part_A[((size_t)scene * 2 * T + (2 * t + ch)) * Pn + blockIdx.x] = sA[o];
    }
  }
}

#undef BRMPPI_SMEM

inline size_t rollout_tile_smem_bytes(const DeviceParams& P, const TilePlan& tp) {
  return tile_smem_layout(P.T, tp.obs_padded, tp.chunks, tp.t_stride).total;
}

using TileKernel = void (*)(const DeviceParams);

inline TileKernel tile_kernel_for(bool precise, int n_discs) {
  switch (n_discs * 2 + (precise ? 1 : 0)) {
    case 2: return rollout_tile<false, 1>;
    case 3: return rollout_tile<true, 1>;
    case 4: return rollout_tile<false, 2>;
    case 5: return rollout_tile<true, 2>;
    case 6: return rollout_tile<false, 3>;
    case 7: return rollout_tile<true, 3>;
    case 8: return rollout_tile<false, 4>;
    default: return rollout_tile<true, 4>;
  }
}

inline cudaError_t configure_rollout_tile(bool precise, int n_discs, size_t smem_bytes) {
  cudaError_t e = cudaFuncSetAttribute(tile_kernel_for(precise, n_discs),
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
  if (e != cudaSuccess) return e;
  // ask for the full shared-memory carve-out: residency here is limited by shared memory and
  // registers, the kernel streams almost nothing through L1
  return cudaFuncSetAttribute(tile_kernel_for(precise, n_discs),
                              cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}

inline cudaError_t launch_rollout_tile(const DeviceParams& d, const TilePlan& tp, bool precise,
                                       size_t smem_bytes, cudaStream_t stream) {
  dim3 grid((unsigned)tp.blocks_per_scene, (unsigned)d.n_scenes);
  tile_kernel_for(precise, d.n_discs)<<<grid, tp.threads, smem_bytes, stream>>>(d);
  return cudaGetLastError();
}

}  // namespace brmppi
