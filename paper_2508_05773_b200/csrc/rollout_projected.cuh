// rollout_projected.cuh -- BR-MPPI proper (Sec. V-A): at every
// prediction step the sampled inputs are PROJECTED onto the barrier-rate equality (9) by the closed form
// (12), the projected input drives the model, the projected auxiliary input drives alpha_i.  Selected by
// BRMPPI_FLAG_PROJECTED; readings in DESIGN.md (reading 30).
//
// One thread per sample, NO = obstacle capacity as a template parameter so that everything -- the rows
// of (9), the N_o x N_o matrix A M^-1 A^T, its Cholesky factor -- lives in registers.  Nothing of a step
// touches HBM: A and b are built from the state, not streamed.
//
// What (9) looks like for the reduced model: with the inputs w = (v, omega), omega = v tan(delta), the model
// is x' = x + dt G(x) w, so row i is   L_g h_i . w + h_i u^alpha_i = -alpha_i h_i - L_f h_i,
//   A = [ L_g h (N_o x 2) | diag(h) ],   M = diag(q_v + rho, q_omega + rho, q_alpha + rho ...),
// and S = A M^-1 A^T = G' M_u^-1 G'^T + diag(h_i^2 / m_alpha) needs three multiply-adds per entry.
//
// The serial chain per step is long (about 1100 instructions, eight obstacle rows of independent work
// in it), so a warp brings its own instruction-level parallelism; 128-thread CTAs put one warp on each
// scheduler of an SM.
#pragma once

#include "rollout_thread.cuh"

namespace brmppi {

// The four standard normals of Philox block (t, n, k, tag): Box-Muller on words (0,1) and (2,3).
template <bool PRECISE>
__device__ __forceinline__ void normals4(uint32_t t, uint32_t n, uint32_t k, uint32_t tag, uint32_t key0,
                                         uint32_t key1, float (&z)[4]) {
  const uint4 w = philox4x32_10(t, n, k, tag, key0, key1);
  const float2 a = box_muller<PRECISE>(w.x, w.y), b = box_muller<PRECISE>(w.z, w.w);
  z[0] = a.x; z[1] = a.y; z[2] = b.x; z[3] = b.y;
}

// Rows of (9) for all obstacles at state X, step t: h_i on the closest disc (lowest index on ties),
// L_g h_i (2), L_f h_i.  Obstacle i: sObs = (ox, oy, 1/rho^2, 2 dt/rho^2) in the vehicle frame, sVel = (dt vel, vel);
// the table is padded to NO entries with null obstacles (1/rho^2 = 0), so the loop has no branch: a null row comes
// out as h = 1, L_g h = 0, L_f h = 0.  ND = the number of vehicle discs when it is 3 (the vehicle of every
// recipe), else BRMPPI_MAX_DISCS with the discs beyond P.n_discs masked.
template <bool PRECISE, int NO, int ND>
__device__ __forceinline__ void barrier_rows(const DeviceParams& P, const State& X, int n_obs, float tf,
                                             const float4* __restrict__ sObs, const float4* __restrict__ sVel,
                                             float (&h)[NO], float (&g0)[NO], float (&g1)[NO], float (&lf)[NO],
                                             float4* trig) {
  float s1, c1, s2, c2;
  sincos_t<PRECISE>(X.psi1, &s1, &c1);
  sincos_t<PRECISE>(X.psi2, &s2, &c2);
  *trig = make_float4(s1, c1, s2, c2);       // the model step out of this state needs the same four
  float cx[ND], cy[ND];
  disc_centres_n<ND>(P, X.x, X.y, s1, c1, s2, c2, cx, cy);
  const float sb = s1 * c2 - c1 * s2, cb = fmaf(c1, c2, s1 * s2);   // sin / cos (psi1 - psi2)
  const float sbL = sb * P.inv_L2, cbL = P.Lh_over_L1 * P.inv_L2 * cb;
#pragma unroll
  for (int i = 0; i < NO; ++i) {
    const float4 o = sObs[i];
    const float4 w = sVel[i];
    const float ox = fmaf(tf, w.x, o.x), oy = fmaf(tf, w.y, o.y);                 // o(t)
    // closest disc: h_j, the offset c_j - o, and the disc's lever arms on the two headings
    // (d c_j / d psi1 = (a1_j - Lh)(-sin psi1, cos psi1), d c_j / d psi2 = a2_j (-sin psi2, cos psi2))
    float hb = CUDART_INF_F, ex = 0.0f, ey = 0.0f, l1 = 0.0f, l2 = 0.0f;
#pragma unroll
    for (int j = 0; j < ND; ++j) {
      const float dx = cx[j] - ox, dy = cy[j] - oy;
      const float hj = (ND < kMaxDiscs || j < P.n_discs) ? fmaf(fmaf(dx, dx, dy * dy), o.z, -1.0f) : CUDART_INF_F;
      const bool take = hj < hb;
      hb = take ? hj : hb; ex = take ? dx : ex; ey = take ? dy : ey;
      l1 = take ? P.disc_a1[j] - P.Lh : l1; l2 = take ? P.disc_a2[j] : l2;
    }
    const float gx = ex * o.w, gy = ey * o.w;                                     // dt grad_c h
    const float dpsi1 = l1 * fmaf(gy, c1, -gx * s1), dpsi2 = l2 * fmaf(gy, c2, -gx * s2);
    h[i] = i < n_obs ? hb : 1.0f;
    g0[i] = fmaf(gx, c1, fmaf(gy, s1, dpsi2 * sbL));
    g1[i] = fmaf(dpsi1, P.inv_L1, -dpsi2 * cbL);
    lf[i] = -fmaf(gx, w.z, gy * w.w);                                             // dt grad_c h . vel
  }
}

template <bool PRECISE, int NO, int ND>
__global__ void __launch_bounds__(kThreadBlock)
rollout_projected(const __grid_constant__ DeviceParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // layout of rollout_thread_per_sample with NO obstacle slots
  const int T = P.T;
  float4* sObs = reinterpret_cast<float4*>(smem_raw);
  float4* sVel = sObs + NO;
  float2* sU = reinterpret_cast<float2*>(sVel + NO);
  double* sRedM = reinterpret_cast<double*>(sU + T);
  int* sRedI = reinterpret_cast<int*>(sRedM + 4);
  float* sRedF = reinterpret_cast<float*>(sRedI + 4);
  float* sA = sRedF + 12;

  const int scene = blockIdx.y;
  const int tid = threadIdx.x;
  const int k = blockIdx.x * kThreadBlock + tid;
  const bool valid = k < P.K;
  const uint32_t n = *P.counter;
  const uint32_t key0 = P.key0 + (uint32_t)scene;
  const uint32_t key1 = P.key1 + (key0 < P.key0 ? 1u : 0u);

  const float4 x0 = reinterpret_cast<const float4*>(P.state)[scene];
  float4 g = reinterpret_cast<const float4*>(P.goal)[scene];
  g.x -= x0.x; g.y -= x0.y;                     // vehicle-centred frame
  const int n_obs = min(P.n_obs[scene], NO);
  for (int i = tid; i < T; i += kThreadBlock)
    sU[i] = reinterpret_cast<const float2*>(P.U)[scene * T + i];
  for (int i = tid; i < NO; i += kThreadBlock) {
    if (i < n_obs) {
      const float* ob = P.obstacles + ((size_t)scene * P.max_obstacles + i) * 5;
      const float rho = ob[2] + P.disc_radius;
      const float ir2 = 1.0f / (rho * rho);
      sObs[i] = make_float4(ob[0] - x0.x, ob[1] - x0.y, ir2, 2.0f * P.dt * ir2);
      sVel[i] = make_float4(P.dt * ob[3], P.dt * ob[4], ob[3], ob[4]);
    } else {                                                 // null obstacle: no gradient, no motion
      sObs[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
      sVel[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    }
  }
  __syncthreads();

  double S = CUDART_INF;
  if (valid) {
    // M^-1 (diagonal), the soft-bound part of p, bounds: PAPER.md:185-192
    const float mv = 1.0f / (P.proj_qv + P.proj_rho), mw = 1.0f / (P.proj_qomega + P.proj_rho),
                ma = 1.0f / (P.proj_qalpha + P.proj_rho);
    const float pv0 = 0.5f * P.proj_rho * (P.v_max + P.v_min);        // rho/2 (z_hi + z_lo): 0 for omega, u^alpha
    State X{0.0f, 0.0f, x0.z, x0.w};
    float alpha[NO];
    {
      const float a0 = sample_alpha(P, n, (uint32_t)(k + P.k_offset), key0, key1);
#pragma unroll
      for (int i = 0; i < NO; ++i) alpha[i] = a0;
    }
    float h[NO], g0[NO], g1[NO], lf[NO];
    float4 trig;
    barrier_rows<PRECISE, NO, ND>(P, X, n_obs, 0.0f, sObs, sVel, h, g0, g1, lf, &trig);
    double cost = 0.0;
    // The draws of step t + 1 do not depend on the state: they are generated during step t, so that the long
    // Philox / Box-Muller chains fill the issue slots the Cholesky chain leaves empty.
    float2 u_next = sample_control<PRECISE>(P, sU[0], 0u, n, (uint32_t)(k + P.k_offset), key0, key1);
    float ua_next[NO];
#pragma unroll
    for (int q = 0; 4 * q < NO; ++q) {
      float z4[4];
      normals4<PRECISE>(0u, n, (uint32_t)(k + P.k_offset), 2u + (uint32_t)q, key0, key1, z4);
#pragma unroll
      for (int e = 0; e < 4; ++e)
        if (4 * q + e < NO) ua_next[4 * q + e] = P.sigma_ualpha * z4[e];
    }
#pragma unroll 1
    for (int t = 0; t < T; ++t) {
      // z_des = [w_des; u~^alpha], w_des = (v~, v~ tan delta~)
      const float2 u = u_next;
      float ua[NO];
#pragma unroll
      for (int i = 0; i < NO; ++i) ua[i] = ua_next[i];
      {
        const uint32_t tn = (uint32_t)min(t + 1, T - 1);
        u_next = sample_control<PRECISE>(P, sU[tn], tn, n, (uint32_t)(k + P.k_offset), key0, key1);
#pragma unroll
        for (int q = 0; 4 * q < NO; ++q) {
          float z4[4];
          normals4<PRECISE>(tn, n, (uint32_t)(k + P.k_offset), 2u + (uint32_t)q, key0, key1, z4);
#pragma unroll
          for (int e = 0; e < 4; ++e)
            if (4 * q + e < NO) ua_next[4 * q + e] = P.sigma_ualpha * z4[e];
        }
      }
      // y = M^-1 p, p = W z_des + rho/2 (z_hi + z_lo)
      const float yv = fmaf(P.proj_qv, u.x, pv0) * mv;
      const float yw = (P.proj_qomega * (u.x * tan_t<PRECISE>(u.y))) * mw;
      float ya[NO], r[NO];
#pragma unroll
      for (int i = 0; i < NO; ++i) {
        ya[i] = (P.proj_qalpha * ua[i]) * ma;
        // (9): L_g h w + h u^alpha = b,  b = -alpha h - L_f h;  r = A y - b.  A null row (i >= n_obs) is
        // u^alpha_i = y_i: r = 0, it changes nothing.
        const float b = i < n_obs ? -fmaf(alpha[i], h[i], lf[i]) : ya[i];
        r[i] = fmaf(g0[i], yv, fmaf(g1[i], yw, fmaf(h[i], ya[i], -b)));
      }
      // S = A M^-1 A^T (lower triangle), Cholesky in place with 1 / L_kk on the diagonal
      float Sm[NO][NO];
#pragma unroll
      for (int i = 0; i < NO; ++i) {
        const float a0 = g0[i] * mv, a1 = g1[i] * mw;
#pragma unroll
        for (int c = 0; c <= i; ++c) Sm[i][c] = fmaf(a0, g0[c], a1 * g1[c]);
        Sm[i][i] = fmaf(h[i] * ma, h[i], Sm[i][i]);
      }
#pragma unroll
      for (int c = 0; c < NO; ++c) {
        const float d0 = Sm[c][c];
        float dkk = d0;
#pragma unroll
        for (int m = 0; m < c; ++m) dkk = fmaf(-Sm[c][m], Sm[c][m], dkk);
        // a row that adds nothing new is dropped: 1 / L_cc = 0 makes its column of L zero and its multiplier
        // zero in both triangular solves (its own entries L_cm are finite and only ever meet that zero)
        const float inv = (dkk > 1e-6f * d0) ? fast_rsqrt(dkk) : 0.0f;
        Sm[c][c] = inv;
#pragma unroll
        for (int i = c + 1; i < NO; ++i) {
          float v = Sm[i][c];
#pragma unroll
          for (int m = 0; m < c; ++m) v = fmaf(-Sm[i][m], Sm[c][m], v);
          Sm[i][c] = v * inv;
        }
      }
#pragma unroll
      for (int i = 0; i < NO; ++i) {              // L w = r
        float v = r[i];
#pragma unroll
        for (int m = 0; m < i; ++m) v = fmaf(-Sm[i][m], r[m], v);
        r[i] = v * Sm[i][i];
      }
#pragma unroll
      for (int i = NO - 1; i >= 0; --i) {         // L^T nu = w
        float v = r[i];
#pragma unroll
        for (int m = i + 1; m < NO; ++m) v = fmaf(-Sm[m][i], r[m], v);
        r[i] = v * Sm[i][i];
      }
      // z* = y - M^-1 A^T nu
      float gv = 0.0f, gw = 0.0f;
#pragma unroll
      for (int i = 0; i < NO; ++i) { gv = fmaf(g0[i], r[i], gv); gw = fmaf(g1[i], r[i], gw); }
      const float vp = fmaf(-mv, gv, yv), wp = fmaf(-mw, gw, yw);
#pragma unroll
      for (int i = 0; i < NO; ++i)
        if (i < n_obs) alpha[i] += fmaf(-ma * h[i], r[i], ya[i]);   // alpha_{tau+1} = alpha_tau + u^alpha_proj
      // x_{tau+1} = x_tau + dt G(x_tau) w_proj
      {
        const float s1 = trig.x, c1 = trig.y, s2 = trig.z, c2 = trig.w;      // of X, from barrier_rows
        const float sb = s1 * c2 - c1 * s2, cb = fmaf(c1, c2, s1 * s2);
        const float a = P.dt * vp;
        State N;
        N.x = fmaf(a, c1, X.x);
        N.y = fmaf(a, s1, X.y);
        N.psi1 = fmaf(P.dt * wp, P.inv_L1, X.psi1);
        N.psi2 = fmaf(P.dt * P.inv_L2, fmaf(vp, sb, -(P.Lh_over_L1 * wp) * cb), X.psi2);
        X = N;
      }
      // rows of (9) at the new state: the alpha cost now, A and b of the next step
      barrier_rows<PRECISE, NO, ND>(P, X, n_obs, (float)(t + 1), sObs, sVel, h, g0, g1, lf, &trig);
      float ca = 0.0f;
#pragma unroll
      for (int i = 0; i < NO; ++i)
        if (i < n_obs && h[i] < P.h_buffer && alpha[i] > 0.0f) ca = fmaf(alpha[i], alpha[i], ca);
      const float stage = goal_cost(P, X, g) + fmaf(P.w_v * vp, vp, P.w_delta * wp * wp) + hitch_cost(P, X, vp) +
                          P.w_alpha * ca;
      cost += (double)stage;
    }
    S = cost + (double)(P.w_term * goal_cost(P, X, g));
    if (P.flags & BRMPPI_FLAG_WRITE_SAMPLES) {
      P.S[(size_t)scene * P.K + k] = (float)S;
      reinterpret_cast<float4*>(P.XT)[(size_t)scene * P.K + k] =
          make_float4(X.x + x0.x, X.y + x0.y, X.psi1, X.psi2);
    }
  }
  // eq. (5) averages the SAMPLED u~ with the projected rollouts' weights
  thread_kernel_epilogue<PRECISE>(P, sU, sRedM, sRedI, sRedF, sA, S, valid, k, scene, n, key0, key1);
}

inline size_t rollout_projected_smem_bytes(const DeviceParams& P) {
  return sizeof(float4) * BRMPPI_PROJECT_MAX_NO + sizeof(float4) * BRMPPI_PROJECT_MAX_NO + sizeof(float2) * P.T +
         sizeof(double) * 4 + sizeof(int) * 4 + sizeof(float) * 12 + sizeof(float) * 4 * 2 * P.T;
}

using ProjectedKernel = void (*)(const DeviceParams);

template <int ND>
inline ProjectedKernel projected_kernel_pick(bool precise, int max_obstacles) {
  const int cap = max_obstacles <= 1 ? 1 : max_obstacles <= 2 ? 2 : max_obstacles <= 4 ? 4 : 8;
  switch (cap * 2 + (precise ? 1 : 0)) {
    case 2: return rollout_projected<false, 1, ND>;
    case 3: return rollout_projected<true, 1, ND>;
    case 4: return rollout_projected<false, 2, ND>;
    case 5: return rollout_projected<true, 2, ND>;
    case 8: return rollout_projected<false, 4, ND>;
    case 9: return rollout_projected<true, 4, ND>;
    case 16: return rollout_projected<false, 8, ND>;
    default: return rollout_projected<true, 8, ND>;
  }
}

// three vehicle discs get their own instantiation; any other count runs the masked four-disc one
inline ProjectedKernel projected_kernel_for(bool precise, int max_obstacles, int n_discs) {
  return n_discs == 3 ? projected_kernel_pick<3>(precise, max_obstacles)
                      : projected_kernel_pick<kMaxDiscs>(precise, max_obstacles);
}

}  // namespace brmppi
