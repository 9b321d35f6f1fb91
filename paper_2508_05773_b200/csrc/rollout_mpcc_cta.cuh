// rollout_mpcc_cta.cuh -- the paper's own model and cost (BRMPPI_FLAG_MPCC, reading 31 and 9.2) as a
// persistent, phase-split CTA kernel: the default for that mode (BRMPPI_FLAG_KERNEL_THREAD_PER_SAMPLE selects
// rollout_mpcc.cuh's one-thread-per-sample kernel).
//
// A tile is 128 samples.  The only serial part of a rollout is the state recursion (noise, Euler step of eq. (6),
// path parameter): four CHAIN warps run it, one thread per sample, and leave every state of the horizon -- with all
// the trigonometry the step needed anyway -- in shared-memory planes, a chunk of kMpccL steps at a time into a
// two-deep ring.  Twelve COST warps take the (sample, step) items of a chunk as the chain finishes it (mbarrier per
// ring slot, full / empty): rates and their derivatives, disc centres, velocities and accelerations, the predictor
// (17) and the hinge for every (obstacle, disc), the path point and the stage cost (13).  A cost thread always serves
// the same sample (384 = 3 x 128), so its cost sum stays in a register for the whole tile; no MUFU is issued by a
// cost thread.  The tile then forms its online-softmax partial like the other kernels, the sampled controls
// regenerated from Philox for the weighted sums.
#pragma once

#include "rollout_mpcc.cuh"
#include "rollout_cta_kernel.cuh"      // mbarrier helpers

namespace brmppi {

constexpr int kMpccThreads = 512;
constexpr int kMpccTile = 128;                         // samples per tile = chain threads
constexpr int kMpccCost = kMpccThreads - kMpccTile;    // 384 cost threads, threads [0, 384)
constexpr int kMpccGroups = kMpccCost / kMpccTile;     // 3 cost threads per sample
constexpr int kMpccL = 6;                              // steps per chunk: kMpccGroups x 2 items per cost thread
constexpr int kMpccRows = kMpccL + 1;                  // a chunk keeps the row after its last step too

// planes of one row (one state of the horizon), each [kMpccTile] floats
enum MpccPlane { MP_X, MP_Y, MP_V, MP_A, MP_T1, MP_T2, MP_PSI, MP_S1, MP_C1, MP_SR, MP_CR,   // read as row t + 1 too
                 MP_S2, MP_C2, MP_TD, MP_J, MP_W, MP_COUNT };

struct MpccCtaSmem { size_t obs, vel, path, U, planes, part, w, red, A, bars, total; };

__host__ __device__ inline MpccCtaSmem mpcc_cta_smem_layout(int T, int max_obstacles, int max_path_segments) {
  MpccCtaSmem L{};
  size_t off = 0;
#define MPCC_TAKE(field, bytes) L.field = off; off = (off + (size_t)(bytes) + 15) / 16 * 16
  const size_t no = (size_t)(max_obstacles > 0 ? max_obstacles : 1);
  MPCC_TAKE(obs, sizeof(float4) * no);
  MPCC_TAKE(vel, sizeof(float4) * no);
  MPCC_TAKE(path, sizeof(float4) * 4 * (size_t)max_path_segments);
  MPCC_TAKE(U, sizeof(float2) * (size_t)(T + 2));
  MPCC_TAKE(planes, sizeof(float) * 2 * kMpccRows * MP_COUNT * kMpccTile);
  MPCC_TAKE(part, sizeof(double) * kMpccGroups * kMpccTile);
  MPCC_TAKE(w, sizeof(float) * kMpccTile);
  MPCC_TAKE(red, sizeof(double) * 4 + sizeof(int) * 4 + sizeof(float) * 12 + 16);
  MPCC_TAKE(A, sizeof(float) * 4 * 2 * (size_t)(T + 1));
  MPCC_TAKE(bars, sizeof(unsigned long long) * 4);
#undef MPCC_TAKE
  L.total = off;
  return L;
}

__device__ __forceinline__ float* mpcc_plane(float* planes, int slot, int row, int plane) {
  return planes + ((size_t)(slot * kMpccRows + row) * MP_COUNT + plane) * kMpccTile;
}

// One (sample, step) item of the cost phase: everything of step t that is not the state recursion.  Returns the
// stage cost (13) with the barrier term; *track = the four tracking terms at (x_{t+1}, psi_{t+1}).
template <int ND>
__device__ __forceinline__ double mpcc_cost_item(const DeviceParams& P, const float4* __restrict__ sObs,
                                                 const float4* __restrict__ sVel, const float4* __restrict__ sPath,
                                                 int n_obs, int M, float dpsi, float inv_dpsi, const float* row0,
                                                 const float* row1, int s, int t, float alpha, float* track) {
  const float x = row0[MP_X * kMpccTile + s], y = row0[MP_Y * kMpccTile + s], v = row0[MP_V * kMpccTile + s],
              a = row0[MP_A * kMpccTile + s], s1 = row0[MP_S1 * kMpccTile + s], c1 = row0[MP_C1 * kMpccTile + s],
              s2 = row0[MP_S2 * kMpccTile + s], c2 = row0[MP_C2 * kMpccTile + s], td = row0[MP_TD * kMpccTile + s];
  const float2 u = make_float2(row0[MP_J * kMpccTile + s], row0[MP_W * kMpccTile + s]);
  const MpccRates R = mpcc_rates(P, v, a, td, s1, c1, s2, c2, u.y);
  const float pen = mpcc_hinge<ND>(P, sObs, sVel, n_obs, ND, (float)t, alpha, x, y, v, a, s1, c1, s2, c2, R);
  // stage cost (13) on (x_{t+1}, u_t, psi_{t+1}): the next row
  const float xn = row1[MP_X * kMpccTile + s], yn = row1[MP_Y * kMpccTile + s], vn = row1[MP_V * kMpccTile + s],
              t1n = row1[MP_T1 * kMpccTile + s], t2n = row1[MP_T2 * kMpccTile + s], psin = row1[MP_PSI * kMpccTile + s],
              s1n = row1[MP_S1 * kMpccTile + s], c1n = row1[MP_C1 * kMpccTile + s], srn = row1[MP_SR * kMpccTile + s],
              crn = row1[MP_CR * kMpccTile + s];
  float nu;
  *track = mpcc_tracking_sc(P, xn, yn, t1n, t2n, vn, s1n, c1n, path_eval(sPath, M, dpsi, inv_dpsi, psin), srn, crn, &nu);
  const float stage = *track + mpcc_stage_rest(P, t1n, t2n, vn, nu, u);
  return (double)stage + (double)P.w_bar * (double)pen;
}

template <bool PRECISE, int ND>
__global__ void __launch_bounds__(kMpccThreads, 1)
rollout_mpcc_cta(const __grid_constant__ DeviceParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const MpccCtaSmem L = mpcc_cta_smem_layout(P.T, P.max_obstacles, P.max_path_segments);
  float4* sObs = reinterpret_cast<float4*>(smem_raw + L.obs);
  float4* sVel = reinterpret_cast<float4*>(smem_raw + L.vel);
  float4* sPath = reinterpret_cast<float4*>(smem_raw + L.path);
  float2* sU = reinterpret_cast<float2*>(smem_raw + L.U);
  float* sPlanes = reinterpret_cast<float*>(smem_raw + L.planes);
  double* sPart = reinterpret_cast<double*>(smem_raw + L.part);
  float* sW = reinterpret_cast<float*>(smem_raw + L.w);
  double* sRedM = reinterpret_cast<double*>(smem_raw + L.red);
  int* sRedI = reinterpret_cast<int*>(sRedM + 4);
  float* sRedF = reinterpret_cast<float*>(sRedI + 4);
  float* sA = reinterpret_cast<float*>(smem_raw + L.A);
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_raw + L.bars);   // full[2], empty[2]

  const int T = P.T, tid = threadIdx.x;
  const int s = tid & (kMpccTile - 1), grp = tid / kMpccTile;       // groups 0..2: cost threads, group 3: the chain
  const bool is_chain = grp == kMpccGroups;
  const int lane = tid & 31, warp = tid >> 5;
  const int n_chunks = (T + kMpccL - 1) / kMpccL;
  const uint32_t n = *P.counter;
  if (tid == 0) {
    mbar_init(smem_addr(&bars[0]), kMpccTile); mbar_init(smem_addr(&bars[1]), kMpccTile);
    mbar_init(smem_addr(&bars[2]), kMpccCost); mbar_init(smem_addr(&bars[3]), kMpccCost);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  uint32_t g = 0;                    // chunks handed over so far (ring position; the same on every thread)
  int loaded_scene = -1;

  for (int tile = blockIdx.x; tile < P.total_tiles; tile += gridDim.x) {
    const int scene = tile / P.tiles_per_scene, part = tile - scene * P.tiles_per_scene;
    const int k = part * kMpccTile + s;
    const bool valid = k < P.K;
    const int kk = valid ? k : P.K - 1;                             // a ragged tile's spare threads redo the last sample
    const uint32_t key0 = P.key0 + (uint32_t)scene;
    const uint32_t key1 = P.key1 + (key0 < P.key0 ? 1u : 0u);
    const float* s7 = P.state7 + 8 * scene;
    const float x0 = s7[0], y0 = s7[1];
    const int n_obs = P.n_obs[scene];
    const int M = P.path_M[scene];
    const float dpsi = P.path_dpsi[scene];
    const float inv_dpsi = 1.0f / dpsi;
    __syncthreads();                                                // the previous tile's epilogue is done with sU / sA
    if (scene != loaded_scene) {
      for (int i = tid; i < T + 2; i += kMpccThreads)
        sU[i] = i < T ? reinterpret_cast<const float2*>(P.U)[scene * T + i] : make_float2(0.0f, 0.0f);
      for (int i = tid; i < n_obs; i += kMpccThreads) {
        const float* ob = P.obstacles + ((size_t)scene * P.max_obstacles + i) * 5;
        const float rho = ob[2] + P.disc_radius;
        sObs[i] = make_float4(ob[0] - x0, ob[1] - y0, 1.0f / (rho * rho), 0.0f);   // vehicle-centred frame
        sVel[i] = make_float4(P.dt * ob[3], P.dt * ob[4], ob[3], ob[4]);
      }
      for (int i = tid; i < 4 * M; i += kMpccThreads) {
        float4 c = reinterpret_cast<const float4*>(P.path_coef)[(size_t)scene * 4 * P.max_path_segments + i];
        if ((i & 3) == 0) c.x -= x0;
        if ((i & 3) == 1) c.x -= y0;
        sPath[i] = c;
      }
      loaded_scene = scene;
    }
    __syncthreads();

    double acc = 0.0;
    if (is_chain) {
      // ---- the state recursion of eq. (6), one thread per sample; rows of kMpccL steps into the ring ----
      const float Lpath = (float)M * dpsi;
      State7 X{0.0f, 0.0f, s7[2], s7[3], s7[4], s7[5], s7[6], s7[7]};
      float s1, c1, sr, cr;
      sincos_t<PRECISE>(X.t1, &s1, &c1);
      sincos_t<PRECISE>(path_eval_component(sPath, M, dpsi, inv_dpsi, X.psi, 2), &sr, &cr);
      float nu = X.v * fmaf(c1, cr, s1 * sr);
      float2 u_odd = make_float2(0.0f, 0.0f);
      int t = 0;
      for (int c = 0; c < n_chunks; ++c) {
        const uint32_t gg = g + (uint32_t)c;
        const int slot = (int)(gg & 1u);
        if (gg >= 2u) mbar_wait(smem_addr(&bars[2 + slot]), ((gg >> 1) - 1u) & 1u);   // the cost threads are done with it
        int r = 0;
#pragma unroll 1
        for (; r < kMpccL && t < T; ++r, ++t) {
          float2 u;
          if ((t & 1) == 0)       // one Philox block serves a pair of steps (reading 6)
            sample_control_pair<PRECISE>(P, sU[t], sU[t + 1], (uint32_t)(t >> 1), n, (uint32_t)(kk + P.k_offset), key0,
                                         key1, &u, &u_odd);
          else
            u = u_odd;
          float s2, c2;
          sincos_t<PRECISE>(X.t2, &s2, &c2);
          const float td = tan_t<PRECISE>(X.de);
          float* row = mpcc_plane(sPlanes, slot, r, 0) + s;
          row[MP_X * kMpccTile] = X.x;   row[MP_Y * kMpccTile] = X.y;   row[MP_V * kMpccTile] = X.v;
          row[MP_A * kMpccTile] = X.a;   row[MP_S1 * kMpccTile] = s1;   row[MP_C1 * kMpccTile] = c1;
          row[MP_S2 * kMpccTile] = s2;   row[MP_C2 * kMpccTile] = c2;   row[MP_TD * kMpccTile] = td;
          row[MP_J * kMpccTile] = u.x;   row[MP_W * kMpccTile] = u.y;
          if (r > 0) {              // this row is also the "next state" of the item before it
            row[MP_T1 * kMpccTile] = X.t1; row[MP_T2 * kMpccTile] = X.t2; row[MP_PSI * kMpccTile] = X.psi;
            row[MP_SR * kMpccTile] = sr;   row[MP_CR * kMpccTile] = cr;
          }
          const MpccRates R = mpcc_rates(P, X.v, X.a, td, s1, c1, s2, c2, u.y);      // W1, W2 are what is used
          State7 N;
          N.x = fmaf(P.dt * X.v, c1, X.x);
          N.y = fmaf(P.dt * X.v, s1, X.y);
          N.v = fmaf(P.dt, X.a, X.v);
          N.a = fmaf(P.dt, u.x, X.a);
          N.t1 = fmaf(P.dt, R.W1, X.t1);
          N.t2 = fmaf(P.dt, R.W2, X.t2);
          N.de = fminf(fmaxf(fmaf(P.dt, u.y, X.de), P.dstate_lo), P.dstate_hi);
          N.psi = fminf(fmaxf(fmaf(P.dt, nu, X.psi), 0.0f), Lpath);
          X = N;
          sincos_t<PRECISE>(X.t1, &s1, &c1);
          sincos_t<PRECISE>(path_eval_component(sPath, M, dpsi, inv_dpsi, X.psi, 2), &sr, &cr);
          nu = X.v * fmaf(c1, cr, s1 * sr);
        }
        {                           // the row after the chunk's last step: read only as a "next state"
          float* row = mpcc_plane(sPlanes, slot, r, 0) + s;
          row[MP_X * kMpccTile] = X.x;   row[MP_Y * kMpccTile] = X.y;   row[MP_V * kMpccTile] = X.v;
          row[MP_T1 * kMpccTile] = X.t1; row[MP_T2 * kMpccTile] = X.t2; row[MP_PSI * kMpccTile] = X.psi;
          row[MP_S1 * kMpccTile] = s1;   row[MP_C1 * kMpccTile] = c1;
          row[MP_SR * kMpccTile] = sr;   row[MP_CR * kMpccTile] = cr;
        }
        mbar_arrive(smem_addr(&bars[slot]));
      }
      if (valid && (P.flags & BRMPPI_FLAG_WRITE_SAMPLES)) {
        float4* out = reinterpret_cast<float4*>(P.XT) + 2 * ((size_t)scene * P.K + k);
        out[0] = make_float4(X.x + x0, X.y + y0, X.v, X.a);
        out[1] = make_float4(X.t1, X.t2, X.de, X.psi);
      }
    } else {
      // ---- cost phase: the (sample, step) items of each chunk as the chain hands it over ----
      const float alpha = sample_alpha(P, n, (uint32_t)(kk + P.k_offset), key0, key1);
      for (int c = 0; c < n_chunks; ++c) {
        const uint32_t gg = g + (uint32_t)c;
        const int slot = (int)(gg & 1u);
        mbar_wait(smem_addr(&bars[slot]), (gg >> 1) & 1u);
#pragma unroll 1
        for (int r = grp; r < kMpccL; r += kMpccGroups) {
          const int t = c * kMpccL + r;
          if (t < T) {
            float track;
            acc += mpcc_cost_item<ND>(P, sObs, sVel, sPath, n_obs, M, dpsi, inv_dpsi, mpcc_plane(sPlanes, slot, r, 0),
                                      mpcc_plane(sPlanes, slot, r + 1, 0), s, t, alpha, &track);
            if (t == T - 1) acc += (double)(P.w_term * track);       // terminal cost: the same four terms at (x_N, psi_N)
          }
        }
        mbar_arrive(smem_addr(&bars[2 + slot]));
      }
      sPart[grp * kMpccTile + s] = acc;
    }
    g += (uint32_t)n_chunks;
    __syncthreads();

    // ---- the tile's online-softmax partial (a7): S_k, block minimum, weights, eta, weighted control sums ----
    double S = CUDART_INF, m = CUDART_INF;
    bool finite = false;
    if (tid < kMpccTile) {
      S = (sPart[s] + sPart[kMpccTile + s]) + sPart[2 * kMpccTile + s];            // fixed order
      finite = valid && (S == S) && (S < CUDART_INF) && (S > -CUDART_INF);
      if (valid && (P.flags & BRMPPI_FLAG_WRITE_SAMPLES)) P.S[(size_t)scene * P.K + k] = (float)S;
      m = finite ? S : CUDART_INF;
      int idx = finite ? k + P.k_offset : 0x7fffffff;
      warp_argmin(m, idx);
      if (lane == 0) { sRedM[warp] = m; sRedI[warp] = idx; }
    }
    __syncthreads();
    int idx = sRedI[0];
    m = sRedM[0];
#pragma unroll
    for (int w = 1; w < 4; ++w)
      if (sRedM[w] < m || (sRedM[w] == m && sRedI[w] < idx)) { m = sRedM[w]; idx = sRedI[w]; }
    if (tid < kMpccTile) {
      const float wk = finite ? expf((float)(-(S - m) * (double)P.inv_lambda)) : 0.0f;   // S - m in fp64, then fp32 exp
      sW[s] = wk;
      const float eta = warp_sum(wk), w2 = warp_sum(wk * wk), nf = warp_sum((valid && !finite) ? 1.0f : 0.0f);
      if (lane == 0) { sRedF[warp] = eta; sRedF[4 + warp] = w2; sRedF[8 + warp] = nf; }
    }
    __syncthreads();
    {   // weighted control sums, the sampled controls regenerated from the counter-based generator: thread ->
        // (sample s, every fourth step pair); the 128 samples of a pair are four warps
      const float wk = sW[s];
      const int sw = warp & 3;
      for (int mp = grp; 2 * mp < T; mp += 4) {
        float2 u0, u1;
        sample_control_pair<PRECISE>(P, sU[2 * mp], sU[2 * mp + 1], (uint32_t)mp, n, (uint32_t)(kk + P.k_offset), key0,
                                     key1, &u0, &u1);
        const float a0 = warp_sum(wk * u0.x), a1 = warp_sum(wk * u0.y), a2 = warp_sum(wk * u1.x), a3 = warp_sum(wk * u1.y);
        if (lane == 0) {
          float* dst = sA + (size_t)sw * 2 * (T + 1) + 4 * mp;
          dst[0] = a0; dst[1] = a1; dst[2] = a2; dst[3] = a3;         // the odd tail of an odd T lands in the padding
        }
      }
    }
    __syncthreads();
    const int P_n = P.n_partials;
    const size_t pbase = (size_t)scene * P_n + part;
    if (tid == 0) {
      P.part_m[pbase] = m;
      P.part_argmin[pbase] = idx;
      P.part_eta[pbase] = (sRedF[0] + sRedF[1]) + (sRedF[2] + sRedF[3]);
      P.part_w2[pbase] = (sRedF[4] + sRedF[5]) + (sRedF[6] + sRedF[7]);
      P.part_nonfinite[pbase] = (int)((sRedF[8] + sRedF[9]) + (sRedF[10] + sRedF[11]));
    }
    for (int o = tid; o < 2 * T; o += kMpccThreads) {
      const int st = 2 * (T + 1);
      const float a = (sA[o] + sA[st + o]) + (sA[2 * st + o] + sA[3 * st + o]);   // fixed order
      P.part_A[((size_t)scene * 2 * T + o) * P_n + part] = a;
    }
  }
}

struct MpccCtaPlan { int tiles_per_scene, total_tiles, grid; size_t smem; };

inline MpccCtaPlan make_mpcc_cta_plan(int K, int T, int n_scenes, int max_obstacles, int max_path_segments, int n_sms) {
  MpccCtaPlan pl{};
  pl.tiles_per_scene = (K + kMpccTile - 1) / kMpccTile;
  pl.total_tiles = pl.tiles_per_scene * n_scenes;
  pl.grid = pl.total_tiles < n_sms ? pl.total_tiles : n_sms;
  pl.smem = mpcc_cta_smem_layout(T, max_obstacles, max_path_segments).total;
  return pl;
}

typedef void (*MpccCtaKernel)(const DeviceParams);

inline MpccCtaKernel mpcc_cta_kernel_for(bool precise, int n_discs) {
  switch (n_discs) {
    case 1: return precise ? rollout_mpcc_cta<true, 1> : rollout_mpcc_cta<false, 1>;
    case 2: return precise ? rollout_mpcc_cta<true, 2> : rollout_mpcc_cta<false, 2>;
    case 3: return precise ? rollout_mpcc_cta<true, 3> : rollout_mpcc_cta<false, 3>;
    default: return precise ? rollout_mpcc_cta<true, 4> : rollout_mpcc_cta<false, 4>;
  }
}

}  // namespace brmppi
