// rollout_mpcc_cta.cuh -- the paper's own model and cost (BRMPPI_FLAG_MPCC, reading 31 and 9.2) as a
// persistent, phase-split CTA kernel: the default for that mode (BRMPPI_FLAG_KERNEL_THREAD_PER_SAMPLE selects
// rollout_mpcc.cuh's one-thread-per-sample kernel).
//
// A tile is S <= 128 samples (S chosen so that the tiles of a launch fill the SMs evenly, make_mpcc_cta_plan).  The
// only serial part of a rollout is the state recursion (noise, Euler step of eq. (6), path parameter): the CHAIN
// threads (the last 128 of the 768-thread CTA, S of them active) run it, one thread per sample, and leave every state of the
// horizon -- with all the trigonometry the step needed anyway -- in shared-memory planes, a chunk of L steps at a
// time into a two-deep ring.  The 640 COST threads take the (sample, step) items of a chunk as the chain finishes it
// (mbarrier per ring slot, full / empty): rates and their derivatives, disc centres, velocities and accelerations,
// the predictor (17) and the hinge for every (obstacle, disc), the path point and the stage cost (13).  G = 640 / S
// (at most 12) cost threads serve each sample, thread g of them the rows g, g + G, .. of every chunk, so a thread's
// cost sum stays in a register for the whole tile; no MUFU is issued by a cost thread.  The tile then forms its
// online-softmax partial like the other kernels, the sampled controls regenerated from Philox for the weighted sums.
#pragma once

#include "rollout_mpcc.cuh"
#include "rollout_cta_kernel.cuh"      // mbarrier helpers

namespace brmppi {

constexpr int kMpccThreads = 768;
constexpr int kMpccTileMax = 128;                      // samples per tile <= chain threads
constexpr int kMpccCost = kMpccThreads - kMpccTileMax; // 640 cost threads, threads [0, 640); the chain is [640, 768)
constexpr int kMpccMaxGroups = 12;                     // cost threads per sample, at most
constexpr int kMpccMaxRows = kMpccMaxGroups + 1;       // a chunk keeps the row after its last step too

// One row (one state of the horizon) is four planes of float4, each [stride]: a thread moves a state with four
// 128-bit accesses, conflict-free (consecutive samples, consecutive 16-byte words).
//   Q0 = (x, y, v, a)   Q1 = (sin t1, cos t1, sin t2, cos t2)   Q2 = (tan delta, t1, t2, psi)
//   Q3 = (sin, cos of the path heading at psi, j, omega)        (j, omega only without the control planes)
constexpr int MP_QUADS = 4;
constexpr int MP_COUNT = 4 * MP_QUADS;                 // floats per sample and row

// Tiling of one launch: S samples per tile, stride = S rounded up to a warp, G cost threads per sample, L steps per chunk.
// noise_planes: the sampled controls of the whole horizon are drawn by all threads before the chain starts and kept
// in shared memory [T][2][stride] (the chain then carries no Philox / Box-Muller latency, and the weighted sums
// read them back); 0 when they do not fit: the chain draws them as it goes and the epilogue regenerates them.
struct MpccCtaPlan { int S, stride, G, L, noise_planes, tiles_per_scene, total_tiles, grid; size_t smem; };

struct MpccCtaSmem { size_t obs, vel, path, U, planes, noise, part, w, red, A, bars, total; };

constexpr size_t kMpccSmemLimit = 227 * 1024;   // opt-in shared memory per CTA on sm_100

__host__ __device__ inline MpccCtaSmem mpcc_cta_smem_layout(int T, int max_obstacles, int max_path_segments,
                                                            int stride, int G, int L, int noise_planes) {
  MpccCtaSmem M{};
  size_t off = 0;
#define MPCC_TAKE(field, bytes) M.field = off; off = (off + (size_t)(bytes) + 15) / 16 * 16
  const size_t no = (size_t)(max_obstacles > 0 ? max_obstacles : 1);
  MPCC_TAKE(obs, sizeof(float4) * no);
  MPCC_TAKE(vel, sizeof(float4) * no);
  MPCC_TAKE(path, sizeof(float4) * 4 * (size_t)max_path_segments);
  MPCC_TAKE(U, sizeof(float2) * (size_t)(T + 2));
  MPCC_TAKE(planes, sizeof(float) * 2 * (size_t)(L + 1) * MP_COUNT * (size_t)stride);
  MPCC_TAKE(noise, noise_planes ? sizeof(float) * 2 * (size_t)(T + 1) * (size_t)stride : 0);
  MPCC_TAKE(part, sizeof(double) * (size_t)G * (size_t)stride);
  MPCC_TAKE(w, sizeof(float) * (size_t)stride);
  MPCC_TAKE(red, sizeof(double) * 4 + sizeof(int) * 4 + sizeof(float) * 12 + 16);
  MPCC_TAKE(A, sizeof(float) * 4 * 2 * (size_t)(T + 1));
  MPCC_TAKE(bars, sizeof(unsigned long long) * 4);
#undef MPCC_TAKE
  M.total = off;
  return M;
}

inline MpccCtaPlan make_mpcc_cta_plan(int K, int T, int n_scenes, int max_obstacles, int max_path_segments, int n_sms) {
  MpccCtaPlan pl{};
  // rounds of the grid over all tiles if every tile were full, then tiles per scene that fill those rounds evenly
  const long long total = (long long)K * n_scenes;
  const long long rounds = (total + (long long)kMpccTileMax * n_sms - 1) / ((long long)kMpccTileMax * n_sms);
  long long per_scene = rounds * n_sms / n_scenes;
  if (per_scene < 1) per_scene = 1;
  int S = (int)((K + per_scene - 1) / per_scene);
  S = S < 16 ? 16 : (S > kMpccTileMax ? kMpccTileMax : S);
  pl.S = S;
  pl.stride = (S + 31) / 32 * 32;
  pl.G = kMpccCost / S > kMpccMaxGroups ? kMpccMaxGroups : kMpccCost / S;
  pl.L = pl.G >= 5 ? pl.G : 2 * pl.G;
  pl.tiles_per_scene = (K + S - 1) / S;
  pl.total_tiles = pl.tiles_per_scene * n_scenes;
  pl.grid = pl.total_tiles < n_sms ? pl.total_tiles : n_sms;
  pl.noise_planes = mpcc_cta_smem_layout(T, max_obstacles, max_path_segments, pl.stride, pl.G, pl.L, 1).total <= kMpccSmemLimit;
  pl.smem = mpcc_cta_smem_layout(T, max_obstacles, max_path_segments, pl.stride, pl.G, pl.L, pl.noise_planes).total;
  return pl;
}

// One (sample, step) item of the cost phase: everything of step t that is not the state recursion.  Returns the
// stage cost (13) with the barrier term; *track = the four tracking terms at (x_{t+1}, psi_{t+1}).  row0 / row1:
// quad 0 of rows t and t + 1, already offset by the sample; st = plane stride (in float4).
template <int ND, bool CULL>
__device__ __forceinline__ float mpcc_cost_item(const DeviceParams& P, const float4* __restrict__ sObs,
                                                 const float4* __restrict__ sVel, const float4* __restrict__ sPath,
                                                 int n_moving, int n_obs, int M, float dpsi, float inv_dpsi, const float4* row0,
                                                 const float4* row1, int st, int t, float alpha, float inv_alpha_cull,
                                                 bool u_in_row, float2 u, float* track, float* pen_out) {
  const float4 q0 = row0[0], q1 = row0[st];                                     // (x, y, v, a), (s1, c1, s2, c2)
  const float td = row0[2 * st].x;
  if (u_in_row) { const float4 q3 = row0[3 * st]; u = make_float2(q3.z, q3.w); }
  const float vh = P.dt * q0.z, ah = P.dt * P.dt * q0.w;                         // step units (mpcc_hinge)
  const MpccRates R = mpcc_rates(P, vh, ah, td, q1.x, q1.y, q1.z, q1.w, P.dt * u.y);
  const float pen = mpcc_hinge<ND, CULL>(P, sObs, sVel, n_moving, n_obs, ND, (float)t, alpha, q0.x, q0.y, vh, ah, q1.x, q1.y,
                                   q1.z, q1.w, R, inv_alpha_cull);
  // stage cost (13) on (x_{t+1}, u_t, psi_{t+1}): the next row
  const float4 n0 = row1[0], n1 = row1[st], n2 = row1[2 * st], n3 = row1[3 * st];
  float nu;
  *track = mpcc_tracking_sc(P, n0.x, n0.y, n2.y, n2.z, n0.z, n1.x, n1.y, path_eval(sPath, M, dpsi, inv_dpsi, n2.w), n3.x,
                            n3.y, &nu);
  *pen_out = pen;
  return *track + mpcc_stage_rest(P, n2.y, n2.z, n0.z, nu, u);
}

template <bool PRECISE, int ND, bool CULL>
__global__ void __launch_bounds__(kMpccThreads, 1)
rollout_mpcc_cta(const __grid_constant__ DeviceParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int T = P.T, tid = threadIdx.x;
  const int S = P.S_tile, st = P.t_stride, G = P.chunks, L = P.chunk_len;
  const bool noise_planes = P.mpcc_noise_planes != 0;
  const MpccCtaSmem lay = mpcc_cta_smem_layout(T, P.max_obstacles, P.max_path_segments, st, G, L, noise_planes);
  float4* sObs = reinterpret_cast<float4*>(smem_raw + lay.obs);
  float4* sVel = reinterpret_cast<float4*>(smem_raw + lay.vel);
  float4* sPath = reinterpret_cast<float4*>(smem_raw + lay.path);
  float2* sU = reinterpret_cast<float2*>(smem_raw + lay.U);
  float4* sPlanes = reinterpret_cast<float4*>(smem_raw + lay.planes);
  float* sNoise = reinterpret_cast<float*>(smem_raw + lay.noise);      // [T + 1][2][st]: j, omega of every step
  double* sPart = reinterpret_cast<double*>(smem_raw + lay.part);
  float* sW = reinterpret_cast<float*>(smem_raw + lay.w);
  double* sRedM = reinterpret_cast<double*>(smem_raw + lay.red);
  int* sRedI = reinterpret_cast<int*>(sRedM + 4);
  float* sRedF = reinterpret_cast<float*>(sRedI + 4);
  float* sA = reinterpret_cast<float*>(smem_raw + lay.A);
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_raw + lay.bars);   // full[2], empty[2]

  // roles: chain thread of sample s, or cost thread `grp` of sample s (cost thread index grp * S + s)
  const int lane = tid & 31, warp = tid >> 5;
  const bool chain_range = tid >= kMpccCost;
  const int grp = chain_range ? 0 : tid / S;
  const int s = chain_range ? tid - kMpccCost : tid - grp * S;
  const bool is_chain = chain_range && s < S, is_cost = !chain_range && grp < G;
  const int n_chunks = (T + L - 1) / L;
  const int row_quads = MP_QUADS * st, slot_quads = (L + 1) * row_quads;
  const uint32_t n = *P.counter;
  if (tid == 0) {
    mbar_init(smem_addr(&bars[0]), S); mbar_init(smem_addr(&bars[1]), S);
    mbar_init(smem_addr(&bars[2]), G * S); mbar_init(smem_addr(&bars[3]), G * S);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  uint32_t g = 0;                    // chunks handed over so far (ring position; the same on every thread)
  int loaded_scene = -1;

  for (int tile = blockIdx.x; tile < P.total_tiles; tile += gridDim.x) {
    const int scene = tile / P.tiles_per_scene, part = tile - scene * P.tiles_per_scene;
    const int k = part * S + s;
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
        // the table holds the moving obstacles first, each class in the caller's order (mpcc_hinge)
        const float* all = P.obstacles + (size_t)scene * P.max_obstacles * 5;
        const float* ob = all + i * 5;
        const bool mov = ob[3] != 0.0f || ob[4] != 0.0f;
        int before_same = 0, n_mov = 0;
        for (int j = 0; j < n_obs; ++j) {
          const bool mj = all[j * 5 + 3] != 0.0f || all[j * 5 + 4] != 0.0f;
          n_mov += mj ? 1 : 0;
          before_same += (j < i && mj == mov) ? 1 : 0;
        }
        const int slot = mov ? before_same : n_mov + before_same;
        const float rho = ob[2] + P.disc_radius;
        // vehicle-centred frame; .w and .z of the two entries: the culling radii of mpcc_hinge, with their margin
        sObs[slot] = make_float4(ob[0] - x0, ob[1] - y0, 1.0f / (rho * rho), fmaf(1.001f, P.mpcc_lmax + rho, 1e-3f));
        sVel[slot] = make_float4(P.dt * ob[3], P.dt * ob[4],
                                 2.0f * P.dt * sqrtf(fmaf(ob[3], ob[3], ob[4] * ob[4])), 0.0f);
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
    if (noise_planes) {
      // ---- the sampled controls of the tile (a1, a2): thread -> (sample slot es, every n_pg-th step pair) ----
      const int pg = tid / st, es = tid - pg * st, n_pg = kMpccThreads / st;
      const int k_es = min(part * S + es, P.K - 1);
      for (int mp = pg; 2 * mp < T; mp += n_pg) {
        float2 u0, u1;
        sample_control_pair<PRECISE>(P, sU[2 * mp], sU[2 * mp + 1], (uint32_t)mp, n, (uint32_t)(k_es + P.k_offset), key0,
                                     key1, &u0, &u1);
        float* dst = sNoise + (size_t)(4 * mp) * st + es;               // the odd tail of an odd T lands in row T
        dst[0] = u0.x; dst[st] = u0.y; dst[2 * st] = u1.x; dst[3 * st] = u1.y;
      }
      __syncthreads();
    }

    if (is_chain) {
      // ---- the state recursion of eq. (6), one thread per sample; rows of L steps into the ring ----
      const float Lpath = (float)M * dpsi;
      State7 X{0.0f, 0.0f, s7[2], s7[3], s7[4], s7[5], s7[6], s7[7]};
      // every function of the current state that a step needs is carried: the four evaluations for the NEXT state
      // (sin / cos of both headings, tan(delta), path heading and its sin / cos) are independent of one another and
      // are issued together at the end of a step, so their latencies overlap instead of adding up
      float s1, c1, s2, c2, sr, cr, td;
      sincos_t<PRECISE>(X.t1, &s1, &c1);
      sincos_t<PRECISE>(X.t2, &s2, &c2);
      td = tan_t<PRECISE>(X.de);
      sincos_t<PRECISE>(path_eval_component(sPath, M, dpsi, inv_dpsi, X.psi, 2), &sr, &cr);
      float2 u_odd = make_float2(0.0f, 0.0f);
      int t = 0;
      for (int c = 0; c < n_chunks; ++c) {
        const uint32_t gg = g + (uint32_t)c;
        const int slot = (int)(gg & 1u);
        if (gg >= 2u) mbar_wait(smem_addr(&bars[2 + slot]), ((gg >> 1) - 1u) & 1u);   // the cost threads are done with it
        float4* row = sPlanes + slot * slot_quads + s;
        const int t_end = min(t + L, T);
#pragma unroll 1
        for (; t < t_end; ++t, row += row_quads) {
          float2 u;
          if (noise_planes)
            u = make_float2(sNoise[(size_t)(2 * t) * st + s], sNoise[(size_t)(2 * t + 1) * st + s]);
          else if ((t & 1) == 0)  // one Philox block serves a pair of steps (reading 6)
            sample_control_pair<PRECISE>(P, sU[t], sU[t + 1], (uint32_t)(t >> 1), n, (uint32_t)(kk + P.k_offset), key0,
                                         key1, &u, &u_odd);
          else
            u = u_odd;
          row[0] = make_float4(X.x, X.y, X.v, X.a);
          row[st] = make_float4(s1, c1, s2, c2);
          row[2 * st] = make_float4(td, X.t1, X.t2, X.psi);
          row[3 * st] = make_float4(sr, cr, u.x, u.y);
          const float vh = P.dt * X.v;
          const float nu = X.v * fmaf(c1, cr, s1 * sr);
          const MpccRates R = mpcc_rates(P, vh, 0.0f, td, s1, c1, s2, c2, 0.0f);     // Ts W1, Ts W2 are what is used
          State7 N;
          N.x = fmaf(vh, c1, X.x);
          N.y = fmaf(vh, s1, X.y);
          N.v = fmaf(P.dt, X.a, X.v);
          N.a = fmaf(P.dt, u.x, X.a);
          N.t1 = X.t1 + R.W1;
          N.t2 = X.t2 + R.W2;
          N.de = fminf(fmaxf(fmaf(P.dt, u.y, X.de), P.dstate_lo), P.dstate_hi);
          N.psi = fminf(fmaxf(fmaf(P.dt, nu, X.psi), 0.0f), Lpath);
          X = N;
          const float thr = path_eval_component(sPath, M, dpsi, inv_dpsi, X.psi, 2);
          sincos_t<PRECISE>(thr, &sr, &cr);
          sincos_t<PRECISE>(X.t1, &s1, &c1);
          sincos_t<PRECISE>(X.t2, &s2, &c2);
          td = tan_t<PRECISE>(X.de);
        }
        // the row after the chunk's last step: read only as a "next state"
        row[0] = make_float4(X.x, X.y, X.v, X.a);
        row[st] = make_float4(s1, c1, s2, c2);
        row[2 * st] = make_float4(td, X.t1, X.t2, X.psi);
        row[3 * st] = make_float4(sr, cr, 0.0f, 0.0f);
        mbar_arrive(smem_addr(&bars[slot]));
      }
      if (valid && (P.flags & BRMPPI_FLAG_WRITE_SAMPLES)) {
        float4* out = reinterpret_cast<float4*>(P.XT) + 2 * ((size_t)scene * P.K + k);
        out[0] = make_float4(X.x + x0, X.y + y0, X.v, X.a);
        out[1] = make_float4(X.t1, X.t2, X.de, X.psi);
      }
    } else if (is_cost) {
      // ---- cost phase: the (sample, step) items of each chunk as the chain hands it over ----
      const float alpha = sample_alpha(P, n, (uint32_t)(kk + P.k_offset), key0, key1);
      int n_moving = 0;
      for (int i = 0; i < n_obs; ++i) n_moving += (sVel[i].x != 0.0f || sVel[i].y != 0.0f) ? 1 : 0;
      // exact culling of far obstacles (mpcc_hinge): off for alpha <= 0 and under BRMPPI_FLAG_NO_CULL
      const float inv_alpha_cull = (CULL && alpha > 0.0f) ? 1.001f / alpha : 0.0f;
      // a thread's T / G items are summed in fp32 (at most a few tens of terms of like size), the stage costs and the
      // hinge sums apart; fp64 takes over where magnitudes mix: w_bar times the hinge sum, the terminal cost, and
      // the sum over the G threads of a sample in phase D
      float acc_stage = 0.0f, acc_pen = 0.0f, term = 0.0f;
      for (int c = 0; c < n_chunks; ++c) {
        const uint32_t gg = g + (uint32_t)c;
        const int slot = (int)(gg & 1u);
        mbar_wait(smem_addr(&bars[slot]), (gg >> 1) & 1u);
#pragma unroll 1
        for (int r = grp; r < L; r += G) {
          const int t = c * L + r;
          if (t < T) {
            float track;
            const float4* row0 = sPlanes + slot * slot_quads + r * row_quads + s;
            float pen;
            acc_stage += mpcc_cost_item<ND, CULL>(P, sObs, sVel, sPath, n_moving, n_obs, M, dpsi, inv_dpsi, row0, row0 + row_quads, st, t,
                                      alpha, inv_alpha_cull, true, make_float2(0.0f, 0.0f), &track, &pen);
            acc_pen += pen;
            if (t == T - 1) term = P.w_term * track;                 // terminal cost: the same four terms at (x_N, psi_N)
          }
        }
        mbar_arrive(smem_addr(&bars[2 + slot]));
      }
      sPart[grp * st + s] = ((double)acc_stage + (double)term) + (double)P.w_bar * (double)acc_pen;
    }
    g += (uint32_t)n_chunks;
    __syncthreads();

    // ---- the tile's online-softmax partial (a7): S_k, block minimum, weights, eta, weighted control sums ----
    // here thread tid < stride stands for sample slot tid (whole warps, so that the warp reductions are complete)
    const int ke = part * S + tid;
    const bool valid_e = tid < S && ke < P.K;
    double Sk = CUDART_INF, m = CUDART_INF;
    bool finite = false;
    if (tid < st) {
      if (tid < S) {
        Sk = sPart[tid];
        for (int q = 1; q < G; ++q) Sk += sPart[q * st + tid];                     // fixed order
      }
      finite = valid_e && (Sk == Sk) && (Sk < CUDART_INF) && (Sk > -CUDART_INF);
      if (valid_e && (P.flags & BRMPPI_FLAG_WRITE_SAMPLES)) P.S[(size_t)scene * P.K + ke] = (float)Sk;
      m = finite ? Sk : CUDART_INF;
      int idx = finite ? ke + P.k_offset : 0x7fffffff;
      warp_argmin(m, idx);
      if (lane == 0) { sRedM[warp] = m; sRedI[warp] = idx; }
    }
    __syncthreads();
    const int n_sw = st >> 5;                                       // warps of sample slots
    int idx = sRedI[0];
    m = sRedM[0];
    for (int w = 1; w < n_sw; ++w)
      if (sRedM[w] < m || (sRedM[w] == m && sRedI[w] < idx)) { m = sRedM[w]; idx = sRedI[w]; }
    if (tid < st) {
      const float wk = finite ? expf((float)(-(Sk - m) * (double)P.inv_lambda)) : 0.0f;   // S - m in fp64, then fp32 exp
      sW[tid] = wk;
      const float eta = warp_sum(wk), w2 = warp_sum(wk * wk), nf = warp_sum((valid_e && !finite) ? 1.0f : 0.0f);
      if (lane == 0) { sRedF[warp] = eta; sRedF[4 + warp] = w2; sRedF[8 + warp] = nf; }
    }
    __syncthreads();
    if (noise_planes) {
      // weighted control sums from the kept controls: a warp takes EIGHT outputs (step, channel) at a time, lanes
      // over the samples; the eight per-lane sums are reduced together by a transposing butterfly (4 + 2 + 1
      // exchanges leave each lane with one output's sum over its 4-lane class, two more finish it): 9 shuffles
      // for 8 outputs instead of 40, and the lane's weights are loaded once
      const int n_warps = kMpccThreads / 32;
      float wl[kMpccTileMax / 32];
#pragma unroll
      for (int i = 0; i < kMpccTileMax / 32; ++i) wl[i] = (lane + 32 * i < st) ? sW[lane + 32 * i] : 0.0f;
#pragma unroll 1
      for (int o0 = 8 * warp; o0 < 2 * T; o0 += 8 * n_warps) {
        float a[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const float* u = sNoise + (size_t)min(o0 + q, 2 * T - 1) * st + lane;
          float acc = 0.0f;
#pragma unroll
          for (int i = 0; i < kMpccTileMax / 32; ++i)
            if (32 * i < st) acc = fmaf(wl[i], u[32 * i], acc);
          a[q] = acc;
        }
        // after the round with mask m a lane keeps the outputs whose bit agrees with its own lane bit
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
        // lane bits (16, 8, 4) -> output bits (4, 2, 1)
        const int q_own = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
        if ((lane & 3) == 0 && o0 + q_own < 2 * T)
          P.part_A[((size_t)scene * 2 * T + o0 + q_own) * P.n_partials + part] = b1;
      }
    } else {
      // the sampled controls regenerated from the counter-based generator: thread -> (sample slot es, every n_pg-th
      // step pair); the samples of a pair are n_sw warps
      const int pg = tid / st, es = tid - pg * st, n_pg = kMpccThreads / st;
      const float wk = sW[es];
      const int k_es = min(part * S + es, P.K - 1);
      const int sw = es >> 5;
      for (int mp = pg; 2 * mp < T; mp += n_pg) {
        float2 u0, u1;
        sample_control_pair<PRECISE>(P, sU[2 * mp], sU[2 * mp + 1], (uint32_t)mp, n, (uint32_t)(k_es + P.k_offset), key0,
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
      float eta = sRedF[0], w2 = sRedF[4], nf = sRedF[8];
      for (int w = 1; w < n_sw; ++w) { eta += sRedF[w]; w2 += sRedF[4 + w]; nf += sRedF[8 + w]; }
      P.part_m[pbase] = m;
      P.part_argmin[pbase] = idx;
      P.part_eta[pbase] = eta;
      P.part_w2[pbase] = w2;
      P.part_nonfinite[pbase] = (int)nf;
    }
    for (int o = tid; o < 2 * T && !noise_planes; o += kMpccThreads) {
      const int sa = 2 * (T + 1);
      float a = sA[o];
      for (int w = 1; w < n_sw; ++w) a += sA[w * sa + o];           // fixed order
      P.part_A[((size_t)scene * 2 * T + o) * P_n + part] = a;
    }
  }
}

typedef void (*MpccCtaKernel)(const DeviceParams);

template <bool CULL>
inline MpccCtaKernel mpcc_cta_kernel_pick(bool precise, int n_discs) {
  switch (n_discs) {
    case 1: return precise ? rollout_mpcc_cta<true, 1, CULL> : rollout_mpcc_cta<false, 1, CULL>;
    case 2: return precise ? rollout_mpcc_cta<true, 2, CULL> : rollout_mpcc_cta<false, 2, CULL>;
    case 3: return precise ? rollout_mpcc_cta<true, 3, CULL> : rollout_mpcc_cta<false, 3, CULL>;
    default: return precise ? rollout_mpcc_cta<true, 4, CULL> : rollout_mpcc_cta<false, 4, CULL>;
  }
}

// cull = false (BRMPPI_FLAG_NO_CULL): the instantiation without the culling test
inline MpccCtaKernel mpcc_cta_kernel_for(bool precise, int n_discs, bool cull) {
  return cull ? mpcc_cta_kernel_pick<true>(precise, n_discs) : mpcc_cta_kernel_pick<false>(precise, n_discs);
}

}  // namespace brmppi
