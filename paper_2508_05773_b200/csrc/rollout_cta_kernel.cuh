// rollout_cta_kernel.cuh -- the persistent-CTA rollout kernel itself (design notes, plan and
// shared-memory layout are in rollout_cta.cuh).
//
// Register discipline: everything that lives for the whole kernel but is touched once per phase
// (start state, goal, obstacle counts, running softmax state) sits in the CtaMisc block of shared
// memory, and every shared-memory section pointer is smem_raw + a constant-bank offset, so the long
// phase-C loop does not have to share the register file with values it never uses.
#pragma once

#include "rollout_cta.cuh"

namespace brmppi {

#define BRMPPI_SMEM(type, off) reinterpret_cast<type*>(smem_raw + (off))

// unroll factor of the phase-C step loop (2 lets h_t / h_{t+1} swap registers without moves)
#ifndef BRMPPI_C_UNROLL
#define BRMPPI_C_UNROLL 2
#endif
constexpr int kCostUnroll = BRMPPI_C_UNROLL;

__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
// BRMPPI_FLAG_PHASE_TIMING: thread 0 adds the SM cycles since the previous stamp to phase slot i
// (clock64: the globaltimer ticks too coarsely for sub-microsecond phases; it only brackets the CTA)
// BAR.SYNC is deferred-blocking: the volatile shared-memory read makes the stamp wait for the
// barrier's release instead of recording the arrival of warp 0.
#define BRMPPI_STAMP(i)                                                      \
  if (P.phase_ns != nullptr && tid == 0) {                                   \
    const unsigned long long seen__ = *reinterpret_cast<volatile unsigned long long*>(&BRMPPI_SMEM(CtaMisc, P.off_misc)->t_begin); \
    const unsigned long long now__ = (unsigned long long)clock64() + (seen__ & 0ull); \
    BRMPPI_SMEM(CtaMisc, P.off_misc)->phase_acc[i] += now__ - t_stamp;       \
    t_stamp = now__;                                                         \
  }

// mbarrier hand-off (chain warps -> cost threads), CTA scope.  One phase per tile: the waiter passes
// the parity of the tile it is in.
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {   // release: this thread's earlier shared stores are visible to the waiter
  asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.acquire.cta.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    if (!done) __nanosleep(32);     // waiting warps must not take issue slots from the chain and the table warp
  } while (!done);
}

// Phase C for one group of kObsGroup obstacles over the steps [t0, t1) of one sample: the
// barrier-rate hinge sum_t sum_{i,j} max(0, (1 - alpha) h_t - h_{t+1})  (a4, a5), and -- for the
// first group (TRACK) -- the goal / heading / hitch stage cost of every state it visits (a6).
//
// Arithmetic form.  With rho = R + r_v and g = |c - o|^2 - rho^2 (so h = g / rho^2):
//     max(0, (1-alpha) h_t - h_{t+1}) = -(1 / rho^2) min(0, zn),   zn = g_{t+1} - (1-alpha) g_t.
// Obstacles are taken two at a time on packed f32x2 operands (add/fma.rn.f32x2: each half rounds
// like the scalar instruction): per (obstacle pair, disc) 2 packed subtractions, 2 packed FMAs for
// g, 1 for zn, 2 scalar FADDs zn - |zn| (= 2 min(0, zn) exactly; the weight carries the 1/2), 1 packed accumulate.
// The table (written by warp 0) interleaves obstacles 2p and 2p+1 field by field, already
// negated -- (-ox, -ox'), (-oy, -oy'), (-1/(2 rho^2), ..), (-rho^2, ..) -- so every packed operand is
// one 64-bit shared-memory load; built from scalars, ptxas re-packs them with two MOVs per use.
// A null (padding) obstacle is all zeros: its weight is 0, so it adds exactly 0.  MOVING: some
// obstacle of the group moves, o(t) = o(0) + t dt vel (a static one has vel == 0, so the update is
// exact for it too).
//
// Exact culling.  thr[i][j] (warp 0, once per scene) is the value of g above which
// disc j cannot violate the rate condition against obstacle i anywhere in a chunk, for ANY alpha the
// sampler can draw (alpha >= alpha_lo gives the largest critical distance): every hinge term of the
// pair is then exactly +0 and the pair of obstacles is skipped for the chunk.  The mask is the union
// over the warp's samples, so the skip is a uniform branch.
// pV, pP1, pP2: this sample's rows of the v, psi1, psi2 planes.
struct GroupCost { double track, bar; };

// One chunk of one sample with the first NACT obstacle pairs of the group evaluated (the others are
// culled for this chunk): loads those pairs, g at the chunk's first state, then the step loop --
// straight-line code, so g_t / g_{t+1} swap registers across the two unrolled steps without moves,
// and a chunk that needs one pair does not carry the registers of four.
template <bool PRECISE, int ND, bool MOVING, bool TRACK, int NACT>
__device__ __forceinline__ GroupCost hinge_chunk(const DeviceParams& P, const float* __restrict__ pV,
                                                 const float* __restrict__ pP1, const float* __restrict__ pP2,
                                                 const float4* __restrict__ obs, const float2* __restrict__ vel,
                                                 float x, float y, int t0, int t1, float one_minus_alpha,
                                                 const float4 g) {
  double bar = 0.0, track = 0.0;
  constexpr int NA = NACT > 0 ? NACT : 1;
  // obstacles in pairs (2p, 2p+1): negated centres, -rho^2, -1/(2 rho^2) and g of the previous state
  f32x2 nox[NA], noy[NA], mrho2[NA], nw[NA], gprev[NA][ND];
  const f32x2 noma = pack2(-one_minus_alpha, -one_minus_alpha);
  float s1, c1;
  sincos_t<PRECISE>(pP1[t0], &s1, &c1);
  if (NACT > 0) {
    // the table is pair-interleaved (see the table warp), so a pair arrives as one 64-bit register
    const ulonglong2* q = reinterpret_cast<const ulonglong2*>(obs);
#pragma unroll
    for (int p = 0; p < NACT; ++p) {
      const ulonglong2 a = q[2 * p], b = q[2 * p + 1];
      nox[p] = a.x; noy[p] = a.y; nw[p] = b.x; mrho2[p] = b.y;
    }
    float s2, c2;
    sincos_t<PRECISE>(pP2[t0], &s2, &c2);
    float cx[ND], cy[ND];
    disc_centres_n<ND>(P, x, y, s1, c1, s2, c2, cx, cy);
    const float tfp = (float)t0;
#pragma unroll
    for (int p = 0; p < NACT; ++p) {
      f32x2 ex = nox[p], ey = noy[p];
      if (MOVING) {   // o(t) = o(0) + t dt vel, negated exactly (a static obstacle has vel == 0)
        const ulonglong2 w = reinterpret_cast<const ulonglong2*>(vel)[p];
        const f32x2 tf2 = pack2(tfp, tfp);
        ex = fma2(tf2, w.x, ex);
        ey = fma2(tf2, w.y, ey);
      }
#pragma unroll
      for (int j = 0; j < ND; ++j) {
        const f32x2 dx = add2(pack2(cx[j], cx[j]), ex), dy = add2(pack2(cy[j], cy[j]), ey);
        gprev[p][j] = fma2(dx, dx, fma2(dy, dy, mrho2[p]));
      }
    }
  }
#pragma unroll kCostUnroll
  for (int t = t0; t < t1; ++t) {
    // (x, y) of state t+1 from state t: the chain's own FMAs on the same operands
    const float v_t = pV[t];
    const float a = P.dt * v_t;
    x = fmaf(a, c1, x);
    y = fmaf(a, s1, y);
    const float psi1 = pP1[t + 1], psi2 = pP2[t + 1];
    sincos_t<PRECISE>(psi1, &s1, &c1);
    if (TRACK) {
      const State X{x, y, psi1, psi2};
      if (PRECISE) track += (double)(goal_cost(P, X, g) + hitch_cost(P, X, v_t));
      else track += (double)tracking_cost_fma(P, X, g, v_t);
    }
    if (NACT > 0) {
      float s2, c2;
      sincos_t<PRECISE>(psi2, &s2, &c2);
      float cx[ND], cy[ND];
      disc_centres_n<ND>(P, x, y, s1, c1, s2, c2, cx, cy);
      const float tfp = (float)(t + 1);
      f32x2 pen = pack2(0.0f, 0.0f);
#pragma unroll
      for (int p = 0; p < NACT; ++p) {
        f32x2 ex = nox[p], ey = noy[p];
        if (MOVING) {
          const ulonglong2 w = reinterpret_cast<const ulonglong2*>(vel)[p];
          const f32x2 tf2 = pack2(tfp, tfp);
          ex = fma2(tf2, w.x, ex);
          ey = fma2(tf2, w.y, ey);
        }
#pragma unroll
        for (int j = 0; j < ND; ++j) {
          const f32x2 dx = add2(pack2(cx[j], cx[j]), ex), dy = add2(pack2(cy[j], cy[j]), ey);
          const f32x2 gn = fma2(dx, dx, fma2(dy, dy, mrho2[p]));
          const f32x2 zn = fma2(gprev[p][j], noma, gn);             // g_{t+1} - (1-alpha) g_t = -z
          float za, zb;
          unpack2(zn, za, zb);
          // + max(0, z) / rho^2: min(0, zn) as (zn - |zn|) / 2 -- exact (0 or 2 zn), one full-rate FADD with the
          // |.| source modifier instead of a half-rate FMNMX; the table's weight carries the 1/2
          pen = fma2(nw[p], pack2(za - fabsf(za), zb - fabsf(zb)), pen);
          gprev[p][j] = gn;
        }
      }
      float pa, pb;
      unpack2(pen, pa, pb);
      bar += (double)(pa + pb);
    }
  }
  return GroupCost{track, bar};
}

template <bool PRECISE, int ND, bool MOVING, bool TRACK>
__device__ __forceinline__ GroupCost barrier_group(const DeviceParams& P, const float* __restrict__ pV,
                                                   const float* __restrict__ pP1, const float* __restrict__ pP2,
                                                   const float4* __restrict__ obs, const float2* __restrict__ vel,
                                                   const float* __restrict__ thr,
                                                   float x, float y, int t0, int t1, float one_minus_alpha,
                                                   const float4 g) {
  constexpr int NP = kObsGroup / 2;
  // pairs to evaluate in this chunk: 1 + the highest pair any sample of the warp needs (the table is
  // ordered by how close an obstacle is to its threshold at the start state, so the needed pairs are
  // mostly a prefix; evaluating a culled pair in between adds exact zeros)
  int n_act = NP;
  if (!(P.flags & BRMPPI_FLAG_NO_CULL)) {
    float s1, c1, s2, c2;
    sincos_t<PRECISE>(pP1[t0], &s1, &c1);
    sincos_t<PRECISE>(pP2[t0], &s2, &c2);
    float cx[ND], cy[ND];
    disc_centres_n<ND>(P, x, y, s1, c1, s2, c2, cx, cy);
    const float tfp = (float)t0;
    unsigned mine = 0u;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
      const ulonglong2 a = reinterpret_cast<const ulonglong2*>(obs)[2 * p];
      const f32x2 mr = reinterpret_cast<const ulonglong2*>(obs)[2 * p + 1].y;
      f32x2 ex = a.x, ey = a.y;
      if (MOVING) {
        const ulonglong2 w = reinterpret_cast<const ulonglong2*>(vel)[p];
        const f32x2 tf2 = pack2(tfp, tfp);
        ex = fma2(tf2, w.x, ex);
        ey = fma2(tf2, w.y, ey);
      }
      bool far = true;
#pragma unroll
      for (int j = 0; j < ND; ++j) {
        const f32x2 dx = add2(pack2(cx[j], cx[j]), ex), dy = add2(pack2(cy[j], cy[j]), ey);
        float ga, gb;
        unpack2(fma2(dx, dx, fma2(dy, dy, mr)), ga, gb);
        far = far && (ga >= thr[(2 * p) * kMaxDiscs + j]) && (gb >= thr[(2 * p + 1) * kMaxDiscs + j]);   // NaN: not far
      }
      mine |= far ? 0u : (1u << p);
    }
    n_act = 32 - __clz((int)__reduce_or_sync(__activemask(), mine));
  }
#define BRMPPI_CHUNK(N) return hinge_chunk<PRECISE, ND, MOVING, TRACK, N>(P, pV, pP1, pP2, obs, vel, x, y, t0, t1, one_minus_alpha, g)
  switch (n_act) {
    case 0: if (TRACK) BRMPPI_CHUNK(0); return GroupCost{0.0, 0.0};
    case 1: BRMPPI_CHUNK(1);
    case 2: BRMPPI_CHUNK(2);
    case 3: BRMPPI_CHUNK(3);
    default: BRMPPI_CHUNK(4);
  }
#undef BRMPPI_CHUNK
}

// Super-ellipse obstacles (eq. (16)), kSeGroup at a time:
//   (x', y') = R(-theta)(c - o(t)),  h = (x'/(m_x + r_v))^e + (y'/(m_y + r_v))^e - 1,  e = 2 or 4,
// and the same barrier-rate hinge as for discs.  The record holds the rows of R(-theta) divided by
// the inflated semi-axes, so u = x'/a_x and v = y'/a_y cost two FMA-pipe instructions each.
// Per (obstacle, disc): 2 subtractions, 4 for (u, v), 4 for u^4 + v^4 - 1 (2 for e = 2), rate
// argument, |.|-add, accumulate = 13 (11).  A null record has weight 0.
struct SeRecord { float ox, oy, a11, a12, a21, a22, wx, wy, e4, half_w, pad0, pad1; };
static_assert(sizeof(SeRecord) == 48, "SeRecord layout");

template <bool PRECISE, int ND, bool TRACK>
__device__ __forceinline__ GroupCost se_group(const DeviceParams& P, const float* __restrict__ pV,
                                              const float* __restrict__ pP1, const float* __restrict__ pP2,
                                              const SeRecord* __restrict__ rec, float x, float y, int t0, int t1,
                                              float one_minus_alpha, const float4 g) {
  double bar = 0.0, track = 0.0;
  float hprev[kSeGroup][ND];
  float s1, c1;
  {
    float s2, c2;
    sincos_t<PRECISE>(pP1[t0], &s1, &c1);
    sincos_t<PRECISE>(pP2[t0], &s2, &c2);
    float cx[ND], cy[ND];
    disc_centres_n<ND>(P, x, y, s1, c1, s2, c2, cx, cy);
    const float tf = (float)t0;
#pragma unroll
    for (int i = 0; i < kSeGroup; ++i) {
      const SeRecord r = rec[i];
      const float ox = fmaf(tf, r.wx, r.ox), oy = fmaf(tf, r.wy, r.oy);
#pragma unroll
      for (int j = 0; j < ND; ++j) {
        const float dx = cx[j] - ox, dy = cy[j] - oy;
        const float u = fmaf(r.a11, dx, r.a12 * dy), v = fmaf(r.a21, dx, r.a22 * dy);
        const float u2 = u * u, v2 = v * v;
        hprev[i][j] = r.e4 != 0.0f ? fmaf(u2, u2, fmaf(v2, v2, -1.0f)) : fmaf(u, u, fmaf(v, v, -1.0f));
      }
    }
  }
  float tf = (float)t0;
  for (int t = t0; t < t1; ++t) {
    const float v_t = pV[t];
    const float a = P.dt * v_t;
    x = fmaf(a, c1, x);
    y = fmaf(a, s1, y);
    const float psi1 = pP1[t + 1], psi2 = pP2[t + 1];
    float s2, c2;
    sincos_t<PRECISE>(psi1, &s1, &c1);
    sincos_t<PRECISE>(psi2, &s2, &c2);
    float cx[ND], cy[ND];
    disc_centres_n<ND>(P, x, y, s1, c1, s2, c2, cx, cy);
    if (TRACK) {   // scenes without disc obstacles: the first super-ellipse group carries the stage cost
      const State X{x, y, psi1, psi2};
      if (PRECISE) track += (double)(goal_cost(P, X, g) + hitch_cost(P, X, v_t));
      else track += (double)tracking_cost_fma(P, X, g, v_t);
    }
    tf += 1.0f;
    float pen = 0.0f;
#pragma unroll
    for (int i = 0; i < kSeGroup; ++i) {
      const SeRecord r = rec[i];
      const float ox = fmaf(tf, r.wx, r.ox), oy = fmaf(tf, r.wy, r.oy);
      float Pi = 0.0f;
#pragma unroll
      for (int j = 0; j < ND; ++j) {
        const float dx = cx[j] - ox, dy = cy[j] - oy;
        const float u = fmaf(r.a11, dx, r.a12 * dy), v = fmaf(r.a21, dx, r.a22 * dy);
        const float u2 = u * u, v2 = v * v;
        const float hn = r.e4 != 0.0f ? fmaf(u2, u2, fmaf(v2, v2, -1.0f)) : fmaf(u, u, fmaf(v, v, -1.0f));   // obstacle-uniform
        const float z = fmaf(one_minus_alpha, hprev[i][j], -hn);
        Pi += z + fabsf(z);                                       // 2 max(0, z), exactly
        hprev[i][j] = hn;
      }
      pen = fmaf(r.half_w, Pi, pen);
    }
    bar += (double)pen;
  }
  return GroupCost{track, bar};
}

// Dispatch on whether any obstacle of the group moves (block-uniform).
template <bool PRECISE, int ND, bool TRACK>
__device__ __forceinline__ GroupCost barrier_group_mv(bool moving, const DeviceParams& P, const float* pV,
                                                      const float* pP1, const float* pP2, const float4* obs,
                                                      const float2* vel, const float* thr, float x, float y,
                                                      int t0, int t1, float oma, const float4 g) {
  if (!moving) return barrier_group<PRECISE, ND, false, TRACK>(P, pV, pP1, pP2, obs, vel, thr, x, y, t0, t1, oma, g);
  return barrier_group<PRECISE, ND, true, TRACK>(P, pV, pP1, pP2, obs, vel, thr, x, y, t0, t1, oma, g);
}

template <bool PRECISE, int ND>
__global__ void __launch_bounds__(kCtaThreads, 1)
rollout_cta(const __grid_constant__ DeviceParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x;
  const int S = P.S_tile;
  const int c = tid / S, s = tid - c * S;     // (chunk or row, sample in tile)
  const int lane = tid & 31, warp = tid >> 5;

  const int tile_first = blockIdx.x * P.tiles_per_cta;
  const int tile_last = min(tile_first + P.tiles_per_cta, P.total_tiles);
  int cur_scene = -1;
  int par = 0;          // parity of the running softmax state in CtaMisc
  uint32_t tile_parity = 0;   // phase parity of the hand-off barriers (one phase per tile)
  unsigned long long t_stamp = 0;
  if (tid == 0) {
    CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
    for (int i = 0; i < kMaxChunks; ++i) mbar_init(smem_addr(&sM->bar_chunk[i]), kMaxTileSamples);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (P.phase_ns != nullptr && tid == 0) {
    for (int i = 0; i < kPhaseSlots; ++i) BRMPPI_SMEM(CtaMisc, P.off_misc)->phase_acc[i] = 0ull;
    t_stamp = (unsigned long long)clock64();
    BRMPPI_SMEM(CtaMisc, P.off_misc)->t_begin = global_ns();
  }

  for (int tile = tile_first; tile < tile_last; ++tile) {
    const int scene = tile / P.tiles_per_scene;
    const int k = (tile - scene * P.tiles_per_scene) * S + s;

    const bool new_scene = (scene != cur_scene);
    if (new_scene) {
      // ---- partial of the scene just finished -> HBM -------------------------------------------
      if (cur_scene >= 0) {
        const int Pn = P.n_partials, T = P.T;
        const CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
        const float* sA = BRMPPI_SMEM(float, P.off_A);
        const int slot = blockIdx.x - (cur_scene * P.tiles_per_scene) / P.tiles_per_cta;
        const size_t pbase = (size_t)cur_scene * Pn + slot;
        if (tid == 0) {
          P.part_m[pbase] = sM->m[par];
          P.part_argmin[pbase] = sM->argmin[par];
          P.part_eta[pbase] = sM->eta[par];
          P.part_w2[pbase] = sM->w2[par];
          P.part_nonfinite[pbase] = sM->nonfinite[par];
        }
        for (int o = tid; o < 2 * T; o += kCtaThreads) {
          const int ch = o >= T ? 1 : 0, t = o - ch * T;
          P.part_A[((size_t)cur_scene * 2 * T + (2 * t + ch)) * Pn + slot] = sA[o];
        }
        __syncthreads();
      }
      cur_scene = scene;
      par = 0;
    }
    // Scene data: the global loads are issued here and consumed after phase A, so their latency
    // (HBM when the caller has flushed L2) hides behind the noise generation.
    float4 x0_in = make_float4(0.f, 0.f, 0.f, 0.f), g_in = x0_in;
    float ob_in[2][5] = {{0.f, 0.f, 1.f, 0.f, 0.f}, {0.f, 0.f, 1.f, 0.f, 0.f}};   // warp 0: obstacles lane, lane + 32
    float4 se_in[2] = {x0_in, x0_in};                                          // warp 0: super-ellipse `lane`
    int n_obs_in = 0, n_se_in = 0;
    if (new_scene) {
      x0_in = reinterpret_cast<const float4*>(P.state)[scene];
      n_obs_in = P.n_obs[scene];
      if (warp == kTableWarp) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int i = lane + 32 * h;
          if (i < P.max_obstacles) {
            const float* ob = P.obstacles + ((size_t)scene * P.max_obstacles + i) * 5;
#pragma unroll
            for (int q = 0; q < 5; ++q) ob_in[h][q] = ob[q];
          }
        }
        if (P.max_superellipses > 0) {
          n_se_in = P.n_se[scene];
          if (lane < P.max_superellipses) {
            const float4* q = reinterpret_cast<const float4*>(P.se + ((size_t)scene * P.max_superellipses + lane) * 8);
            se_in[0] = q[0]; se_in[1] = q[1];
          }
        }
      }
      if (tid == 0) g_in = reinterpret_cast<const float4*>(P.goal)[scene];
    }

    BRMPPI_STAMP(0)
    // ---- phase A: noise, perturb + clamp (a1, a2) ---------------------------------------------
    {
      const int TS = P.t_stride, T = P.T;
      const int R = kCtaThreads / S;
      const uint32_t n = *P.counter;
      const uint32_t key0 = P.key0 + (uint32_t)scene;
      const uint32_t key1 = P.key1 + (key0 < P.key0 ? 1u : 0u);
      const float2* Unom = reinterpret_cast<const float2*>(P.U) + (size_t)scene * T;   // read-only here
      // items (sample si, step pair mi) dealt round-robin over all 512 threads: item = tid,
      // tid + 512, ...; (si, mi) = (item % S, item / S) kept up to date incrementally
      float* planes = BRMPPI_SMEM(float, P.off_planes);
      const int n_pairs = (T + 1) >> 1;
      // On a tile that starts a scene the table warp writes the obstacle tables instead (below), and
      // the other 480 threads share the items.
      const int n_noise = new_scene ? kCtaThreads - 32 : kCtaThreads;
      const int nid = (new_scene && warp > kTableWarp) ? tid - 32 : tid;
      const int ds = n_noise % S, dm = n_noise / S;
      const int k0 = k - s;                                  // sample index of the tile's first sample
      int mi = nid / S, si = nid - mi * S;
      if (new_scene && warp == kTableWarp) mi = n_pairs;
      (void)R;
#pragma unroll 2
      for (; mi < n_pairs; ) {
        const int t = 2 * mi, t1 = min(t + 1, T - 1);
        float2 u0, u1;
        sample_control_pair<PRECISE>(P, __ldg(Unom + t), __ldg(Unom + t1), (uint32_t)mi, n, (uint32_t)(k0 + si + P.k_offset), key0, key1, &u0, &u1);
        float* pV = planes + si * TS;
        float* pD = pV + S * TS;
        float* pP1 = pD + S * TS;
        pV[t] = u0.x; pD[t] = u0.y;
        pP1[t + 1] = (P.dt * u0.x) * P.inv_L1 * tan_t<PRECISE>(u0.y);       // dpsi1 of step t, parked at t+1
        if (t + 1 < T) {
          pV[t + 1] = u1.x; pD[t + 1] = u1.y;
          pP1[t + 2] = (P.dt * u1.x) * P.inv_L1 * tan_t<PRECISE>(u1.y);
        }
        si += ds; mi += dm;
        if (si >= S) { si -= S; ++mi; }
      }
      if (c == 0) BRMPPI_SMEM(float, P.off_alpha)[s] = sample_alpha(P, n, (uint32_t)(k + P.k_offset), key0, key1);
    }
    if (new_scene && warp == kTableWarp) {
      // The scene's obstacle tables, by the one warp that generates no noise on this tile.
      CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
      // obstacle table for phase C, in the vehicle-centred frame, ordered by how close an obstacle is
      // to its culling threshold at the start state (the obstacles a chunk has to evaluate are then
      // mostly the first pairs of the table), null padding behind.
      // Obstacles 2p and 2p+1 are interleaved field by field -- (-ox, -ox'), (-oy, -oy'),
      // (-1/(2 rho^2), ..), (-rho^2, ..); velocities (-dt vx, ..), (-dt vy, ..) -- so that phase C
      // loads each pair of fields as one packed f32x2 operand.
      // Lane l holds obstacles l and l + 32 in registers and ranks them by counting over shuffles.
      //
      // Culling thresholds: with Dl the largest change of the centre distance per
      // step and d_crit(alpha) = (Dl + sqrt((1 - alpha) Dl^2 + alpha^2 rho^2)) / alpha, largest at
      // alpha_lo, the pair (obstacle, disc) has all its hinge terms exactly 0 over a chunk of L steps
      // when it starts at distance d0 >= L Dl + 1.02 d_crit + 0.05, i.e. g0 = d0^2 - rho^2 >= thr.
      float4* sObs = BRMPPI_SMEM(float4, P.off_obs);
      float2* sVel = BRMPPI_SMEM(float2, P.off_vel);
      float* sThr = BRMPPI_SMEM(float, P.off_thr);
      const int n_obs = n_obs_in;
      const float a_lo = P.alpha_lo;
      const float steps = (float)P.chunk_len;
      // (sort keys and thresholds only have to be on the safe side, not exact: MUFU approximations,
      // with their 1e-6 relative error covered by the 1.00001 factors)
      float dcx[kMaxDiscs], dcy[kMaxDiscs];                // disc centres at the start state
      {
        const float s1 = fast_sin(x0_in.z), c1 = fast_cos(x0_in.z), s2 = fast_sin(x0_in.w), c2 = fast_cos(x0_in.w);
#pragma unroll
        for (int j = 0; j < kMaxDiscs; ++j) {
          dcx[j] = fmaf(P.disc_a1[j], c1, fmaf(P.disc_a2[j], c2, -P.Lh * c1));
          dcy[j] = fmaf(P.disc_a1[j], s1, fmaf(P.disc_a2[j], s2, -P.Lh * s1));
        }
      }
      const float inv_a_lo = a_lo > 0.0f ? 1.00001f * fast_rcp(a_lo) : 0.0f;
      bool val[2], mov[2];
      float key[2], th[2][kMaxDiscs];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        val[h] = lane + 32 * h < n_obs;
        mov[h] = val[h] && (ob_in[h][3] != 0.0f || ob_in[h][4] != 0.0f);
        const float ox = ob_in[h][0] - x0_in.x, oy = ob_in[h][1] - x0_in.y;
        const float rho = ob_in[h][2] + P.disc_radius;
        // obstacle displacement per step, rounded up
        const float spd = 1.0001f * P.dt * fast_sqrt(fmaf(ob_in[h][3], ob_in[h][3], ob_in[h][4] * ob_in[h][4]));
        key[h] = CUDART_INF_F;
#pragma unroll
        for (int j = 0; j < kMaxDiscs; ++j) {
          float t = CUDART_INF_F;
          if (a_lo > 0.0f) {
            const float dl = fmaf(P.dt, P.disc_speed[j], spd);
            const float d_crit = (dl + 1.00001f * fast_sqrt(fmaf((1.0f - a_lo) * dl, dl, a_lo * a_lo * rho * rho))) * inv_a_lo;
            const float r_cull = fmaf(steps, dl, fmaf(1.02f, d_crit, 0.05f));
            t = fmaf(1.00001f * r_cull, r_cull, -(rho * rho));
          }
          th[h][j] = t;
          if (j < P.n_discs) {
            const float ex = dcx[j] - ox, ey = dcy[j] - oy;
            const float margin = fmaf(ex, ex, fmaf(ey, ey, -(rho * rho))) - t;
            key[h] = fminf(key[h], a_lo > 0.0f ? margin : fmaf(ex, ex, ey * ey));
          }
        }
      }
      int rank[2] = {0, 0};
      for (int j = 0; j < n_obs; ++j) {
        const float kj = __shfl_sync(0xffffffffu, (j >> 5) ? key[1] : key[0], j & 31);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int i = lane + 32 * h;
          rank[h] += (kj < key[h] || (kj == key[h] && j < i)) ? 1 : 0;   // j sorts before i
        }
      }
      unsigned moving_groups = 0u;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        if (val[h]) {
          const int dst = rank[h];
          const float rho = ob_in[h][2] + P.disc_radius;
          float* ob = reinterpret_cast<float*>(sObs) + (dst >> 1) * 8 + (dst & 1);
          ob[0] = -(ob_in[h][0] - x0_in.x);
          ob[2] = -(ob_in[h][1] - x0_in.y);
          ob[4] = -(0.5f / (rho * rho));                 // -1 / (2 rho^2): the hinge is formed as zn - |zn| = 2 min(0, zn)
          ob[6] = -(rho * rho);
          float* vl = reinterpret_cast<float*>(sVel) + (dst >> 1) * 4 + (dst & 1);
          vl[0] = -(P.dt * ob_in[h][3]);
          vl[2] = -(P.dt * ob_in[h][4]);
#pragma unroll
          for (int j = 0; j < kMaxDiscs; ++j) sThr[dst * kMaxDiscs + j] = th[h][j];
          if (mov[h]) moving_groups |= 1u << (dst / kObsGroup);
        }
      }
      moving_groups = __reduce_or_sync(0xffffffffu, moving_groups);
      for (int i = n_obs + lane; i < P.obs_padded; i += 32) {   // null obstacles: weight 0, never "near"
        float* ob = reinterpret_cast<float*>(sObs) + (i >> 1) * 8 + (i & 1);
        ob[0] = 0.0f; ob[2] = 0.0f; ob[4] = 0.0f; ob[6] = 0.0f;
        float* vl = reinterpret_cast<float*>(sVel) + (i >> 1) * 4 + (i & 1);
        vl[0] = 0.0f; vl[2] = 0.0f;
#pragma unroll
        for (int j = 0; j < kMaxDiscs; ++j) sThr[i * kMaxDiscs + j] = -CUDART_INF_F;
      }
      // super-ellipse table: rows of R(-theta) over the inflated semi-axes; null records weigh 0
      const int n_se = n_se_in;
      SeRecord* sSE = BRMPPI_SMEM(SeRecord, P.off_se);
      if (lane < P.se_padded) {
        SeRecord r = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (lane < n_se) {
          float st, ct;
          sincosf(se_in[1].x, &st, &ct);
          const float iax = 1.0f / (se_in[0].z + P.disc_radius), iay = 1.0f / (se_in[0].w + P.disc_radius);
          r.ox = se_in[0].x - x0_in.x; r.oy = se_in[0].y - x0_in.y;
          r.a11 = ct * iax; r.a12 = st * iax; r.a21 = -st * iay; r.a22 = ct * iay;
          r.wx = P.dt * se_in[1].y; r.wy = P.dt * se_in[1].z;
          r.e4 = se_in[1].w == 4.0f ? 1.0f : 0.0f;
          r.half_w = 0.5f;
        }
        sSE[lane] = r;
      }
      if (lane == 0) {
        sM->moving_groups = moving_groups;
        sM->n_groups = n_obs > 0 ? (n_obs + kObsGroup - 1) / kObsGroup : 1;
        sM->n_se_groups = (n_se + kSeGroup - 1) / kSeGroup;
      }
    }
    if (new_scene) {
      CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
      float* sA = BRMPPI_SMEM(float, P.off_A);
      for (int i = tid; i < 2 * P.T; i += kCtaThreads) sA[i] = 0.0f;
      if (tid == 0) {
        g_in.x -= x0_in.x; g_in.y -= x0_in.y;          // vehicle-centred frame
        sM->x0 = x0_in;
        sM->g = g_in;
        sM->n_obs = n_obs_in;
        sM->m[0] = CUDART_INF; sM->argmin[0] = 0x7fffffff; sM->eta[0] = 0.0f; sM->w2[0] = 0.0f; sM->nonfinite[0] = 0;
      }
    }
    __syncthreads();
    BRMPPI_STAMP(1)

    // ---- phase B: serial Euler chain of eq. (6), one sample per thread (a3), on the CTA's LAST four
    //      warps -- one per scheduler, and the ones the arbiter prefers (highest warp id first), so
    //      the in-order chain keeps its issue slots while the cost threads of the chunks already
    //      handed over run underneath it.  Only the psi2 recursion is a true chain; the thread also
    //      integrates psi1, x, y (short independent dependency chains that fill its issue
    //      bubbles).  After every chunk of L steps the chain threads arrive on bar_chunk[chunk]. ---
    const int k0 = k - s;                                    // sample index of the tile's first sample
    if (warp >= kCtaWarps - kChainWarps) {
      CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
      const int sc = tid - kChainFirstThread;
      const int n_handoff = P.chunks - 1;                    // the last chunk stays with the chain threads
      if (sc < S) {
        const int TS = P.t_stride, T = P.T, L = P.chunk_len;
        const float* pV = BRMPPI_SMEM(float, P.off_planes) + sc * TS;
        float* pP1 = BRMPPI_SMEM(float, P.off_planes) + (2 * S + sc) * TS;
        float* pP2 = pP1 + S * TS;
        float2* sXY = BRMPPI_SMEM(float2, P.off_xy);        // [C][S] chunk-start (x, y)
        const float4 x0 = sM->x0;
        float x = 0.0f, y = 0.0f, psi1 = x0.z, psi2 = x0.w;
        pP1[0] = psi1;
        pP2[0] = psi2;
        const float* pD = pV + S * TS;
        float effort = 0.0f;                                   // w_v v^2 + w_delta delta^2 summed over the horizon
        float v = pV[0], b = pP1[1];
        const long long t_chain = (P.phase_ns != nullptr && sc == 0) ? clock64() : 0ll;
        for (int cc = 0, t = 0; t < T; ++cc) {
          sXY[cc * S + sc] = make_float2(x, y);
          const int te = min(t + L, T);
          for (; t < te; ++t) {
            // next step's inputs first: the loads do not wait behind this step's stores
            const int tn = min(t + 1, T - 1);
            const float v_next = pV[tn], b_next = pP1[tn + 1];
            const float d = pD[t];
            effort = fmaf(P.w_v * v, v, fmaf(P.w_delta * d, d, effort));
            const float a = P.dt * v;
            float s1, c1, sb, cb;
            sincos_t<PRECISE>(psi1 - psi2, &sb, &cb);
            sincos_t<PRECISE>(psi1, &s1, &c1);
            x = fmaf(a, c1, x);
            y = fmaf(a, s1, y);
            psi1 += b;
            psi2 = fmaf(a * P.inv_L2, sb, fmaf(-(b * P.Lh_over_L2), cb, psi2));
            pP1[t + 1] = psi1;
            pP2[t + 1] = psi2;
            v = v_next; b = b_next;
          }
          if (cc < n_handoff) mbar_arrive(smem_addr(&sM->bar_chunk[cc]));
        }
        sXY[P.chunks * S + sc] = make_float2(x, y);   // x_T
        BRMPPI_SMEM(float, P.off_scratch)[sc] = effort;
        if (P.phase_ns != nullptr && sc == 0) sM->phase_acc[kChainSlot] += (unsigned long long)(clock64() - t_chain);
      } else {
        for (int cc = 0; cc < n_handoff; ++cc) mbar_arrive(smem_addr(&sM->bar_chunk[cc]));
      }
    }

    // ---- phase C: barrier, barrier-rate hinge, goal / heading / hitch cost (a4-a6).  Worker thread
    //      (chunk, sample) = (tid / S, tid % S) takes chunks 0 .. C-2 as soon as the chain has handed
    //      the chunk over; the chain thread of a sample takes its last chunk. -------------------------
    int cq = -1, sq = 0;
    {
      const int n_worker_items = (P.chunks - 1) * S;
      if (tid < n_worker_items) { cq = c; sq = s; }
      else if (tid >= kChainFirstThread && tid - kChainFirstThread < S) { cq = P.chunks - 1; sq = tid - kChainFirstThread; }
      if (cq >= 0) {
        CtaMisc* sMb = BRMPPI_SMEM(CtaMisc, P.off_misc);
        if (tid < n_worker_items) {   // warp-uniform: the latest chunk any lane of this warp works on
          const int last = min((warp << 5) + 31, n_worker_items - 1);
          mbar_wait(smem_addr(&sMb->bar_chunk[last / S]), tile_parity);
        }
      }
    }
    if (cq >= 0) {
      const int c = cq, s = sq, k = k0 + sq;     // this thread's (chunk, sample in tile, sample index)
      const int TS = P.t_stride, T = P.T;
      const int t0 = c * P.chunk_len, t1 = min(t0 + P.chunk_len, T);
      const CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
      const float* pV = BRMPPI_SMEM(float, P.off_planes) + s * TS;
      const float* pP1 = pV + 2 * S * TS;
      const float* pP2 = pP1 + S * TS;
      const float4* sObs = BRMPPI_SMEM(float4, P.off_obs);
      const float2* sVel = BRMPPI_SMEM(float2, P.off_vel);
      const float one_minus_alpha = 1.0f - BRMPPI_SMEM(float, P.off_alpha)[s];
      const float4 g = sM->g;
      const unsigned moving_groups = sM->moving_groups;
      const int n_groups = sM->n_groups;
      const float2 xy = BRMPPI_SMEM(float2, P.off_xy)[c * S + s];
      double track = 0.0, bar = 0.0;
      const int n_se_groups = sM->n_se_groups;
      const SeRecord* sSE = BRMPPI_SMEM(SeRecord, P.off_se);
      if (sM->n_obs == 0 && n_se_groups > 0) {
        // no disc obstacles: the first super-ellipse group carries the stage cost
        const GroupCost gc = se_group<PRECISE, ND, true>(P, pV, pP1, pP2, sSE, xy.x, xy.y, t0, t1, one_minus_alpha, g);
        track = gc.track; bar = gc.bar;
        for (int grp = 1; grp < n_se_groups; ++grp)
          bar += se_group<PRECISE, ND, false>(P, pV, pP1, pP2, sSE + grp * kSeGroup, xy.x, xy.y, t0, t1, one_minus_alpha, g).bar;
      } else {
        const float* sThr = BRMPPI_SMEM(float, P.off_thr);
        const GroupCost gc = barrier_group_mv<PRECISE, ND, true>((moving_groups & 1u) != 0u, P, pV, pP1, pP2, sObs, sVel, sThr, xy.x, xy.y, t0, t1, one_minus_alpha, g);
        track = gc.track; bar = gc.bar;
        for (int grp = 1; grp < n_groups; ++grp) {
          const int ib = grp * kObsGroup;
          bar += barrier_group_mv<PRECISE, ND, false>(((moving_groups >> grp) & 1u) != 0u, P, pV, pP1, pP2, sObs + ib, sVel + ib, sThr + ib * kMaxDiscs, xy.x, xy.y, t0, t1, one_minus_alpha, g).bar;
        }
        for (int grp = 0; grp < n_se_groups; ++grp)
          bar += se_group<PRECISE, ND, false>(P, pV, pP1, pP2, sSE + grp * kSeGroup, xy.x, xy.y, t0, t1, one_minus_alpha, g).bar;
      }
      if (t1 == T) {   // terminal cost r_N(x_N), eq. (7); final state out
        const float2 xT = BRMPPI_SMEM(float2, P.off_xy)[P.chunks * S + s];
        const State X{xT.x, xT.y, pP1[T], pP2[T]};
        track += (double)(P.w_term * goal_cost(P, X, g));
        if ((P.flags & BRMPPI_FLAG_WRITE_SAMPLES) && k < P.K) {
          const float4 x0 = sM->x0;
          reinterpret_cast<float4*>(P.XT)[(size_t)scene * P.K + k] = make_float4(X.x + x0.x, X.y + x0.y, X.psi1, X.psi2);
        }
      }
      BRMPPI_SMEM(double, P.off_cost)[c * S + s] = track + (double)P.w_bar * bar;
    }
    __syncthreads();
    BRMPPI_STAMP(3)

    // ---- phase D: tile reduction against the running online-softmax state (a7) --------------
    double Sk = CUDART_INF;
    bool valid = false, finite = false;
    if (warp < kChainWarps) {
      CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
      valid = (tid < S) && (k < P.K);
      if (valid) {
        const double* sCost = BRMPPI_SMEM(double, P.off_cost);
        Sk = (double)BRMPPI_SMEM(float, P.off_scratch)[s];                   // effort, from the chain
        for (int cc = 0; cc < P.chunks; ++cc) Sk += sCost[cc * S + s];
        if (P.flags & BRMPPI_FLAG_WRITE_SAMPLES) P.S[(size_t)scene * P.K + k] = (float)Sk;
      }
      finite = valid && (Sk == Sk) && (Sk < CUDART_INF) && (Sk > -CUDART_INF);
      double m = finite ? Sk : CUDART_INF;
      int idx = finite ? k + P.k_offset : 0x7fffffff;     // global sample index (K-sharded solves)
      warp_argmin(m, idx);
      if (lane == 0) { sM->redM[warp] = m; sM->redI[warp] = idx; }
    }
    __syncthreads();
    float scale_old;
    {
      // every thread folds the four warp minima and the running minimum the same way
      CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
      double m_new = sM->m[par];
      int idx_new = sM->argmin[par];
      const double m_old = m_new;
#pragma unroll
      for (int w = 0; w < kChainWarps; ++w) {
        const double mw = sM->redM[w];
        const int iw = sM->redI[w];
        if (mw < m_new || (mw == m_new && iw < idx_new)) { m_new = mw; idx_new = iw; }
      }
      scale_old = (m_old < CUDART_INF) ? expf((float)(-(m_old - m_new) * (double)P.inv_lambda)) : 0.0f;
      if (warp < kChainWarps) {
        // S - m in fp64, then fp32 exp (SURVEY §7 hard part 2)
        const float w = finite ? expf((float)(-(Sk - m_new) * (double)P.inv_lambda)) : 0.0f;
        if (tid < S) BRMPPI_SMEM(float, P.off_w)[tid] = w;
        const float eta_w = warp_sum(w), w2_w = warp_sum(w * w);
        const float nf_w = warp_sum((valid && !finite) ? 1.0f : 0.0f);
        if (lane == 0) { sM->redF[0][warp] = eta_w; sM->redF[1][warp] = w2_w; sM->redF[2][warp] = nf_w; }
      }
      if (tid == 0) { sM->m[par ^ 1] = m_new; sM->argmin[par ^ 1] = idx_new; }
    }
    __syncthreads();
    BRMPPI_STAMP(4)

    // ---- phase E: running weighted control sums A[t] (a7) -----------------------------------
    {
      const int TS = P.t_stride, T = P.T;
      CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
      if (tid == 0) {
        float eta_t = 0.0f, w2_t = 0.0f, nf_t = 0.0f;
#pragma unroll
        for (int w = 0; w < kChainWarps; ++w) { eta_t += sM->redF[0][w]; w2_t += sM->redF[1][w]; nf_t += sM->redF[2][w]; }
        sM->eta[par ^ 1] = fmaf(sM->eta[par], scale_old, eta_t);
        sM->w2[par ^ 1] = fmaf(sM->w2[par], scale_old * scale_old, w2_t);
        sM->nonfinite[par ^ 1] = sM->nonfinite[par] + (int)nf_t;
      }
      float* sA = BRMPPI_SMEM(float, P.off_A);
      const float* sW = BRMPPI_SMEM(float, P.off_w);
      const float* sV = BRMPPI_SMEM(float, P.off_planes);
      const int n_out = 2 * T;
      if (n_out * 2 <= kCtaThreads) {
        // G threads per output, each over the samples s = g, g + G, ...; fixed-order combine
        float* sScr = BRMPPI_SMEM(float, P.off_scratch);
        const int G = kCtaThreads / n_out;
        const int g = tid / n_out, o = tid - g * n_out;
        if (g < G) {
          const int ch = o >= T ? 1 : 0, t = o - ch * T;
          const float* plane = sV + ch * S * TS + t;
          // four independent partial sums: the shared-memory loads of consecutive samples overlap
          float a0 = 0.0f, a1 = 0.0f, a2 = 0.0f, a3 = 0.0f;
          int ss = g;
          for (; ss + 3 * G < S; ss += 4 * G) {
            a0 = fmaf(sW[ss], plane[ss * TS], a0);
            a1 = fmaf(sW[ss + G], plane[(ss + G) * TS], a1);
            a2 = fmaf(sW[ss + 2 * G], plane[(ss + 2 * G) * TS], a2);
            a3 = fmaf(sW[ss + 3 * G], plane[(ss + 3 * G) * TS], a3);
          }
          for (; ss < S; ss += G) a0 = fmaf(sW[ss], plane[ss * TS], a0);
          sScr[tid] = (a0 + a1) + (a2 + a3);
        }
        __syncthreads();
        if (tid < n_out) {
          float acc = 0.0f;
          for (int gg = 0; gg < G; ++gg) acc += sScr[gg * n_out + tid];
          sA[tid] = fmaf(sA[tid], scale_old, acc);
        }
      } else {
        for (int o = tid; o < n_out; o += kCtaThreads) {
          const int ch = o >= T ? 1 : 0, t = o - ch * T;
          const float* plane = sV + ch * S * TS + t;
          float acc = 0.0f;
          for (int ss = 0; ss < S; ++ss) acc = fmaf(sW[ss], plane[ss * TS], acc);
          sA[o] = fmaf(sA[o], scale_old, acc);
        }
      }
    }
    par ^= 1;
    tile_parity ^= 1u;
    __syncthreads();
    BRMPPI_STAMP(5)
  }

  // ---- partial of the last scene -> HBM -----------------------------------------------------
  if (cur_scene >= 0) {
    const int Pn = P.n_partials, T = P.T;
    const CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
    const float* sA = BRMPPI_SMEM(float, P.off_A);
    const int slot = blockIdx.x - (cur_scene * P.tiles_per_scene) / P.tiles_per_cta;
    const size_t pbase = (size_t)cur_scene * Pn + slot;
    if (tid == 0) {
      P.part_m[pbase] = sM->m[par];
      P.part_argmin[pbase] = sM->argmin[par];
      P.part_eta[pbase] = sM->eta[par];
      P.part_w2[pbase] = sM->w2[par];
      P.part_nonfinite[pbase] = sM->nonfinite[par];
    }
    for (int o = tid; o < 2 * T; o += kCtaThreads) {
      const int ch = o >= T ? 1 : 0, t = o - ch * T;
      P.part_A[((size_t)cur_scene * 2 * T + (2 * t + ch)) * Pn + slot] = sA[o];
    }
  }
  if (P.phase_ns != nullptr && tid == 0) {
    const CtaMisc* sM = BRMPPI_SMEM(CtaMisc, P.off_misc);
    const unsigned long long now = (unsigned long long)clock64();
    unsigned long long* out = P.phase_ns + (size_t)blockIdx.x * (kPhaseSlots + 2);
    for (int i = 0; i < kPhaseSlots; ++i) out[i] = sM->phase_acc[i];
    out[6] += now - t_stamp;            // partial to HBM
    out[kPhaseSlots] = sM->t_begin;
    out[kPhaseSlots + 1] = global_ns();
  }
}

#undef BRMPPI_STAMP
#undef BRMPPI_SMEM

using CtaKernel = void (*)(const DeviceParams);

inline CtaKernel cta_kernel_for(bool precise, int n_discs) {
  switch (n_discs * 2 + (precise ? 1 : 0)) {
    case 2: return rollout_cta<false, 1>;
    case 3: return rollout_cta<true, 1>;
    case 4: return rollout_cta<false, 2>;
    case 5: return rollout_cta<true, 2>;
    case 6: return rollout_cta<false, 3>;
    case 7: return rollout_cta<true, 3>;
    case 8: return rollout_cta<false, 4>;
    default: return rollout_cta<true, 4>;
  }
}

// The dynamic shared-memory limit is an attribute of the FUNCTION on a device, not of a context: it is
// always raised to the opt-in maximum, so that a second context with a smaller tile never lowers it
// under a live one.
inline cudaError_t configure_rollout_cta(bool precise, int n_discs, size_t smem_bytes) {
  if (smem_bytes > kSmemMax) return cudaErrorInvalidValue;
  cudaError_t e = cudaFuncSetAttribute(cta_kernel_for(precise, n_discs),
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
  if (e != cudaSuccess) return e;
  // the kernel streams almost nothing through L1: ask for the full shared-memory carve-out
  return cudaFuncSetAttribute(cta_kernel_for(precise, n_discs),
                              cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}

inline cudaError_t launch_rollout_cta(const DeviceParams& d, const CtaPlan& pl, bool precise,
                                      cudaStream_t stream) {
  cta_kernel_for(precise, d.n_discs)<<<(unsigned)pl.grid, kCtaThreads, pl.smem, stream>>>(d);
  return cudaGetLastError();
}

}  // namespace brmppi
