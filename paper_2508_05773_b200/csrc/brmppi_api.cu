// brmppi_api.cu -- host side of the C ABI declared in include/brmppi.h: validation, workspace
// layout, launches, CUDA-graph capture.  Every step of the hot path runs in the kernels included
// below; this file only marshals arguments and enqueues work.  There is no CPU fallback.
#include <cuda_runtime.h>
#include <math_constants.h>

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/brmppi.h"
#include "brmppi_device.cuh"
#include "peaks.cuh"
#include "rollout_thread.cuh"
#include "rollout_projected.cuh"
#include "rollout_mpcc.cuh"
#include "rollout_mpcc_cta.cuh"
#include "rollout_cta.cuh"
#include "rollout_cta_kernel.cuh"
#include "update.cuh"
#include "project.cuh"

using namespace brmppi;

namespace {

thread_local char g_errbuf[256];
thread_local cudaError_t g_last_cuda = cudaSuccess;

inline int cuda_fail(cudaError_t e) {
  g_last_cuda = e;
  return BRMPPI_ERR_CUDA;
}
#define CU(expr)                                         \
  do {                                                   \
    cudaError_t e__ = (expr);                            \
    if (e__ != cudaSuccess) return cuda_fail(e__);       \
  } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

bool finite_all(const float* v, int n) {
  for (int i = 0; i < n; ++i)
    if (!std::isfinite(v[i])) return false;
  return true;
}

bool hitch_params_valid(const brmppi_params* p) {
  const float f[] = {p->hitch_alpha, p->hitch_qv, p->hitch_qdelta, p->hitch_max, p->hitch_kappa};
  if (!finite_all(f, 5)) return false;
  return p->hitch_alpha > 0.f && p->hitch_alpha <= 1.f && p->hitch_qv > 0.f && p->hitch_qdelta > 0.f &&
         p->hitch_kappa >= 0.f;
}

bool params_valid(const brmppi_params* p) {
  if (!p) return false;
  if (p->K < 1 || p->K > (1 << 27)) return false;
  if (p->T < 1 || p->T > BRMPPI_MAX_T) return false;
  if (p->n_iter < 1 || p->n_scenes < 1 || p->n_scenes > 65535) return false;
  if ((long long)p->K * p->n_scenes > 0x7fffffffLL) return false;
  if (p->k_offset < 0 || (long long)p->k_offset + p->K > 0x7fffffffLL) return false;
  if (p->max_obstacles < 0 || p->max_obstacles > BRMPPI_MAX_OBSTACLES) return false;
  if (p->max_superellipses < 0 || p->max_superellipses > BRMPPI_MAX_SUPERELLIPSES) return false;
  if (p->max_superellipses > 0 && (p->flags & BRMPPI_FLAG_KERNEL_THREAD_PER_SAMPLE)) return false;   // default kernel only
  if (p->n_discs < 1 || p->n_discs > BRMPPI_MAX_DISCS) return false;
  for (int j = 0; j < p->n_discs; ++j) {
    if (p->discs[j].body != 0 && p->discs[j].body != 1) return false;
    if (!std::isfinite(p->discs[j].offset)) return false;
  }
  const float f[] = {p->disc_radius, p->dt, p->L1, p->L2, p->Lh, p->v_min, p->v_max, p->delta_min,
                     p->delta_max, p->sigma_v, p->sigma_delta, p->alpha_lo, p->alpha_hi, p->w_pos,
                     p->w_head, p->w_v, p->w_delta, p->w_hitch, p->hitch_max, p->w_bar, p->w_term,
                     p->lambda};
  if (!finite_all(f, (int)(sizeof(f) / sizeof(f[0])))) return false;
  if (!(p->dt > 0.f) || !(p->L1 > 0.f) || !(p->L2 > 0.f) || !(p->lambda > 0.f)) return false;
  if (p->disc_radius < 0.f || p->sigma_v < 0.f || p->sigma_delta < 0.f) return false;
  if (!std::isfinite(p->hitch_kappa) || p->hitch_kappa < 0.f) return false;
  if (p->hitch_filter != 0 && p->hitch_filter != 1) return false;
  if (p->hitch_filter && !hitch_params_valid(p)) return false;
  if (p->v_min > p->v_max || p->delta_min > p->delta_max) return false;
  if (p->delta_min <= -1.5f || p->delta_max >= 1.5f) return false;   // tan(delta) must stay finite
  if (p->alpha_lo > p->alpha_hi) return false;
  const unsigned known = BRMPPI_FLAG_WRITE_SAMPLES | BRMPPI_FLAG_PRECISE_MATH |
                         BRMPPI_FLAG_KERNEL_THREAD_PER_SAMPLE | BRMPPI_FLAG_PHASE_TIMING |
                         BRMPPI_FLAG_NO_CULL | BRMPPI_FLAG_PROJECTED | BRMPPI_FLAG_MPCC;
  if (p->flags & ~known) return false;
  if (p->flags & BRMPPI_FLAG_MPCC) {
    if ((p->flags & BRMPPI_FLAG_PROJECTED) || p->max_superellipses > 0 || p->hitch_filter) return false;
    if (p->max_path_segments < 1 || p->max_path_segments > BRMPPI_MAX_PATH_SEGMENTS) return false;
    const float q[] = {p->j_min, p->j_max, p->omega_min, p->omega_max, p->sigma_j, p->sigma_omega, p->Qc, p->Ql,
                       p->Qth1, p->Qth2, p->Rj, p->Rw, p->mu, p->nu_bar};
    if (!finite_all(q, 14)) return false;
    if (p->j_min > p->j_max || p->omega_min > p->omega_max || p->sigma_j < 0.f || p->sigma_omega < 0.f) return false;
  }
  if (p->flags & BRMPPI_FLAG_PROJECTED) {
    if (p->max_obstacles > BRMPPI_PROJECT_MAX_NO || p->max_superellipses > 0) return false;
    const float q[] = {p->proj_qv, p->proj_qomega, p->proj_qalpha, p->proj_rho, p->sigma_ualpha, p->ualpha_max,
                       p->w_alpha, p->h_buffer};
    if (!finite_all(q, 8)) return false;
    if (!(p->proj_qv > 0.f) || !(p->proj_qomega > 0.f) || !(p->proj_qalpha > 0.f)) return false;
    if (p->proj_rho < 0.f || p->sigma_ualpha < 0.f || p->ualpha_max < 0.f || p->w_alpha < 0.f) return false;
  }
  return true;
}

struct Layout {
  size_t state, goal, n_obs, obstacles, n_se, se, U, counter, u0, part_m, part_argmin, part_eta, part_w2,
      part_nf, part_A, diag, S, XT, phase, hitch, state7, path_M, path_dpsi, path_coef, total;
};

// Launch plan: which rollout kernel, how the sample axis is tiled, how many partials.
struct Plan {
  bool cta_kernel;
  bool mpcc_cta;          // BRMPPI_FLAG_MPCC without KERNEL_THREAD_PER_SAMPLE: the phase-split kernel of rollout_mpcc_cta.cuh
  int n_partials;
  CtaPlan cta;
  MpccCtaPlan mpcc;
};

// SM count of the current device (the persistent kernel launches one CTA per SM); 148 -- a B200 --
// when no device is visible, so that brmppi_workspace_bytes still answers on a CPU-only box.
int device_sm_count() {
  int dev = 0, n = 0;
  if (cudaGetDevice(&dev) == cudaSuccess &&
      cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
    return n;
  cudaGetLastError();
  return 148;
}

Plan make_plan(const brmppi_params& p) {
  Plan pl{};
  pl.cta_kernel = !(p.flags & (BRMPPI_FLAG_KERNEL_THREAD_PER_SAMPLE | BRMPPI_FLAG_PROJECTED | BRMPPI_FLAG_MPCC));
  pl.mpcc_cta = (p.flags & BRMPPI_FLAG_MPCC) && !(p.flags & BRMPPI_FLAG_KERNEL_THREAD_PER_SAMPLE);
  if (pl.cta_kernel) {
    pl.cta = make_cta_plan(p.K, p.T, p.n_scenes, p.max_obstacles, p.max_superellipses, device_sm_count());
    pl.n_partials = pl.cta.n_partials;
  } else if (pl.mpcc_cta) {
    pl.mpcc = make_mpcc_cta_plan(p.K, p.T, p.n_scenes, p.max_obstacles, p.max_path_segments, device_sm_count());
    pl.n_partials = pl.mpcc.tiles_per_scene;
  } else {
    pl.n_partials = (p.K + kThreadBlock - 1) / kThreadBlock;
  }
  return pl;
}

Layout make_layout(const brmppi_params& p, const Plan& pl) {
  Layout L{};
  size_t off = 0;
  const size_t ns = (size_t)p.n_scenes, P = (size_t)pl.n_partials, T = (size_t)p.T;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
  L.state = take(ns * 16);
  L.goal = take(ns * 16);
  L.n_obs = take(ns * 4);
  L.obstacles = take(ns * (size_t)(p.max_obstacles > 0 ? p.max_obstacles : 1) * 20);
  L.n_se = take(ns * 4);
  L.se = take(ns * (size_t)(p.max_superellipses > 0 ? p.max_superellipses : 1) * 32);
  L.U = take(ns * T * 8);
  L.counter = take(4);
  L.u0 = take(ns * 8);
  L.hitch = take(ns * 16);
  if (p.flags & BRMPPI_FLAG_MPCC) {
    L.state7 = take(ns * 32);
    L.path_M = take(ns * 4);
    L.path_dpsi = take(ns * 4);
    L.path_coef = take(ns * (size_t)p.max_path_segments * 64);
  }
  L.part_m = take(ns * P * 8);
  L.part_argmin = take(ns * P * 4);
  L.part_eta = take(ns * P * 4);
  L.part_w2 = take(ns * P * 4);
  L.part_nf = take(ns * P * 4);
  L.part_A = take(ns * 2 * T * P * 4);
  L.diag = take(ns * sizeof(brmppi_diag));
  if (p.flags & BRMPPI_FLAG_WRITE_SAMPLES) {
    L.S = take(ns * (size_t)p.K * 4);
    L.XT = take(ns * (size_t)p.K * ((p.flags & BRMPPI_FLAG_MPCC) ? 32 : 16));
  }
  if ((p.flags & BRMPPI_FLAG_PHASE_TIMING) && pl.cta_kernel)
    L.phase = take((size_t)pl.cta.grid * (kPhaseSlots + 2) * sizeof(unsigned long long));
  L.total = off;
  return L;
}

}  // namespace

struct brmppi_ctx {
  brmppi_params p;
  DeviceParams d;
  Plan plan;
  Layout layout;
  cudaStream_t stream;
  unsigned char* state_set;
  unsigned char* goal_set;
  unsigned long long launches;
  unsigned int n_host;          // host mirror of the device iteration counter
  cudaGraphExec_t solve_graph, step_graph, solve_host_graph, solve_io_graph;
  float* pinned_u0;             // [n_scenes][2] staging for brmppi_step
  float* pinned_U;              // [n_scenes][T][2] page-locked host copy of U that the last merge_update of
  float* pinned_U_dev;          //   brmppi_solve_get_controls writes (device address of the same memory)
  float* path_len;              // [n_scenes] M dpsi of the reference path (BRMPPI_FLAG_MPCC), host
  unsigned char* pinned_in[2];  // single-scene contexts: page-locked images of the workspace's input span
  cudaEvent_t pinned_in_done[2];//   (state .. obstacles), used in turn by brmppi_set_inputs
  int pinned_in_next;
  size_t smem_rollout, smem_update;
};

namespace {

int launch_rollout(brmppi_ctx* c) {
  const DeviceParams& d = c->d;
  const bool precise = (c->p.flags & BRMPPI_FLAG_PRECISE_MATH) != 0;
  if (c->plan.cta_kernel) {
    CU(launch_rollout_cta(d, c->plan.cta, precise, c->stream));
  } else if (c->plan.mpcc_cta) {
    mpcc_cta_kernel_for(precise, d.n_discs, !(c->p.flags & BRMPPI_FLAG_NO_CULL))<<<(unsigned)c->plan.mpcc.grid, kMpccThreads, c->smem_rollout, c->stream>>>(d);
    CU(cudaGetLastError());
  } else if (c->p.flags & BRMPPI_FLAG_MPCC) {
    dim3 grid((unsigned)c->plan.n_partials, (unsigned)d.n_scenes);
    if (precise)
      rollout_mpcc<true><<<grid, kThreadBlock, c->smem_rollout, c->stream>>>(d);
    else
      rollout_mpcc<false><<<grid, kThreadBlock, c->smem_rollout, c->stream>>>(d);
    CU(cudaGetLastError());
  } else if (c->p.flags & BRMPPI_FLAG_PROJECTED) {
    dim3 grid((unsigned)c->plan.n_partials, (unsigned)d.n_scenes);
    projected_kernel_for(precise, d.max_obstacles, d.n_discs)<<<grid, kThreadBlock, c->smem_rollout, c->stream>>>(d);
    CU(cudaGetLastError());
  } else {
    dim3 grid((unsigned)c->plan.n_partials, (unsigned)d.n_scenes);
    if (precise)
      rollout_thread_per_sample<true><<<grid, kThreadBlock, c->smem_rollout, c->stream>>>(d);
    else
      rollout_thread_per_sample<false><<<grid, kThreadBlock, c->smem_rollout, c->stream>>>(d);
    CU(cudaGetLastError());
  }
  return BRMPPI_OK;
}

// to_host: the update also writes the new nominal into the context's page-locked host copy of U
int launch_update(brmppi_ctx* c, bool to_host = false) {
  DeviceParams d = c->d;
  d.U_host = to_host ? c->pinned_U_dev : nullptr;
  dim3 ugrid((unsigned)((2 * d.T + kUpdateOutputsPerBlock - 1) / kUpdateOutputsPerBlock),
             (unsigned)d.n_scenes);
  merge_update<kMergeLocal><<<ugrid, kUpdateBlock, c->smem_update, c->stream>>>(d, nullptr, 0);
  CU(cudaGetLastError());
  return BRMPPI_OK;
}

int enqueue_iteration(brmppi_ctx* c, bool to_host = false) {
  int r = launch_rollout(c);
  if (r) return r;
  return launch_update(c, to_host);
}

// to_host: the LAST iteration's update leaves the result in page-locked host memory as well
int enqueue_solve(brmppi_ctx* c, bool to_host = false) {
  for (int it = 0; it < c->p.n_iter; ++it) {
    int r = enqueue_iteration(c, to_host && it == c->p.n_iter - 1);
    if (r) return r;
  }
  return BRMPPI_OK;
}

int ready(const brmppi_ctx* c) {
  for (int s = 0; s < c->p.n_scenes; ++s)
    if (!c->state_set[s] || !c->goal_set[s]) return BRMPPI_ERR_NOT_READY;
  return BRMPPI_OK;
}

template <class F>
int capture(brmppi_ctx* c, cudaGraphExec_t* exec, F&& body) {
  cudaGraph_t graph = nullptr;
  CU(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
  int r = body();
  cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
  if (r) { if (graph) cudaGraphDestroy(graph); return r; }
  if (e != cudaSuccess) return cuda_fail(e);
  e = cudaGraphInstantiate(exec, graph, 0);
  cudaGraphDestroy(graph);
  if (e != cudaSuccess) return cuda_fail(e);
  return BRMPPI_OK;
}

}  // namespace

// Static device scratch of brmppi_hitch_filter_static (include/brmppi.h): staging for at most
// BRMPPI_HITCH_STATIC_MAX_N problems, 36 bytes each.  In host code the name g_hitch_static is a host-side stand-in,
// not a device address: the address comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_hitch_static[(size_t)BRMPPI_HITCH_STATIC_MAX_N * 36];

namespace {
constexpr int kStaticMaxDevices = 64;
std::atomic<unsigned char*> g_hitch_static_addr[kStaticMaxDevices];

int hitch_static_address(unsigned char** out) {
  int dev = 0;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) return BRMPPI_ERR_INVALID_ARG;
  unsigned char* ptr = g_hitch_static_addr[dev].load(std::memory_order_acquire);
  if (!ptr) {
    CU(cudaGetSymbolAddress((void**)&ptr, g_hitch_static));
    if (!ptr) return BRMPPI_ERR_NULL;
    g_hitch_static_addr[dev].store(ptr, std::memory_order_release);   // the same value from any thread
  }
  *out = ptr;
  return BRMPPI_OK;
}
}  // namespace

template <int KIND>
static cudaError_t launch_peak(int blocks, cudaStream_t s, long long* spans, float* sink) {
  peak_kernel<KIND><<<blocks, 256, 0, s>>>(1.0f, spans, sink);
  return cudaGetLastError();
}

extern "C" {

size_t brmppi_workspace_bytes(const brmppi_params* p) {
  if (!params_valid(p)) return 0;
  return make_layout(*p, make_plan(*p)).total;
}

int brmppi_create(const brmppi_params* p, void* dev_workspace, size_t workspace_bytes,
                  void* cuda_stream, brmppi_ctx** out) {
  if (!p || !dev_workspace || !out) return BRMPPI_ERR_NULL;
  *out = nullptr;
  if (!params_valid(p)) return BRMPPI_ERR_INVALID_ARG;
  if ((uintptr_t)dev_workspace % 256 != 0) return BRMPPI_ERR_UNALIGNED;
  int dev = 0;
  CU(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  CU(cudaGetDeviceProperties(&prop, dev));

  brmppi_ctx* c = new (std::nothrow) brmppi_ctx();
  if (!c) return BRMPPI_ERR_NULL;
  c->p = *p;
  c->plan = make_plan(*p);
  c->layout = make_layout(*p, c->plan);
  if (workspace_bytes < c->layout.total) { delete c; return BRMPPI_ERR_WORKSPACE_TOO_SMALL; }
  c->stream = (cudaStream_t)cuda_stream;
  c->state_set = (unsigned char*)calloc((size_t)p->n_scenes, 1);
  c->goal_set = (unsigned char*)calloc((size_t)p->n_scenes, 1);
  c->launches = 0;
  c->n_host = 0;
  c->solve_graph = nullptr;
  c->step_graph = nullptr;
  c->solve_host_graph = nullptr;
  c->solve_io_graph = nullptr;
  c->pinned_u0 = nullptr;
  c->pinned_U = nullptr;
  c->pinned_U_dev = nullptr;
  c->path_len = (float*)calloc((size_t)p->n_scenes, sizeof(float));
  c->pinned_in[0] = c->pinned_in[1] = nullptr;
  c->pinned_in_done[0] = c->pinned_in_done[1] = nullptr;
  c->pinned_in_next = 0;

  DeviceParams& d = c->d;
  memset(&d, 0, sizeof(d));
  d.K = p->K; d.T = p->T; d.n_scenes = p->n_scenes; d.max_obstacles = p->max_obstacles;
  d.n_discs = p->n_discs; d.k_offset = p->k_offset;
  for (int j = 0; j < p->n_discs; ++j) {
    d.disc_body[j] = p->discs[j].body; d.disc_offset[j] = p->discs[j].offset;
    d.disc_a1[j] = p->discs[j].body == 0 ? p->discs[j].offset : 0.0f;
    d.disc_a2[j] = p->discs[j].body == 0 ? 0.0f : p->discs[j].offset;
  }
  d.disc_radius = p->disc_radius;
  {
    // Speed bound of every disc centre under the Euler map of eq. (6): the rear
    // axle moves |v| dt per step, headings turn by at most |v| dt tan|delta| / L1 (tractor) and
    // (|v| dt / L2)(1 + |Lh| tan|delta| / L1) (trailer), and |e(psi') - e(psi)| <= |psi' - psi|.
    const double V = std::fmax(std::fabs((double)p->v_min), std::fabs((double)p->v_max));
    const double td = std::tan(std::fmax(std::fabs((double)p->delta_min), std::fabs((double)p->delta_max)));
    const double w1 = V * td / p->L1, w2 = V / p->L2 * (1.0 + std::fabs((double)p->Lh) * td / p->L1);
    const double v_hitch = V + std::fabs((double)p->Lh) * w1;
    for (int j = 0; j < p->n_discs; ++j) {
      const double a = p->discs[j].offset;
      const double sp = p->discs[j].body == 0 ? V + std::fabs(a - p->Lh) * w1 : v_hitch + std::fabs(a) * w2;
      d.disc_speed[j] = (float)(1.001 * sp);
    }
  }
  d.dt = p->dt; d.inv_L1 = 1.0f / p->L1; d.inv_L2 = 1.0f / p->L2; d.Lh = p->Lh;
  d.Lh_over_L1 = p->Lh / p->L1; d.Lh_over_L2 = p->Lh / p->L2;
  d.v_min = p->v_min; d.v_max = p->v_max; d.delta_min = p->delta_min; d.delta_max = p->delta_max;
  d.sigma_v = p->sigma_v; d.sigma_delta = p->sigma_delta;
  if (p->flags & BRMPPI_FLAG_MPCC) {
    // the sampled inputs are (j, omega): their box and sigmas take the control slots of the sampler
    d.v_min = p->j_min; d.v_max = p->j_max; d.delta_min = p->omega_min; d.delta_max = p->omega_max;
    d.sigma_v = p->sigma_j; d.sigma_delta = p->sigma_omega;
    d.dstate_lo = p->delta_min; d.dstate_hi = p->delta_max;
    d.Qc = p->Qc; d.Ql = p->Ql; d.Qth1 = p->Qth1; d.Qth2 = p->Qth2; d.Rj = p->Rj; d.Rw = p->Rw;
    d.mu = p->mu; d.nu_bar = p->nu_bar; d.max_path_segments = p->max_path_segments;
    d.mpcc_lmax = 0.0f;
    for (int j = 0; j < p->n_discs; ++j)
      d.mpcc_lmax = std::fmax(d.mpcc_lmax, std::fabs(d.disc_a1[j] - p->Lh) + std::fabs(d.disc_a2[j]));
  }
  d.alpha_lo = p->alpha_lo; d.alpha_span = p->alpha_hi - p->alpha_lo;
  d.w_pos = p->w_pos; d.w_head = p->w_head; d.w_v = p->w_v; d.w_delta = p->w_delta;
  d.w_hitch = p->w_hitch; d.hitch_max = p->hitch_max; d.hitch_kappa = p->hitch_kappa; d.w_bar = p->w_bar; d.w_term = p->w_term;
  d.inv_lambda = 1.0f / p->lambda;
  d.hitch_filter = p->hitch_filter; d.hitch_alpha = p->hitch_alpha;
  d.hitch_qv = p->hitch_qv; d.hitch_qdelta = p->hitch_qdelta;
  d.proj_qv = p->proj_qv; d.proj_qomega = p->proj_qomega; d.proj_qalpha = p->proj_qalpha; d.proj_rho = p->proj_rho;
  d.sigma_ualpha = p->sigma_ualpha; d.ualpha_max = p->ualpha_max; d.w_alpha = p->w_alpha; d.h_buffer = p->h_buffer;
  d.key0 = (uint32_t)(p->seed & 0xFFFFFFFFull); d.key1 = (uint32_t)(p->seed >> 32);
  d.flags = p->flags;
  d.n_partials = c->plan.n_partials;
  if (c->plan.cta_kernel) {
    const CtaPlan& cp = c->plan.cta;
    d.S_tile = cp.S_tile; d.tiles_per_scene = cp.tiles_per_scene; d.total_tiles = cp.total_tiles;
    d.tiles_per_cta = cp.tiles_per_cta;
    d.chunks = cp.chunks; d.chunk_len = cp.chunk_len; d.t_stride = cp.ts; d.obs_padded = cp.obs_padded;
    const CtaSmem ts = cta_smem_layout(d.T, cp.S_tile, cp.chunks, cp.ts, cp.obs_padded, cp.se_padded);
    d.se_padded = cp.se_padded; d.off_se = (int)ts.se;
    d.off_obs = (int)ts.obs; d.off_vel = (int)ts.vel; d.off_thr = (int)ts.thr; d.off_A = (int)ts.A;
    d.off_scratch = (int)ts.scratch; d.off_w = (int)ts.w; d.off_alpha = (int)ts.alpha;
    d.off_cost = (int)ts.cost; d.off_xy = (int)ts.xy;
    d.off_planes = (int)ts.planes; d.off_misc = (int)ts.misc;
  }
  if (c->plan.mpcc_cta) {
    const MpccCtaPlan& mp = c->plan.mpcc;
    d.S_tile = mp.S; d.t_stride = mp.stride; d.chunks = mp.G; d.chunk_len = mp.L; d.mpcc_noise_planes = mp.noise_planes;
    d.tiles_per_scene = mp.tiles_per_scene; d.total_tiles = mp.total_tiles;
  }
  unsigned char* base = (unsigned char*)dev_workspace;
  const Layout& L = c->layout;
  d.state = (float*)(base + L.state); d.goal = (float*)(base + L.goal);
  d.n_obs = (int*)(base + L.n_obs); d.obstacles = (float*)(base + L.obstacles);
  d.n_se = (int*)(base + L.n_se); d.se = (float*)(base + L.se); d.max_superellipses = p->max_superellipses;
  d.U = (float*)(base + L.U); d.counter = (uint32_t*)(base + L.counter);
  d.u0_applied = (float*)(base + L.u0);
  d.hitch_ref = (float*)(base + L.hitch);
  if (p->flags & BRMPPI_FLAG_MPCC) {
    d.state7 = (float*)(base + L.state7); d.path_M = (int*)(base + L.path_M);
    d.path_dpsi = (float*)(base + L.path_dpsi); d.path_coef = (float*)(base + L.path_coef);
  }
  d.part_m = (double*)(base + L.part_m); d.part_argmin = (int*)(base + L.part_argmin);
  d.part_eta = (float*)(base + L.part_eta); d.part_w2 = (float*)(base + L.part_w2);
  d.part_nonfinite = (int*)(base + L.part_nf); d.part_A = (float*)(base + L.part_A);
  d.diag = (brmppi_diag*)(base + L.diag);
  if (p->flags & BRMPPI_FLAG_WRITE_SAMPLES) { d.S = (float*)(base + L.S); d.XT = (float*)(base + L.XT); }
  if ((p->flags & BRMPPI_FLAG_PHASE_TIMING) && c->plan.cta_kernel) d.phase_ns = (unsigned long long*)(base + L.phase);

  c->smem_update = 0;
  cudaError_t e = cudaSuccess;
  if (c->plan.cta_kernel) {
    c->smem_rollout = c->plan.cta.smem;
    e = configure_rollout_cta((p->flags & BRMPPI_FLAG_PRECISE_MATH) != 0, p->n_discs, c->smem_rollout);
  } else if (c->plan.mpcc_cta) {
    c->smem_rollout = c->plan.mpcc.smem;
    e = cudaFuncSetAttribute(mpcc_cta_kernel_for((p->flags & BRMPPI_FLAG_PRECISE_MATH) != 0, p->n_discs,
                                                 !(p->flags & BRMPPI_FLAG_NO_CULL)),
                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin);
  } else {
    c->smem_rollout = (p->flags & BRMPPI_FLAG_PROJECTED) ? rollout_projected_smem_bytes(d)
                      : (p->flags & BRMPPI_FLAG_MPCC)    ? rollout_mpcc_smem_bytes(d)
                                                         : rollout_thread_smem_bytes(d);
    // per function and device, not per context: always the opt-in maximum, never lowered
    if (p->flags & BRMPPI_FLAG_PROJECTED)
      e = cudaFuncSetAttribute(projected_kernel_for((p->flags & BRMPPI_FLAG_PRECISE_MATH) != 0, p->max_obstacles, p->n_discs),
                               cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(rollout_mpcc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(rollout_mpcc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(rollout_thread_per_sample<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(rollout_thread_per_sample<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin);
  }
  if (e == cudaSuccess && c->smem_update > 48 * 1024)
    e = cudaFuncSetAttribute(merge_update<kMergeLocal>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_update);
  if (e == cudaSuccess && (c->smem_rollout > prop.sharedMemPerBlockOptin || c->smem_update > prop.sharedMemPerBlockOptin))
    e = cudaErrorInvalidValue;
  // zero: n_obs, U, counter, diag, u0 (state/goal stay unset until the caller provides them)
  if (e == cudaSuccess) e = cudaMemsetAsync(base, 0, L.part_m, c->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(base + L.diag, 0, (size_t)p->n_scenes * sizeof(brmppi_diag), c->stream);
  if (e == cudaSuccess) e = cudaHostAlloc((void**)&c->pinned_u0, sizeof(float) * 2 * (size_t)p->n_scenes, cudaHostAllocMapped);
  if (e == cudaSuccess) e = cudaHostGetDevicePointer((void**)&d.u0_host, c->pinned_u0, 0);
  if (e == cudaSuccess) e = cudaHostAlloc((void**)&c->pinned_U, sizeof(float) * 2 * (size_t)p->T * (size_t)p->n_scenes, cudaHostAllocMapped);
  if (e == cudaSuccess) e = cudaHostGetDevicePointer((void**)&c->pinned_U_dev, c->pinned_U, 0);
  d.U_host = nullptr;
  if (p->n_scenes == 1 && !(p->flags & BRMPPI_FLAG_MPCC)) {
    const size_t span = L.obstacles + (size_t)(p->max_obstacles > 0 ? p->max_obstacles : 1) * 20 - L.state;
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
      e = cudaHostAlloc((void**)&c->pinned_in[i], span, cudaHostAllocDefault);
      if (e == cudaSuccess) { memset(c->pinned_in[i], 0, span); e = cudaEventCreateWithFlags(&c->pinned_in_done[i], cudaEventDisableTiming); }
    }
  }
  if (e != cudaSuccess) {
    free(c->state_set); free(c->goal_set); free(c->path_len);
    for (int i = 0; i < 2; ++i) {
      if (c->pinned_in[i]) cudaFreeHost(c->pinned_in[i]);
      if (c->pinned_in_done[i]) cudaEventDestroy(c->pinned_in_done[i]);
    }
    if (c->pinned_u0) cudaFreeHost(c->pinned_u0);
    if (c->pinned_U) cudaFreeHost(c->pinned_U);
    delete c;
    return cuda_fail(e);
  }
  *out = c;
  return BRMPPI_OK;
}

int brmppi_destroy(brmppi_ctx* c) {
  if (!c) return BRMPPI_ERR_NULL;
  if (c->solve_graph) cudaGraphExecDestroy(c->solve_graph);
  if (c->step_graph) cudaGraphExecDestroy(c->step_graph);
  if (c->solve_host_graph) cudaGraphExecDestroy(c->solve_host_graph);
  if (c->solve_io_graph) cudaGraphExecDestroy(c->solve_io_graph);
  if (c->pinned_u0) cudaFreeHost(c->pinned_u0);
    if (c->pinned_U) cudaFreeHost(c->pinned_U);
  for (int i = 0; i < 2; ++i) {
    if (c->pinned_in[i]) cudaFreeHost(c->pinned_in[i]);
    if (c->pinned_in_done[i]) cudaEventDestroy(c->pinned_in_done[i]);
  }
  free(c->state_set);
  free(c->goal_set);
  free(c->path_len);
  delete c;
  return BRMPPI_OK;
}

static int check_scene(const brmppi_ctx* c, int scene) {
  if (!c) return BRMPPI_ERR_NULL;
  if (scene < 0 || scene >= c->p.n_scenes) return BRMPPI_ERR_INVALID_ARG;
  return BRMPPI_OK;
}

static float wrap_pi(float a) {
  const double two_pi = 6.283185307179586476925286766559;
  return (float)((double)a - two_pi * std::nearbyint((double)a / two_pi));
}

int brmppi_set_state(brmppi_ctx* c, int scene, const float x[4]) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!x) return BRMPPI_ERR_NULL;
  if (c->p.flags & BRMPPI_FLAG_MPCC) return BRMPPI_ERR_INVALID_ARG;
  if (!finite_all(x, 4)) return BRMPPI_ERR_NONFINITE_INPUT;
  const float v[4] = {x[0], x[1], wrap_pi(x[2]), wrap_pi(x[3])};
  CU(cudaMemcpyAsync(c->d.state + 4 * scene, v, sizeof(v), cudaMemcpyHostToDevice, c->stream));
  c->state_set[scene] = 1;
  return BRMPPI_OK;
}

int brmppi_set_state7(brmppi_ctx* c, int scene, const float x[7], float psi) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!x) return BRMPPI_ERR_NULL;
  if (!(c->p.flags & BRMPPI_FLAG_MPCC)) return BRMPPI_ERR_INVALID_ARG;
  if (!c->goal_set[scene]) return BRMPPI_ERR_NOT_READY;          // the path comes first: psi is checked against it
  if (!finite_all(x, 7) || !std::isfinite(psi)) return BRMPPI_ERR_NONFINITE_INPUT;
  if (psi < 0.f || psi > c->path_len[scene]) return BRMPPI_ERR_INVALID_ARG;
  if (x[6] < c->p.delta_min || x[6] > c->p.delta_max) return BRMPPI_ERR_INVALID_ARG;
  const float v[8] = {x[0], x[1], x[2], x[3], wrap_pi(x[4]), wrap_pi(x[5]), x[6], psi};
  CU(cudaMemcpyAsync(c->d.state7 + 8 * scene, v, sizeof(v), cudaMemcpyHostToDevice, c->stream));
  CU(cudaStreamSynchronize(c->stream));     // v is a stack buffer
  c->state_set[scene] = 1;
  return BRMPPI_OK;
}

int brmppi_set_reference_path(brmppi_ctx* c, int scene, int M, float dpsi, const float* coef) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!coef) return BRMPPI_ERR_NULL;
  if (!(c->p.flags & BRMPPI_FLAG_MPCC)) return BRMPPI_ERR_INVALID_ARG;
  if (M < 1 || M > c->p.max_path_segments) return BRMPPI_ERR_INVALID_ARG;
  if (!std::isfinite(dpsi) || !finite_all(coef, 16 * M)) return BRMPPI_ERR_NONFINITE_INPUT;
  if (!(dpsi > 0.f)) return BRMPPI_ERR_INVALID_ARG;
  CU(cudaMemcpyAsync(c->d.path_coef + (size_t)scene * c->p.max_path_segments * 16, coef, sizeof(float) * 16 * (size_t)M,
                     cudaMemcpyHostToDevice, c->stream));
  CU(cudaMemcpyAsync(c->d.path_M + scene, &M, sizeof(int), cudaMemcpyHostToDevice, c->stream));
  CU(cudaMemcpyAsync(c->d.path_dpsi + scene, &dpsi, sizeof(float), cudaMemcpyHostToDevice, c->stream));
  CU(cudaStreamSynchronize(c->stream));     // M and dpsi are stack values
  c->path_len[scene] = (float)M * dpsi;
  c->goal_set[scene] = 1;                   // the path stands where the goal does on the other paths
  c->state_set[scene] = 0;                  // psi has to be given again against the new path
  return BRMPPI_OK;
}

int brmppi_set_goal(brmppi_ctx* c, int scene, const float g[4]) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!g) return BRMPPI_ERR_NULL;
  if (c->p.flags & BRMPPI_FLAG_MPCC) return BRMPPI_ERR_INVALID_ARG;
  if (!finite_all(g, 4)) return BRMPPI_ERR_NONFINITE_INPUT;
  CU(cudaMemcpyAsync(c->d.goal + 4 * scene, g, 16, cudaMemcpyHostToDevice, c->stream));
  c->goal_set[scene] = 1;
  return BRMPPI_OK;
}

int brmppi_set_obstacles(brmppi_ctx* c, int scene, int n, const brmppi_obstacle* obs) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (n < 0) return BRMPPI_ERR_INVALID_ARG;
  if (n > c->p.max_obstacles) return BRMPPI_ERR_TOO_MANY_OBSTACLES;
  if (n > 0 && !obs) return BRMPPI_ERR_NULL;
  for (int i = 0; i < n; ++i) {
    if (!finite_all(&obs[i].cx, 5)) return BRMPPI_ERR_NONFINITE_INPUT;
    if (!(obs[i].radius > 0.f)) return BRMPPI_ERR_INVALID_ARG;
  }
  if (n > 0)
    CU(cudaMemcpyAsync(c->d.obstacles + (size_t)scene * c->p.max_obstacles * 5, obs,
                       sizeof(brmppi_obstacle) * (size_t)n, cudaMemcpyHostToDevice, c->stream));
  CU(cudaMemcpyAsync(c->d.n_obs + scene, &n, sizeof(int), cudaMemcpyHostToDevice, c->stream));
  return BRMPPI_OK;
}

// every check of brmppi_set_state + brmppi_set_goal + brmppi_set_obstacles, nothing changed
static int check_inputs(brmppi_ctx* c, int scene, const float x[4], const float g[4], int n, const brmppi_obstacle* obs) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!x || !g) return BRMPPI_ERR_NULL;
  if (c->p.flags & BRMPPI_FLAG_MPCC) return BRMPPI_ERR_INVALID_ARG;
  if (!finite_all(x, 4) || !finite_all(g, 4)) return BRMPPI_ERR_NONFINITE_INPUT;
  if (n < 0) return BRMPPI_ERR_INVALID_ARG;
  if (n > c->p.max_obstacles) return BRMPPI_ERR_TOO_MANY_OBSTACLES;
  if (n > 0 && !obs) return BRMPPI_ERR_NULL;
  for (int i = 0; i < n; ++i) {
    if (!finite_all(&obs[i].cx, 5)) return BRMPPI_ERR_NONFINITE_INPUT;
    if (!(obs[i].radius > 0.f)) return BRMPPI_ERR_INVALID_ARG;
  }
  return BRMPPI_OK;
}

// the image of the workspace's input span (state | goal | n_obs | obstacles, each where the layout puts it); obstacle
// slots beyond n keep what the image held: never read
static void fill_input_image(const brmppi_ctx* c, unsigned char* img, const float x[4], const float g[4], int n,
                             const brmppi_obstacle* obs) {
  const Layout& L = c->layout;
  const float v[4] = {x[0], x[1], wrap_pi(x[2]), wrap_pi(x[3])};
  memcpy(img + (L.state - L.state), v, 16);
  memcpy(img + (L.goal - L.state), g, 16);
  memcpy(img + (L.n_obs - L.state), &n, sizeof(int));
  if (n > 0) memcpy(img + (L.obstacles - L.state), obs, sizeof(brmppi_obstacle) * (size_t)n);
}

int brmppi_set_inputs(brmppi_ctx* c, int scene, const float x[4], const float g[4], int n,
                      const brmppi_obstacle* obs) {
  int r = check_inputs(c, scene, x, g, n, obs);       // first, so that a failure changes nothing
  if (r) return r;
  if (!c->pinned_in[0]) {                    // several scenes: the three copies
    r = brmppi_set_state(c, scene, x);
    if (!r) r = brmppi_set_goal(c, scene, g);
    if (!r) r = brmppi_set_obstacles(c, scene, n, obs);
    return r;
  }
  // one scene: the image of the input span in page-locked memory, one copy
  const Layout& L = c->layout;
  const int b = c->pinned_in_next;
  c->pinned_in_next ^= 1;
  CU(cudaEventSynchronize(c->pinned_in_done[b]));       // the copy that last used this buffer has been made
  unsigned char* img = c->pinned_in[b];
  fill_input_image(c, img, x, g, n, obs);
  const size_t span = L.obstacles + sizeof(brmppi_obstacle) * (size_t)n - L.state;
  CU(cudaMemcpyAsync((unsigned char*)c->d.state, img, span, cudaMemcpyHostToDevice, c->stream));
  CU(cudaEventRecord(c->pinned_in_done[b], c->stream));
  c->state_set[scene] = 1;
  c->goal_set[scene] = 1;
  return BRMPPI_OK;
}

int brmppi_set_superellipses(brmppi_ctx* c, int scene, int n, const brmppi_superellipse* se) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (n < 0) return BRMPPI_ERR_INVALID_ARG;
  if (n > c->p.max_superellipses) return BRMPPI_ERR_TOO_MANY_OBSTACLES;
  if (n > 0 && !se) return BRMPPI_ERR_NULL;
  float rec[BRMPPI_MAX_SUPERELLIPSES][8];
  for (int i = 0; i < n; ++i) {
    if (!finite_all(&se[i].cx, 7)) return BRMPPI_ERR_NONFINITE_INPUT;
    if (!(se[i].mx > 0.f) || !(se[i].my > 0.f)) return BRMPPI_ERR_INVALID_ARG;
    if (se[i].exponent != 2 && se[i].exponent != 4) return BRMPPI_ERR_INVALID_ARG;
    memcpy(rec[i], &se[i].cx, 7 * sizeof(float));
    rec[i][7] = (float)se[i].exponent;
  }
  if (n > 0)
    CU(cudaMemcpyAsync(c->d.se + (size_t)scene * c->p.max_superellipses * 8, rec, sizeof(float) * 8 * (size_t)n,
                       cudaMemcpyHostToDevice, c->stream));
  CU(cudaMemcpyAsync(c->d.n_se + scene, &n, sizeof(int), cudaMemcpyHostToDevice, c->stream));
  CU(cudaStreamSynchronize(c->stream));     // rec is a stack buffer
  return BRMPPI_OK;
}

int brmppi_set_nominal(brmppi_ctx* c, int scene, const float* U) {
  int r = check_scene(c, scene);
  if (r) return r;
  float* dst = c->d.U + (size_t)scene * c->p.T * 2;
  const size_t bytes = sizeof(float) * 2 * (size_t)c->p.T;
  if (!U) { CU(cudaMemsetAsync(dst, 0, bytes, c->stream)); return BRMPPI_OK; }
  if (!finite_all(U, 2 * c->p.T)) return BRMPPI_ERR_NONFINITE_INPUT;
  for (int t = 0; t < c->p.T; ++t) {    // c->d holds the box of the mode's controls: (v, delta) or (j, omega)
    if (U[2 * t] < c->d.v_min || U[2 * t] > c->d.v_max) return BRMPPI_ERR_INVALID_ARG;
    if (U[2 * t + 1] < c->d.delta_min || U[2 * t + 1] > c->d.delta_max) return BRMPPI_ERR_INVALID_ARG;
  }
  CU(cudaMemcpyAsync(dst, U, bytes, cudaMemcpyHostToDevice, c->stream));
  return BRMPPI_OK;
}

int brmppi_set_counter(brmppi_ctx* c, unsigned int n) {
  if (!c) return BRMPPI_ERR_NULL;
  CU(cudaMemcpyAsync(c->d.counter, &n, sizeof(n), cudaMemcpyHostToDevice, c->stream));
  c->n_host = n;
  return BRMPPI_OK;
}

int brmppi_reset(brmppi_ctx* c) {
  if (!c) return BRMPPI_ERR_NULL;
  CU(cudaMemsetAsync(c->d.U, 0, sizeof(float) * 2 * (size_t)c->p.T * (size_t)c->p.n_scenes, c->stream));
  return brmppi_set_counter(c, 0u);
}

int brmppi_solve(brmppi_ctx* c) {
  if (!c) return BRMPPI_ERR_NULL;
  int r = ready(c);
  if (r) return r;
  if (c->stream == nullptr) {           // the legacy default stream cannot be captured
    r = enqueue_solve(c);
    if (r) return r;
  } else {
    if (!c->solve_graph) {
      r = capture(c, &c->solve_graph, [&] { return enqueue_solve(c); });
      if (r) return r;
    }
    CU(cudaGraphLaunch(c->solve_graph, c->stream));
  }
  c->launches += 2ull * (unsigned)c->p.n_iter;
  c->n_host += (unsigned)c->p.n_iter;
  return BRMPPI_OK;
}

int brmppi_solve_get_controls(brmppi_ctx* c, float* U_out) {
  if (!c || !U_out) return BRMPPI_ERR_NULL;
  int r = ready(c);
  if (r) return r;
  if (c->stream == nullptr) {           // the legacy default stream cannot be captured
    r = enqueue_solve(c, true);
    if (r) return r;
  } else {
    if (!c->solve_host_graph) {
      r = capture(c, &c->solve_host_graph, [&] { return enqueue_solve(c, true); });
      if (r) return r;
    }
    CU(cudaGraphLaunch(c->solve_host_graph, c->stream));
  }
  c->launches += 2ull * (unsigned)c->p.n_iter;
  c->n_host += (unsigned)c->p.n_iter;
  // the last update wrote U straight into the page-locked host copy (mapped under unified addressing): no copy
  // node behind the graph, the sync makes it visible
  CU(cudaStreamSynchronize(c->stream));
  memcpy(U_out, c->pinned_U, sizeof(float) * 2 * (size_t)c->p.T * (size_t)c->p.n_scenes);
  return BRMPPI_OK;
}

int brmppi_solve_host(brmppi_ctx* c, const float x[4], const float g[4], int n, const brmppi_obstacle* obs,
                      float* U_out) {
  if (!c || !U_out) return BRMPPI_ERR_NULL;
  int r = check_inputs(c, 0, x, g, n, obs);
  if (r) return r;
  if (!c->pinned_in[0] || c->stream == nullptr) {       // several scenes, or no stream to capture on: the two calls
    r = brmppi_set_inputs(c, 0, x, g, n, obs);
    return r ? r : brmppi_solve_get_controls(c, U_out);
  }
  // ONE graph launch: copy of the input image (page-locked, fixed address: staging buffer 0) into the workspace,
  // the solve, the last update writing U into page-locked host memory
  CU(cudaEventSynchronize(c->pinned_in_done[0]));        // a brmppi_set_inputs copy out of this buffer has been made
  fill_input_image(c, c->pinned_in[0], x, g, n, obs);
  c->state_set[0] = 1;
  c->goal_set[0] = 1;
  if (!c->solve_io_graph) {
    const Layout& L = c->layout;
    const size_t span = L.obstacles + sizeof(brmppi_obstacle) * (size_t)(c->p.max_obstacles > 0 ? c->p.max_obstacles : 1) - L.state;
    r = capture(c, &c->solve_io_graph, [&] {
      CU(cudaMemcpyAsync((unsigned char*)c->d.state, c->pinned_in[0], span, cudaMemcpyHostToDevice, c->stream));
      return enqueue_solve(c, true);
    });
    if (r) return r;
  }
  CU(cudaGraphLaunch(c->solve_io_graph, c->stream));
  c->launches += 2ull * (unsigned)c->p.n_iter;
  c->n_host += (unsigned)c->p.n_iter;
  CU(cudaStreamSynchronize(c->stream));
  memcpy(U_out, c->pinned_U, sizeof(float) * 2 * (size_t)c->p.T);
  return BRMPPI_OK;
}

size_t brmppi_shard_words(const brmppi_ctx* c) {
  return c ? (size_t)c->p.n_scenes * (size_t)(kShardHeader + 2 * c->p.T) : 0;
}

int brmppi_shard_export(brmppi_ctx* c, float* dev_shard) {
  if (!c || !dev_shard) return BRMPPI_ERR_NULL;
  if ((uintptr_t)dev_shard % 8 != 0) return BRMPPI_ERR_UNALIGNED;
  int r = ready(c);
  if (r) return r;
  r = launch_rollout(c);
  if (r) return r;
  dim3 ugrid((unsigned)(2 * c->d.T), (unsigned)c->d.n_scenes);
  merge_update<kMergeExport><<<ugrid, kUpdateBlock, 0, c->stream>>>(c->d, dev_shard, 0);
  CU(cudaGetLastError());
  c->launches += 2;
  return BRMPPI_OK;
}

int brmppi_shard_import(brmppi_ctx* c, int n_shards, const float* dev_shards) {
  if (!c || !dev_shards) return BRMPPI_ERR_NULL;
  if (n_shards < 1) return BRMPPI_ERR_INVALID_ARG;
  if ((uintptr_t)dev_shards % 8 != 0) return BRMPPI_ERR_UNALIGNED;
  dim3 ugrid((unsigned)(2 * c->d.T), (unsigned)c->d.n_scenes);
  merge_update<kMergeImport><<<ugrid, kUpdateBlock, 0, c->stream>>>(c->d, const_cast<float*>(dev_shards), n_shards);
  CU(cudaGetLastError());
  c->launches += 1;
  c->n_host += 1;
  return BRMPPI_OK;
}

int brmppi_shift(brmppi_ctx* c) {
  if (!c) return BRMPPI_ERR_NULL;
  shift_plant<false><<<(unsigned)c->p.n_scenes, kShiftBlock, 0, c->stream>>>(c->d);
  CU(cudaGetLastError());
  c->launches += 1;
  return BRMPPI_OK;
}

int brmppi_step(brmppi_ctx* c, float* u0_out) {
  if (!c) return BRMPPI_ERR_NULL;
  int r = ready(c);
  if (r) return r;
  if (c->stream == nullptr) return BRMPPI_ERR_INVALID_ARG;   // graph replay needs a real stream
  if (!c->step_graph) {
    r = capture(c, &c->step_graph, [&] {
      int rr = enqueue_solve(c);
      if (rr) return rr;
      // the plant step writes the applied control straight into the page-locked host buffer (mapped
      // under unified addressing): the graph needs no copy node, the sync below makes it visible
      shift_plant<true><<<(unsigned)c->p.n_scenes, kShiftBlock, 0, c->stream>>>(c->d);
      CU(cudaGetLastError());
      return (int)BRMPPI_OK;
    });
    if (r) return r;
  }
  CU(cudaGraphLaunch(c->step_graph, c->stream));
  c->launches += 2ull * (unsigned)c->p.n_iter + 1ull;
  c->n_host += (unsigned)c->p.n_iter;
  CU(cudaStreamSynchronize(c->stream));
  if (u0_out) memcpy(u0_out, c->pinned_u0, sizeof(float) * 2 * (size_t)c->p.n_scenes);
  return BRMPPI_OK;
}

static int d2h(brmppi_ctx* c, void* dst, const void* src, size_t bytes) {
  CU(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return BRMPPI_OK;
}

int brmppi_get_controls(brmppi_ctx* c, int scene, float* U_out) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!U_out) return BRMPPI_ERR_NULL;
  return d2h(c, U_out, c->d.U + (size_t)scene * c->p.T * 2, sizeof(float) * 2 * (size_t)c->p.T);
}

int brmppi_get_state(brmppi_ctx* c, int scene, float x_out[4]) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!x_out) return BRMPPI_ERR_NULL;
  if (c->p.flags & BRMPPI_FLAG_MPCC) return BRMPPI_ERR_INVALID_ARG;
  return d2h(c, x_out, c->d.state + 4 * scene, 16);
}

int brmppi_get_state7(brmppi_ctx* c, int scene, float x_out[8]) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!x_out) return BRMPPI_ERR_NULL;
  if (!(c->p.flags & BRMPPI_FLAG_MPCC)) return BRMPPI_ERR_INVALID_ARG;
  return d2h(c, x_out, c->d.state7 + 8 * scene, 32);
}

int brmppi_get_obstacles(brmppi_ctx* c, int scene, int* n_out, brmppi_obstacle* out) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!n_out) return BRMPPI_ERR_NULL;
  r = d2h(c, n_out, c->d.n_obs + scene, sizeof(int));
  if (r) return r;
  if (out && *n_out > 0)
    return d2h(c, out, c->d.obstacles + (size_t)scene * c->p.max_obstacles * 5,
               sizeof(brmppi_obstacle) * (size_t)*n_out);
  return BRMPPI_OK;
}

int brmppi_get_superellipses(brmppi_ctx* c, int scene, int* n_out, brmppi_superellipse* out) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!n_out) return BRMPPI_ERR_NULL;
  r = d2h(c, n_out, c->d.n_se + scene, sizeof(int));
  if (r) return r;
  if (out && *n_out > 0) {
    float rec[BRMPPI_MAX_SUPERELLIPSES][8];
    r = d2h(c, rec, c->d.se + (size_t)scene * c->p.max_superellipses * 8, sizeof(float) * 8 * (size_t)*n_out);
    if (r) return r;
    for (int i = 0; i < *n_out; ++i) { memcpy(&out[i].cx, rec[i], 7 * sizeof(float)); out[i].exponent = (int)rec[i][7]; }
  }
  return BRMPPI_OK;
}

int brmppi_get_costs(brmppi_ctx* c, int scene, float* S_out) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!S_out) return BRMPPI_ERR_NULL;
  if (!(c->p.flags & BRMPPI_FLAG_WRITE_SAMPLES)) return BRMPPI_ERR_NOT_READY;
  return d2h(c, S_out, c->d.S + (size_t)scene * c->p.K, sizeof(float) * (size_t)c->p.K);
}

int brmppi_get_final_states(brmppi_ctx* c, int scene, float* X_out) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!X_out) return BRMPPI_ERR_NULL;
  if (!(c->p.flags & BRMPPI_FLAG_WRITE_SAMPLES)) return BRMPPI_ERR_NOT_READY;
  if (c->p.flags & BRMPPI_FLAG_MPCC) return BRMPPI_ERR_INVALID_ARG;
  return d2h(c, X_out, c->d.XT + (size_t)scene * c->p.K * 4, sizeof(float) * 4 * (size_t)c->p.K);
}

int brmppi_get_final_states7(brmppi_ctx* c, int scene, float* X_out) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!X_out) return BRMPPI_ERR_NULL;
  if (!(c->p.flags & BRMPPI_FLAG_WRITE_SAMPLES)) return BRMPPI_ERR_NOT_READY;
  if (!(c->p.flags & BRMPPI_FLAG_MPCC)) return BRMPPI_ERR_INVALID_ARG;
  return d2h(c, X_out, c->d.XT + (size_t)scene * c->p.K * 8, sizeof(float) * 8 * (size_t)c->p.K);
}

int brmppi_get_diag(brmppi_ctx* c, int scene, brmppi_diag* out) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!out) return BRMPPI_ERR_NULL;
  r = d2h(c, out, c->d.diag + scene, sizeof(brmppi_diag));
  out->n = c->n_host;
  return r;
}

int brmppi_time_kernels(brmppi_ctx* c, int reps, float out_ms[2]) {
  if (!c || !out_ms) return BRMPPI_ERR_NULL;
  if (reps < 1 || reps > 4096) return BRMPPI_ERR_INVALID_ARG;
  int r = ready(c);
  if (r) return r;
  // Two trains of launches, everything enqueued back to back with ONE synchronisation at the end so
  // that the stream never runs dry: `reps` rollout launches between two events, then `reps` update
  // launches between two events (the update is a pure function of the partials, so repeating it
  // leaves U as one iteration would).  A train's mean is the kernel's device time plus the
  // kernel-to-kernel gap, as inside the captured graph; an event between every two kernels would
  // add its own drain-and-timestamp gap (about 3 us here) to each interval.  kWarm leading
  // launches of each train are left out.
  const int kWarm = 2;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  cudaError_t e = cudaSuccess;
  int made = 0;
  for (; made < 4 && e == cudaSuccess; ++made) e = cudaEventCreate(&ev[made]);
  for (int it = 0; it < reps + kWarm && e == cudaSuccess && r == 0; ++it) {
    if (it == kWarm) e = cudaEventRecord(ev[0], c->stream);
    if (e == cudaSuccess) r = launch_rollout(c);
    c->launches += 1;
  }
  if (e == cudaSuccess && r == 0) e = cudaEventRecord(ev[1], c->stream);
  for (int it = 0; it < reps + kWarm && e == cudaSuccess && r == 0; ++it) {
    if (it == kWarm) e = cudaEventRecord(ev[2], c->stream);
    if (e == cudaSuccess) r = launch_update(c);
    c->launches += 1;
    c->n_host += 1;
  }
  if (e == cudaSuccess && r == 0) e = cudaEventRecord(ev[3], c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  float roll = 0.f, upd = 0.f;
  if (e == cudaSuccess && r == 0) e = cudaEventElapsedTime(&roll, ev[0], ev[1]);
  if (e == cudaSuccess && r == 0) e = cudaEventElapsedTime(&upd, ev[2], ev[3]);
  for (int i = 0; i < made; ++i) cudaEventDestroy(ev[i]);
  if (r) return r;
  if (e != cudaSuccess) return cuda_fail(e);
  out_ms[0] = roll / (float)reps;
  out_ms[1] = upd / (float)reps;
  return BRMPPI_OK;
}

int brmppi_get_phase_times(brmppi_ctx* c, float out_us[8]) {
  if (!c || !out_us) return BRMPPI_ERR_NULL;
  if (!c->d.phase_ns) return BRMPPI_ERR_NOT_READY;
  const int grid = c->plan.cta.grid, W = kPhaseSlots + 2;
  unsigned long long* h = (unsigned long long*)malloc(sizeof(unsigned long long) * (size_t)grid * W);
  if (!h) return BRMPPI_ERR_NULL;
  int r = d2h(c, h, c->d.phase_ns, sizeof(unsigned long long) * (size_t)grid * W);
  if (r == BRMPPI_OK) {
    // phase slots are SM cycles (clock64); each CTA's own lifetime on the globaltimer converts them
    double acc[kPhaseSlots] = {0};
    unsigned long long tmin = ~0ull, tmax = 0ull, life = 0ull;
    for (int b = 0; b < grid; ++b) {
      const unsigned long long t0 = h[b * W + kPhaseSlots], t1 = h[b * W + kPhaseSlots + 1];
      double cyc = 0.0;   // the chain slot runs under the cost slot: not part of the CTA's timeline sum
      for (int i = 0; i < kPhaseSlots; ++i) if (i != kChainSlot) cyc += (double)h[b * W + i];
      const double ns_per_cycle = cyc > 0.0 ? (double)(t1 - t0) / cyc : 0.0;
      for (int i = 0; i < kPhaseSlots; ++i) acc[i] += (double)h[b * W + i] * ns_per_cycle;
      if (t0 < tmin) tmin = t0;
      if (t1 > tmax) tmax = t1;
      if (t1 - t0 > life) life = t1 - t0;
    }
    for (int i = 0; i < kPhaseSlots; ++i) out_us[i] = (float)(acc[i] / grid * 1e-3);
    out_us[7] = (float)((double)(tmax - tmin) * 1e-3);
    (void)life;
  }
  free(h);
  return r;
}

unsigned long long brmppi_launch_count(const brmppi_ctx* c) { return c ? c->launches : 0ull; }

const char* brmppi_strerror(int status) {
  switch (status) {
    case BRMPPI_OK: return "ok";
    case BRMPPI_ERR_NULL: return "null pointer";
    case BRMPPI_ERR_INVALID_ARG: return "invalid argument";
    case BRMPPI_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case BRMPPI_ERR_TOO_MANY_OBSTACLES: return "too many obstacles";
    case BRMPPI_ERR_NONFINITE_INPUT: return "non-finite input";
    case BRMPPI_ERR_NOT_READY: return "not ready (state/goal unset, or sample outputs not enabled)";
    case BRMPPI_ERR_UNALIGNED: return "workspace not 256-byte aligned";
    case BRMPPI_ERR_TOO_LARGE: return "size exceeds the capacity of the library's static device scratch";
    case BRMPPI_ERR_CUDA:
      snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error: %s", cudaGetErrorString(g_last_cuda));
      return g_errbuf;
    default: return "unknown status";
  }
}

int brmppi_debug_philox(void* cuda_stream, unsigned long long seed, unsigned int n, int K, int T,
                        unsigned int tag, unsigned int* dev_out) {
  if (!dev_out) return BRMPPI_ERR_NULL;
  if (K < 1 || T < 1) return BRMPPI_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const size_t total = (size_t)K * T;
  debug_philox<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(
      (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32), n, K, T, tag, (uint4*)dev_out);
  CU(cudaGetLastError());
  CU(cudaStreamSynchronize(s));
  return BRMPPI_OK;
}

int brmppi_debug_philox_raw(void* cuda_stream, int n, const unsigned int* dev_ctr, const unsigned int* dev_key,
                            int use_curand, unsigned int* dev_out) {
  if (n < 0 || (use_curand != 0 && use_curand != 1)) return BRMPPI_ERR_INVALID_ARG;
  if (n == 0) return BRMPPI_OK;
  if (!dev_ctr || !dev_key || !dev_out) return BRMPPI_ERR_NULL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const unsigned grid = (unsigned)((n + 255) / 256);
  if (use_curand)
    debug_philox_raw<true><<<grid, 256, 0, s>>>(n, (const uint4*)dev_ctr, (const uint2*)dev_key, (uint4*)dev_out);
  else
    debug_philox_raw<false><<<grid, 256, 0, s>>>(n, (const uint4*)dev_ctr, (const uint2*)dev_key, (uint4*)dev_out);
  CU(cudaGetLastError());
  CU(cudaStreamSynchronize(s));
  return BRMPPI_OK;
}

int brmppi_debug_sample_controls(void* cuda_stream, const brmppi_params* p, unsigned int n,
                                 const float* dev_U_nominal, float* dev_u, float* dev_alpha) {
  if (!p || !dev_U_nominal) return BRMPPI_ERR_NULL;
  if (!params_valid(p)) return BRMPPI_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceParams d;
  memset(&d, 0, sizeof(d));
  d.K = p->K; d.T = p->T;
  d.v_min = p->v_min; d.v_max = p->v_max; d.delta_min = p->delta_min; d.delta_max = p->delta_max;
  d.sigma_v = p->sigma_v; d.sigma_delta = p->sigma_delta;
  if (p->flags & BRMPPI_FLAG_MPCC) {
    d.v_min = p->j_min; d.v_max = p->j_max; d.delta_min = p->omega_min; d.delta_max = p->omega_max;
    d.sigma_v = p->sigma_j; d.sigma_delta = p->sigma_omega;
  }
  d.alpha_lo = p->alpha_lo; d.alpha_span = p->alpha_hi - p->alpha_lo;
  d.key0 = (uint32_t)(p->seed & 0xFFFFFFFFull); d.key1 = (uint32_t)(p->seed >> 32);
  const size_t total = (size_t)p->K * p->T;
  const unsigned grid = (unsigned)((total + 255) / 256);
  if (p->flags & BRMPPI_FLAG_PRECISE_MATH)
    debug_sample_controls<true><<<grid, 256, 0, s>>>(d, n, (const float2*)dev_U_nominal, (float2*)dev_u, dev_alpha);
  else
    debug_sample_controls<false><<<grid, 256, 0, s>>>(d, n, (const float2*)dev_U_nominal, (float2*)dev_u, dev_alpha);
  CU(cudaGetLastError());
  CU(cudaStreamSynchronize(s));
  return BRMPPI_OK;
}

int brmppi_get_hitch_filter(brmppi_ctx* c, int scene, float u_ref[2], int* status) {
  int r = check_scene(c, scene);
  if (r) return r;
  if (!u_ref || !status) return BRMPPI_ERR_NULL;
  float h[4];
  r = d2h(c, h, c->d.hitch_ref + (size_t)scene * 4, sizeof(h));
  if (r) return r;
  u_ref[0] = h[0]; u_ref[1] = h[1];
  memcpy(status, &h[2], sizeof(int));
  return BRMPPI_OK;
}

size_t brmppi_hitch_filter_scratch_bytes(int n) { return n > 0 ? (size_t)n * 36 + 256 : 0; }

int brmppi_hitch_filter(void* cuda_stream, const brmppi_params* p, int n, const float* x,
                        const float* u_ref, float* u_out, int* status_out, void* dev_scratch,
                        size_t scratch_bytes) {
  if (!p) return BRMPPI_ERR_NULL;
  if (n < 0) return BRMPPI_ERR_INVALID_ARG;
  const float f[] = {p->dt, p->L1, p->L2, p->Lh, p->v_min, p->v_max, p->delta_min, p->delta_max};
  if (!finite_all(f, 8) || !hitch_params_valid(p) || !(p->dt > 0.f) || !(p->L1 > 0.f) || !(p->L2 > 0.f) ||
      p->v_min > p->v_max || p->delta_min > p->delta_max || p->delta_min <= -1.5f || p->delta_max >= 1.5f)
    return BRMPPI_ERR_INVALID_ARG;
  if (n == 0) return BRMPPI_OK;
  if (!x || !u_ref || !u_out || !dev_scratch) return BRMPPI_ERR_NULL;
  if (scratch_bytes < brmppi_hitch_filter_scratch_bytes(n)) return BRMPPI_ERR_WORKSPACE_TOO_SMALL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceParams d;
  memset(&d, 0, sizeof(d));
  d.dt = p->dt; d.inv_L1 = 1.0f / p->L1; d.inv_L2 = 1.0f / p->L2; d.Lh = p->Lh;
  d.Lh_over_L1 = p->Lh / p->L1; d.Lh_over_L2 = p->Lh / p->L2;
  d.v_min = p->v_min; d.v_max = p->v_max; d.delta_min = p->delta_min; d.delta_max = p->delta_max;
  d.hitch_max = p->hitch_max; d.hitch_kappa = p->hitch_kappa; d.hitch_alpha = p->hitch_alpha;
  d.hitch_qv = p->hitch_qv; d.hitch_qdelta = p->hitch_qdelta;
  // the caller's scratch: x [n][4] | u_ref [n][2] | u_out [n][2] | status [n]
  const size_t N = (size_t)n;
  unsigned char* buf = (unsigned char*)align_up((size_t)(uintptr_t)dev_scratch, 256);
  float4* dx = (float4*)buf;
  float2* dr = (float2*)(buf + N * 16);
  float2* du = (float2*)(buf + N * 24);
  int* ds = (int*)(buf + N * 32);
  CU(cudaMemcpyAsync(dx, x, N * 16, cudaMemcpyHostToDevice, s));
  CU(cudaMemcpyAsync(dr, u_ref, N * 8, cudaMemcpyHostToDevice, s));
  hitch_filter_batch<<<(unsigned)((N + 127) / 128), 128, 0, s>>>(d, n, dx, dr, du, ds);
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(u_out, du, N * 8, cudaMemcpyDeviceToHost, s));
  if (status_out) CU(cudaMemcpyAsync(status_out, ds, N * 4, cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  return BRMPPI_OK;
}

int brmppi_hitch_filter_static(void* cuda_stream, const brmppi_params* p, int n, const float* x,
                               const float* u_ref, float* u_out, int* status_out) {
  if (!p) return BRMPPI_ERR_NULL;
  if (n < 0) return BRMPPI_ERR_INVALID_ARG;
  if (n > BRMPPI_HITCH_STATIC_MAX_N) return BRMPPI_ERR_TOO_LARGE;
  const float f[] = {p->dt, p->L1, p->L2, p->Lh, p->v_min, p->v_max, p->delta_min, p->delta_max};
  if (!finite_all(f, 8) || !hitch_params_valid(p) || !(p->dt > 0.f) || !(p->L1 > 0.f) || !(p->L2 > 0.f) ||
      p->v_min > p->v_max || p->delta_min > p->delta_max || p->delta_min <= -1.5f || p->delta_max >= 1.5f)
    return BRMPPI_ERR_INVALID_ARG;
  if (n == 0) return BRMPPI_OK;
  if (!x || !u_ref || !u_out) return BRMPPI_ERR_NULL;
  unsigned char* buf = nullptr;
  int r = hitch_static_address(&buf);
  if (r) return r;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceParams d;
  memset(&d, 0, sizeof(d));
  d.dt = p->dt; d.inv_L1 = 1.0f / p->L1; d.inv_L2 = 1.0f / p->L2; d.Lh = p->Lh;
  d.Lh_over_L1 = p->Lh / p->L1; d.Lh_over_L2 = p->Lh / p->L2;
  d.v_min = p->v_min; d.v_max = p->v_max; d.delta_min = p->delta_min; d.delta_max = p->delta_max;
  d.hitch_max = p->hitch_max; d.hitch_kappa = p->hitch_kappa; d.hitch_alpha = p->hitch_alpha;
  d.hitch_qv = p->hitch_qv; d.hitch_qdelta = p->hitch_qdelta;
  // the static array: x [n][4] | u_ref [n][2] | u_out [n][2] | status [n]
  const size_t N = (size_t)n;
  float4* dx = (float4*)buf;
  float2* dr = (float2*)(buf + N * 16);
  float2* du = (float2*)(buf + N * 24);
  int* ds = (int*)(buf + N * 32);
  CU(cudaMemcpyAsync(dx, x, N * 16, cudaMemcpyHostToDevice, s));
  CU(cudaMemcpyAsync(dr, u_ref, N * 8, cudaMemcpyHostToDevice, s));
  hitch_filter_batch<<<(unsigned)((N + 127) / 128), 128, 0, s>>>(d, n, dx, dr, du, ds);
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(u_out, du, N * 8, cudaMemcpyDeviceToHost, s));
  if (status_out) CU(cudaMemcpyAsync(status_out, ds, N * 4, cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  return BRMPPI_OK;
}

size_t brmppi_project_scratch_bytes(int n, int n_o) {
  if (n <= 0 || n_o < 1 || n_o > BRMPPI_PROJECT_MAX_NO) return 0;
  const size_t N = (size_t)n, d = (size_t)n_o + 2;
  return sizeof(float) * (N * n_o * d + N * n_o + 2 * N * d + 16) + 256;
}

int brmppi_project(void* cuda_stream, int n, int n_o, const float* A, const float* b, const float* z_des,
                   const float* w, float rho, const float* z_lo, const float* z_hi, float* z_out,
                   int device_ptrs, void* dev_scratch, size_t scratch_bytes) {
  if (n < 0 || n_o < 1 || n_o > BRMPPI_PROJECT_MAX_NO || (device_ptrs != 0 && device_ptrs != 1))
    return BRMPPI_ERR_INVALID_ARG;
  if (!w || !z_lo || !z_hi) return BRMPPI_ERR_NULL;
  const int d = n_o + 2;
  if (!finite_all(w, d) || !finite_all(z_lo, d) || !finite_all(z_hi, d) || !std::isfinite(rho) || rho < 0.f)
    return BRMPPI_ERR_INVALID_ARG;
  ProjConst pc;
  memset(&pc, 0, sizeof(pc));
  for (int j = 0; j < d; ++j) {
    if (!(w[j] > 0.f)) return BRMPPI_ERR_INVALID_ARG;
    pc.w[j] = w[j]; pc.lo[j] = z_lo[j]; pc.hi[j] = z_hi[j];
  }
  pc.rho = rho;
  if (n == 0) return BRMPPI_OK;
  if (!A || !b || !z_des || !z_out) return BRMPPI_ERR_NULL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (device_ptrs) {
    CU(launch_project_dyn(n_o, n, A, b, z_des, pc, z_out, s));
    return BRMPPI_OK;
  }
  if (!dev_scratch) return BRMPPI_ERR_NULL;
  if (scratch_bytes < brmppi_project_scratch_bytes(n, n_o)) return BRMPPI_ERR_WORKSPACE_TOO_SMALL;
  const size_t N = (size_t)n, nA = N * n_o * d, nb = N * n_o, nz = N * d;
  // sections of the caller's scratch, kept 16-byte aligned
  auto up4 = [](size_t x) { return (x + 3) & ~(size_t)3; };
  float* dA = (float*)align_up((size_t)(uintptr_t)dev_scratch, 256);
  float* db = dA + up4(nA);
  float* dz = db + up4(nb);
  float* dout = dz + up4(nz);
  CU(cudaMemcpyAsync(dA, A, sizeof(float) * nA, cudaMemcpyHostToDevice, s));
  CU(cudaMemcpyAsync(db, b, sizeof(float) * nb, cudaMemcpyHostToDevice, s));
  CU(cudaMemcpyAsync(dz, z_des, sizeof(float) * nz, cudaMemcpyHostToDevice, s));
  CU(launch_project_dyn(n_o, n, dA, db, dz, pc, dout, s));
  CU(cudaMemcpyAsync(z_out, dout, sizeof(float) * nz, cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  return BRMPPI_OK;
}

size_t brmppi_measure_peaks_scratch_bytes(void) { return sizeof(long long) * 3 * 4 * 1024 + 256; }

int brmppi_measure_peaks(void* cuda_stream, void* dev_scratch, size_t scratch_bytes, float out[16]) {
  if (!out || !dev_scratch) return BRMPPI_ERR_NULL;
  if (scratch_bytes < brmppi_measure_peaks_scratch_bytes()) return BRMPPI_ERR_WORKSPACE_TOO_SMALL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int dev = 0;
  CU(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  CU(cudaGetDeviceProperties(&prop, dev));
  const int blocks = prop.multiProcessorCount * 4;   // 4 x 256 threads resident per SM, one wave
  if (blocks > 4 * 1024 - 8) return BRMPPI_ERR_INVALID_ARG;
  float* sink = (float*)align_up((size_t)(uintptr_t)dev_scratch, 256);   // 4 floats, then the spans
  long long* spans = (long long*)(sink + 8);
  long long* h = (long long*)malloc(sizeof(long long) * 3 * (size_t)blocks);
  if (!h) return BRMPPI_ERR_NULL;
  // where each kind's rate goes in out[]: 0..4 as before, 5..7 = SM count and clocks, 8..15 = the rest
  const int slot[PEAK_KINDS] = {0, 1, 2, 3, 4, 8, 9, 10, 11, 12, 13, 14, 15};
  cudaError_t e = cudaSuccess;
  for (int kind = 0; kind < PEAK_KINDS && e == cudaSuccess; ++kind) {
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {   // last repetition is the one kept
      switch (kind) {
        case PEAK_FFMA: e = launch_peak<PEAK_FFMA>(blocks, s, spans, sink); break;
        case PEAK_ALU: e = launch_peak<PEAK_ALU>(blocks, s, spans, sink); break;
        case PEAK_MUFU: e = launch_peak<PEAK_MUFU>(blocks, s, spans, sink); break;
        case PEAK_MIX: e = launch_peak<PEAK_MIX>(blocks, s, spans, sink); break;
        case PEAK_IMAD_WIDE: e = launch_peak<PEAK_IMAD_WIDE>(blocks, s, spans, sink); break;
        case PEAK_FMNMX: e = launch_peak<PEAK_FMNMX>(blocks, s, spans, sink); break;
        case PEAK_FFMA2: e = launch_peak<PEAK_FFMA2>(blocks, s, spans, sink); break;
        case PEAK_FFMA2_DISTINCT: e = launch_peak<PEAK_FFMA2_DISTINCT>(blocks, s, spans, sink); break;
        case PEAK_FADD2: e = launch_peak<PEAK_FADD2>(blocks, s, spans, sink); break;
        case PEAK_FFMA_FMNMX: e = launch_peak<PEAK_FFMA_FMNMX>(blocks, s, spans, sink); break;
        case PEAK_FFMA2_FMNMX: e = launch_peak<PEAK_FFMA2_FMNMX>(blocks, s, spans, sink); break;
        case PEAK_IMAD_LO: e = launch_peak<PEAK_IMAD_LO>(blocks, s, spans, sink); break;
        default: e = launch_peak<PEAK_IMAD_HI>(blocks, s, spans, sink); break;
      }
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(h, spans, sizeof(long long) * 3 * (size_t)blocks, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) break;
    // Rate = instructions per SM / (first block start .. last block end, on the nanosecond
    // globaltimer) converted to SM cycles with the clock each block saw while running
    // (clock64 span / globaltimer span).  Per-block clock64 spans alone over-estimate: blocks
    // that win the arbitration finish early while the SM is still busy with the others.
    long long gmin = h[1], gmax = h[2];
    double mhz_sum = 0.0;
    for (int b = 0; b < blocks; ++b) {
      gmin = h[3 * b + 1] < gmin ? h[3 * b + 1] : gmin;
      gmax = h[3 * b + 2] > gmax ? h[3 * b + 2] : gmax;
      mhz_sum += (double)h[3 * b] * 1e3 / (double)(h[3 * b + 2] - h[3 * b + 1]);
    }
    const double mhz_kernel = mhz_sum / blocks;
    const double wall_ns = (double)(gmax - gmin);
    const double per_thread = (double)kPeakIters * kPeakReps * kPeakChains * peak_instr_per_slot(kind);
    out[slot[kind]] = (float)(per_thread * 1024.0 / (wall_ns * 1e-3 * mhz_kernel));   // thread-instr / clk / SM
    if (kind == PEAK_FFMA) out[7] = (float)mhz_kernel;
  }
  if (e == cudaSuccess) {
    clock_rate_kernel<<<1, 1, 0, s>>>(sink);
    e = cudaGetLastError();
    float mhz[2] = {0, 0};
    if (e == cudaSuccess) e = cudaMemcpyAsync(mhz, sink, sizeof(float) * 2, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    out[5] = (float)prop.multiProcessorCount;
    out[6] = mhz[0];
  }
  free(h);
  if (e != cudaSuccess) return cuda_fail(e);
  return BRMPPI_OK;
}

}  // extern "C"
