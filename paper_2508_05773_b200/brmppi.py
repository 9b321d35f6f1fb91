"""Thin Python binding of the C ABI in include/brmppi.h -- same names, argument marshalling only.

PyTorch provides device memory (the workspace tensor) and the CUDA stream; every step of the hot
path runs in libbrmppi.so's kernels.  There is no CPU fallback: if the CUDA library is missing or
no device is present, construction raises."""
import ctypes as C

import numpy as np

from . import build as _build

MAX_DISCS = 4
FLAG_WRITE_SAMPLES = 1
FLAG_PRECISE_MATH = 2
FLAG_KERNEL_THREAD_PER_SAMPLE = 4
FLAG_PHASE_TIMING = 8
FLAG_NO_CULL = 16
FLAG_PROJECTED = 32
FLAG_MPCC = 64

OK = 0
ERR_NULL, ERR_INVALID_ARG, ERR_WORKSPACE_TOO_SMALL, ERR_TOO_MANY_OBSTACLES = -1, -2, -3, -4
ERR_NONFINITE_INPUT, ERR_NOT_READY, ERR_CUDA, ERR_UNALIGNED = -5, -6, -7, -8
ERR_TOO_LARGE = -9
HITCH_STATIC_MAX_N = 16384

EXPORTS = [
    "brmppi_workspace_bytes", "brmppi_create", "brmppi_destroy", "brmppi_set_state",
    "brmppi_set_goal", "brmppi_set_obstacles", "brmppi_set_superellipses", "brmppi_get_superellipses", "brmppi_set_nominal", "brmppi_set_counter",
    "brmppi_reset", "brmppi_solve", "brmppi_solve_get_controls", "brmppi_solve_host", "brmppi_shift", "brmppi_step", "brmppi_get_controls",
    "brmppi_get_state", "brmppi_get_obstacles", "brmppi_get_costs", "brmppi_get_final_states",
    "brmppi_get_diag", "brmppi_get_phase_times", "brmppi_time_kernels", "brmppi_launch_count", "brmppi_strerror", "brmppi_debug_philox",
    "brmppi_debug_sample_controls", "brmppi_measure_peaks", "brmppi_get_hitch_filter", "brmppi_hitch_filter", "brmppi_project",
    "brmppi_debug_philox_raw", "brmppi_hitch_filter_scratch_bytes", "brmppi_project_scratch_bytes",
    "brmppi_measure_peaks_scratch_bytes", "brmppi_shard_words", "brmppi_shard_export", "brmppi_shard_import",
    "brmppi_set_state7", "brmppi_set_reference_path", "brmppi_get_state7", "brmppi_get_final_states7",
    "brmppi_hitch_filter_static", "brmppi_set_inputs",
]


class Obstacle(C.Structure):
    _fields_ = [("cx", C.c_float), ("cy", C.c_float), ("radius", C.c_float),
                ("vx", C.c_float), ("vy", C.c_float)]


class Superellipse(C.Structure):
    _fields_ = [("cx", C.c_float), ("cy", C.c_float), ("mx", C.c_float), ("my", C.c_float),
                ("theta", C.c_float), ("vx", C.c_float), ("vy", C.c_float), ("exponent", C.c_int)]


class Disc(C.Structure):
    _fields_ = [("body", C.c_int), ("offset", C.c_float)]


class CParams(C.Structure):
    _fields_ = [("K", C.c_int), ("T", C.c_int), ("n_iter", C.c_int), ("n_scenes", C.c_int),
                ("max_obstacles", C.c_int), ("n_discs", C.c_int), ("discs", Disc * MAX_DISCS),
                ("disc_radius", C.c_float),
                ("dt", C.c_float), ("L1", C.c_float), ("L2", C.c_float), ("Lh", C.c_float),
                ("v_min", C.c_float), ("v_max", C.c_float),
                ("delta_min", C.c_float), ("delta_max", C.c_float),
                ("sigma_v", C.c_float), ("sigma_delta", C.c_float),
                ("alpha_lo", C.c_float), ("alpha_hi", C.c_float),
                ("w_pos", C.c_float), ("w_head", C.c_float), ("w_v", C.c_float),
                ("w_delta", C.c_float), ("w_hitch", C.c_float), ("hitch_max", C.c_float),
                ("w_bar", C.c_float), ("w_term", C.c_float), ("lam", C.c_float),
                ("seed", C.c_ulonglong), ("flags", C.c_uint), ("max_superellipses", C.c_int),
                ("hitch_kappa", C.c_float), ("hitch_filter", C.c_int), ("hitch_alpha", C.c_float),
                ("hitch_qv", C.c_float), ("hitch_qdelta", C.c_float),
                ("proj_qv", C.c_float), ("proj_qomega", C.c_float), ("proj_qalpha", C.c_float), ("proj_rho", C.c_float),
                ("sigma_ualpha", C.c_float), ("ualpha_max", C.c_float), ("w_alpha", C.c_float), ("h_buffer", C.c_float),
                ("k_offset", C.c_int),
                ("j_min", C.c_float), ("j_max", C.c_float), ("omega_min", C.c_float), ("omega_max", C.c_float),
                ("sigma_j", C.c_float), ("sigma_omega", C.c_float),
                ("Qc", C.c_float), ("Ql", C.c_float), ("Qth1", C.c_float), ("Qth2", C.c_float),
                ("Rj", C.c_float), ("Rw", C.c_float), ("mu", C.c_float), ("nu_bar", C.c_float),
                ("max_path_segments", C.c_int)]


class Diag(C.Structure):
    _fields_ = [("S_min", C.c_float), ("argmin", C.c_int), ("eta", C.c_float), ("ess", C.c_float),
                ("n", C.c_ulonglong), ("nonfinite", C.c_int)]


class BrmppiError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"brmppi status {status}: {text}")
        self.status = status


_lib = None
_fp = C.POINTER(C.c_float)


def lib():
    """Load libbrmppi.so (building it in-tree first if its sources are newer)."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp = C.c_void_p
        L.brmppi_workspace_bytes.argtypes = [C.POINTER(CParams)]
        L.brmppi_workspace_bytes.restype = C.c_size_t
        L.brmppi_create.argtypes = [C.POINTER(CParams), vp, C.c_size_t, vp, C.POINTER(vp)]
        L.brmppi_destroy.argtypes = [vp]
        L.brmppi_set_state.argtypes = [vp, C.c_int, _fp]
        L.brmppi_set_goal.argtypes = [vp, C.c_int, _fp]
        L.brmppi_set_state7.argtypes = [vp, C.c_int, _fp, C.c_float]
        L.brmppi_set_reference_path.argtypes = [vp, C.c_int, C.c_int, C.c_float, _fp]
        L.brmppi_get_state7.argtypes = [vp, C.c_int, _fp]
        L.brmppi_get_final_states7.argtypes = [vp, C.c_int, _fp]
        L.brmppi_set_obstacles.argtypes = [vp, C.c_int, C.c_int, C.POINTER(Obstacle)]
        L.brmppi_set_inputs.argtypes = [vp, C.c_int, vp, vp, C.c_int, vp]     # addresses passed as integers
        L.brmppi_set_superellipses.argtypes = [vp, C.c_int, C.c_int, C.POINTER(Superellipse)]
        L.brmppi_get_superellipses.argtypes = [vp, C.c_int, C.POINTER(C.c_int), C.POINTER(Superellipse)]
        L.brmppi_set_nominal.argtypes = [vp, C.c_int, _fp]
        L.brmppi_set_counter.argtypes = [vp, C.c_uint]
        L.brmppi_reset.argtypes = [vp]
        L.brmppi_solve.argtypes = [vp]
        L.brmppi_solve_get_controls.argtypes = [vp, vp]
        L.brmppi_solve_host.argtypes = [vp, vp, vp, C.c_int, vp, vp]
        L.brmppi_shift.argtypes = [vp]
        L.brmppi_shard_words.argtypes = [vp]
        L.brmppi_shard_words.restype = C.c_size_t
        L.brmppi_shard_export.argtypes = [vp, vp]
        L.brmppi_shard_import.argtypes = [vp, C.c_int, vp]
        L.brmppi_step.argtypes = [vp, _fp]
        L.brmppi_get_controls.argtypes = [vp, C.c_int, _fp]
        L.brmppi_get_state.argtypes = [vp, C.c_int, _fp]
        L.brmppi_get_obstacles.argtypes = [vp, C.c_int, C.POINTER(C.c_int), C.POINTER(Obstacle)]
        L.brmppi_get_costs.argtypes = [vp, C.c_int, _fp]
        L.brmppi_get_final_states.argtypes = [vp, C.c_int, _fp]
        L.brmppi_get_diag.argtypes = [vp, C.c_int, C.POINTER(Diag)]
        L.brmppi_get_phase_times.argtypes = [vp, _fp]
        L.brmppi_time_kernels.argtypes = [vp, C.c_int, _fp]
        L.brmppi_launch_count.argtypes = [vp]
        L.brmppi_launch_count.restype = C.c_ulonglong
        L.brmppi_strerror.argtypes = [C.c_int]
        L.brmppi_strerror.restype = C.c_char_p
        L.brmppi_debug_philox.argtypes = [vp, C.c_ulonglong, C.c_uint, C.c_int, C.c_int, C.c_uint, vp]
        L.brmppi_debug_philox_raw.argtypes = [vp, C.c_int, vp, vp, C.c_int, vp]
        L.brmppi_debug_sample_controls.argtypes = [vp, C.POINTER(CParams), C.c_uint, vp, vp, vp]
        L.brmppi_measure_peaks_scratch_bytes.argtypes = []
        L.brmppi_measure_peaks_scratch_bytes.restype = C.c_size_t
        L.brmppi_measure_peaks.argtypes = [vp, vp, C.c_size_t, _fp]
        L.brmppi_project_scratch_bytes.argtypes = [C.c_int, C.c_int]
        L.brmppi_project_scratch_bytes.restype = C.c_size_t
        L.brmppi_project.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp, _fp, C.c_float, _fp, _fp, vp, C.c_int, vp, C.c_size_t]
        L.brmppi_get_hitch_filter.argtypes = [vp, C.c_int, _fp, C.POINTER(C.c_int)]
        L.brmppi_hitch_filter_scratch_bytes.argtypes = [C.c_int]
        L.brmppi_hitch_filter_scratch_bytes.restype = C.c_size_t
        L.brmppi_hitch_filter.argtypes = [vp, C.POINTER(CParams), C.c_int, _fp, _fp, _fp, C.POINTER(C.c_int), vp, C.c_size_t]
        L.brmppi_hitch_filter_static.argtypes = [vp, C.POINTER(CParams), C.c_int, _fp, _fp, _fp, C.POINTER(C.c_int)]
        _lib = L
    return _lib


def strerror(status):
    return lib().brmppi_strerror(int(status)).decode()


def _check(status):
    if status != OK:
        raise BrmppiError(status, strerror(status))


def make_cparams(p, n_scenes=1, max_obstacles=8, flags=0, max_superellipses=0, k_offset=0,
                 max_path_segments=64) -> CParams:
    """scenes.Params (plain data) -> brmppi_params."""
    c = CParams()
    c.K, c.T, c.n_iter, c.n_scenes = int(p.K), int(p.T), int(p.n_iter), int(n_scenes)
    c.max_obstacles, c.n_discs = int(max_obstacles), len(p.discs)
    for j, (body, off) in enumerate(p.discs):
        c.discs[j].body, c.discs[j].offset = int(body), float(off)
    for name in ("disc_radius", "dt", "L1", "L2", "Lh", "v_min", "v_max", "delta_min", "delta_max",
                 "sigma_v", "sigma_delta", "alpha_lo", "alpha_hi", "w_pos", "w_head", "w_v",
                 "w_delta", "w_hitch", "hitch_max", "w_bar", "w_term", "lam"):
        setattr(c, name, float(getattr(p, name)))
    c.seed, c.flags = int(p.seed) & 0xFFFFFFFFFFFFFFFF, int(flags)
    c.max_superellipses = int(max_superellipses)
    c.hitch_kappa = float(getattr(p, "hitch_kappa", 0.0))
    c.hitch_filter = int(getattr(p, "hitch_filter", 0))
    c.hitch_alpha = float(getattr(p, "hitch_alpha", 0.5))
    c.hitch_qv = float(getattr(p, "hitch_qv", 1.0))
    c.hitch_qdelta = float(getattr(p, "hitch_qdelta", 1.0))
    for name, default in (("proj_qv", 1.0), ("proj_qomega", 4.0), ("proj_qalpha", 0.5), ("proj_rho", 0.25),
                          ("sigma_ualpha", 0.3), ("ualpha_max", 1.0), ("w_alpha", 10.0), ("h_buffer", 0.5)):
        setattr(c, name, float(getattr(p, name, default)))
    c.k_offset = int(k_offset)
    for name, default in (("j_min", -2.0), ("j_max", 2.0), ("omega_min", -0.9), ("omega_max", 0.9), ("sigma_j", 0.8),
                          ("sigma_omega", 0.3), ("Qc", 2.0), ("Ql", 0.5), ("Qth1", 0.5), ("Qth2", 0.5), ("Rj", 0.01),
                          ("Rw", 0.1), ("mu", 0.2), ("nu_bar", 1.5)):
        setattr(c, name, float(getattr(p, name, default)))
    c.max_path_segments = int(max_path_segments)
    return c


def _f32(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a.reshape(shape) if shape is not None else a


def _p(a):
    return a.ctypes.data_as(_fp)


class Solver:
    """One brmppi_ctx plus the torch-owned workspace and stream it lives on."""

    def __init__(self, params, n_scenes=1, max_obstacles=8, flags=0, stream=None, device="cuda:0",
                 max_superellipses=0, k_offset=0, max_path_segments=64):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("brmppi needs a CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.params = params
        self.cparams = make_cparams(params, n_scenes, max_obstacles, flags, max_superellipses, k_offset,
                                    max_path_segments)
        self.mpcc = bool(flags & FLAG_MPCC)
        self.max_superellipses = int(max_superellipses)
        self.n_scenes, self.K, self.T = int(n_scenes), int(params.K), int(params.T)
        self.max_obstacles = int(max_obstacles)
        L = lib()
        nbytes = L.brmppi_workspace_bytes(C.byref(self.cparams))
        if nbytes == 0:
            raise BrmppiError(ERR_INVALID_ARG, strerror(ERR_INVALID_ARG))
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        self._ctx = C.c_void_p()
        torch.cuda.synchronize(self.device)
        _check(L.brmppi_create(C.byref(self.cparams), C.c_void_p(ptr), C.c_size_t(nbytes),
                               C.c_void_p(self.stream.cuda_stream), C.byref(self._ctx)))

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.stream.synchronize()
            lib().brmppi_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- inputs -------------------------------------------------------------------------
    def set_state(self, x, scene=0):
        _check(lib().brmppi_set_state(self._ctx, scene, _p(_f32(x, (4,)))))

    def set_goal(self, g, scene=0):
        _check(lib().brmppi_set_goal(self._ctx, scene, _p(_f32(g, (4,)))))

    def set_obstacles(self, obstacles, scene=0):
        obs = _f32(obstacles).reshape(-1, 5)
        n = obs.shape[0]
        ptr = obs.ctypes.data_as(C.POINTER(Obstacle)) if n else None
        _check(lib().brmppi_set_obstacles(self._ctx, scene, n, ptr))

    def set_inputs(self, x, g, obstacles, scene=0):
        """State, goal and obstacles of one scene in one call (one host-to-device copy in a single-scene context)."""
        x, g, obs = _f32(x, (4,)), _f32(g, (4,)), _f32(obstacles).reshape(-1, 5)
        n = obs.shape[0]
        adr = lambda a: a.__array_interface__["data"][0]       # cheaper than building ctypes pointer objects
        _check(lib().brmppi_set_inputs(self._ctx, scene, adr(x), adr(g), n, adr(obs) if n else None))

    def set_superellipses(self, superellipses, scene=0):
        """rows (cx, cy, mx, my, theta, vx, vy, exponent)"""
        se = np.asarray(superellipses, dtype=np.float64).reshape(-1, 8)
        arr = (Superellipse * max(len(se), 1))()
        for i, r in enumerate(se):
            arr[i] = Superellipse(*[float(x) for x in r[:7]], int(round(r[7])))
        _check(lib().brmppi_set_superellipses(self._ctx, scene, len(se), arr if len(se) else None))

    def get_superellipses(self, scene=0):
        n = C.c_int(0)
        arr = (Superellipse * max(self.max_superellipses, 1))()
        _check(lib().brmppi_get_superellipses(self._ctx, scene, C.byref(n), arr))
        return np.array([[a.cx, a.cy, a.mx, a.my, a.theta, a.vx, a.vy, a.exponent] for a in arr[:n.value]]).reshape(-1, 8)

    def set_nominal(self, U=None, scene=0):
        _check(lib().brmppi_set_nominal(self._ctx, scene, None if U is None else _p(_f32(U, (self.T, 2)))))

    def set_counter(self, n):
        _check(lib().brmppi_set_counter(self._ctx, int(n)))

    def reset(self):
        _check(lib().brmppi_reset(self._ctx))

    def set_reference_path(self, coef, dpsi, scene=0):
        """FLAG_MPCC: coef [M][4][4] cubic coefficients of (p^{x,r}, p^{y,r}, theta^{1,r}, theta^{2,r})."""
        coef = _f32(coef)
        M = coef.shape[0]
        _check(lib().brmppi_set_reference_path(self._ctx, scene, int(M), float(dpsi), _p(_f32(coef, (M, 4, 4)))))

    def set_state7(self, x, psi, scene=0):
        _check(lib().brmppi_set_state7(self._ctx, scene, _p(_f32(x, (7,))), float(psi)))

    def set_scene(self, scene_obj, scene=0):
        if self.mpcc:                     # a scenes.PathScene
            self.set_reference_path(scene_obj.coef, scene_obj.dpsi, scene)
            self.set_state7(scene_obj.x0, scene_obj.psi0, scene)
            self.set_obstacles(scene_obj.obstacles, scene)
            return
        self.set_state(scene_obj.x0, scene)
        self.set_goal(scene_obj.goal, scene)
        self.set_obstacles(scene_obj.obstacles, scene)
        if self.max_superellipses > 0:
            se = getattr(scene_obj, "superellipses", None)
            self.set_superellipses(np.zeros((0, 8)) if se is None else se, scene)

    # ---- work ---------------------------------------------------------------------------
    def solve(self):
        _check(lib().brmppi_solve(self._ctx))

    def solve_get_controls(self, out=None):
        """solve() and the new nominal of every scene, [n_scenes][T][2], in one call (no copy behind the solve)."""
        if out is None:
            out = np.empty((self.n_scenes, self.T, 2), dtype=np.float32)
        assert out.dtype == np.float32 and out.flags.c_contiguous and out.size == self.n_scenes * self.T * 2
        _check(lib().brmppi_solve_get_controls(self._ctx, C.c_void_p(out.ctypes.data)))
        return out

    def solve_host(self, x, g, obstacles, out=None):
        """set_inputs(x, g, obstacles) + solve_get_controls() as one call (one graph launch in a single-scene context)."""
        x, g, obs = _f32(x, (4,)), _f32(g, (4,)), _f32(obstacles).reshape(-1, 5)
        n = obs.shape[0]
        if out is None:
            out = np.empty((self.n_scenes, self.T, 2), dtype=np.float32)
        assert out.dtype == np.float32 and out.flags.c_contiguous and out.size == self.n_scenes * self.T * 2
        adr = lambda a: a.__array_interface__["data"][0]
        _check(lib().brmppi_solve_host(self._ctx, adr(x), adr(g), n, adr(obs) if n else None, adr(out)))
        return out

    def shift(self):
        _check(lib().brmppi_shift(self._ctx))

    # ---- K-sharded solves -------------------------------------------------------
    def shard_words(self):
        return int(lib().brmppi_shard_words(self._ctx))

    def shard_export(self, record):
        """Rollout of this context's samples, merged into one record (float32 CUDA tensor of shard_words())."""
        assert record.is_cuda and record.is_contiguous() and record.numel() >= self.shard_words()
        _check(lib().brmppi_shard_export(self._ctx, C.c_void_p(record.data_ptr())))

    def shard_import(self, records, n_shards):
        """Merge n_shards records (float32 CUDA tensor [n_shards][shard_words()], in shard order) into U."""
        assert records.is_cuda and records.is_contiguous() and records.numel() >= n_shards * self.shard_words()
        _check(lib().brmppi_shard_import(self._ctx, int(n_shards), C.c_void_p(records.data_ptr())))

    def step(self):
        u0 = np.zeros((self.n_scenes, 2), dtype=np.float32)
        _check(lib().brmppi_step(self._ctx, _p(u0)))
        return u0

    def synchronize(self):
        self.stream.synchronize()

    # ---- outputs ------------------------------------------------------------------------
    def get_controls(self, scene=0):
        U = np.zeros((self.T, 2), dtype=np.float32)
        _check(lib().brmppi_get_controls(self._ctx, scene, _p(U)))
        return U

    def get_state(self, scene=0):
        x = np.zeros(4, dtype=np.float32)
        _check(lib().brmppi_get_state(self._ctx, scene, _p(x)))
        return x

    def get_state7(self, scene=0):
        """FLAG_MPCC: (p_x, p_y, v, a, theta1, theta2, delta, psi)."""
        x = np.zeros(8, dtype=np.float32)
        _check(lib().brmppi_get_state7(self._ctx, scene, _p(x)))
        return x

    def get_final_states7(self, scene=0):
        X = np.zeros((self.K, 8), dtype=np.float32)
        _check(lib().brmppi_get_final_states7(self._ctx, scene, _p(X)))
        return X

    def get_obstacles(self, scene=0):
        n = C.c_int(0)
        buf = np.zeros((max(self.max_obstacles, 1), 5), dtype=np.float32)
        _check(lib().brmppi_get_obstacles(self._ctx, scene, C.byref(n), buf.ctypes.data_as(C.POINTER(Obstacle))))
        return buf[:n.value].copy()

    def get_costs(self, scene=0):
        S = np.zeros(self.K, dtype=np.float32)
        _check(lib().brmppi_get_costs(self._ctx, scene, _p(S)))
        return S

    def get_final_states(self, scene=0):
        X = np.zeros((self.K, 4), dtype=np.float32)
        _check(lib().brmppi_get_final_states(self._ctx, scene, _p(X)))
        return X

    def get_diag(self, scene=0):
        d = Diag()
        _check(lib().brmppi_get_diag(self._ctx, scene, C.byref(d)))
        return dict(S_min=d.S_min, argmin=d.argmin, eta=d.eta, ess=d.ess, n=d.n, nonfinite=d.nonfinite)

    def get_hitch_filter(self, scene=0):
        """(u_ref, status) of the hitch-angle stabiliser in the last step()."""
        u = np.zeros(2, dtype=np.float32)
        st = C.c_int()
        _check(lib().brmppi_get_hitch_filter(self._ctx, scene, _p(u), C.byref(st)))
        return u, int(st.value)

    def time_kernels(self, reps=20):
        """Mean device ms per launch of (rollout kernel, merge/update kernel)."""
        out = np.zeros(2, dtype=np.float32)
        _check(lib().brmppi_time_kernels(self._ctx, int(reps), _p(out)))
        return float(out[0]), float(out[1])

    def get_phase_times(self):
        """Per-phase microseconds of the last rollout launch (FLAG_PHASE_TIMING)."""
        out = np.zeros(8, dtype=np.float32)
        _check(lib().brmppi_get_phase_times(self._ctx, _p(out)))
        names = ("prologue", "A_noise", "B_chain", "C_cost", "D_reduce", "E_update", "partial_out", "span")
        return dict(zip(names, (float(x) for x in out)))

    def launch_count(self):
        return int(lib().brmppi_launch_count(self._ctx))


def debug_philox(seed, n, K, T, tag=0):
    """Raw Philox words of the in-kernel generator: uint32 array [K][T][4]."""
    import torch
    out = torch.empty(K * T * 4, dtype=torch.int32, device="cuda")
    st = torch.cuda.current_stream()
    _check(lib().brmppi_debug_philox(C.c_void_p(st.cuda_stream), int(seed) & 0xFFFFFFFFFFFFFFFF, int(n),
                                     int(K), int(T), int(tag), C.c_void_p(out.data_ptr())))
    return out.cpu().numpy().view(np.uint32).reshape(K, T, 4)


def debug_philox_raw(ctr, key, use_curand=False):
    """Philox4x32-10 blocks for arbitrary (counter [n][4], key [n][2]) uint32 arrays: through the library's
    generator, or through the toolkit's raw curand_Philox4x32_10 device function.  uint32 [n][4]."""
    import torch
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    n = ctr.shape[0]
    assert key.shape[0] == n
    dc = torch.from_numpy(ctr.view(np.int32)).cuda()
    dk = torch.from_numpy(key.view(np.int32)).cuda()
    out = torch.empty((max(n, 1), 4), dtype=torch.int32, device="cuda")
    st = torch.cuda.current_stream()
    st.synchronize()
    _check(lib().brmppi_debug_philox_raw(C.c_void_p(st.cuda_stream), n, C.c_void_p(dc.data_ptr()), C.c_void_p(dk.data_ptr()),
                                         1 if use_curand else 0, C.c_void_p(out.data_ptr())))
    return out[:n].cpu().numpy().view(np.uint32)


def debug_sample_controls(params, n, U_nominal=None, flags=0):
    """Perturbed, clamped controls u[K][T][2] and alpha[K] exactly as the kernels draw them."""
    import torch
    cp = make_cparams(params, 1, 0, flags)
    u = torch.empty(params.K * params.T * 2, dtype=torch.float32, device="cuda")
    a = torch.empty(params.K, dtype=torch.float32, device="cuda")
    Un = torch.from_numpy(_f32(np.zeros((params.T, 2)) if U_nominal is None else U_nominal, (params.T, 2))).cuda()
    st = torch.cuda.current_stream()
    st.synchronize()
    _check(lib().brmppi_debug_sample_controls(C.c_void_p(st.cuda_stream), C.byref(cp), int(n), C.c_void_p(Un.data_ptr()),
                                              C.c_void_p(u.data_ptr()), C.c_void_p(a.data_ptr())))
    return u.cpu().numpy().reshape(params.K, params.T, 2), a.cpu().numpy()


def _scratch(nbytes):
    import torch
    return torch.empty(max(int(nbytes), 1), dtype=torch.uint8, device="cuda")


def hitch_filter(params, x, u_ref):
    """Hitch-angle stabiliser (Sec. V-D) for n (state, reference control) pairs: (u[n][2], status[n])."""
    import torch
    x = _f32(x).reshape(-1, 4)
    r = _f32(u_ref).reshape(-1, 2)
    n = x.shape[0]
    assert r.shape[0] == n
    cp = make_cparams(params, 1, 0, 0)
    u = np.zeros((n, 2), dtype=np.float32)
    status = np.zeros(n, dtype=np.int32)
    nb = lib().brmppi_hitch_filter_scratch_bytes(n)
    scratch = _scratch(nb)
    st = torch.cuda.current_stream()
    st.synchronize()
    _check(lib().brmppi_hitch_filter(C.c_void_p(st.cuda_stream), C.byref(cp), n, _p(x), _p(r), _p(u),
                                     status.ctypes.data_as(C.POINTER(C.c_int)), C.c_void_p(scratch.data_ptr()), C.c_size_t(nb)))
    return u, status


def hitch_filter_static(params, x, u_ref):
    """hitch_filter through the library's static device scratch (no device allocation anywhere on the call:
    brmppi_hitch_filter_static); n <= HITCH_STATIC_MAX_N, else BrmppiError with status ERR_TOO_LARGE."""
    import torch
    x = _f32(x).reshape(-1, 4)
    r = _f32(u_ref).reshape(-1, 2)
    n = x.shape[0]
    assert r.shape[0] == n
    cp = make_cparams(params, 1, 0, 0)
    u = np.zeros((n, 2), dtype=np.float32)
    status = np.zeros(n, dtype=np.int32)
    st = torch.cuda.current_stream()
    st.synchronize()
    _check(lib().brmppi_hitch_filter_static(C.c_void_p(st.cuda_stream), C.byref(cp), n, _p(x), _p(r), _p(u),
                                            status.ctypes.data_as(C.POINTER(C.c_int))))
    return u, status


def project(A, b, z_des, w, rho, z_lo, z_hi, out=None, scratch=None):
    """Closed-form projection (12) for a batch.  numpy arrays (or CPU torch tensors, e.g. page-locked ones) ->
    HOST-pointer call through a caller-owned device scratch, returns numpy [n][d]; torch CUDA tensors (float32,
    contiguous) -> DEVICE-pointer call on the current stream, returns a tensor."""
    import torch
    st = torch.cuda.current_stream()
    on_device = isinstance(A, torch.Tensor) and A.is_cuda
    n, n_o, d = A.shape
    w, z_lo, z_hi = _f32(w, (d,)), _f32(z_lo, (d,)), _f32(z_hi, (d,))
    if on_device:
        for t in (A, b, z_des):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
        if out is None:
            out = torch.empty((n, d), dtype=torch.float32, device=A.device)
        ptr = lambda t: C.c_void_p(t.data_ptr())
        _check(lib().brmppi_project(C.c_void_p(st.cuda_stream), n, n_o, ptr(A), ptr(b), ptr(z_des), _p(w),
                                    float(rho), _p(z_lo), _p(z_hi), ptr(out), 1, None, 0))
        return out
    if isinstance(A, torch.Tensor):            # CPU tensors (page-locked staging): no copies on the way in
        for t in (A, b, z_des):
            assert t.dtype == torch.float32 and t.is_contiguous()
        ptr = lambda t: C.c_void_p(t.data_ptr())
        if out is None:
            out = torch.empty((n, d), dtype=torch.float32).pin_memory()
        ret = out.numpy()
    else:
        A, b, z_des = _f32(A), _f32(b, (n, n_o)), _f32(z_des, (n, d))
        ptr = lambda a: C.c_void_p(a.ctypes.data)
        out = np.zeros((n, d), dtype=np.float32) if out is None else out
        ret = out
    nb = lib().brmppi_project_scratch_bytes(n, n_o)
    if scratch is None:
        scratch = _scratch(nb)
        st.synchronize()
    _check(lib().brmppi_project(C.c_void_p(st.cuda_stream), n, n_o, ptr(A), ptr(b), ptr(z_des), _p(w),
                                float(rho), _p(z_lo), _p(z_hi), ptr(out), 0, C.c_void_p(scratch.data_ptr()),
                                C.c_size_t(scratch.numel())))
    return ret


def measure_peaks():
    import torch
    out = np.zeros(16, dtype=np.float32)
    nb = lib().brmppi_measure_peaks_scratch_bytes()
    scratch = _scratch(nb)
    st = torch.cuda.current_stream()
    st.synchronize()
    _check(lib().brmppi_measure_peaks(C.c_void_p(st.cuda_stream), C.c_void_p(scratch.data_ptr()), C.c_size_t(nb), _p(out)))
    return dict(ffma=float(out[0]), alu=float(out[1]), mufu=float(out[2]), mix=float(out[3]),
                imad_wide=float(out[4]), n_sms=int(out[5]), sm_mhz=float(out[6]),
                sm_mhz_under_ffma=float(out[7]), fmnmx=float(out[8]), ffma2=float(out[9]),
                ffma2_distinct_operands=float(out[10]), fadd2=float(out[11]), ffma_fmnmx_mix=float(out[12]),
                ffma2_fmnmx_mix=float(out[13]), imad_lo=float(out[14]), imad_hi=float(out[15]))
