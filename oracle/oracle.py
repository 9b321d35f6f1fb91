"""ctypes front-end of the CPU oracle (oracle/brmppi_oracle.c).  TEST INFRASTRUCTURE ONLY:
imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs,
never by paper_2508_05773_b200/.  Argument marshalling only -- all arithmetic is in the C file."""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "brmppi_oracle.c")
# oracle/oracle32.py executes this file a second time with _ORACLE_FP32 set: the same front-end over the fp32 re-run
# build of the same C source (SURVEY 8(c) reading 23: prints the fp32 noise floor, never a parity reference)
_FP32 = bool(globals().get("_ORACLE_FP32", False))
_LIB = os.path.join(_HERE, "liboracle32.so" if _FP32 else "liboracle.so")
_REAL_C = C.c_float if _FP32 else C.c_double
_REAL_NP = np.float32 if _FP32 else np.float64
ORC_MAX_DISCS = 4


def _zeros(shape):
    return np.zeros(shape, dtype=_REAL_NP)


def build(force: bool = False) -> str:
    """gcc -O2 build of liboracle.so next to its source (rebuilt when the source is newer)."""
    hdr = os.path.join(_HERE, "brmppi_oracle.h")
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(f) > os.path.getmtime(_LIB) for f in (_SRC, hdr))
    if force or stale:
        mode = ["-DORC_FP32", "-fsingle-precision-constant", "-Wno-overflow"] if _FP32 else []
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off"] + mode + ["-fPIC", "-shared", "-o", _LIB, _SRC,
                                                                      "-lm", "-lpthread"]
        subprocess.check_call(cmd)
    return _LIB


class _Params(C.Structure):
    _fields_ = [("K", C.c_int), ("T", C.c_int), ("n_discs", C.c_int),
                ("disc_body", C.c_int * ORC_MAX_DISCS), ("disc_offset", _REAL_C * ORC_MAX_DISCS),
                ("disc_radius", _REAL_C),
                ("dt", _REAL_C), ("L1", _REAL_C), ("L2", _REAL_C), ("Lh", _REAL_C),
                ("v_min", _REAL_C), ("v_max", _REAL_C),
                ("delta_min", _REAL_C), ("delta_max", _REAL_C),
                ("sigma_v", _REAL_C), ("sigma_delta", _REAL_C),
                ("alpha_lo", _REAL_C), ("alpha_hi", _REAL_C),
                ("w_pos", _REAL_C), ("w_head", _REAL_C), ("w_v", _REAL_C),
                ("w_delta", _REAL_C), ("w_hitch", _REAL_C), ("hitch_max", _REAL_C),
                ("w_bar", _REAL_C), ("w_term", _REAL_C), ("lam", _REAL_C), ("hitch_kappa", _REAL_C),
                ("hitch_alpha", _REAL_C), ("hitch_qv", _REAL_C), ("hitch_qdelta", _REAL_C),
                ("seed", C.c_uint64)]


class _ProjParams(C.Structure):
    _fields_ = [("q_v", _REAL_C), ("q_omega", _REAL_C), ("q_alpha", _REAL_C), ("rho", _REAL_C),
                ("sigma_ualpha", _REAL_C), ("ualpha_max", _REAL_C), ("w_alpha", _REAL_C),
                ("h_buffer", _REAL_C)]


class _MpccParams(C.Structure):
    _fields_ = [("j_min", _REAL_C), ("j_max", _REAL_C), ("omega_min", _REAL_C), ("omega_max", _REAL_C),
                ("sigma_j", _REAL_C), ("sigma_omega", _REAL_C), ("delta_lo", _REAL_C), ("delta_hi", _REAL_C),
                ("Qc", _REAL_C), ("Ql", _REAL_C), ("Qth1", _REAL_C), ("Qth2", _REAL_C),
                ("Rj", _REAL_C), ("Rw", _REAL_C), ("mu", _REAL_C), ("nu_bar", _REAL_C),
                ("M", C.c_int), ("dpsi", _REAL_C), ("coef", C.POINTER(_REAL_C))]


_lib = None
_dp = C.POINTER(_REAL_C)
_u32p = C.POINTER(C.c_uint32)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
        L.orc_philox4x32_10.restype = None
        L.orc_uniform.argtypes = [C.c_uint32]
        L.orc_uniform.restype = _REAL_C
        L.orc_normals.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _dp]
        L.orc_normals.restype = None
        L.orc_alpha.argtypes = [C.POINTER(_Params), C.c_uint32, C.c_uint32]
        L.orc_alpha.restype = _REAL_C
        L.orc_wrap.argtypes = [_REAL_C]
        L.orc_wrap.restype = _REAL_C
        L.orc_kinematic_step.argtypes = [C.POINTER(_Params), _dp, _REAL_C, _REAL_C, _dp]
        L.orc_kinematic_step.restype = None
        L.orc_disc_centre.argtypes = [C.POINTER(_Params), _dp, C.c_int, _dp]
        L.orc_disc_centre.restype = None
        L.orc_barrier.argtypes = [C.POINTER(_Params), _dp, _dp, _REAL_C]
        L.orc_barrier.restype = _REAL_C
        L.orc_goal_cost.argtypes = [C.POINTER(_Params), _dp, _dp]
        L.orc_goal_cost.restype = _REAL_C
        L.orc_rollout.argtypes = [C.POINTER(_Params), _dp, _dp, C.c_int, _dp, _dp, _REAL_C,
                                  _dp, _dp, _dp]
        L.orc_rollout.restype = _REAL_C
        L.orc_sample.argtypes = [C.POINTER(_Params), C.c_uint32, C.c_uint32, _dp, _dp, C.c_int, _dp,
                                 _dp, _dp, _dp]
        L.orc_sample.restype = _REAL_C
        L.orc_weights_update.argtypes = [C.c_int, C.c_int, _REAL_C, _dp, _dp, _dp, _dp,
                                         C.POINTER(C.c_int), _dp, _dp]
        L.orc_weights_update.restype = C.c_int
        L.orc_iteration.argtypes = [C.POINTER(_Params), C.c_uint32, _dp, _dp, C.c_int, _dp, _dp,
                                    _dp, _dp, _dp, _dp, _dp, C.POINTER(C.c_int), _dp, _dp, C.c_int]
        L.orc_iteration.restype = C.c_int
        L.orc_barrier_se.argtypes = [C.POINTER(_Params), _dp, _dp, _dp]
        L.orc_barrier_se.restype = _REAL_C
        L.orc_rollout_se.argtypes = [C.POINTER(_Params), _dp, _dp, C.c_int, _dp, C.c_int, _dp, _dp,
                                     _REAL_C, _dp, _dp, _dp]
        L.orc_rollout_se.restype = _REAL_C
        L.orc_sample_se.argtypes = [C.POINTER(_Params), C.c_uint32, C.c_uint32, _dp, _dp, C.c_int, _dp,
                                    C.c_int, _dp, _dp, _dp, _dp]
        L.orc_sample_se.restype = _REAL_C
        L.orc_iteration_se.argtypes = [C.POINTER(_Params), C.c_uint32, _dp, _dp, C.c_int, _dp, C.c_int, _dp,
                                       _dp, _dp, _dp, _dp, _dp, _dp, C.POINTER(C.c_int), _dp, _dp, C.c_int]
        L.orc_iteration_se.restype = C.c_int
        L.orc_advance_se.argtypes = [C.POINTER(_Params), C.c_int, _dp]
        L.orc_advance_se.restype = None
        L.orc_shift.argtypes = [C.c_int, _dp]
        L.orc_shift.restype = None
        L.orc_plant_step.argtypes = [C.POINTER(_Params), _dp, _dp, C.c_int, _dp]
        L.orc_plant_step.restype = None
        L.orc_hitch_barrier.argtypes = [C.POINTER(_Params), _dp, _REAL_C]
        L.orc_hitch_barrier.restype = _REAL_C
        L.orc_hitch_rate_cond.argtypes = [C.POINTER(_Params), _dp, _dp]
        L.orc_hitch_rate_cond.restype = _REAL_C
        L.orc_hitch_constraint.argtypes = [C.POINTER(_Params), _dp, _dp, _dp, _dp]
        L.orc_hitch_constraint.restype = None
        L.orc_hitch_filter.argtypes = [C.POINTER(_Params), _dp, _dp, _dp]
        L.orc_hitch_filter.restype = C.c_int
        PP = C.POINTER(_ProjParams)
        ip = C.POINTER(C.c_int)
        L.orc_project.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp, _dp, _REAL_C, _dp, _dp, _dp]
        L.orc_project.restype = C.c_int
        L.orc_ualpha_normals.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_int, _dp]
        L.orc_ualpha_normals.restype = None
        L.orc_barrier_row.argtypes = [C.POINTER(_Params), _dp, _dp, C.c_int, _dp, ip, _dp, _dp]
        L.orc_barrier_row.restype = None
        L.orc_affine_step.argtypes = [C.POINTER(_Params), _dp, _dp, _dp]
        L.orc_affine_step.restype = None
        L.orc_rollout_projected.argtypes = [C.POINTER(_Params), PP, _dp, _dp, C.c_int, _dp, _dp, _dp, _REAL_C,
                                            _dp, _dp, _dp, _dp, _dp]
        L.orc_rollout_projected.restype = _REAL_C
        L.orc_sample_projected.argtypes = [C.POINTER(_Params), PP, C.c_uint32, C.c_uint32, _dp, _dp, C.c_int, _dp,
                                           _dp, _dp, _dp]
        L.orc_sample_projected.restype = _REAL_C
        L.orc_iteration_projected.argtypes = [C.POINTER(_Params), PP, C.c_uint32, _dp, _dp, C.c_int, _dp, _dp,
                                              _dp, _dp, _dp, _dp, _dp, ip, _dp, _dp, C.c_int]
        L.orc_iteration_projected.restype = C.c_int
        MP = C.POINTER(_MpccParams)
        L.orc7_step.argtypes = [C.POINTER(_Params), MP, _dp, _dp, _dp]
        L.orc7_step.restype = None
        L.orc_path_eval.argtypes = [MP, _REAL_C, _dp]
        L.orc_path_eval.restype = None
        L.orc7_progress.argtypes = [MP, _dp, _REAL_C]
        L.orc7_progress.restype = _REAL_C
        L.orc7_errors.argtypes = [MP, _dp, _REAL_C, _dp]
        L.orc7_errors.restype = None
        L.orc7_hhat.argtypes = [C.POINTER(_Params), _dp, _dp, _dp, C.c_int, C.c_int, _dp]
        L.orc7_hhat.restype = _REAL_C
        L.orc7_rollout.argtypes = [C.POINTER(_Params), MP, _dp, _REAL_C, C.c_int, _dp, _dp, _REAL_C, _dp, _dp]
        L.orc7_rollout.restype = _REAL_C
        L.orc7_sample.argtypes = [C.POINTER(_Params), MP, C.c_uint32, C.c_uint32, _dp, _REAL_C, C.c_int, _dp, _dp, _dp, _dp]
        L.orc7_sample.restype = _REAL_C
        L.orc7_iteration.argtypes = [C.POINTER(_Params), MP, C.c_uint32, _dp, _REAL_C, C.c_int, _dp, _dp, _dp, _dp, _dp,
                                     _dp, _dp, ip, _dp, _dp, C.c_int]
        L.orc7_iteration.restype = C.c_int
        _lib = L
    return _lib


def _pparams(p) -> _ProjParams:
    s = _ProjParams()
    s.q_v, s.q_omega, s.q_alpha, s.rho = float(p.proj_qv), float(p.proj_qomega), float(p.proj_qalpha), float(p.proj_rho)
    s.sigma_ualpha, s.ualpha_max = float(p.sigma_ualpha), float(p.ualpha_max)
    s.w_alpha, s.h_buffer = float(p.w_alpha), float(p.h_buffer)
    return s


def _cparams(p) -> _Params:
    """scenes.Params (plain data) -> C struct."""
    s = _Params()
    s.K, s.T, s.n_discs = int(p.K), int(p.T), len(p.discs)
    for j, (body, off) in enumerate(p.discs):
        s.disc_body[j] = int(body)
        s.disc_offset[j] = float(off)
    for name in ("disc_radius", "dt", "L1", "L2", "Lh", "v_min", "v_max", "delta_min",
                 "delta_max", "sigma_v", "sigma_delta", "alpha_lo", "alpha_hi", "w_pos", "w_head",
                 "w_v", "w_delta", "w_hitch", "hitch_max", "w_bar", "w_term", "lam", "hitch_kappa",
                 "hitch_alpha", "hitch_qv", "hitch_qdelta"):
        setattr(s, name, float(getattr(p, name)))
    s.seed = int(p.seed) & 0xFFFFFFFFFFFFFFFF
    return s


def _d(a, shape=None):
    a = np.ascontiguousarray(a, dtype=_REAL_NP)
    if shape is not None:
        a = a.reshape(shape)
    return a


def _ptr(a):
    return a.ctypes.data_as(_dp)


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def uniform(w):
    return lib().orc_uniform(int(w) & 0xFFFFFFFF)


def normals(seed, n, k, t):
    z = _zeros(2)
    lib().orc_normals(int(seed), int(n), int(k), int(t), _ptr(z))
    return z


def alpha(p, n, k):
    cp = _cparams(p)
    return lib().orc_alpha(C.byref(cp), int(n), int(k))


def wrap(a):
    return lib().orc_wrap(float(a))


def kinematic_step(p, x, v, delta):
    cp = _cparams(p)
    x = _d(x, (4,))
    xn = _zeros(4)
    lib().orc_kinematic_step(C.byref(cp), _ptr(x), float(v), float(delta), _ptr(xn))
    return xn


def disc_centre(p, x, j):
    cp = _cparams(p)
    x = _d(x, (4,))
    c = _zeros(2)
    lib().orc_disc_centre(C.byref(cp), _ptr(x), int(j), _ptr(c))
    return c


def barrier(p, c, o, R):
    cp = _cparams(p)
    c, o = _d(c, (2,)), _d(o, (2,))
    return lib().orc_barrier(C.byref(cp), _ptr(c), _ptr(o), float(R))


def goal_cost(p, x, goal):
    cp = _cparams(p)
    x, goal = _d(x, (4,)), _d(goal, (4,))
    return lib().orc_goal_cost(C.byref(cp), _ptr(x), _ptr(goal))


def _se(superellipses):
    """(n, 8) float64: cx, cy, m_x, m_y, theta, vx, vy, e."""
    if superellipses is None:
        return _zeros((0, 8))
    return _d(superellipses).reshape(-1, 8)


def barrier_se(p, c, o, se):
    cp = _cparams(p)
    c, o, se = _d(c, (2,)), _d(o, (2,)), _d(se, (8,))
    return lib().orc_barrier_se(C.byref(cp), _ptr(c), _ptr(o), _ptr(se))


def rollout(p, x0, goal, obstacles, u, alpha_k, want_traj=False, superellipses=None):
    """One sample.  Returns dict(S, xT, pen, traj)."""
    cp = _cparams(p)
    x0, goal = _d(x0, (4,)), _d(goal, (4,))
    obstacles = _d(obstacles).reshape(-1, 5)
    u = _d(u, (p.T, 2))
    xT = _zeros(4)
    traj = _zeros((p.T + 1, 4)) if want_traj else None
    pen = _REAL_C(0.0)
    se = _se(superellipses)
    S = lib().orc_rollout_se(C.byref(cp), _ptr(x0), _ptr(goal), obstacles.shape[0], _ptr(obstacles),
                             se.shape[0], _ptr(se), _ptr(u), float(alpha_k), _ptr(xT),
                             _ptr(traj) if want_traj else None, C.cast(C.byref(pen), _dp))
    return dict(S=S, xT=xT, pen=pen.value, traj=traj)


def sample(p, n, k, x0, goal, obstacles, U_in, superellipses=None):
    """Sample k of iteration n alone: dict(S, xT, u)."""
    cp = _cparams(p)
    x0, goal = _d(x0, (4,)), _d(goal, (4,))
    obstacles = _d(obstacles).reshape(-1, 5)
    U_in = _d(U_in, (p.T, 2))
    u = _zeros((p.T, 2))
    xT = _zeros(4)
    se = _se(superellipses)
    S = lib().orc_sample_se(C.byref(cp), int(n), int(k), _ptr(x0), _ptr(goal), obstacles.shape[0],
                            _ptr(obstacles), se.shape[0], _ptr(se), _ptr(U_in), _ptr(u), _ptr(xT))
    return dict(S=S, xT=xT, u=u)


def weights_update(S, u, lam):
    """S[K], u[K][T][2] -> dict(U, w, argmin, gap, eta, nonfinite)."""
    S = _d(S)
    K = S.shape[0]
    u = _d(u).reshape(K, -1, 2)
    T = u.shape[1]
    U = _zeros((T, 2))
    w = _zeros(K)
    am = C.c_int(0)
    gap = _REAL_C(0.0)
    eta = _REAL_C(0.0)
    nf = lib().orc_weights_update(K, T, float(lam), _ptr(S), _ptr(u), _ptr(U), _ptr(w),
                                  C.byref(am), C.cast(C.byref(gap), _dp),
                                  C.cast(C.byref(eta), _dp))
    return dict(U=U, w=w, argmin=am.value, gap=gap.value, eta=eta.value, nonfinite=nf)


def iteration(p, n, x0, goal, obstacles, U_in, n_threads=1, want_samples=False, superellipses=None):
    """One MPPI iteration with global counter n.  Returns dict(U, S, XT, argmin, gap, eta,
    nonfinite[, u, w])."""
    cp = _cparams(p)
    K, T = p.K, p.T
    x0, goal = _d(x0, (4,)), _d(goal, (4,))
    obstacles = _d(obstacles).reshape(-1, 5)
    U_in = _d(U_in, (T, 2))
    U = _zeros((T, 2))
    S = _zeros(K)
    XT = _zeros((K, 4))
    u = _zeros((K, T, 2)) if want_samples else None
    w = _zeros(K) if want_samples else None
    am = C.c_int(0)
    gap = _REAL_C(0.0)
    eta = _REAL_C(0.0)
    se = _se(superellipses)
    nf = lib().orc_iteration_se(C.byref(cp), int(n), _ptr(x0), _ptr(goal), obstacles.shape[0],
                             _ptr(obstacles), se.shape[0], _ptr(se), _ptr(U_in), _ptr(U), _ptr(S), _ptr(XT),
                             _ptr(u) if want_samples else None, _ptr(w) if want_samples else None,
                             C.byref(am), C.cast(C.byref(gap), _dp), C.cast(C.byref(eta), _dp),
                             int(n_threads))
    out = dict(U=U, S=S, XT=XT, argmin=am.value, gap=gap.value, eta=eta.value, nonfinite=nf)
    if want_samples:
        out["u"], out["w"] = u, w
    return out


def solve(p, n0, x0, goal, obstacles, U_in, n_threads=1, superellipses=None):
    """p.n_iter iterations starting at counter n0, no shift in between (CFG2).  Returns the list
    of per-iteration results; the last one's U is the solve's output."""
    U = _d(U_in, (p.T, 2)).copy()
    outs = []
    for it in range(p.n_iter):
        r = iteration(p, n0 + it, x0, goal, obstacles, U, n_threads=n_threads, superellipses=superellipses)
        U = r["U"]
        outs.append(r)
    return outs


def advance_se(p, superellipses):
    cp = _cparams(p)
    se = _se(superellipses).copy()
    lib().orc_advance_se(C.byref(cp), se.shape[0], _ptr(se))
    return se


def shift(U):
    U = _d(U).copy()
    lib().orc_shift(U.shape[0], _ptr(U))
    return U


def plant_step(p, x0, u0, obstacles):
    cp = _cparams(p)
    x = _d(x0, (4,)).copy()
    u0 = _d(u0, (2,))
    obs = _d(obstacles).reshape(-1, 5).copy()
    lib().orc_plant_step(C.byref(cp), _ptr(x), _ptr(u0), obs.shape[0], _ptr(obs))
    return x, obs


def hitch_barrier(p, x, v):
    """eq. (18)."""
    return lib().orc_hitch_barrier(C.byref(_cparams(p)), _ptr(_d(x, (4,))), float(v))


def hitch_rate_cond(p, x, u):
    return lib().orc_hitch_rate_cond(C.byref(_cparams(p)), _ptr(_d(x, (4,))), _ptr(_d(u, (2,))))


def hitch_constraint(p, x, u_ref):
    """(c0, a): c(u) ~ c0 + a . (u - u_ref), reading 28."""
    c0 = _REAL_C()
    a = _zeros(2)
    lib().orc_hitch_constraint(C.byref(_cparams(p)), _ptr(_d(x, (4,))), _ptr(_d(u_ref, (2,))),
                               C.byref(c0), _ptr(a))
    return c0.value, a


def hitch_filter(p, x, u_ref):
    """CBF-QP of Sec. V-D: (u*, status)."""
    u = _zeros(2)
    st = lib().orc_hitch_filter(C.byref(_cparams(p)), _ptr(_d(x, (4,))), _ptr(_d(u_ref, (2,))), _ptr(u))
    return u, int(st)


# ---- projected rollout, Sec. V-A ---------------------------------------------
def project(A, b, z_des, w, rho, z_lo, z_hi):
    """Eq. (12) by the C oracle: (z*, number of dropped rows)."""
    A = _d(A)
    m, d = A.shape
    z = _zeros(d)
    dropped = lib().orc_project(m, d, _ptr(A), _ptr(_d(b, (m,))), _ptr(_d(z_des, (d,))), _ptr(_d(w, (d,))),
                                float(rho), _ptr(_d(z_lo, (d,))), _ptr(_d(z_hi, (d,))), _ptr(z))
    return z, int(dropped)


def ualpha_normals(seed, n, k, t, n_obs):
    z = _zeros(max(n_obs, 1))
    lib().orc_ualpha_normals(int(seed) & 0xFFFFFFFFFFFFFFFF, int(n), int(k), int(t), int(n_obs), _ptr(z))
    return z[:n_obs]


def barrier_row(p, x, obstacle, t):
    """(h, active disc, L_g h [2], L_f h) of one obstacle at state x, step t."""
    h, Lf, j = _REAL_C(), _REAL_C(), C.c_int()
    Lg = _zeros(2)
    lib().orc_barrier_row(C.byref(_cparams(p)), _ptr(_d(x, (4,))), _ptr(_d(obstacle, (5,))), int(t), C.byref(h),
                          C.byref(j), _ptr(Lg), C.byref(Lf))
    return h.value, j.value, Lg, Lf.value


def affine_step(p, x, w):
    xn = _zeros(4)
    lib().orc_affine_step(C.byref(_cparams(p)), _ptr(_d(x, (4,))), _ptr(_d(w, (2,))), _ptr(xn))
    return xn


def rollout_projected(p, x0, goal, obstacles, u, ualpha, alpha0):
    obs = _d(obstacles).reshape(-1, 5)
    n_obs, T = obs.shape[0], p.T
    u = _d(u, (T, 2))
    ua = _d(ualpha).reshape(T, n_obs) if n_obs else _zeros((T, 1))
    xT, traj = _zeros(4), _zeros((T + 1, 4))
    z = _zeros((T, 2 + n_obs))
    al = _zeros((T + 1, max(n_obs, 1)))
    Ab = _zeros((T, max(n_obs, 1), 4))
    S = lib().orc_rollout_projected(C.byref(_cparams(p)), C.byref(_pparams(p)), _ptr(_d(x0, (4,))), _ptr(_d(goal, (4,))),
                                    n_obs, _ptr(obs), _ptr(u), _ptr(ua), float(alpha0), _ptr(xT), _ptr(traj), _ptr(z),
                                    _ptr(al), _ptr(Ab))
    return dict(S=S, xT=xT, traj=traj, z=z, alpha=al[:, :n_obs], Ab=Ab[:, :n_obs])


def sample_projected(p, n, k, x0, goal, obstacles, U_in):
    obs = _d(obstacles).reshape(-1, 5)
    u, xT = _zeros((p.T, 2)), _zeros(4)
    S = lib().orc_sample_projected(C.byref(_cparams(p)), C.byref(_pparams(p)), int(n), int(k), _ptr(_d(x0, (4,))),
                                   _ptr(_d(goal, (4,))), obs.shape[0], _ptr(obs), _ptr(_d(U_in, (p.T, 2))), _ptr(u), _ptr(xT))
    return dict(S=S, u=u, xT=xT)


def iteration_projected(p, n, x0, goal, obstacles, U_in, n_threads=1, want_samples=False):
    obs = _d(obstacles).reshape(-1, 5)
    K, T = p.K, p.T
    U_out, S, XT, w = _zeros((T, 2)), _zeros(K), _zeros((K, 4)), _zeros(K)
    u_all = _zeros((K, T, 2))
    argmin, gap, eta = C.c_int(), _REAL_C(), _REAL_C()
    nonfinite = lib().orc_iteration_projected(C.byref(_cparams(p)), C.byref(_pparams(p)), int(n), _ptr(_d(x0, (4,))),
                                              _ptr(_d(goal, (4,))), obs.shape[0], _ptr(obs), _ptr(_d(U_in, (T, 2))),
                                              _ptr(U_out), _ptr(S), _ptr(XT), _ptr(u_all), _ptr(w), C.byref(argmin),
                                              C.byref(gap), C.byref(eta), int(n_threads))
    out = dict(U=U_out, S=S, XT=XT, w=w, argmin=argmin.value, gap=gap.value, eta=eta.value, nonfinite=nonfinite)
    if want_samples:
        out["u"] = u_all
    return out


def solve_projected(p, n0, x0, goal, obstacles, U_in, n_threads=1):
    """n_iter projected iterations from counter n0; list of per-iteration results."""
    U = _d(U_in, (p.T, 2)).copy()
    outs = []
    for it in range(p.n_iter):
        r = iteration_projected(p, n0 + it, x0, goal, obstacles, U, n_threads=n_threads)
        U = r["U"].copy()
        outs.append(r)
    return outs


# ---- the paper's own model and tracking cost: eq. (6), (13)-(15), (17) ------------------------------
def _mparams(p, coef, dpsi):
    """(struct, keep-alive array): coef [M][4][4]."""
    coef = _d(coef)
    s = _MpccParams()
    for name in ("j_min", "j_max", "omega_min", "omega_max", "sigma_j", "sigma_omega", "Qc", "Ql", "Qth1", "Qth2",
                 "Rj", "Rw", "mu", "nu_bar"):
        setattr(s, name, float(getattr(p, name)))
    s.delta_lo, s.delta_hi = float(p.delta_min), float(p.delta_max)
    s.M, s.dpsi = int(coef.shape[0]), float(dpsi)
    s.coef = _ptr(coef)
    return s, coef


def step7(p, coef, dpsi, x, u):
    mp, keep = _mparams(p, coef, dpsi)
    xn = _zeros(7)
    lib().orc7_step(C.byref(_cparams(p)), C.byref(mp), _ptr(_d(x, (7,))), _ptr(_d(u, (2,))), _ptr(xn))
    return xn


def path_eval(p, coef, dpsi, psi):
    mp, keep = _mparams(p, coef, dpsi)
    out = _zeros(4)
    lib().orc_path_eval(C.byref(mp), float(psi), _ptr(out))
    return out


def progress7(p, coef, dpsi, x, psi):
    mp, keep = _mparams(p, coef, dpsi)
    return lib().orc7_progress(C.byref(mp), _ptr(_d(x, (7,))), float(psi))


def errors7(p, coef, dpsi, x, psi):
    mp, keep = _mparams(p, coef, dpsi)
    e = _zeros(4)
    lib().orc7_errors(C.byref(mp), _ptr(_d(x, (7,))), float(psi), _ptr(e))
    return e


def hhat7(p, x, u, obstacle, t, j):
    """(hhat, h) of eq. (17) for disc j against one obstacle at step t."""
    h = _REAL_C()
    hh = lib().orc7_hhat(C.byref(_cparams(p)), _ptr(_d(x, (7,))), _ptr(_d(u, (2,))), _ptr(_d(obstacle, (5,))), int(t), int(j),
                         C.byref(h))
    return hh, h.value


def rollout7(p, coef, dpsi, x0, psi0, obstacles, u, alpha):
    mp, keep = _mparams(p, coef, dpsi)
    obs = _d(obstacles).reshape(-1, 5)
    xT, traj = _zeros(8), _zeros((p.T + 1, 8))
    S = lib().orc7_rollout(C.byref(_cparams(p)), C.byref(mp), _ptr(_d(x0, (7,))), float(psi0), obs.shape[0], _ptr(obs),
                           _ptr(_d(u, (p.T, 2))), float(alpha), _ptr(xT), _ptr(traj))
    return dict(S=S, xT=xT, traj=traj)


def sample7(p, coef, dpsi, n, k, x0, psi0, obstacles, U_in):
    mp, keep = _mparams(p, coef, dpsi)
    obs = _d(obstacles).reshape(-1, 5)
    u, xT = _zeros((p.T, 2)), _zeros(8)
    S = lib().orc7_sample(C.byref(_cparams(p)), C.byref(mp), int(n), int(k), _ptr(_d(x0, (7,))), float(psi0), obs.shape[0],
                          _ptr(obs), _ptr(_d(U_in, (p.T, 2))), _ptr(u), _ptr(xT))
    return dict(S=S, u=u, xT=xT)


def iteration7(p, coef, dpsi, n, x0, psi0, obstacles, U_in, n_threads=1, want_samples=False):
    mp, keep = _mparams(p, coef, dpsi)
    obs = _d(obstacles).reshape(-1, 5)
    K, T = p.K, p.T
    U_out, S, XT, w = _zeros((T, 2)), _zeros(K), _zeros((K, 8)), _zeros(K)
    u_all = _zeros((K, T, 2))
    argmin, gap, eta = C.c_int(), _REAL_C(), _REAL_C()
    nonfinite = lib().orc7_iteration(C.byref(_cparams(p)), C.byref(mp), int(n), _ptr(_d(x0, (7,))), float(psi0), obs.shape[0],
                                     _ptr(obs), _ptr(_d(U_in, (T, 2))), _ptr(U_out), _ptr(S), _ptr(XT), _ptr(u_all), _ptr(w),
                                     C.byref(argmin), C.byref(gap), C.byref(eta), int(n_threads))
    out = dict(U=U_out, S=S, XT=XT, w=w, argmin=argmin.value, gap=gap.value, eta=eta.value, nonfinite=nonfinite)
    if want_samples:
        out["u"] = u_all
    return out


def solve7(p, coef, dpsi, n0, x0, psi0, obstacles, U_in, n_threads=1):
    U = _d(U_in, (p.T, 2)).copy()
    outs = []
    for it in range(p.n_iter):
        r = iteration7(p, coef, dpsi, n0 + it, x0, psi0, obstacles, U, n_threads=n_threads)
        U = r["U"].copy()
        outs.append(r)
    return outs
