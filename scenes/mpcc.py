"""Seeded reference paths and scenes for the paper's own formulation (7-state model, contouring cost; SURVEY §8(f)
rank 3).  The paper fits "a third-order spline to the Hybrid A* output"; the planner and its output
are not available, so the path here is a cubic spline through a few seeded waypoints between the start pose and
the bay pose, re-parameterised by arc length.  Input recipe only: it produces the coefficient table
[M][4 components (p^x, p^y, theta1, theta2)][c0..c3] on uniform knots that oracle and library both read."""
from dataclasses import dataclass

import numpy as np
from scipy.interpolate import CubicSpline

from .parking import Scene, scene_static, _draw_obstacles, _r32


@dataclass
class PathScene:
    x0: np.ndarray          # (7,): px, py, v, a, theta1, theta2, delta
    psi0: float
    obstacles: np.ndarray   # (N, 5)
    coef: np.ndarray        # (M, 4, 4) fp32-representable
    dpsi: float
    params: object
    name: str = ""


def spline_table(way_xy, M, trailer_lag):
    """Arc-length cubic splines of a smooth curve through `way_xy`: (coef [M][4][4], dpsi)."""
    way_xy = np.asarray(way_xy, dtype=np.float64)
    u = np.linspace(0.0, 1.0, len(way_xy))
    cx, cy = CubicSpline(u, way_xy[:, 0]), CubicSpline(u, way_xy[:, 1])
    uu = np.linspace(0.0, 1.0, 4001)
    x, y = cx(uu), cy(uu)
    s = np.concatenate([[0.0], np.cumsum(np.hypot(np.diff(x), np.diff(y)))])
    L = float(s[-1])
    knots = np.linspace(0.0, L, M + 1)
    xk, yk = np.interp(knots, s, x), np.interp(knots, s, y)
    th = np.unwrap(np.arctan2(np.gradient(y, s), np.gradient(x, s)))
    th1 = np.interp(knots, s, th)
    th2 = np.interp(np.clip(knots - trailer_lag, 0.0, L), s, th)          # the trailer's heading lags the tractor's
    dpsi = float(np.float32(L / M))
    kk = dpsi * np.arange(M + 1)
    coef = np.zeros((M, 4, 4))
    for c, vals in enumerate((xk, yk, th1, th2)):
        sp = CubicSpline(kk, vals)
        coef[:, c, :] = sp.c[::-1, :].T                                    # scipy stores the highest power first
    return _r32(coef), dpsi


def scene_mpcc(seed=0, K=16384, T=80, dt=0.05, n_obs=8, M=24):
    """CFG2-shaped scene for the 7-state model: start pose and bay pose of `scene_static`, a smooth reference path
    between them, static discs and three pedestrians placed like CFG2's but clear of the path's start."""
    base = scene_static(seed, max(n_obs - 3, 0), K=K, T=T, dt=dt, n_iter=1)
    rng = np.random.default_rng(4000 + seed)
    a, b = base.x0[:2], base.goal[:2]
    mid = 0.5 * (a + b) + rng.uniform(-4.0, 4.0, 2)
    ahead = a + 5.0 * np.array([np.cos(base.x0[2]), np.sin(base.x0[2])])
    coef, dpsi = spline_table([a, ahead, mid, b], M, trailer_lag=4.0)
    obs = list(base.obstacles)
    peds = _draw_obstacles(rng, min(3, n_obs), 20.0, 0.4, 0.4, [base.x0[:3], base.goal[:3]], base.params.disc_radius + 2.0)
    for o in peds:
        speed, ang = rng.uniform(0.0, 1.5), rng.uniform(-np.pi, np.pi)
        o[3], o[4] = speed * np.cos(ang), speed * np.sin(ang)
    obs = np.array(obs + peds, dtype=np.float64).reshape(-1, 5)[:n_obs]
    th0 = float(coef[0, 2, 0])
    x0 = np.array([coef[0, 0, 0], coef[0, 1, 0], 0.5, 0.0, th0, th0, 0.0])
    return PathScene(_r32(x0), 0.0, _r32(obs), coef, dpsi, base.params.with_(K=K, T=T, dt=dt), f"mpcc/seed{seed}")
