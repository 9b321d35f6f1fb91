"""Seeded synthetic parking scenes standing in for the paper's CarMaker parking-lot scenario
(PAPER.md:245-247), which is not available: a 12 m tractor-trailer, up to eight obstacles
(parked-car-sized discs plus crossing pedestrians), a bay pose to reach.  BASELINE.json configs
0-4; recipe restated in DESIGN.md.  Plain geometry only: a vehicle at a straight pose
(zero hitch angle) is the segment from 8 m behind to 4 m ahead of the tractor rear axle, and an
obstacle is accepted when its centre keeps a given distance from that segment.

Every returned real number is rounded to fp32 so both implementations get identical inputs.
Obstacle rows are (cx, cy, R, vx, vy)."""
from dataclasses import dataclass
from typing import List

import numpy as np

from .params import Params, default_params

VEH_REAR = 8.0    # trailer rear, metres behind the hitch/rear axle (L2)
VEH_FRONT = 4.0   # tractor front axle, metres ahead (L1)


@dataclass
class Scene:
    x0: np.ndarray          # (4,) float64 holding fp32 values: x, y, psi1, psi2
    goal: np.ndarray        # (4,)
    obstacles: np.ndarray   # (N, 5)
    params: Params
    name: str = ""
    goal_next: np.ndarray = None   # second waypoint of a forward-then-reverse schedule (CFG2)
    superellipses: np.ndarray = None   # (M, 8): cx, cy, m_x, m_y, theta, vx, vy, exponent (eq. 16)


def _r32(a):
    return np.asarray(a, dtype=np.float32).astype(np.float64)


def _seg_dist(px, py, pose):
    """Distance from point (px, py) to the straight-vehicle segment of `pose` = (x, y, psi)."""
    x, y, psi = pose
    ax, ay = np.cos(psi), np.sin(psi)
    s = np.clip((px - x) * ax + (py - y) * ay, -VEH_REAR, VEH_FRONT)
    return float(np.hypot(px - (x + s * ax), py - (y + s * ay)))


def vehicle_disc_centres(pose, discs):
    """Disc centres of a STRAIGHT vehicle (psi1 == psi2) -- used only by scene acceptance tests."""
    x, y, psi = pose
    return np.array([[x + off * np.cos(psi), y + off * np.sin(psi)] for _, off in discs])


def _draw_obstacles(rng, n, half, r_lo, r_hi, poses, margin):
    obs = []
    while len(obs) < n:
        R = rng.uniform(r_lo, r_hi) if r_hi > r_lo else r_lo
        cx, cy = rng.uniform(-half, half, size=2)
        if all(_seg_dist(cx, cy, p) >= R + margin for p in poses):
            obs.append([cx, cy, R, 0.0, 0.0])
    return obs


def scene_cfg0(seed: int = 0) -> Scene:
    """CFG0: K=256, T=30, dt=0.1, start at origin, goal (-10,0,0,0) reversing, one static disc
    R=1 m, centre uniform in [-10,10]^2, re-drawn while it overlaps the vehicle at start/goal."""
    p = default_params(K=256, T=30, dt=0.1, n_iter=1, seed=seed)
    rng = np.random.default_rng(seed)
    x0 = np.zeros(4)
    goal = np.array([-10.0, 0.0, 0.0, 0.0])
    obs = _draw_obstacles(rng, 1, 10.0, 1.0, 1.0, [x0[:3], goal[:3]], p.disc_radius)
    return Scene(_r32(x0), _r32(goal), _r32(obs), p, f"cfg0/seed{seed}")


def scene_static(seed: int, n_obs: int, K: int, T: int, dt: float = 0.05, n_iter: int = 1) -> Scene:
    """CFG1 recipe with a free obstacle count (CFG3/CFG4 reuse it): 40x40 m lot, start pose
    uniform in the lot with heading U[-pi,pi) and zero hitch; bay pose uniform in the lot inset
    7 m, goal = bay centre shifted 2 m along the bay axis (centres the [-8,+4] m vehicle in a
    14 m bay); static discs R~U[0.5,1.5] whose centres keep R + r_v + 2 m from the vehicle
    segment at start and at goal."""
    p = default_params(K=K, T=T, dt=dt, n_iter=n_iter, seed=seed)
    rng = np.random.default_rng(1000 + seed)
    half = 20.0
    sx, sy = rng.uniform(-half, half, size=2)
    spsi = rng.uniform(-np.pi, np.pi)
    bx, by = rng.uniform(-half + 7.0, half - 7.0, size=2)
    bth = rng.uniform(-np.pi, np.pi)
    x0 = np.array([sx, sy, spsi, spsi])
    goal = np.array([bx + 2.0 * np.cos(bth), by + 2.0 * np.sin(bth), bth, bth])
    obs = _draw_obstacles(rng, n_obs, half, 0.5, 1.5, [x0[:3], goal[:3]], p.disc_radius + 2.0)
    return Scene(_r32(x0), _r32(goal), _r32(obs), p, f"static{n_obs}/seed{seed}")


def scene_cfg1(seed: int = 0) -> Scene:
    s = scene_static(seed, 8, K=4096, T=50, dt=0.05)
    s.name = f"cfg1/seed{seed}"
    return s


def scene_cfg2(seed: int = 0) -> Scene:
    """CFG2: K=16384, T=80, dt=0.05, 3 iterations; 5 static discs as CFG1 + 3 pedestrians
    (R=0.4 m, speed U[0,1.5] m/s, direction U[-pi,pi)); two-waypoint goal schedule: a
    pull-forward pose 6 m ahead of the bay mouth along the bay axis, then the bay pose."""
    s = scene_static(seed, 5, K=16384, T=80, dt=0.05, n_iter=3)
    rng = np.random.default_rng(2000 + seed)
    peds = _draw_obstacles(rng, 3, 20.0, 0.4, 0.4, [s.x0[:3], s.goal[:3]], s.params.disc_radius + 2.0)
    for o in peds:
        speed = rng.uniform(0.0, 1.5)
        ang = rng.uniform(-np.pi, np.pi)
        o[3], o[4] = speed * np.cos(ang), speed * np.sin(ang)
    obs = np.vstack([s.obstacles, _r32(peds)])
    bay = s.goal.copy()
    fwd = bay.copy()
    fwd[0] += 6.0 * np.cos(bay[2])
    fwd[1] += 6.0 * np.sin(bay[2])
    return Scene(s.x0, _r32(fwd), obs, s.params, f"cfg2/seed{seed}", goal_next=bay)


def scene_cfg2_superellipse(seed: int = 0) -> Scene:
    """CFG2 with the paper's obstacle models: the five static obstacles
    become parked cars -- super-ellipses with e = 4, semi-axes 2.25 x 0.9 m (a 4.5 x 1.8 m car),
    orientation U[-pi, pi), centre where CFG2's generator would put a disc of the car's
    circumscribed radius -- and the three pedestrians super-ellipses with e = 2, m_x = m_y = 0.4 m,
    same constant velocities as in CFG2."""
    s = scene_cfg2(seed)
    rng = np.random.default_rng(3000 + seed)
    half_len, half_wid = 2.25, 0.9
    rad = float(np.hypot(half_len, half_wid))
    cars = _draw_obstacles(rng, 5, 20.0, rad, rad, [s.x0[:3], s.goal_next[:3], s.goal[:3]], s.params.disc_radius + 1.0)
    se = [[c[0], c[1], half_len, half_wid, rng.uniform(-np.pi, np.pi), 0.0, 0.0, 4.0] for c in cars]
    for o in s.obstacles[5:]:
        se.append([o[0], o[1], o[2], o[2], 0.0, o[3], o[4], 2.0])
    return Scene(s.x0, s.goal, np.zeros((0, 5)), s.params, f"cfg2se/seed{seed}", goal_next=s.goal_next,
                 superellipses=_r32(se))


def scene_cfg3(seed: int = 0) -> Scene:
    s = scene_static(seed, 8, K=8192, T=60, dt=0.05)
    s.name = f"cfg3/seed{seed}"
    return s


def scene_batch(n_scenes: int = 64, K: int = 16384, T: int = 80) -> List[Scene]:
    """CFG4 batched launch: independent CFG2-shaped scenes, seeds 0..n_scenes-1."""
    out = []
    for s in range(n_scenes):
        sc = scene_cfg2(s)
        sc.params = sc.params.with_(K=K, T=T, n_iter=1, seed=s)
        out.append(sc)
    return out
