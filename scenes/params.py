"""Problem parameters as plain data (BASELINE.json configs[0]; SURVEY.md §8(c) defaults).

The paper never prints its cost weights (tuned by falsification); the values
here are this build's defaults (item 18) and are runtime parameters."""
from dataclasses import dataclass, fields, replace
from typing import Tuple

import numpy as np


def _f32(x: float) -> float:
    """Round to the nearest fp32 value: every real-valued input of the problem is DEFINED as an
    fp32 number, so the fp64 oracle and the fp32 library start from bit-identical inputs."""
    return float(np.float32(x))


@dataclass(frozen=True)
class Params:
    K: int = 256
    T: int = 30
    n_iter: int = 1
    dt: float = 0.1
    # vehicle: tractor wheelbase, trailer length, hitch offset (12 m overall), CFG0
    L1: float = 4.0
    L2: float = 8.0
    Lh: float = 0.0
    disc_radius: float = 1.3
    # (body, offset): body 0 = tractor axis (psi1), 1 = trailer axis (psi2); metres from hitch
    discs: Tuple[Tuple[int, float], ...] = ((0, 2.0), (1, -2.0), (1, -6.0))
    v_min: float = -2.0
    v_max: float = 2.0
    delta_min: float = -0.6
    delta_max: float = 0.6
    sigma_v: float = 0.5
    sigma_delta: float = 0.2
    alpha_lo: float = 0.1
    alpha_hi: float = 1.0
    w_pos: float = 0.05
    w_head: float = 0.5
    w_v: float = 0.01
    w_delta: float = 0.1
    w_hitch: float = 10.0
    hitch_max: float = 1.2
    hitch_kappa: float = 0.0      # velocity-dependent hitch limit hitch_max - kappa |v| (eq. 18); 0 = fixed limit
    # hitch-angle stabiliser, Sec. V-D (reading 28); off by default
    hitch_filter: int = 0         # 1: brmppi_step passes U[0] through the CBF-QP before the plant step
    hitch_alpha: float = 0.5      # alpha of condition (3), in (0, 1]
    hitch_qv: float = 1.0         # Q_h = diag(q_v, q_delta)
    hitch_qdelta: float = 1.0
    # projected rollout, Sec. V-A (reading 30); read only in projected mode
    proj_qv: float = 1.0          # W = Diag(Q1, Q2): Q1 = diag(proj_qv, proj_qomega), Q2 = proj_qalpha I
    proj_qomega: float = 4.0
    proj_qalpha: float = 0.5
    proj_rho: float = 0.25        # soft-bound weight rho of (11a)
    sigma_ualpha: float = 0.3     # standard deviation of the sampled auxiliary inputs u~^alpha
    ualpha_max: float = 1.0       # u^alpha in [-ualpha_max, ualpha_max]
    w_alpha: float = 10.0         # cost on positive alpha inside the buffer zone h < h_buffer
    h_buffer: float = 0.5
    # the paper's own model and tracking cost, eq. (6), (13)-(15), (17) (reading 31); read only in MPCC mode
    j_min: float = -2.0           # jerk bounds, m/s^3
    j_max: float = 2.0
    omega_min: float = -0.9       # steering-rate bounds, rad/s
    omega_max: float = 0.9
    sigma_j: float = 0.8
    sigma_omega: float = 0.3
    Qc: float = 2.0               # weights of (13): contouring, lag, the two headings, effort, progress
    Ql: float = 0.5
    Qth1: float = 0.5
    Qth2: float = 0.5
    Rj: float = 0.01
    Rw: float = 0.1
    mu: float = 0.2
    nu_bar: float = 1.5           # desired progress rate along the path, m/s
    w_bar: float = 1.0e3
    w_term: float = 10.0
    lam: float = 1.0
    seed: int = 0

    def with_(self, **kw) -> "Params":
        return replace(self, **kw).rounded()

    def rounded(self) -> "Params":
        kw = {}
        for f in fields(self):
            v = getattr(self, f.name)
            if isinstance(v, float):
                kw[f.name] = _f32(v)
        kw["discs"] = tuple((int(b), _f32(o)) for b, o in self.discs)
        return replace(self, **kw)


def default_params(**kw) -> Params:
    return Params(**kw).rounded()
