"""Pins of the oracle's hitch-angle stabiliser, Sec. V-D (reading 28).

None of these retypes the oracle's formulas: the rate condition is tied to the exact discrete
condition (2) through the separately pinned Euler step, the gradient to finite differences, the QP to
scipy's SLSQP, a dense grid search and the textbook half-plane projection, and the whole filter to the
property the paper states for it (h_h >= 0 stays enforced)."""
import math

import numpy as np
import pytest
from scipy.optimize import minimize

from oracle import oracle as O
from scenes import default_params


def P(**kw):
    base = dict(dt=0.05, hitch_max=1.2, hitch_kappa=0.0, hitch_alpha=0.5, hitch_qv=1.0, hitch_qdelta=1.0)
    base.update(kw)
    return default_params().with_(**base)


def test_barrier_hand_value():
    # eq. (18): 1.2 - 0.2 * |-1| - |0.9 - 0.4| = 0.5
    p = P(hitch_kappa=0.2)
    assert O.hitch_barrier(p, [3.0, -1.0, 0.9, 0.4], -1.0) == pytest.approx(0.5, abs=1e-7)
    # symmetric in the sign of the hitch angle and of the speed
    assert O.hitch_barrier(p, [0, 0, 0.4, 0.9], 1.0) == pytest.approx(0.5, abs=1e-7)
    # wrapped: psi1 - psi2 = 2 pi - 0.3 is a hitch angle of -0.3
    assert O.hitch_barrier(p, [0, 0, math.pi - 0.1, -math.pi + 0.2], 0.0) == pytest.approx(1.2 - 0.3, abs=1e-7)


def test_rate_cond_is_exact_discrete_condition():
    """Where the hitch angle keeps its sign over the step, |beta| is linear there and the first-order
    expansion is exact: c(u) = h_h(x_{k+1}) - (1 - alpha) h_h(x_k), i.e. condition (2) with reading 1's
    sign, evaluated through orc_kinematic_step."""
    rng = np.random.default_rng(5)
    for _ in range(200):
        p = P(hitch_kappa=float(rng.uniform(0, 0.3)), hitch_alpha=float(rng.uniform(0.1, 1.0)),
              Lh=float(rng.uniform(0.0, 1.0)))
        beta = rng.uniform(0.2, 1.5) * rng.choice([-1, 1])
        psi2 = rng.uniform(-1.0, 1.0)
        x = [rng.uniform(-5, 5), rng.uniform(-5, 5), psi2 + beta, psi2]
        u = [rng.uniform(-2, 2), rng.uniform(-0.6, 0.6)]
        xn = O.kinematic_step(p, x, u[0], u[1])
        want = O.hitch_barrier(p, xn, u[0]) - (1.0 - p.hitch_alpha) * O.hitch_barrier(p, x, u[0])
        assert O.hitch_rate_cond(p, x, u) == pytest.approx(want, abs=1e-12)


def test_constraint_is_first_order_taylor():
    rng = np.random.default_rng(6)
    for _ in range(200):
        p = P(hitch_kappa=float(rng.uniform(0, 0.3)), Lh=float(rng.uniform(0.0, 1.0)))
        x = [0.0, 0.0, rng.uniform(-1.4, 1.4), 0.0]
        u = np.array([rng.uniform(0.2, 2.0) * rng.choice([-1, 1]), rng.uniform(-0.6, 0.6)])
        c0, a = O.hitch_constraint(p, x, u)
        assert c0 == O.hitch_rate_cond(p, x, u)
        for i in range(2):
            e = np.zeros(2)
            e[i] = 1e-6
            fd = (O.hitch_rate_cond(p, x, u + e) - O.hitch_rate_cond(p, x, u - e)) / 2e-6
            assert a[i] == pytest.approx(fd, abs=1e-8)


def test_speed_term_sign_at_zero_speed():
    # d|v|/dv := 0 at v = 0 (reading 28); the steering has no authority at standstill
    p = P(hitch_kappa=0.2)
    _, a = O.hitch_constraint(p, [0, 0, 0.7, 0], [0.0, 0.3])
    _, a0 = O.hitch_constraint(P(hitch_kappa=0.0), [0, 0, 0.7, 0], [0.0, 0.3])
    assert a[1] == 0.0 and a[0] == pytest.approx(a0[0], abs=1e-15)


def _cases(rng, n):
    for _ in range(n):
        p = P(hitch_kappa=float(rng.uniform(0, 0.3)), hitch_alpha=float(rng.uniform(0.1, 1.0)),
              hitch_qv=float(rng.uniform(0.2, 5.0)), hitch_qdelta=float(rng.uniform(0.2, 5.0)),
              hitch_max=float(rng.uniform(0.6, 1.3)), Lh=float(rng.uniform(0.0, 1.0)))
        beta = rng.uniform(-1.5, 1.5)
        x = [0.0, 0.0, beta + 0.3, 0.3]
        u = np.array([rng.uniform(-2.2, 2.2), rng.uniform(-0.7, 0.7)])   # may lie outside the box
        yield p, x, u


def _J(p, u, u_ref):
    return p.hitch_qv * (u[0] - u_ref[0]) ** 2 + p.hitch_qdelta * (u[1] - u_ref[1]) ** 2


def test_qp_against_scipy_slsqp():
    rng = np.random.default_rng(7)
    seen = {0: 0, 1: 0, 2: 0}
    for p, x, u_ref in _cases(rng, 300):
        c0, a = O.hitch_constraint(p, x, u_ref)
        u, st = O.hitch_filter(p, x, u_ref)
        seen[st] += 1
        lo = np.array([p.v_min, p.delta_min])
        hi = np.array([p.v_max, p.delta_max])
        assert np.all(u >= lo) and np.all(u <= hi)
        if st == 2:
            # box and half-plane do not meet: the linear programme max a.u over the box is below 0
            best = c0 + sum(max(a[i] * (lo[i] - u_ref[i]), a[i] * (hi[i] - u_ref[i])) for i in range(2))
            assert best < 0
            assert c0 + a @ (u - u_ref) == pytest.approx(best, abs=1e-12)
            continue
        res = minimize(lambda z: _J(p, z, u_ref), np.clip(u_ref, lo, hi), method="SLSQP",
                       jac=lambda z: 2 * np.array([p.hitch_qv, p.hitch_qdelta]) * (z - u_ref),
                       bounds=list(zip(lo, hi)),
                       constraints=[{"type": "ineq", "fun": lambda z: c0 + a @ (z - u_ref), "jac": lambda z: a}],
                       options={"ftol": 1e-14, "maxiter": 200})
        assert c0 + a @ (u - u_ref) >= -1e-10
        if res.success:
            assert _J(p, u, u_ref) <= _J(p, res.x, u_ref) + 1e-7
            assert np.allclose(u, res.x, atol=2e-4)
        if st == 0:
            assert np.array_equal(u, np.clip(u_ref, lo, hi))
    assert min(seen.values()) >= 5, seen        # every branch exercised


def test_qp_against_grid_search():
    rng = np.random.default_rng(8)
    for p, x, u_ref in list(_cases(rng, 40)):
        c0, a = O.hitch_constraint(p, x, u_ref)
        u, st = O.hitch_filter(p, x, u_ref)
        if st == 2:
            continue
        V, D = np.meshgrid(np.linspace(p.v_min, p.v_max, 801), np.linspace(p.delta_min, p.delta_max, 801), indexing="ij")
        feas = c0 + a[0] * (V - u_ref[0]) + a[1] * (D - u_ref[1]) >= 0
        if not feas.any():
            continue
        Jg = np.where(feas, p.hitch_qv * (V - u_ref[0]) ** 2 + p.hitch_qdelta * (D - u_ref[1]) ** 2, np.inf)
        i = np.unravel_index(np.argmin(Jg), Jg.shape)
        assert _J(p, u, u_ref) <= Jg[i] + 1e-12                   # nothing feasible on the grid is better
        assert Jg[i] - _J(p, u, u_ref) <= 0.02 * (1.0 + _J(p, u, u_ref))    # ... and the grid gets that close


def test_qp_halfplane_projection_when_box_is_far():
    """Active constraint, box inactive: the Q-norm projection on a half-plane,
    u = u_ref - c0 Q^-1 a / (a' Q^-1 a) (textbook), and the constraint holds with equality."""
    p = P(v_min=-50.0, v_max=50.0, delta_min=-1.4, delta_max=1.4, hitch_qv=2.0, hitch_qdelta=0.5)
    x = [0, 0, 1.19, 0.0]
    u_ref = np.array([-1.5, -0.3])
    c0, a = O.hitch_constraint(p, x, u_ref)
    assert c0 < 0
    u, st = O.hitch_filter(p, x, u_ref)
    Qi = np.array([1 / p.hitch_qv, 1 / p.hitch_qdelta])
    assert st == 1
    assert np.allclose(u, u_ref - c0 * Qi * a / (a @ (Qi * a)), atol=1e-12)
    assert c0 + a @ (u - u_ref) == pytest.approx(0.0, abs=1e-13)


def test_inactive_deep_inside_safe_set():
    p = P()
    u, st = O.hitch_filter(p, [1.0, 2.0, 0.1, 0.0], [-1.0, 0.2])
    assert st == 0 and np.array_equal(u, np.array([-1.0, 0.2], dtype=np.float64))


def test_at_the_limit_the_hitch_angle_stops_growing():
    """h_h = 0 (|beta| = hitch_max, kappa = 0): the filtered control's linearised hitch rate does not
    point outwards, whatever the reference asks for."""
    p = P()
    for beta in (1.2, -1.2):
        for u_ref in ([-2.0, 0.5], [-2.0, -0.5], [2.0, 0.5], [2.0, -0.5]):
            x = [0, 0, beta * (1 + 0e-9), 0.0]
            p2 = p.with_(hitch_max=abs(beta))
            u, st = O.hitch_filter(p2, x, u_ref)
            if st == 2:
                continue
            c0, a = O.hitch_constraint(p2, x, u_ref)
            assert c0 + a @ (u - np.array(u_ref)) >= -1e-12
            xn = O.kinematic_step(p2, x, u[0], u[1])
            # exact step: growth of |beta| is bounded by the second-order remainder of the expansion in u
            assert abs(xn[2] - xn[3]) - abs(beta) <= 0.5 * p2.dt * 4.0 * np.sum((u - np.array(u_ref)) ** 2) + 1e-9


@pytest.mark.parametrize("kappa", [0.0, 0.1])
def test_closed_loop_forward_invariance(kappa):
    """enforcing h_h >= 0 keeps |hitch| <= hitch_max - kappa |v|.  A reversing reference with
    constant steering jackknifes the unfiltered vehicle; the filtered one stays inside the limit (up to the
    linearisation remainder per step)."""
    p = P(hitch_max=0.8, hitch_kappa=kappa, hitch_alpha=0.3)
    u_ref = np.array([-1.5, 0.3])
    x_f = np.array([0.0, 0.0, 0.0, 0.0])
    x_n = x_f.copy()
    worst_f = worst_n = -1e9
    active = 0
    for _ in range(600):
        u, st = O.hitch_filter(p, x_f, u_ref)
        assert st != 2
        active += st == 1
        x_f = np.array(O.kinematic_step(p, x_f, u[0], u[1]))
        x_n = np.array(O.kinematic_step(p, x_n, u_ref[0], u_ref[1]))
        worst_f = max(worst_f, -O.hitch_barrier(p, x_f, u[0]))
        worst_n = max(worst_n, abs(O.wrap(x_n[2] - x_n[3])) - p.hitch_max)
    assert worst_n > 0.3            # unfiltered: the limit is exceeded by far
    # filtered: h_h >= -0.02 rad throughout.  The slack is the second-order remainder of reading 28's
    # expansion in u (dt |dv| |d tan(delta)| / L1 ~ 6e-3 per step), which settles at remainder / alpha.
    # With kappa > 0 the speed moves further from the reference and the remainder grows with it.
    assert worst_f < (2e-2 if kappa == 0.0 else 5e-2)
    assert active > 100
