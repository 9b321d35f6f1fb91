"""Pins of oracle/projection.py (eq. (11)-(12)) against what the mathematics fixes."""
import numpy as np
import pytest
from scipy.linalg import null_space
from scipy.optimize import minimize

from oracle import projection as OP
from scenes.projection import projection_batch


def problems(seed, n, n_o, dense=False):
    B = projection_batch(seed, n, n_o, dense)
    for i in range(n):
        yield B["A"][i], B["b"][i], B["z_des"][i], B["w"], B["rho"], B["z_lo"], B["z_hi"]


@pytest.mark.parametrize("n_o", [1, 2, 3, 8])
@pytest.mark.parametrize("dense", [False, True])
def test_feasible_and_stationary_on_the_null_space(n_o, dense):
    for A, b, zd, w, rho, lo, hi in problems(3 + n_o, 20, n_o, dense):
        z = OP.project(A, b, zd, w, rho, lo, hi)
        assert np.abs(A @ z - b).max() < 1e-10                                   # (11b)
        N = null_space(A)                                                        # 2 feasible directions
        assert N.shape[1] == 2
        J0 = OP.objective(z, zd, w, rho, lo, hi)
        for k in range(2):                                                       # d/dt J(z + t N_k) = 0 at t = 0
            e = 1e-5 * N[:, k]
            fd = (OP.objective(z + e, zd, w, rho, lo, hi) - OP.objective(z - e, zd, w, rho, lo, hi)) / 2e-5
            assert abs(fd) < 1e-6 * (1 + abs(J0))
        rng = np.random.default_rng(0)
        for _ in range(5):                                                       # and it is the minimum
            t = rng.normal(0, 0.5, 2)
            assert OP.objective(z + N @ t, zd, w, rho, lo, hi) > J0


@pytest.mark.parametrize("n_o", [1, 4, 8])
def test_against_scipy_slsqp(n_o):
    for A, b, zd, w, rho, lo, hi in problems(11 + n_o, 8, n_o):
        z = OP.project(A, b, zd, w, rho, lo, hi)
        res = minimize(lambda x: OP.objective(x, zd, w, rho, lo, hi), zd, method="SLSQP",
                       constraints=[{"type": "eq", "fun": lambda x: A @ x - b, "jac": lambda x: A}],
                       options={"ftol": 1e-15, "maxiter": 500})
        assert res.success
        assert np.allclose(z, res.x, atol=2e-5)


@pytest.mark.parametrize("n_o", [1, 3, 8])
def test_rho_zero_is_the_weighted_minimum_norm_projection(n_o):
    """(10): min ||z - z_des||_W s.t. A z = b.  With y = W^(1/2)(z - z_des): y = pinv(A W^(-1/2))(b - A z_des)."""
    for A, b, zd, w, _, lo, hi in problems(20 + n_o, 10, n_o, dense=True):
        z = OP.project(A, b, zd, w, 0.0, lo, hi)
        y = np.linalg.pinv(A / np.sqrt(w)[None, :]) @ (b - A @ zd)
        assert np.allclose(z, zd + y / np.sqrt(w), atol=1e-10)


def test_scalar_case_by_hand():
    """N_o = 1, A = [1 2 | 2], b = 3, W = I, rho = 0, z_des = 0: the nearest point of the plane
    x + 2y + 2z = 3 to the origin is 3 (1, 2, 2) / 9."""
    z = OP.project([[1.0, 2.0, 2.0]], [3.0], [0, 0, 0], [1, 1, 1], 0.0, [-1, -1, -1], [1, 1, 1])
    assert np.allclose(z, np.array([1.0, 2.0, 2.0]) / 3.0, atol=1e-14)
    # rho -> inf pulls towards the centre of the bounds, here (1, 0, 0); nearest point of the plane to it:
    z = OP.project([[1.0, 2.0, 2.0]], [3.0], [0, 0, 0], [1, 1, 1], 1e9, [0, -1, -1], [2, 1, 1])
    assert np.allclose(z, np.array([1.0, 0, 0]) + 2.0 * np.array([1.0, 2.0, 2.0]) / 9.0, atol=1e-7)


def test_already_feasible_target_is_kept_when_rho_is_zero():
    A = np.array([[0.3, -0.2, 1.5, 0.0], [0.1, 0.4, 0.0, -0.7]])
    zd = np.array([1.0, -0.3, 0.2, 0.5])
    z = OP.project(A, A @ zd, zd, [1, 2, 3, 4], 0.0, -np.ones(4), np.ones(4))
    assert np.allclose(z, zd, atol=1e-14)
