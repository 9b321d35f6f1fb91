"""CPU oracle of BR-MPPI's closed-form projection, eq. (11)-(12).  TEST INFRASTRUCTURE
ONLY (imported by tests/ alone; never by paper_2508_05773_b200/).  fp64 numpy, the formula as printed:

    min_z ||z - z_des||_W^2 + rho/2 (||z - z_lo||^2 + ||z_hi - z||^2)   s.t.  A z = b              (11)
    z* = M^-1 [ p - A^T (A M^-1 A^T)^-1 (A M^-1 p - b) ],  M = W + rho I,  p = W z_des + rho/2 (z_hi + z_lo)   (12)

z = [u_proj (2), u_proj^alpha (N_o)], A is N_o x (2 + N_o), W = Diag(Q1, Q2) is passed as its diagonal.
A library solve serves as the inverse of the N_o x N_o matrix; nothing is blocked, fused or reordered.

Pins (tests/test_oracle_projection.py): feasibility A z* = b; stationarity of the *printed objective* (11a)
on the null space of A (scipy null_space, finite differences of the objective itself); scipy SLSQP on (11);
rho = 0 against the pseudo-inverse form of the weighted minimum-norm projection; the N_o = 1 scalar case
worked by hand.  How (9) builds A and b from the rollout state (the Lie derivatives of the reduced model)
is NOT part of this file: that integration is not built.
"""
import numpy as np


def project(A, b, z_des, w_diag, rho, z_lo, z_hi):
    """Eq. (12).  A [N_o, d], b [N_o], z_des / w_diag / z_lo / z_hi [d]; returns z* [d]."""
    A = np.asarray(A, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    z_des = np.asarray(z_des, dtype=np.float64)
    W = np.diag(np.asarray(w_diag, dtype=np.float64))
    d = A.shape[1]
    M = W + float(rho) * np.eye(d)
    p = W @ z_des + 0.5 * float(rho) * (np.asarray(z_hi, dtype=np.float64) + np.asarray(z_lo, dtype=np.float64))
    Minv = np.linalg.inv(M)
    S = A @ Minv @ A.T
    nu = np.linalg.solve(S, A @ Minv @ p - b)
    return Minv @ (p - A.T @ nu)


def objective(z, z_des, w_diag, rho, z_lo, z_hi):
    """(11a) as printed."""
    z = np.asarray(z, dtype=np.float64)
    e = z - np.asarray(z_des, dtype=np.float64)
    return float(e @ (np.asarray(w_diag, dtype=np.float64) * e)
                 + 0.5 * rho * (np.sum((z - z_lo) ** 2) + np.sum((z_hi - z) ** 2)))
