"""Seeded inputs for the projection (11)-(12): problems shaped like (9)-(10b), PAPER.md:167-181 --
A = [L_g h (N_o x 2) | diag(h)], b_i = -alpha_i h_i - L_f h_i -- with magnitudes of a parking scene
(barrier values of discs a few metres away, gradients scaled by the step).  Input recipe only: holds none of
the method's arithmetic (the entries are drawn, not derived from a model)."""
import numpy as np


def projection_batch(seed, n, n_o, dense=False):
    rng = np.random.default_rng(seed)
    d = 2 + n_o
    A = np.zeros((n, n_o, d))
    A[:, :, :2] = rng.normal(0.0, 0.3, (n, n_o, 2))
    h = rng.uniform(0.05, 4.0, (n, n_o)) * rng.choice([1.0, 1.0, 1.0, -0.2], (n, n_o))
    A[:, np.arange(n_o), 2 + np.arange(n_o)] = h
    if dense:                                  # any full-row-rank A: eq. (12) does not need the structure
        A += rng.normal(0.0, 0.2, A.shape)
    alpha = rng.uniform(0.1, 1.0, (n, n_o))
    b = -alpha * h - rng.normal(0.0, 0.2, (n, n_o))
    z_des = np.concatenate([rng.uniform(-2, 2, (n, 1)), rng.uniform(-0.6, 0.6, (n, 1)),
                            rng.normal(0.0, 0.3, (n, n_o))], axis=1)
    w = np.concatenate([[1.0, 4.0], np.full(n_o, 0.5)])
    z_lo = np.concatenate([[-2.0, -0.6], np.full(n_o, -1.0)])
    z_hi = np.concatenate([[2.0, 0.6], np.full(n_o, 1.0)])
    f32 = lambda a: np.asarray(a, dtype=np.float32).astype(np.float64)     # fp32-representable, like Params
    return dict(A=f32(A), b=f32(b), z_des=f32(z_des), w=f32(w), rho=0.25, z_lo=f32(z_lo), z_hi=f32(z_hi))
