"""fp32 noise floor of every parity quantity (SURVEY 8(c) reading 23).  TEST INFRASTRUCTURE ONLY.

For each path of the library, the oracle's fp32 re-run build (oracle/oracle32.py: the same C source with float
arithmetic, rounding after every operation) is compared with the fp64 oracle on the seeded inputs the parity tests
use, in the measure those tests use, and the result is printed next to the tolerance.  A floor above a tolerance
means that the tolerance is unattainable in fp32 for that quantity: the report says so instead of hiding it, and the
parity test of that quantity carries a stated, derived widening.

Not reported: the hitch-angle QP (orc_hitch_filter) and the projection (12) (orc_project).  The first is defined in
the oracle by enumerating candidate points and testing their feasibility at 1e-12 relative -- a definition that is
only meaningful in fp64; the second is compared on conditioning-scaled tolerances of its own
(tests/test_gpu_projection.py).  Their parity rules are stated in those tests.

    python -m oracle.fp32_floor          # prints the table (markdown); tests/test_oracle_fp32_floor.py asserts on it
"""
import numpy as np

import scenes
from oracle import oracle as O64
from oracle import oracle32 as O32

RTOL = 1e-4     # the north star's tolerance on x_T, S_k and U


def _rel(a, b, floor):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return np.abs(a - b) / np.maximum(np.abs(b), floor)


def _row(name, quantity, err, note=""):
    err = np.asarray(err).ravel()
    worst, p99 = float(err.max()), float(np.quantile(err, 0.99))
    over = float((err > RTOL).mean())
    return dict(path=name, quantity=quantity, floor_max=worst, floor_p99=p99, tolerance=RTOL, share_over=over,
                attainable=worst <= RTOL, note=note)


def penalty_rows(name, sc, p, n_threads=8, se=None):
    U0 = np.zeros((p.T, 2))
    kw = dict(superellipses=se) if se is not None else {}
    a = O64.solve(p, 0, sc.x0, sc.goal, sc.obstacles, U0, n_threads=n_threads, **kw)[-1]
    b = O32.solve(p, 0, sc.x0, sc.goal, sc.obstacles, U0, n_threads=n_threads, **kw)[-1]
    floors = np.array([p.v_max, p.delta_max])
    return [_row(name, "x_T", _rel(b["XT"], a["XT"], 1.0)), _row(name, "S_k", _rel(b["S"], a["S"], 1.0)),
            _row(name, "U", _rel(b["U"], a["U"], floors[None, :]),
                 "after %d iteration(s); pure fp32 also rounds S_k (~1e4) and S_k - min S before the exponential, "
                 "which the kernels keep in fp64 (SURVEY 7 hard part 2)" % p.n_iter)]


def projected_rows(name, sc, p, n_threads=8):
    U0 = np.zeros((p.T, 2))
    a = O64.solve_projected(p, 0, sc.x0, sc.goal, sc.obstacles, U0, n_threads=n_threads)[-1]
    b = O32.solve_projected(p, 0, sc.x0, sc.goal, sc.obstacles, U0, n_threads=n_threads)[-1]
    floors = np.array([p.v_max, p.delta_max])
    note = "samples pinned to an obstacle boundary (h -> 0) amplify rounding: the rule of tests/test_gpu_projected.py"
    return [_row(name, "x_T", _rel(b["XT"], a["XT"], 1.0).max(axis=1), note), _row(name, "S_k", _rel(b["S"], a["S"], 1.0), note),
            _row(name, "U", _rel(b["U"], a["U"], floors[None, :]))]


def mpcc_rows(name, sc, p, n_threads=8):
    U0 = np.zeros((p.T, 2))
    a = O64.solve7(p, sc.coef, sc.dpsi, 0, sc.x0, sc.psi0, sc.obstacles, U0, n_threads=n_threads)[-1]
    b = O32.solve7(p, sc.coef, sc.dpsi, 0, sc.x0, sc.psi0, sc.obstacles, U0, n_threads=n_threads)[-1]
    floors = np.array([p.j_max, p.omega_max])
    note = "S_k of tens with w_bar = 1e3 per hinge term: active terms amplify (tests/test_gpu_mpcc.py widens by them)"
    return [_row(name, "x_T", _rel(b["XT"], a["XT"], 1.0)), _row(name, "S_k", _rel(b["S"], a["S"], 1.0), note),
            _row(name, "U", _rel(b["U"], a["U"], floors[None, :]), "lambda = 1, effective sample size of tens")]


def report(K=1024, n_threads=8):
    rows = []
    sc = scenes.scene_cfg1(0)
    rows += penalty_rows("penalty path, cfg1 shape", sc, sc.params.with_(K=K, n_iter=1), n_threads)
    sc = scenes.scene_cfg2(0)
    rows += penalty_rows("penalty path, cfg2 shape, 3 iterations", sc, sc.params.with_(K=K), n_threads)
    sc = scenes.scene_cfg2_superellipse(0)
    rows += penalty_rows("super-ellipses (eq. 16), cfg2se shape", sc, sc.params.with_(K=K, n_iter=1), n_threads, se=sc.superellipses)
    sc = scenes.scene_cfg2(0)
    rows += projected_rows("projected rollout (Sec. V-A), cfg2 shape", sc, sc.params.with_(K=K, n_iter=1), n_threads)
    sc = scenes.scene_mpcc(0, K=K, T=80, dt=0.05, n_obs=8, M=24)
    rows += mpcc_rows("7-state model + (13), (17), cfg2mpcc shape", sc, sc.params.with_(n_iter=1), n_threads)
    return rows


def markdown(rows):
    out = ["| path | quantity | fp32 floor (max) | fp32 floor (99 %) | tolerance | share above | attainable in fp32 | note |",
           "|---|---|---|---|---|---|---|---|"]
    for r in rows:
        out.append("| %s | %s | %.2e | %.2e | %.0e | %.3f | %s | %s |" % (
            r["path"], r["quantity"], r["floor_max"], r["floor_p99"], r["tolerance"], r["share_over"],
            "yes" if r["attainable"] else "NO for the samples above it", r["note"]))
    return "\n".join(out)


if __name__ == "__main__":
    print(markdown(report()))
