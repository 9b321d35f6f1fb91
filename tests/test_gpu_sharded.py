"""K-sharded solve (brmppi_shard_export / brmppi_shard_import) on ONE GPU: G contexts that each own
K/G of the samples of the same solve, records exchanged by a plain concatenation (what an all-gather delivers),
against a single context with all K samples and against the oracle.  Per-sample results are bit-identical (a
sample's cost depends on its own draws and on U only); U differs from the single context's only in the order of
the fp32 merge."""
import numpy as np
import pytest

import scenes
from paper_2508_05773_b200 import sharded

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    from paper_2508_05773_b200 import brmppi
    brmppi.lib()
    return brmppi


def sharded_solve(B, sc, p, G, flags):
    import torch
    shards = []
    for r in range(G):
        k0, Kr = sharded.shard_range(p.K, r, G)
        s = B.Solver(p.with_(K=Kr), 1, max(len(sc.obstacles), 1), flags | B.FLAG_WRITE_SAMPLES, k_offset=k0)
        s.set_scene(sc)
        shards.append(s)
    words = shards[0].shard_words()
    records = torch.empty((G, words), dtype=torch.float32, device="cuda")
    for _ in range(p.n_iter):
        for r, s in enumerate(shards):
            s.shard_export(records[r])
            s.synchronize()
        for s in shards:
            s.shard_import(records, G)
            s.synchronize()
    out = dict(U=[s.get_controls() for s in shards], S=np.concatenate([s.get_costs() for s in shards]),
               XT=np.concatenate([s.get_final_states() for s in shards]), diag=[s.get_diag() for s in shards])
    for s in shards:
        s.close()
    return out


@pytest.mark.parametrize("flags", [0, 4, 32], ids=["tile", "thread", "projected"])
@pytest.mark.parametrize("G", [2, 3])
def test_shards_equal_the_single_context(B, O, G, flags):
    sc = scenes.scene_cfg2(1)
    p = sc.params.with_(K=1000, T=40, n_iter=2)
    single = B.Solver(p, 1, 8, flags | B.FLAG_WRITE_SAMPLES)
    single.set_scene(sc)
    single.solve()
    ref = dict(U=single.get_controls(), S=single.get_costs(), XT=single.get_final_states(), diag=single.get_diag())
    single.close()
    got = sharded_solve(B, sc, p, G, flags)
    for U in got["U"][1:]:
        assert np.array_equal(U, got["U"][0])               # every shard merges the same records in the same order
    floors = np.array([p.v_max, p.delta_max])[None, :]
    assert (np.abs(got["U"][0] - ref["U"]) <= 2e-6 * floors).all()
    # second-iteration costs: per sample, from a nominal that differs by the merge order only
    assert (np.abs(got["S"] - ref["S"]) <= 1e-5 * np.maximum(np.abs(ref["S"]), 1.0)).all()
    assert got["diag"][0]["argmin"] == ref["diag"]["argmin"] and got["diag"][0]["n"] == 2
    assert got["diag"][0]["eta"] == pytest.approx(ref["diag"]["eta"], rel=1e-4)


def test_first_iteration_samples_are_bit_identical_and_match_the_oracle(B, O):
    sc = scenes.scene_cfg1(2)
    p = sc.params.with_(K=777, T=30, n_iter=1)
    single = B.Solver(p, 1, 8, B.FLAG_WRITE_SAMPLES)
    single.set_scene(sc)
    single.solve()
    S1, X1 = single.get_costs(), single.get_final_states()
    single.close()
    got = sharded_solve(B, sc, p, 3, 0)
    assert np.array_equal(got["S"], S1) and np.array_equal(got["XT"], X1)
    ref = O.solve(p, 0, sc.x0, sc.goal, sc.obstacles, np.zeros((p.T, 2)), n_threads=4)[-1]
    floors = np.array([p.v_max, p.delta_max])[None, :]
    assert (np.abs(got["U"][0] - ref["U"]) <= 1e-4 * np.maximum(np.abs(ref["U"]), floors)).all()
    assert got["diag"][0]["argmin"] == ref["argmin"]


def test_shard_errors(B):
    import ctypes as C
    import torch
    sc = scenes.scene_cfg0(0)
    s = B.Solver(sc.params, 1, 1, 0)
    assert s.shard_words() == 8 + 2 * sc.params.T
    rec = torch.empty(s.shard_words(), dtype=torch.float32, device="cuda")
    assert B.lib().brmppi_shard_export(s._ctx, C.c_void_p(rec.data_ptr())) == B.ERR_NOT_READY      # no state / goal yet
    s.set_scene(sc)
    assert B.lib().brmppi_shard_export(s._ctx, None) == B.ERR_NULL
    assert B.lib().brmppi_shard_import(s._ctx, 0, C.c_void_p(rec.data_ptr())) == B.ERR_INVALID_ARG
    assert B.lib().brmppi_shard_export(s._ctx, C.c_void_p(rec.data_ptr() + 4)) == B.ERR_UNALIGNED
    s.close()
    with pytest.raises(B.BrmppiError):
        B.Solver(sc.params, 1, 1, 0, k_offset=-1)
