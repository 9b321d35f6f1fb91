"""K-sharded BR-MPPI solve over several GPUs: one process per GPU, every
rank owns a contiguous range of the K samples of ONE solve, and one iteration exchanges a single record of
8 + 2T floats per scene and rank (the online-softmax state of eq. (5): min, argmin, eta, sum w^2, A[2T]).

All arithmetic is in libbrmppi.so (brmppi_shard_export / brmppi_shard_import); this module owns the plumbing:
the sample ranges and the all-gather of the records over torch.distributed (NCCL on GPUs; the same code runs
over gloo with CPU tensors, which is how the exchange is tested without GPUs)."""


def shard_range(K, rank, world):
    """(first global sample index, number of samples) of `rank`: contiguous, disjoint, covering 0..K-1."""
    k0 = K * rank // world
    return k0, K * (rank + 1) // world - k0


def gather_records(dist, record, world=None, group=None):
    """All-gather of one record per rank -> tensor [world][record.numel()] in RANK order (the merge order)."""
    import torch
    world = dist.get_world_size(group) if world is None else world
    out = [torch.empty_like(record) for _ in range(world)]
    dist.all_gather(out, record.contiguous(), group=group)
    return torch.stack(out, dim=0)


class ShardedSolver:
    """One brmppi context per rank holding K/world samples of the same solve.  Inputs (state, goal, obstacles,
    nominal) must be set identically on every rank; U comes out bit-identical on all of them."""

    def __init__(self, brmppi, params, dist, n_scenes=1, max_obstacles=8, flags=0, device="cuda:0", group=None):
        import torch
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.k0, self.Kr = shard_range(params.K, self.rank, self.world)
        if self.Kr < 1:
            raise ValueError("more ranks than samples")
        self.params = params
        self.solver = brmppi.Solver(params.with_(K=self.Kr), n_scenes, max_obstacles, flags, device=device,
                                    k_offset=self.k0)
        self.record = torch.empty(self.solver.shard_words(), dtype=torch.float32, device=device)
        self._torch = torch

    def __getattr__(self, name):            # set_state / set_goal / set_obstacles / get_controls / ... of the shard
        return getattr(self.solver, name)

    def solve(self):
        torch = self._torch
        for _ in range(self.params.n_iter):
            self.solver.shard_export(self.record)
            with torch.cuda.stream(self.solver.stream):          # the collective follows the export on its stream
                records = gather_records(self.dist, self.record, self.world, self.group)
            self.solver.shard_import(records, self.world)
            records.record_stream(self.solver.stream)

    def close(self):
        self.solver.close()
