"""Output-sharded projection over several GPUs ("a future multi-GPU modification",
L572, rule L342 "all records of the same output on the same [device]": no output is ever merged).

One process per GPU.  Every rank builds its plan with `shard_rank` / `shard_count`: the planner assigns the output segments
to ranks by longest-processing-time on their FLOP cost (dmrg_partition_outputs; every rank computes the same table) and keeps
only the records of the outputs it owns.  One projection = the local grouped launch into a zeroed vector + ONE all-reduce
(sum) of that vector over NCCL -- every element has exactly one non-zero contributor, so the sum is exact and bitwise
independent of the reduction order.  The Davidson BLAS-2 part runs replicated on every rank (dmrg_davidson_step_given_w),
which keeps the iteration state identical everywhere without further collectives.

This module is plumbing only (torch.distributed); the arithmetic is in the kernels behind the plan."""
from __future__ import annotations


def sharded_apply(apply_local, x, y, dist=None, group=None):
    """y = H x with the outputs sharded over the ranks of `dist`: `apply_local(x, y)` writes the segments this rank owns
    into y (zeroed here first), the all-reduce fills in the others.  Works for any tensor type `dist` supports."""
    y.zero_()
    apply_local(x, y)
    if dist is not None and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(y, op=dist.ReduceOp.SUM, group=group)
    return y


class ShardedDavidson:
    """Alg. 3 with the projection sharded by outputs: line 2 = local launch + all-reduce, lines 3-14 replicated."""

    def __init__(self, plan, dist=None, group=None):
        self.plan, self.dist, self.group = plan, dist, group

    def step(self, V, W, k: int):
        n = self.plan.n
        sharded_apply(lambda a, b: self.plan.apply_H(a, b), V[k - 1, :n], W[k - 1, :n], self.dist, self.group)
        return self.plan.davidson_step_given_w(V, W, k)
