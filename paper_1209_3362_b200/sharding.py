"""Multi-GPU host logic of time-chunk sharding (include/nfs.h: nfs_push_halo, nfs_export_partials,
nfs_import_partials).

The structure function is a sum over frame pairs, so one stack splits over G ranks by the LATER
frame of each pair: rank g owns the frames [g N / G, (g+1) N / G) and first receives the Lmax frames before them as a
halo; every pair is then counted on exactly one rank.  The ranks' partial sums (pair sums per lag, sum |F|^2, sum F, pair
and frame counts) are added by ONE all-reduce, after which every rank holds the result of the whole stack.  This module
holds only the plan and the collective call, so that both are covered by world_size-2 gloo tests on CPU; the arithmetic
is in the kernels.
"""
from dataclasses import dataclass


@dataclass(frozen=True)
class Shard:
    rank: int
    halo_start: int   # first halo frame (== own_start when the rank has no halo)
    own_start: int    # first own frame
    own_end: int      # one past the last own frame

    @property
    def n_halo(self):
        return self.own_start - self.halo_start

    @property
    def n_own(self):
        return self.own_end - self.own_start


def shard_plan(n_frames: int, world: int, lag_max: int):
    """Contiguous time chunks of (almost) equal length, each preceded by a halo of min(lag_max, frames before it)
    frames.  With more ranks than frames some chunks are empty (own_start == own_end); such a rank pushes nothing, and
    merge() still works on it: its context exports zeros and imports the total (include/nfs.h)."""
    assert n_frames >= 1 and world >= 1 and lag_max >= 1
    out = []
    for g in range(world):
        a = (g * n_frames) // world
        b = ((g + 1) * n_frames) // world
        out.append(Shard(g, max(0, a - lag_max), a, b))
    return out


def pairs_on_shard(sh: Shard, lag: int) -> int:
    """Frame pairs (s - lag, s) whose later frame s is owned by the shard (the earlier one may lie anywhere before:
    the halo is assumed complete, which shard_plan guarantees for lag <= lag_max)."""
    lo = max(sh.own_start, lag)
    return max(0, sh.own_end - lo)


def all_reduce_sum(buf, dist=None):
    """SUM all-reduce of a tensor in place (NCCL over NVLink for CUDA tensors, gloo on CPU); identity without a
    process group.  Returns the tensor."""
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)
    return buf


def push_shard(nfs, stack, sh: Shard, chunk: int = 0):
    """Feeds a rank's part of a device-resident stack to its context: the halo, then the own frames."""
    if sh.n_halo > 0:
        nfs.push_halo(stack[sh.halo_start:sh.own_start])
    if sh.n_own > 0:
        step = chunk or sh.n_own
        for i in range(sh.own_start, sh.own_end, step):
            nfs.push(stack[i:min(i + step, sh.own_end)])


def merge(nfs, dist=None):
    """The one collective of the sharded path: export this rank's partial sums, add them over the ranks, import the
    total.  Afterwards nfs.finalize() returns the result of the whole stack on every rank."""
    buf = nfs.export_partials()
    all_reduce_sum(buf, dist)
    nfs.import_partials(buf)
    return buf.numel() * 8
