"""P-sharded sigma-build over several GPUs (SURVEY 8(e) option 2; "distributing these chunks across multiple GPUs",
PAPER.md:395): one process and one `risp_ctx` per GPU, set up with `shard_rank` / `shard_count`, the trial vectors replicated.
Each rank holds every shard_count-th kept shell pair (both integral passes and the pair-sparse halves of the J transforms) and
the K-tensor slices of every shard_count-th auxiliary centre (Eq. 22-23), so the 3000-atom K tensors need no host streaming
from 2 GPUs on.  Two collectives per batch, both through `torch.distributed` (NCCL over NVLink on GPUs, gloo in the CPU test):

    R_mQ   all-reduce between the passes   nauxJ x 32 doubles   (< 2 MB)
    sigma  all-reduce at the end           m x nocc x nvir doubles

Argument marshalling and the two collectives only; every arithmetic step runs in the library's kernels.
"""
from __future__ import annotations


def sharded_matvec(ctx, X, group=None):
    """sigma = A X on this rank, identical on all ranks after the final all-reduce.  `ctx` is this rank's sharded RispContext
    (anything with matvec_shard_begin / matvec_shard_end), X the replicated trial vectors [m][nocc][nvir], m <= 32."""
    import torch.distributed as dist
    R = ctx.matvec_shard_begin(X)
    dist.all_reduce(R, op=dist.ReduceOp.SUM, group=group)
    sigma = ctx.matvec_shard_end(X, R)
    dist.all_reduce(sigma, op=dist.ReduceOp.SUM, group=group)
    return sigma


def shard_of_pair(kept_index: int, shard_count: int) -> int:
    """rank that owns the kept shell pair with this running index (round robin, as risp_setup deals them)"""
    return kept_index % max(shard_count, 1)


def shard_of_aux_centre(centre_index: int, shard_count: int) -> int:
    """rank that owns the K-tensor slices of this auxiliary centre"""
    return centre_index % max(shard_count, 1)
