"""Data-parallel plumbing of the E_loc path (the model and the Hamiltonian tensors are
replicated on every GPU, the batch of unique samples is split; the only exchange is the reduction of the
per-rank statistics).  One process per GPU under `torch.distributed` (NCCL on the GPUs, gloo in the CPU tests).
No arithmetic of the method lives here: row partitions, the mini-batch a rank takes at a step, the
reduction of the five statistics `[sum n, sum n Re E, sum n Im E, sum n |E|^2, max |ratio|]` (include/nqs.h), and
the gradient exchange of PAPER.md:146 ("gradients from each node are averaged"): every rank evaluates Eq. 7 on its
shard with the GLOBAL baseline and normalisation (`global_stats` of nqs_energy_grad), so the all-reduce SUM of the
per-rank gradients is the gradient of the whole batch.
"""
import torch
import torch.distributed as dist


def shard_rows(n_rows: int, world: int, rank: int):
    """Contiguous, even partition of the unique samples by row: rank r owns rows [lo, hi)."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    return n_rows * rank // world, n_rows * (rank + 1) // world


def minibatch_of_step(step: int, rank: int, world: int, n_minibatches: int) -> int:
    """Weak scaling over gradient-accumulation mini-batches: at step k rank r processes
    mini-batch (k * world + r) mod n_minibatches, so one step covers `world` distinct mini-batches."""
    return (step * world + rank) % n_minibatches


def all_reduce_stats(stats, group=None):
    """Combine per-rank statistics in place: the first four entries add, the last one is a maximum.
    `stats` is a float64 tensor of 5 entries on the backend's device (CPU for gloo, CUDA for NCCL)."""
    if stats.dtype != torch.float64 or stats.numel() != 5:
        raise ValueError("stats must be 5 float64 values")
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        head, tail = stats[:4].clone(), stats[4:].clone()
        dist.all_reduce(head, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(tail, op=dist.ReduceOp.MAX, group=group)
        stats[:4] = head
        stats[4:] = tail
    return stats


def max_over_ranks(value: float, device="cpu", group=None) -> float:
    """Timing rule of bench.py: a multi-rank number is the maximum over ranks."""
    t = torch.tensor([value], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def all_reduce_gradient(grad, group=None):
    """Sum the per-rank gradients in place (each computed with the global statistics, see module docstring).
    `grad` is a float tensor on the backend's device."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(grad, op=dist.ReduceOp.SUM, group=group)
    return grad
