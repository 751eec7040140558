"""N-GPU form of the path: sub-graph predictions are independent, so rank r evaluates the
sub-domains k with k mod world == r (mlip_energy_forces_shard applies the same rule inside the library) and ONE
all-reduce sums the partial energy and the partial forces. Host logic only; torch.distributed does the exchange
(NCCL on GPUs, gloo in the CPU tests)."""
from __future__ import annotations


def subdomains_of(rank: int, world: int, n_sub: int) -> list[int]:
    """Sub-domains owned by `rank`: k mod world == rank (the rule of mlip_energy_forces_shard)."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    return [k for k in range(n_sub) if k % world == rank]


def all_reduce_results(*tensors):
    """Sum every partial result (E [1] float64, F [N,3] float32, optionally sigma [3,3] float64) over all ranks in
    place. No-op when torch.distributed is not initialised (single process)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        for t in tensors:
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return tensors
