"""Multi-GPU plumbing: the N_HP + N_LP solves of one configuration are independent, so the
path shards over noise sources -- every rank holds the packed gauge field and takes whole batches of right-hand sides; the
only exchange is one gather of the [16][T] loops (16 KB per source).  No arithmetic of the method lives here.

torch.distributed does the transport: NCCL over NVLink for CUDA tensors, gloo for the CPU tests.
"""
import torch
import torch.distributed as dist


def source_batches(n_sources, nrhs, rank, world):
    """Batches (first_source, count) owned by `rank`: sources are cut into consecutive batches of `nrhs` (the last one may be
    shorter) and dealt round-robin, so every rank gets whole batches and the batch count differs by at most one."""
    if n_sources < 0 or nrhs < 1 or world < 1 or not (0 <= rank < world):
        raise ValueError("bad sharding arguments")
    batches = [(first, min(nrhs, n_sources - first)) for first in range(0, n_sources, nrhs)]
    return batches[rank::world]


def owned_sources(n_sources, nrhs, rank, world):
    return [first + k for first, count in source_batches(n_sources, nrhs, rank, world) for k in range(count)]


def gather_loops(local_loops, n_sources, nrhs, group=None):
    """All ranks: local_loops[k] ([16][T][2] doubles) belongs to owned_sources(...)[k].  Returns [n_sources][16][T][2] in source
    order on every rank.  One all_gather of equally sized (padded) blocks."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    counts = [len(owned_sources(n_sources, nrhs, r, world)) for r in range(world)]
    if local_loops.shape[0] != counts[rank]:
        raise ValueError("rank %d holds %d loops, owns %d sources" % (rank, local_loops.shape[0], counts[rank]))
    tail = tuple(local_loops.shape[1:])
    if world == 1:
        return local_loops.clone()
    pad = max(counts)
    block = torch.zeros((pad,) + tail, dtype=local_loops.dtype, device=local_loops.device)
    block[:counts[rank]] = local_loops
    blocks = [torch.empty_like(block) for _ in range(world)]
    dist.all_gather(blocks, block, group=group)
    out = torch.empty((n_sources,) + tail, dtype=local_loops.dtype, device=local_loops.device)
    for r in range(world):
        ids = owned_sources(n_sources, nrhs, r, world)
        if ids:
            out[torch.tensor(ids, device=out.device)] = blocks[r][:counts[r]]
    return out
