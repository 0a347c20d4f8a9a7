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


class LoopGather:
    """The gather of gather_loops() with everything that does not depend on the data prepared once: block sizes, the padded
    send block, the receive buffer and the index that puts the received rows into source order (one index_select per call,
    no host-to-device copy and no synchronisation inside a timed loop)."""

    def __init__(self, n_sources, nrhs, tail, dtype, device, group=None):
        self.group = group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.n_sources = n_sources
        self.counts = [len(owned_sources(n_sources, nrhs, r, self.world)) for r in range(self.world)]
        self.pad = max(self.counts) if self.counts else 0
        tail = tuple(tail)
        self.block = torch.zeros((self.pad,) + tail, dtype=dtype, device=device)
        self.recv = torch.empty((self.world * self.pad,) + tail, dtype=dtype, device=device)
        perm = [0] * n_sources
        for r in range(self.world):
            for k, src in enumerate(owned_sources(n_sources, nrhs, r, self.world)):
                perm[src] = r * self.pad + k
        self.perm = torch.tensor(perm, dtype=torch.long, device=device)

    def __call__(self, local_loops):
        if local_loops.shape[0] != self.counts[self.rank]:
            raise ValueError("rank %d holds %d loops, owns %d sources" % (self.rank, local_loops.shape[0], self.counts[self.rank]))
        if self.world == 1:
            return local_loops.index_select(0, self.perm)
        self.block[:self.counts[self.rank]] = local_loops
        dist.all_gather_into_tensor(self.recv, self.block, group=self.group)
        return self.recv.index_select(0, self.perm)


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
