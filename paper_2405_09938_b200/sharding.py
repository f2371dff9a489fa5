"""Multi-GPU plan: pulses are independent units, so the path shards by
pulse with NO data-path collective -- each rank owns the whole (procedural) scene and writes a
disjoint [c][pulse-slab][n] block.  The optional gather below is plumbing over
torch.distributed (NCCL on GPUs, gloo in the CPU tests); the paper's own scheme divides tiles
between devices and lets "a final thread gather the sparse raw data".
"""
from __future__ import annotations


def pulse_slab(n_pulses: int, rank: int, world_size: int) -> tuple[int, int]:
    """Contiguous, balanced split of [0, n_pulses): the first n_pulses % world ranks get one extra."""
    if world_size < 1 or not (0 <= rank < world_size) or n_pulses < 0:
        raise ValueError("bad rank/world_size/n_pulses")
    base, extra = divmod(n_pulses, world_size)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def gather_slabs(local, n_pulses: int, group=None):
    """All-gather per-rank slabs [C][p_r][Ns] into the full [C][P][Ns] tensor on every rank.

    Slabs may be ragged (P not divisible by world size); they are padded to the largest slab for
    the collective and trimmed afterwards.
    """
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    sizes = [pulse_slab(n_pulses, r, world) for r in range(world)]
    pmax = max(e - b for b, e in sizes)
    C, p_loc, ns = local.shape
    pad = local
    if p_loc < pmax:
        pad = torch.zeros((C, pmax, ns), dtype=local.dtype, device=local.device)
        pad[:, :p_loc] = local
    # complex tensors travel as real pairs (gloo has no complex all_gather)
    buf = torch.view_as_real(pad.contiguous())
    parts = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf, group=group)
    out = torch.empty((C, n_pulses, ns), dtype=local.dtype, device=local.device)
    for r, (b, e) in enumerate(sizes):
        out[:, b:e] = torch.view_as_complex(parts[r])[:, : e - b]
    return out
