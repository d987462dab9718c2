"""Walker sharding across ranks (the paper's own parallel model is independent walks
over MPI ranks).  Walkers are independent units: every rank owns a contiguous range, holds its
own context (tables replicated, stored rho(G) with its walkers), and no collective runs inside energy or
move calls.  The only exchange is the optional gather of per-walker energies below."""
import numpy as np


def walker_range(n_walkers, rank, world):
    """Contiguous [lo, hi) of `n_walkers` for `rank` of `world`; sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world) or n_walkers < 0:
        raise ValueError("bad sharding arguments")
    base, extra = divmod(n_walkers, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def owner_of(walker, n_walkers, world):
    """Rank that owns global walker index `walker`, and its local index there."""
    for r in range(world):
        lo, hi = walker_range(n_walkers, r, world)
        if lo <= walker < hi:
            return r, walker - lo
    raise IndexError("walker index out of range")


def gather_energies(local_energies, n_walkers, group=None):
    """All ranks' per-walker energies in global walker order (numpy float64 array of length n_walkers).
    `local_energies`: this rank's torch tensor (CPU for gloo, CUDA for nccl)."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    sizes = [walker_range(n_walkers, r, world)[1] - walker_range(n_walkers, r, world)[0] for r in range(world)]
    assert local_energies.numel() == sizes[rank], "local energies do not match this rank's walker range"
    pad = max(sizes)
    buf = torch.zeros(pad, dtype=torch.float64, device=local_energies.device)
    buf[:sizes[rank]] = local_energies.to(torch.float64)
    out = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(out, buf, group=group)
    return np.concatenate([o[:s].cpu().numpy() for o, s in zip(out, sizes)])
