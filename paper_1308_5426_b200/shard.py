"""Multi-GPU plumbing: ensembles are independent, so they are sharded over ranks with no data-path collective
(pt_create_ex(..., ens_base)).  This module holds the host-side logic only: which ensembles a
rank owns, and how per-ensemble results are put back in global order.  It needs torch.distributed (NCCL on the
GPUs, gloo in the CPU tests) and no CUDA extension."""
import numpy as np


def ensemble_shard(n_ens_total, world_size, rank):
    """Contiguous block of ensembles of `rank`: returns (ens_base, n_ens_local); the first
    n_ens_total % world_size ranks take one more.  n_ens_local may be 0 when world_size > n_ens_total."""
    if n_ens_total < 0 or world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("bad shard arguments")
    q, r = divmod(n_ens_total, world_size)
    n_local = q + (1 if rank < r else 0)
    base = rank * q + min(rank, r)
    return base, n_local


def gather_ensembles(local, n_ens_total, dist, device=None):
    """All ranks contribute their [n_ens_local, ...] int64 array (ensemble-major, as returned by PT.energy() or one
    field of PT.observables()); every rank receives the [n_ens_total, ...] array in global ensemble order.
    One all_gather of equally padded blocks; exact (integers)."""
    import torch
    world, rank = dist.get_world_size(), dist.get_rank()
    local = np.ascontiguousarray(local, dtype=np.int64)
    base, n_local = ensemble_shard(n_ens_total, world, rank)
    if local.shape[0] != n_local:
        raise ValueError("rank %d holds %d ensembles, expected %d" % (rank, local.shape[0], n_local))
    tail = local.shape[1:]
    n_max = -(-n_ens_total // world)
    buf = np.zeros((n_max,) + tail, dtype=np.int64)
    buf[:n_local] = local
    t = torch.from_numpy(buf)
    if device is not None:
        t = t.to(device)
    out = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(out, t)
    parts = []
    for r in range(world):
        _, n_r = ensemble_shard(n_ens_total, world, r)
        parts.append(out[r].cpu().numpy()[:n_r])
    return np.concatenate(parts, axis=0) if parts else np.zeros((0,) + tail, dtype=np.int64)


def max_over_ranks(value, dist, device=None):
    """Max over ranks of a float (device-timed milliseconds)."""
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
