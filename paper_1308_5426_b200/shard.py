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


def all_gather_blocks(local_padded, n_total, dist, out=None):
    """The exchange step of a slot-sharded ensemble: every rank contributes its block of ensemble_shard(n_total, world,
    rank) values, stored at the front of a tensor padded to ceil(n_total / world) entries; returns the n_total values in
    global order (one all_gather; works for torch tensors on any device / backend)."""
    import torch
    world = dist.get_world_size()
    parts = [torch.empty_like(local_padded) for _ in range(world)]
    dist.all_gather(parts, local_padded)
    if out is None:
        out = torch.empty(n_total, dtype=local_padded.dtype, device=local_padded.device)
    pos = 0
    for r in range(world):
        _, n_r = ensemble_shard(n_total, world, r)
        out[pos:pos + n_r] = parts[r][:n_r]
        pos += n_r
    return out


class ShardedEnsemble:
    """ONE ensemble of n_rep replicas spread over the ranks of a process group: rank r sweeps
    a contiguous block of configurations (pt_create_shard); at every swap event the ranks all-gather their running
    energies (n_rep int64: the only data that ever crosses GPUs) and every rank takes the same swap decisions
    (pt_swap_external), so that only temperature labels move.  `dist` may be None (single process, all replicas)."""

    def __init__(self, pt, L, q, sigma, n_rep, betas, seed, dist=None, ens_base=0):
        import torch
        self.torch, self.dist = torch, dist
        self.world = dist.get_world_size() if dist is not None else 1
        self.rank = dist.get_rank() if dist is not None else 0
        self.n_rep = n_rep
        self.base, self.n_local = ensemble_shard(n_rep, self.world, self.rank)
        if self.n_local < 1:
            raise ValueError("more ranks than replicas")
        self.g = pt.PT(L, q, sigma, 1, n_rep, betas, seed, ens_base=ens_base, shard=(self.base, self.n_local))
        # sweeps, the copy of the local energies, the all-gather and the swap kernel are all enqueued on ONE stream (the
        # current torch stream, which NCCL collectives follow): a swap event costs no host round trip
        self.g.use_torch_stream(torch.cuda.current_stream())
        self.n_max = -(-n_rep // self.world)
        self._loc = torch.zeros(self.n_max, dtype=torch.int64, device="cuda")
        self._flat = torch.zeros(self.world * self.n_max, dtype=torch.int64, device="cuda")
        self._all = torch.zeros(n_rep, dtype=torch.int64, device="cuda")
        idx = []   # position of storage index x in the padded gather buffer
        for r in range(self.world):
            _, n_r = ensemble_shard(n_rep, self.world, r)
            idx += [r * self.n_max + k for k in range(n_r)]
        self._index = torch.tensor(idx, dtype=torch.int64, device="cuda")

    def gather_energies(self):
        """All configurations' running energies in storage order, on the device (the exchange step), enqueued."""
        torch = self.torch
        self.g.energy_storage_dev_async(self._loc[: self.n_local])
        if self.dist is None:
            self._all.copy_(self._loc[: self.n_rep])
            return self._all
        self.dist.all_gather_into_tensor(self._flat, self._loc)
        torch.index_select(self._flat, 0, self._index, out=self._all)
        return self._all

    def sweeps(self, n, swap_every=1):
        done = 0
        while done < n:
            chunk = n - done
            event = False
            if swap_every > 0:
                to_event = swap_every - (self.g.sweep_counter() % swap_every)
                if to_event <= chunk:
                    chunk, event = to_event, True
            self.g.sweeps_async(chunk, 0)
            if event:
                self.g.swap_external_async(self.gather_energies())
            done += chunk
        self.g.sync()

    def close(self):
        self.g.close()


def merge_shards(results, perms, bases, counts):
    """Host-side assembly of per-slot results of the shards of one ensemble: results[r] is an array [n_rep, ...] in
    slot order as returned by shard r (PT.energy()[0], PT.get_spins()[0]); slot t is taken from the shard that holds
    storage index perm[t]."""
    perm = np.asarray(perms[0]).reshape(-1)
    out = np.zeros_like(np.asarray(results[0]))
    for t, st in enumerate(perm):
        for r, (b, c) in enumerate(zip(bases, counts)):
            if b <= st < b + c:
                out[t] = np.asarray(results[r])[t]
    return out


def sum_observables(obs_list):
    """Field-wise sum of the shards' accumulators (each slot's samples were gathered by whichever shard held its
    configuration); the multi-word integers (sum_E2, sum_E4, sum_Nmax4) are added as whole integers."""
    first = obs_list[0]
    shape = first["n_samples"].shape
    out = {}
    for k in first:
        if k in ("sum_E2_lo", "sum_E2_hi", "sum_E4", "sum_Nmax4_lo", "sum_Nmax4_hi", "near_ties"):
            continue
        out[k] = sum(o[k] for o in obs_list)
    out["near_ties"] = first["near_ties"].copy()
    m64 = (1 << 64) - 1
    for lo, hi in (("sum_E2_lo", "sum_E2_hi"), ("sum_Nmax4_lo", "sum_Nmax4_hi")):
        out[lo] = np.zeros(shape, dtype=np.uint64)
        out[hi] = np.zeros(shape, dtype=np.int64)
        for idx in np.ndindex(*shape):
            v = sum((int(o[hi][idx]) << 64) + int(o[lo][idx]) for o in obs_list)
            out[lo][idx] = v & m64
            out[hi][idx] = v >> 64
    out["sum_E4"] = np.zeros(shape + (4,), dtype=np.uint64)
    for idx in np.ndindex(*shape):
        v = sum(sum(int(o["sum_E4"][idx + (k,)]) << (64 * k) for k in range(4)) for o in obs_list)
        for k in range(4):
            out["sum_E4"][idx + (k,)] = (v >> (64 * k)) & m64
    return out
