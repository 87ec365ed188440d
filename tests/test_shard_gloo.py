"""N > 1 path on CPU: two gloo ranks each run their shard of the ensembles (the oracle stands in for the GPU
library: same ens_base semantics as pt_create_ex) and the gathered results must equal the unsharded run."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_ens_total, out_dir):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from oracle import pt_oracle
    from paper_1308_5426_b200 import inputs, shard
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        L, q, sigma, n_rep, seed = 64, 3, 0.5, 4, 9
        b = inputs.geometric_betas(0.8, 2.0, n_rep)
        base, n_local = shard.ensemble_shard(n_ens_total, world, rank)
        if n_local > 0:
            o = pt_oracle.Oracle(L, q, sigma, n_local, n_rep, b, seed, ens_base=base)
            o.sweeps(30, 1)
            E, obs = o.energy(), o.observables()
            acc, sE = obs["flip_accepts"], obs["sum_E"]
        else:
            E = acc = sE = np.zeros((0, n_rep), dtype=np.int64)
        E_all = shard.gather_ensembles(E, n_ens_total, dist)
        acc_all = shard.gather_ensembles(acc, n_ens_total, dist)
        sE_all = shard.gather_ensembles(sE, n_ens_total, dist)
        # exchange step of a slot-sharded ensemble: uneven blocks, padded all_gather, global order
        import torch
        for n_total in (7, 8, 2):
            b0, nl = shard.ensemble_shard(n_total, world, rank)
            n_max = -(-n_total // world)
            loc = torch.full((n_max,), -1, dtype=torch.int64)
            loc[:nl] = torch.arange(b0, b0 + nl) * 1000003
            got = shard.all_gather_blocks(loc, n_total, dist)
            assert torch.equal(got, torch.arange(n_total) * 1000003), (rank, n_total, got)
        t_max = shard.max_over_ranks(10.0 + rank, dist)
        assert t_max == 10.0 + world - 1
        if rank == 0:
            np.savez(os.path.join(out_dir, "gathered.npz"), E=E_all, acc=acc_all, sE=sE_all)
    finally:
        dist.destroy_process_group()


def test_ensemble_shard_partition():
    from paper_1308_5426_b200 import shard
    for n in (0, 1, 5, 40):
        for world in (1, 2, 3, 8):
            blocks = [shard.ensemble_shard(n, world, r) for r in range(world)]
            assert sum(b[1] for b in blocks) == n
            pos = 0
            for base, cnt in blocks:
                assert base == pos
                pos += cnt
            assert max(b[1] for b in blocks) - min(b[1] for b in blocks) <= 1
    with pytest.raises(ValueError):
        shard.ensemble_shard(4, 2, 2)


@pytest.mark.parametrize("n_ens_total", [4, 3])
def test_two_ranks_reproduce_the_unsharded_run(tmp_path, oracle, n_ens_total):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), n_ens_total, str(tmp_path)), nprocs=world, join=True)
    got = np.load(os.path.join(str(tmp_path), "gathered.npz"))
    from paper_1308_5426_b200 import inputs
    L, q, sigma, n_rep, seed = 64, 3, 0.5, 4, 9
    whole = oracle.Oracle(L, q, sigma, n_ens_total, n_rep, inputs.geometric_betas(0.8, 2.0, n_rep), seed)
    whole.sweeps(30, 1)
    obs = whole.observables()
    np.testing.assert_array_equal(got["E"], whole.energy())
    np.testing.assert_array_equal(got["acc"], obs["flip_accepts"])
    np.testing.assert_array_equal(got["sE"], obs["sum_E"])
    # different ensembles really are different streams
    assert not np.array_equal(got["E"][0], got["E"][1])
