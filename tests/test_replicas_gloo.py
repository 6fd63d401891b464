"""N > 1 = replicas only: rank i owns realizations [i*R, (i+1)*R), no collective
on the data path.  World-size-2 `gloo` run on CPU: each rank follows its shard with the oracle (no GPU
here), the integer sums are gathered, and the union must equal one run over all 2R realizations --
i.e. the shard bookkeeping of bench.py (workloads.replica_range -> first_real) tiles a run exactly,
and the max-over-ranks timing reduction works.
"""
import os
import socket

import numpy as np
import pytest


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, L, N, R, seed, mcs, out):
    import torch
    import torch.distributed as dist
    from oracle import rsos_oracle
    from paper_1605_02620_b200.utils import workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    first_real, r = workloads.replica_range(rank, world, R)
    o = rsos_oracle.Oracle(L, N, r, seed, first_real=first_real, threads=1)
    o.advance(mcs)
    s1, s2, acc = o.sums()
    mine = torch.from_numpy(np.stack([s1.astype(np.int64), s2.astype(np.int64), acc.astype(np.int64)]))
    gathered = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(gathered, mine)                       # harness-side gather only: the data path has no collective
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)              # bench.py's max-over-ranks timing
    if rank == 0:
        np.save(out, torch.cat(gathered, dim=1).numpy())
        assert float(t.item()) == float(world)
    dist.barrier()
    dist.destroy_process_group()


def test_two_replica_ranks_tile_a_run(tmp_path, oracle_mod):
    import torch.multiprocessing as mp
    L, N, R, seed, mcs, world = 128, 1, 3, 9, 3, 2
    out = str(tmp_path / "sums.npy")
    mp.spawn(_worker, args=(world, _free_port(), L, N, R, seed, mcs, out), nprocs=world, join=True)
    got = np.load(out)
    whole = oracle_mod.Oracle(L, N, world * R, seed)
    whole.advance(mcs)
    s1, s2, acc = whole.sums()
    assert (got[0] == s1.astype(np.int64)).all()
    assert (got[1] == s2.astype(np.int64)).all()
    assert (got[2] == acc.astype(np.int64)).all()


def test_replica_range_bounds():
    from paper_1605_02620_b200.utils import workloads
    assert workloads.replica_range(0, 8, 128) == (0, 128)
    assert workloads.replica_range(7, 8, 128) == (896, 128)
    with pytest.raises(ValueError):
        workloads.replica_range(8, 8, 128)
