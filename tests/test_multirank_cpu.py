"""The N>1 path on the CPU: world_size 2 over gloo.

Slices are independent problems, so ranks shard them with no data-path collective; what
the multi-rank code adds is host logic only: the slice ranges, the per-rank seeding bench.py uses, and the
MAX-over-ranks reduction of the timings.  No CUDA call is made here."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_slices, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    import paper_2109_02174_b200 as pkg
    from paper_2109_02174_b200 import inputs as I

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = pkg.shard_slices(n_slices, rank, world)
        # every rank checksums the inputs of its own slices (cfg 1 geometry, per-slice seeded noise)
        sums = torch.zeros(n_slices, dtype=torch.float64)
        clean = I.config_slice(1)
        for s in mine:
            sums[s] = float(I.gaussian_noise(clean, 0.01, 4100 + s).sum())
        dist.all_reduce(sums, op=dist.ReduceOp.SUM)          # disjoint shards: SUM == gather
        owned = torch.zeros(n_slices, dtype=torch.int64)
        owned[list(mine)] = 1
        dist.all_reduce(owned, op=dist.ReduceOp.SUM)
        # bench.py's timing reduction: max over ranks
        t = torch.tensor([10.0 + rank, 5.0 - rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        if rank == 0:
            np.save(out, np.concatenate([sums.numpy(), owned.numpy().astype(np.float64), t.numpy()]))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_world_size_2_gloo_slice_sharding(tmp_path):
    import torch.multiprocessing as mp

    from paper_2109_02174_b200 import inputs as I

    world, n_slices = 2, 5
    out = str(tmp_path / "res.npy")
    mp.spawn(_worker, args=(world, _free_port(), n_slices, out), nprocs=world, join=True)
    res = np.load(out)
    sums, owned, t = res[:n_slices], res[n_slices:2 * n_slices], res[2 * n_slices:]
    assert np.array_equal(owned, np.ones(n_slices))           # every slice has exactly one owner
    clean = I.config_slice(1)
    want = np.array([I.gaussian_noise(clean, 0.01, 4100 + s).sum() for s in range(n_slices)])
    assert np.allclose(sums, want, rtol=1e-14)                # same bytes as a single-rank run would see
    assert list(t) == [11.0, 5.0]                             # max over ranks
