"""N > 1 host logic: batch sharding and the gather of the
per-model results, on CPU with the gloo backend, world_size 2 (and a ragged 3)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1910_01070_b200.sharding import gather_rows, shard_bounds


def test_shard_bounds_cover_the_batch_once():
    for n in (0, 1, 2, 7, 64, 255, 256, 4096):
        for world in (1, 2, 3, 8):
            blocks = [shard_bounds(n, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(blocks, blocks[1:]))
            sizes = [e - b for b, e in blocks]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_bounds(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_models, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        params = torch.arange(n_models * 3, dtype=torch.float64).reshape(n_models, 3)
        b, e = shard_bounds(n_models, rank, world)
        # stand-in for the per-rank hot path: any function of a model's own parameters
        local_logl = -(params[b:e] ** 2).sum(dim=1)
        local_spec = params[b:e, :2].float() * 0.5
        logl = gather_rows(local_logl, n_models)
        spec = gather_rows(local_spec, n_models)
        assert torch.equal(logl, -(params ** 2).sum(dim=1))
        assert torch.equal(spec, params[:, :2].float() * 0.5)
        # the timing reduction bench.py uses: max over ranks
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert t.item() == float(world)
        np.save(os.path.join(out_dir, f"ok{rank}.npy"), logl.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,n_models", [(2, 64), (2, 7), (3, 8)])
def test_gather_over_gloo(tmp_path, world, n_models):
    port = _free_port()
    mp.spawn(_worker, args=(world, port, n_models, str(tmp_path)), nprocs=world, join=True)
    outs = [np.load(tmp_path / f"ok{r}.npy") for r in range(world)]
    for o in outs[1:]:
        assert np.array_equal(o, outs[0])
