"""The N > 1 path on CPU: world_size-2 gloo processes shard the baselines.
Each rank grids ITS baselines (here with the float64 oracle standing in for the device kernels:
this test is about the host logic, not the kernels), the grids are summed with the product's
all-reduce helper, and the result must equal the single-process grid; the degridded visibilities
gathered over ranks must equal the single-process prediction."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1909_07226_b200 import sharding


def test_baseline_ranges_cover_exactly_once():
    for B in (0, 1, 7, 28, 1128, 8128):
        for world in (1, 2, 3, 8):
            seen = np.zeros(B, dtype=int)
            sizes = []
            for r in range(world):
                b, e = sharding.baseline_range(B, world, r)
                seen[b:e] += 1
                sizes.append(e - b)
            assert np.all(seen == 1) and max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.baseline_range(10, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import idg_oracle as orc
        from paper_1909_07226_b200 import synth
        w = synth.make_workload("tiny")
        uvw, vis, bl, b0 = sharding.shard_inputs(w.uvw, w.vis, w.baselines, world, rank)
        meta, planned, skipped = orc.plan(w.params, uvw.numpy(), w.freqs, bl)
        at, tp = w.aterms.numpy(), w.taper.numpy()
        g = orc.grid(w.params, meta, uvw.numpy(), w.freqs, vis.numpy(), at, tp)
        grid = torch.from_numpy(g.astype(np.complex64))
        sharding.allreduce_grid(grid)
        model = grid.clone()
        sharding.broadcast_grid(model, src=0)
        assert torch.equal(model, grid)          # every rank holds the same summed grid
        pred = orc.degrid(w.params, meta, uvw.numpy(), w.freqs, model.numpy().astype(np.complex128), at, tp,
                          len(bl))
        allv = sharding.gather_visibilities(torch.from_numpy(pred.astype(np.complex64)), w.B)
        cnt = torch.tensor([planned, skipped], dtype=torch.int64)
        dist.all_reduce(cnt)
        if rank == 0:
            np.save(os.path.join(out_dir, "grid.npy"), grid.numpy())
            np.save(os.path.join(out_dir, "vis.npy"), allv.numpy())
            np.save(os.path.join(out_dir, "cnt.npy"), cnt.numpy())
    finally:
        dist.destroy_process_group()


def test_two_ranks_equal_one(tmp_path):
    from oracle import idg_oracle as orc
    from paper_1909_07226_b200 import synth
    orc.lib()                                    # build once, before the workers race for it
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    w = synth.make_workload("tiny")
    meta, planned, skipped = orc.plan(w.params, w.uvw.numpy(), w.freqs, w.baselines)
    at, tp = w.aterms.numpy(), w.taper.numpy()
    g = orc.grid(w.params, meta, w.uvw.numpy(), w.freqs, w.vis.numpy(), at, tp)
    got = np.load(tmp_path / "grid.npy")
    assert np.linalg.norm(got - g) / np.linalg.norm(g) < 1e-6           # complex64 partial sums
    assert tuple(np.load(tmp_path / "cnt.npy")) == (planned, skipped)
    pred = orc.degrid(w.params, meta, w.uvw.numpy(), w.freqs, got.astype(np.complex128), at, tp, w.B)
    v = np.load(tmp_path / "vis.npy")
    assert v.shape == pred.shape
    assert np.linalg.norm(v - pred) / np.linalg.norm(pred) < 1e-6
