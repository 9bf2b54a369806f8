"""-m gpu, needs TWO devices (skipped otherwise): the sharded path of DESIGN.md section 11 with the CUDA kernels and
NCCL -- every rank plans and grids its contiguous baseline range (sharding.baseline_range), the [4][L][L] grids are
summed with one all-reduce, every rank degrids its range from the reduced grid, the visibilities are gathered.  The
2-rank grid and visibilities must equal the 1-rank result (FP32 sums in another order: 1e-6).
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dev = torch.device("cuda", rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    try:
        from paper_1909_07226_b200 import binding as idg
        from paper_1909_07226_b200 import sharding, synth
        full = synth.make_workload("lofar", n_baselines=64, baseline_offset=500, n_time=128)
        # the rank's contiguous baseline range of ONE data set (A-terms, taper and frequencies replicated)
        uvw, vis, bl, b0 = sharding.shard_inputs(full.uvw, full.vis, full.baselines, world, rank)
        import dataclasses
        w = dataclasses.replace(full, uvw=uvw, vis=vis, baselines=bl).to(dev)
        plan = idg.idg_plan_create(w.params, w.uvw, w.freqs, w.baselines, w.n_stations)
        L = w.params.grid_size
        grid = torch.zeros((4, L, L), dtype=torch.complex64, device=dev)
        idg.idg_grid(plan, w.uvw, w.vis, w.aterms, w.taper, grid)
        sharding.allreduce_grid(grid)
        out = torch.zeros_like(w.vis)
        idg.idg_degrid(plan, w.uvw, grid, w.aterms, w.taper, out)
        allv = sharding.gather_visibilities(out, full.B)
        torch.cuda.synchronize()
        if rank == 0:
            np.save(os.path.join(out_dir, "grid.npy"), grid.cpu().numpy())
            np.save(os.path.join(out_dir, "vis.npy"), allv.cpu().numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two CUDA devices")
def test_two_nccl_ranks_equal_one_rank(tmp_path):
    from paper_1909_07226_b200 import binding as idg
    from paper_1909_07226_b200 import synth
    mp.spawn(_worker, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
    w = synth.make_workload("lofar", n_baselines=64, baseline_offset=500, n_time=128).to("cuda:0")
    plan = idg.idg_plan_create(w.params, w.uvw, w.freqs, w.baselines, w.n_stations)
    L = w.params.grid_size
    grid = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda:0")
    idg.idg_grid(plan, w.uvw, w.vis, w.aterms, w.taper, grid)
    out = torch.zeros_like(w.vis)
    idg.idg_degrid(plan, w.uvw, grid, w.aterms, w.taper, out)
    torch.cuda.synchronize()
    g1, v1 = grid.cpu().numpy(), out.cpu().numpy()
    g2, v2 = np.load(tmp_path / "grid.npy"), np.load(tmp_path / "vis.npy")
    assert np.linalg.norm(g2 - g1) / np.linalg.norm(g1) < 1e-6
    assert v2.shape == v1.shape
    assert np.linalg.norm(v2 - v1) / np.linalg.norm(v1) < 1e-6
