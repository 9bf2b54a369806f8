"""-m gpu: parity at the FULL size of BASELINE.json's configurations, in the launch configuration bench.py times.

configs[1] (LOFAR-like) is small enough for the float64 oracle to run every subgrid (about 15 s on 16 host cores),
so there the whole grid, every subgrid, the adder on the full plan and every degridded visibility are compared
element by element (Alg. 1 / Alg. 2).  configs[2]/[3] (SKA-low-like, 133 M visibilities) get a
STRATIFIED sample of subgrids: short and long baselines, every w layer, halved channel groups, subgrids at the
edge of the covered part of the grid.
"""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import idg_oracle as orc
from paper_1909_07226_b200 import binding as idg
from paper_1909_07226_b200 import synth
from tests import helpers as H

pytestmark = pytest.mark.gpu
TOL = 1e-4


def _host_arrays(w):
    return dict(uvw=w.uvw.cpu().numpy(), freqs=w.freqs, vis=w.vis.cpu().numpy(),
                aterms=w.aterms.cpu().numpy(), taper=w.taper.cpu().numpy())


def test_lofar_full_every_subgrid_every_visibility():
    """configs[1] end to end over all 4512 subgrids: the [4][2048][2048] grid against orc.grid, every subgrid
    against the oracle's, the adder against oracle_adder on the full plan, all 4.6 M degridded visibilities
    against orc.degrid; worst subgrid and worst visibility asserted, not only the totals."""
    w = synth.make_workload("lofar")
    wc = w.to("cuda")
    d = _host_arrays(w)
    prm = w.params
    N, L = prm.subgrid_size, prm.grid_size
    plan = idg.idg_plan_create(prm, wc.uvw, w.freqs, w.baselines, w.n_stations)
    meta, planned, skipped = orc.plan(prm, d["uvw"], d["freqs"], w.baselines)
    assert plan.metadata().tobytes() == meta.tobytes() and plan.size() == (len(meta), planned, skipped)
    P = len(meta)
    assert P > 4000 and planned == w.B * w.T * w.C

    # ---- Alg. 1, stage by stage and as one call
    ref_sub = orc.subgrid_fft(orc.gridder(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"]), -1)
    sub = plan.subgrids()
    idg.idg_gridder(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, sub)
    idg.idg_subgrid_fft(plan, sub, -1)
    torch.cuda.synchronize()
    got_sub = sub.cpu().numpy()
    err = np.linalg.norm((got_sub - ref_sub).reshape(P, -1), axis=1) / np.linalg.norm(ref_sub.reshape(P, -1), axis=1)
    assert err.max() < TOL, (int(err.argmax()), float(err.max()))
    # adder on the full plan: the GPU's own subgrids through oracle_adder (float64) against idg_adder
    ref_add = orc.adder(meta, got_sub.astype(np.complex128), np.zeros((4, L, L), dtype=np.complex128))
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    idg.idg_adder(plan, sub, g)
    torch.cuda.synchronize()
    got_add = g.cpu().numpy()
    assert H.rel_l2(got_add, ref_add) < 1e-6
    assert np.max(np.abs(got_add - ref_add)) < 1e-5 * np.max(np.abs(ref_add))        # element-wise too
    assert np.array_equal(got_add == 0, ref_add == 0)                                   # untouched pixels stay untouched
    # the whole grid through idg_grid against the oracle's Alg. 1
    ref_grid = orc.adder(meta, ref_sub, np.zeros((4, L, L), dtype=np.complex128))
    g.zero_()
    idg.idg_grid(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, g)
    torch.cuda.synchronize()
    got_grid = g.cpu().numpy()
    assert H.rel_l2(got_grid, ref_grid) < TOL
    for q in range(4):                                                                  # per polarisation plane
        assert H.rel_l2(got_grid[q], ref_grid[q]) < TOL

    # ---- Alg. 2 on the oracle's grid: every visibility
    model = ref_grid.astype(np.complex64)
    ref_vis = orc.degrid(prm, meta, d["uvw"], d["freqs"], model.astype(np.complex128), d["aterms"], d["taper"], w.B)
    out = torch.full(wc.vis.shape, 7.0, dtype=torch.complex64, device="cuda")
    idg.idg_degrid(plan, wc.uvw, torch.from_numpy(model).cuda(), wc.aterms, wc.taper, out)
    torch.cuda.synchronize()
    got_vis = out.cpu().numpy()
    assert H.rel_l2(got_vis, ref_vis) < TOL
    # worst block and worst single visibility (4 polarisations together)
    num = np.linalg.norm(got_vis - ref_vis, axis=-1)
    den = np.linalg.norm(ref_vis, axis=-1)
    assert np.max(num / den) < 1e-3, float(np.max(num / den))
    worst_block = 0.0
    for r in meta:
        sl = (int(r["baseline"]), slice(int(r["time_begin"]), int(r["time_begin"] + r["n_time"])),
              slice(int(r["chan_begin"]), int(r["chan_begin"] + r["n_chan"])))
        worst_block = max(worst_block, float(np.linalg.norm(num[sl]) / np.linalg.norm(den[sl])))
    assert worst_block < TOL, worst_block


def _stratified_sample(meta, bl_len, n_target, rng):
    """Indices of a stratified sample of the plan: every w layer, every channel-group size, the shortest and the
    longest baselines, the subgrids farthest from the grid centre, and a uniform remainder."""
    P = len(meta)
    pick = set()
    per = max(2, n_target // 8 // max(1, len(np.unique(meta["w_index"]))))
    for wi in np.unique(meta["w_index"]):
        idx = np.nonzero(meta["w_index"] == wi)[0]
        pick.update(rng.choice(idx, size=min(per, len(idx)), replace=False).tolist())
    for nc in np.unique(meta["n_chan"]):
        idx = np.nonzero(meta["n_chan"] == nc)[0]
        pick.update(rng.choice(idx, size=min(n_target // 8, len(idx)), replace=False).tolist())
    order = np.argsort(bl_len[meta["baseline"]], kind="stable")
    pick.update(order[: n_target // 8].tolist())                     # shortest baselines
    pick.update(order[-(n_target // 8):].tolist())                   # longest baselines
    L2 = (meta["x0"].astype(np.int64) - meta["x0"].mean()) ** 2 + (meta["y0"].astype(np.int64) - meta["y0"].mean()) ** 2
    pick.update(np.argsort(L2)[-(n_target // 8):].tolist())          # edge of the covered part of the grid
    short_t = np.nonzero(meta["n_time"] < meta["n_time"].max())[0]   # blocks cut short by the box rule
    if len(short_t):
        pick.update(rng.choice(short_t, size=min(n_target // 8, len(short_t)), replace=False).tolist())
    while len(pick) < n_target:
        pick.update(rng.choice(P, size=n_target - len(pick), replace=False).tolist())
    return np.array(sorted(pick), dtype=np.int64)


def test_ska_full_size_stratified_sample():
    """configs[2] + [3] at full size (8128 baselines, 133 M visibilities, 8192^2 grid, ~266 k subgrids): plan
    bit-exact; >= 256 stratified subgrids through gridder + FFT and through Alg. 2 against the oracle; the adder
    and the fused splitter + inverse FFT on sampled windows against the oracle's adder / splitter."""
    w = synth.make_workload("ska", device="cuda")
    d = dict(uvw=w.uvw.cpu().numpy(), freqs=w.freqs, vis=None, aterms=w.aterms.cpu().numpy(), taper=w.taper.cpu().numpy())
    prm = w.params
    N, L = prm.subgrid_size, prm.grid_size
    plan = idg.idg_plan_create(prm, w.uvw, w.freqs, w.baselines, w.n_stations)
    meta, planned, skipped = orc.plan(prm, d["uvw"], d["freqs"], w.baselines)
    assert plan.metadata().tobytes() == meta.tobytes() and plan.size() == (len(meta), planned, skipped)
    P = len(meta)
    assert P > 250000
    rng = np.random.default_rng(41)
    bl_len = np.linalg.norm(d["uvw"][:, 0, :], axis=1)
    pick = _stratified_sample(meta, bl_len, 256, rng)
    assert len(pick) >= 256
    assert set(np.unique(meta["w_index"][pick]).tolist()) == set(np.unique(meta["w_index"]).tolist())
    assert set(np.unique(meta["n_chan"][pick]).tolist()) == set(np.unique(meta["n_chan"]).tolist())
    sample = np.ascontiguousarray(meta[pick])
    # only the sampled baselines' visibilities travel to the host
    need_b = np.unique(sample["baseline"])
    remap = {int(b): i for i, b in enumerate(need_b)}
    vis_small = w.vis[torch.from_numpy(need_b).cuda()].cpu().numpy()
    uvw_small = d["uvw"][need_b]
    sample_small = sample.copy()
    sample_small["baseline"] = [remap[int(b)] for b in sample["baseline"]]

    sub = plan.subgrids()
    idg.idg_gridder(plan, w.uvw, w.vis, w.aterms, w.taper, sub)
    idg.idg_subgrid_fft(plan, sub, -1)
    torch.cuda.synchronize()
    got = sub[torch.from_numpy(pick).cuda()].cpu().numpy()
    ref = orc.subgrid_fft(orc.gridder(prm, sample_small, uvw_small, d["freqs"], vis_small, d["aterms"], d["taper"]), -1)
    err = np.linalg.norm((got - ref).reshape(len(pick), -1), axis=1) / np.linalg.norm(ref.reshape(len(pick), -1), axis=1)
    assert err.max() < TOL, (int(pick[err.argmax()]), float(err.max()))

    # adder: sampled windows against oracle_adder fed with every subgrid that touches them
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    idg.idg_adder(plan, sub, g)
    torch.cuda.synchronize()
    for p in pick[:: max(1, len(pick) // 24)]:
        x0, y0 = int(meta[p]["x0"]), int(meta[p]["y0"])
        touch = np.nonzero((np.abs(meta["x0"] - x0) < N) & (np.abs(meta["y0"] - y0) < N))[0]
        m_loc = meta[touch].copy()
        m_loc["x0"] -= x0 - N                                   # window [x0 - N, x0 + 2N) -> local grid of 3N
        m_loc["y0"] -= y0 - N
        loc = orc.adder(m_loc, sub[torch.from_numpy(touch).cuda()].cpu().numpy().astype(np.complex128),
                        np.zeros((4, 3 * N, 3 * N), dtype=np.complex128))
        got_w = g[:, y0:y0 + N, x0:x0 + N].cpu().numpy()
        assert H.rel_l2(got_w, loc[:, N:2 * N, N:2 * N]) < 1e-5

    # Alg. 2 on a random model grid, sampled blocks; splitter + IFFT fused kernel on the sampled subgrids
    model = torch.view_as_complex(torch.randn((4, L, L, 2), device="cuda", generator=torch.Generator("cuda").manual_seed(5)))
    out = torch.zeros_like(w.vis)
    idg.idg_degrid(plan, w.uvw, model, w.aterms, w.taper, out)
    torch.cuda.synchronize()
    # the oracle needs the model grid only under the sampled windows: its splitter output for subgrid p is the
    # window grid[:, y0:y0+N, x0:x0+N], cut here by plain slicing
    windows = np.stack([model[:, int(r["y0"]):int(r["y0"]) + N, int(r["x0"]):int(r["x0"]) + N].cpu().numpy()
                        for r in sample]).astype(np.complex128)
    imgs = orc.subgrid_fft(windows, +1)
    # fused splitter + inverse FFT (what idg_degrid ran) on the sampled subgrids
    idg.idg_splitter_ifft(plan, model, sub)
    torch.cuda.synchronize()
    got_img = sub[torch.from_numpy(pick).cuda()].cpu().numpy()
    assert max(H.rel_l2(got_img[i], imgs[i]) for i in range(len(pick))) < 1e-5
    ref_v = orc.degridder(prm, sample_small, uvw_small, d["freqs"], imgs, d["aterms"], d["taper"], len(need_b))
    got_all = out[torch.from_numpy(need_b).cuda()].cpu().numpy()
    worst = 0.0
    for r in sample_small:
        sl = (int(r["baseline"]), slice(int(r["time_begin"]), int(r["time_begin"] + r["n_time"])),
              slice(int(r["chan_begin"]), int(r["chan_begin"] + r["n_chan"])))
        worst = max(worst, H.rel_l2(got_all[sl], ref_v[sl]))
    assert worst < TOL, worst
