"""-m gpu: the CUDA path (through the C ABI, paper_1909_07226_b200.binding) against the float64
oracle on the same seeded inputs.  Bars (BASELINE.json north_star): plan metadata bit-exact;
grid and degridded visibilities within relative L2 1e-4 (FP32 accumulation); adder / splitter are
pure data movement plus FP32 adds and are held to 1e-6 / bit-exact."""
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


def _cuda(w):
    return w.to("cuda")


def _np(w):
    return dict(uvw=w.uvw.cpu().numpy(), freqs=w.freqs, vis=w.vis.cpu().numpy(),
                aterms=w.aterms.cpu().numpy(), taper=w.taper.cpu().numpy())


def _plan_both(w, prm=None):
    prm = w.params if prm is None else prm
    wc = _cuda(w)
    plan = idg.idg_plan_create(prm, wc.uvw, w.freqs, w.baselines, w.n_stations)
    meta_o, planned_o, skipped_o = orc.plan(prm, w.uvw.cpu().numpy(), w.freqs, w.baselines)
    meta_g = plan.metadata()
    assert plan.size() == (len(meta_o), planned_o, skipped_o)
    assert meta_g.tobytes() == meta_o.tobytes()          # bit-exact, all 48 bytes of every entry
    return plan, wc, meta_o


# ---------------------------------------------------------------------------------------------
# planner
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("w_step", [0.0, 150.0])
def test_plan_bit_exact_tiny(w_step):
    w = synth.make_workload("tiny")
    _plan_both(w, dataclasses.replace(w.params, w_step=w_step))


def test_plan_bit_exact_channel_halving_and_skips():
    w = synth.make_workload("lofar", n_baselines=80, baseline_offset=1040, n_time=128)
    w.freqs = 140e6 + 3e6 * np.arange(16)                     # 32 % bandwidth forces halving
    prm = dataclasses.replace(w.params, grid_size=1024)       # long baselines leave the grid
    plan, _, meta = _plan_both(w, prm)
    assert meta["n_chan"].min() < 16 and plan.size()[2] > 0


def test_plan_bit_exact_ska_slice_w_layers():
    w = synth.make_workload("ska", n_baselines=300, baseline_offset=7800, n_time=256)
    _, _, meta = _plan_both(w)
    assert len(np.unique(meta["w_index"])) > 3


def test_plan_bit_exact_force_blocks():
    w = synth.make_workload("sweep", n_baselines=16, n_time=96, max_timesteps=32, max_channels=64,
                            aterm_interval=24)
    _, _, meta = _plan_both(w)
    assert np.all(meta["n_time"] == 24) and np.all(meta["n_chan"] == 64)


def test_plan_lofar_full_bit_exact():
    w = synth.make_workload("lofar")
    _, _, meta = _plan_both(w)
    assert len(meta) > 4000


# ---------------------------------------------------------------------------------------------
# stages on the tiny configuration (BASELINE.json configs[0])
# ---------------------------------------------------------------------------------------------

@pytest.fixture(scope="module")
def tiny_case():
    w = synth.make_workload("tiny")
    prm = dataclasses.replace(w.params, w_step=150.0)
    plan, wc, meta = _plan_both(w, prm)
    return dict(w=w, wc=wc, prm=prm, plan=plan, meta=meta, d=_np(w))


def test_kernel_launch_counter(tiny_case):
    """idg_kernel_launches (what bench.py reports as gpu_launches) counts one per stage call, three / two for
    idg_grid / idg_degrid."""
    c = tiny_case
    wc, plan = c["wc"], c["plan"]
    L = c["prm"].grid_size
    sub = plan.subgrids()
    grid = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    out = torch.zeros_like(wc.vis)
    n0 = idg.idg_kernel_launches()
    idg.idg_gridder(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, sub)
    assert idg.idg_kernel_launches() - n0 == 1
    idg.idg_subgrid_fft(plan, sub, -1)
    idg.idg_adder(plan, sub, grid)
    idg.idg_splitter(plan, grid, sub)
    idg.idg_subgrid_fft(plan, sub, +1)
    idg.idg_degridder(plan, wc.uvw, sub, wc.aterms, wc.taper, out)
    assert idg.idg_kernel_launches() - n0 == 6
    idg.idg_grid(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, grid)
    assert idg.idg_kernel_launches() - n0 == 9
    idg.idg_degrid(plan, wc.uvw, grid, wc.aterms, wc.taper, out)        # splitter + inverse FFT are one kernel there
    assert idg.idg_kernel_launches() - n0 == 11
    torch.cuda.synchronize()


def test_gridder_stage(tiny_case):
    c = tiny_case
    ref = orc.gridder(c["prm"], c["meta"], c["d"]["uvw"], c["d"]["freqs"], c["d"]["vis"], c["d"]["aterms"], c["d"]["taper"])
    sub = torch.zeros(ref.shape, dtype=torch.complex64, device="cuda")
    idg.idg_gridder(c["plan"], c["wc"].uvw, c["wc"].vis, c["wc"].aterms, c["wc"].taper, sub)
    torch.cuda.synchronize()
    assert H.rel_l2(sub.cpu().numpy(), ref) < TOL
    # per subgrid too: no single block may hide behind the others
    got = sub.cpu().numpy()
    worst = max(H.rel_l2(got[p], ref[p]) for p in range(len(ref)))
    assert worst < TOL, worst


@pytest.mark.parametrize("N", [16, 24, 32, 48])
@pytest.mark.parametrize("direction", [-1, 1])
def test_subgrid_fft_stage(N, direction):
    rng = np.random.default_rng(100 + N)
    P = 37                                                     # ragged: not a multiple of anything
    x = (rng.standard_normal((P, 4, N, N)) + 1j * rng.standard_normal((P, 4, N, N))).astype(np.complex64)
    meta = np.zeros(P, dtype=idg.META_DTYPE)
    meta["n_time"] = 1; meta["n_chan"] = 1
    prm = synth.PlanParams(grid_size=64, subgrid_size=N, kernel_size=4, max_timesteps=1, max_channels=1,
                           aterm_interval=1, flags=0, image_size=0.01, w_step=0.0)
    plan = idg.idg_plan_from_metadata(prm, meta, np.array([1e8]), 1, 1, 1)
    t = torch.from_numpy(x).cuda()
    idg.idg_subgrid_fft(plan, t, direction)
    torch.cuda.synchronize()
    ref = orc.subgrid_fft(x.astype(np.complex128), direction)
    assert H.rel_l2(t.cpu().numpy(), ref) < 2e-6


def _random_meta(rng, P, N, L):
    meta = np.zeros(P, dtype=idg.META_DTYPE)
    meta["x0"] = rng.integers(0, L - N + 1, P)
    meta["y0"] = rng.integers(0, L - N + 1, P)
    meta["x0"][:4] = [0, L - N, 0, L - N]                     # the four corners of the grid
    meta["y0"][:4] = [0, 0, L - N, L - N]
    meta["x0"][4:200] = L // 2 - N // 2 + rng.integers(-3, 4, 196)   # a heavily overlapped core
    meta["y0"][4:200] = L // 2 - N // 2 + rng.integers(-3, 4, 196)
    meta["n_time"] = 1; meta["n_chan"] = 1
    return meta


@pytest.mark.parametrize("N,L", [(16, 80), (24, 250), (32, 256), (48, 200)])
def test_adder_and_splitter_stage(N, L):
    rng = np.random.default_rng(N)
    P = 300
    meta = _random_meta(rng, P, N, L)
    prm = synth.PlanParams(grid_size=L, subgrid_size=N, kernel_size=4, max_timesteps=1, max_channels=1,
                           aterm_interval=1, flags=0, image_size=0.01, w_step=0.0)
    plan = idg.idg_plan_from_metadata(prm, meta, np.array([1e8]), 1, 1, 1)
    sub = (rng.standard_normal((P, 4, N, N)) + 1j * rng.standard_normal((P, 4, N, N))).astype(np.complex64)
    grid0 = (rng.standard_normal((4, L, L)) + 1j * rng.standard_normal((4, L, L))).astype(np.complex64)
    g = torch.from_numpy(grid0.copy()).cuda()
    idg.idg_adder(plan, torch.from_numpy(sub).cuda(), g)
    torch.cuda.synchronize()
    ref = orc.adder(meta, sub.astype(np.complex128), grid0.astype(np.complex128))
    assert H.rel_l2(g.cpu().numpy(), ref) < 1e-6
    out = torch.zeros((P, 4, N, N), dtype=torch.complex64, device="cuda")
    idg.idg_splitter(plan, torch.from_numpy(grid0).cuda(), out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), orc.splitter(meta, grid0, N).astype(np.complex64))  # bit-exact copy
    # rows a4 + a5 fused (what idg_degrid runs): bit-identical to the two calls, and within tolerance of the oracle
    idg.idg_subgrid_fft(plan, out, +1)
    fused = torch.zeros_like(out)
    idg.idg_splitter_ifft(plan, torch.from_numpy(grid0).cuda(), fused)
    torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(fused), torch.view_as_real(out))
    ref_i = orc.subgrid_fft(orc.splitter(meta, grid0.astype(np.complex128), N), +1)
    assert H.rel_l2(fused.cpu().numpy(), ref_i) < 1e-6


def test_degridder_stage(tiny_case):
    c = tiny_case
    rng = np.random.default_rng(21)
    N = c["prm"].subgrid_size
    P = len(c["meta"])
    img = (rng.standard_normal((P, 4, N, N)) + 1j * rng.standard_normal((P, 4, N, N))).astype(np.complex64)
    ref = orc.degridder(c["prm"], c["meta"], c["d"]["uvw"], c["d"]["freqs"], img.astype(np.complex128),
                        c["d"]["aterms"], c["d"]["taper"], c["w"].B)
    out = torch.zeros(c["wc"].vis.shape, dtype=torch.complex64, device="cuda")
    idg.idg_degridder(c["plan"], c["wc"].uvw, torch.from_numpy(img).cuda(), c["wc"].aterms, c["wc"].taper, out)
    torch.cuda.synchronize()
    assert H.rel_l2(out.cpu().numpy(), ref) < TOL


def test_grid_and_degrid_end_to_end_tiny(tiny_case):
    c = tiny_case
    L = c["prm"].grid_size
    ref = orc.grid(c["prm"], c["meta"], c["d"]["uvw"], c["d"]["freqs"], c["d"]["vis"], c["d"]["aterms"], c["d"]["taper"])
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    idg.idg_grid(c["plan"], c["wc"].uvw, c["wc"].vis, c["wc"].aterms, c["wc"].taper, g)
    torch.cuda.synchronize()
    assert H.rel_l2(g.cpu().numpy(), ref) < TOL
    # accumulates: a second call doubles the grid
    idg.idg_grid(c["plan"], c["wc"].uvw, c["wc"].vis, c["wc"].aterms, c["wc"].taper, g)
    torch.cuda.synchronize()
    assert H.rel_l2(g.cpu().numpy(), 2.0 * ref) < TOL
    # degrid the oracle's grid (rounded to complex64, the type the GPU receives)
    model = ref.astype(np.complex64)
    refv = orc.degrid(c["prm"], c["meta"], c["d"]["uvw"], c["d"]["freqs"], model.astype(np.complex128),
                      c["d"]["aterms"], c["d"]["taper"], c["w"].B)
    out = torch.full(c["wc"].vis.shape, 7.0, dtype=torch.complex64, device="cuda")
    idg.idg_degrid(c["plan"], c["wc"].uvw, torch.from_numpy(model).cuda(), c["wc"].aterms, c["wc"].taper, out)
    torch.cuda.synchronize()
    assert H.rel_l2(out.cpu().numpy(), refv) < TOL


# ---------------------------------------------------------------------------------------------
# golden hand-worked plans through the CUDA planner (tests/golden/plan_hand_worked.txt)
# ---------------------------------------------------------------------------------------------

def test_plan_golden_hand_worked():
    from tests.test_plan import check_golden_plan, load_golden_plans
    for name, prm, uvw, f, exp, exp_planned, exp_skipped in load_golden_plans():
        plan = idg.idg_plan_create(prm, torch.from_numpy(uvw).cuda(), f, np.array([[0, 1]], dtype=np.int32), 2)
        P, planned, skipped = plan.size()
        check_golden_plan(plan.metadata(), planned, skipped, exp, exp_planned, exp_skipped)


# ---------------------------------------------------------------------------------------------
# every subgrid size, ragged blocks (odd timestep counts, 1..5 channels, channel counts that are not
# a multiple of the degridder's per-thread channel group), edge-of-grid subgrids
# ---------------------------------------------------------------------------------------------

def _ragged_case(N, seed):
    """A hand-made plan over a small random data set: blocks of odd sizes at random positions."""
    rng = np.random.default_rng(seed)
    B, T, C, S, L, n_st = 6, 40, 11, 0.04, 192, 5
    freqs = 120e6 + 300e3 * np.arange(C)
    bl = np.array([[i % n_st, (i * 2 + 1) % n_st] for i in range(B)], dtype=np.int32)
    uvw = (rng.standard_normal((B, T, 3)) * np.array([900.0, 900.0, 60.0])).astype(np.float32)
    vis = (rng.standard_normal((B, T, C, 4)) + 1j * rng.standard_normal((B, T, C, 4))).astype(np.complex64)
    n_slots = 3
    aterms = synth.random_aterms(rng, n_slots, n_st, N)
    taper = synth.prolate_taper(N)
    rows = []
    for b in range(B):
        t0 = 0
        while t0 < T:
            nt = int(min(T - t0, rng.choice([1, 3, 7, 13])))
            c0 = 0
            while c0 < C:
                nc = int(min(C - c0, rng.choice([1, 2, 3, 5])))
                if rng.random() < 0.85:                      # leave some samples unplanned
                    k = freqs[c0:c0 + nc].mean() / H.C0
                    xc = int(np.floor(uvw[b, t0:t0 + nt, 0].mean() * k * S + 0.5)) + int(rng.integers(-2, 3))
                    yc = int(np.floor(uvw[b, t0:t0 + nt, 1].mean() * k * S + 0.5)) + int(rng.integers(-2, 3))
                    x0 = int(np.clip(xc + L // 2 - N // 2, 0, L - N))
                    y0 = int(np.clip(yc + L // 2 - N // 2, 0, L - N))
                    rows.append((b, bl[b, 0], bl[b, 1], t0, nt, c0, nc, int(rng.integers(0, n_slots)), x0, y0,
                                 int(rng.integers(-1, 2)), 0))
                c0 += nc
            t0 += nt
    rows[0] = rows[0][:8] + (0, 0) + rows[0][10:]            # corners of the grid
    rows[1] = rows[1][:8] + (L - N, L - N) + rows[1][10:]
    meta = np.array(rows, dtype=idg.META_DTYPE)
    prm = synth.PlanParams(grid_size=L, subgrid_size=N, kernel_size=N // 4, max_timesteps=16, max_channels=8,
                           aterm_interval=1, flags=0, image_size=S, w_step=3.0)
    return prm, meta, uvw, freqs, vis, aterms, taper, B, T, n_st


@pytest.mark.parametrize("N", [16, 24, 32, 48])
def test_all_sizes_ragged_blocks_every_stage_and_end_to_end(N):
    prm, meta, uvw, freqs, vis, aterms, taper, B, T, n_st = _ragged_case(N, 7 + N)
    plan = idg.idg_plan_from_metadata(prm, meta, freqs, B, T, n_st)
    P = len(meta)
    d_uvw, d_vis = torch.from_numpy(uvw).cuda(), torch.from_numpy(vis).cuda()
    d_at, d_tp = torch.from_numpy(aterms).cuda(), torch.from_numpy(taper).cuda()
    # gridder
    ref_img = orc.gridder(prm, meta, uvw, freqs, vis, aterms, taper)
    sub = torch.zeros((P, 4, N, N), dtype=torch.complex64, device="cuda")
    idg.idg_gridder(plan, d_uvw, d_vis, d_at, d_tp, sub)
    torch.cuda.synchronize()
    got = sub.cpu().numpy()
    assert max(H.rel_l2(got[p], ref_img[p]) for p in range(P)) < TOL
    # Alg. 1 end to end
    L = prm.grid_size
    ref_grid = orc.grid(prm, meta, uvw, freqs, vis, aterms, taper)
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    idg.idg_grid(plan, d_uvw, d_vis, d_at, d_tp, g)
    torch.cuda.synchronize()
    assert H.rel_l2(g.cpu().numpy(), ref_grid) < TOL
    # Alg. 2 end to end on a random model grid; unplanned samples must read 0
    rng = np.random.default_rng(N)
    model = (rng.standard_normal((4, L, L)) + 1j * rng.standard_normal((4, L, L))).astype(np.complex64)
    ref_vis = orc.degrid(prm, meta, uvw, freqs, model.astype(np.complex128), aterms, taper, B)
    out = torch.full(d_vis.shape, 3.0, dtype=torch.complex64, device="cuda")
    idg.idg_degrid(plan, d_uvw, torch.from_numpy(model).cuda(), d_at, d_tp, out)
    torch.cuda.synchronize()
    got_v = out.cpu().numpy()
    assert H.rel_l2(got_v, ref_vis) < TOL
    covered = np.zeros(vis.shape[:3], dtype=bool)
    for r in meta:
        covered[r["baseline"], r["time_begin"]:r["time_begin"] + r["n_time"],
                r["chan_begin"]:r["chan_begin"] + r["n_chan"]] = True
    assert np.all(got_v[~covered] == 0)
    # per visibility: no planned sample may hide behind the others
    num = np.linalg.norm((got_v - ref_vis)[covered], axis=-1)
    den = np.linalg.norm(ref_vis[covered], axis=-1)
    assert np.max(num / den) < 1e-3


def test_empty_plan_is_a_no_op():
    prm = synth.PlanParams(grid_size=64, subgrid_size=16, kernel_size=4, max_timesteps=4, max_channels=1,
                           aterm_interval=4, flags=0, image_size=0.01, w_step=0.0)
    meta = np.zeros(0, dtype=idg.META_DTYPE)
    plan = idg.idg_plan_from_metadata(prm, meta, np.array([1e8]), 1, 4, 2)
    assert plan.size() == (0, 0, 4)
    uvw = torch.zeros((1, 4, 3), device="cuda")
    vis = torch.ones((1, 4, 1, 4), dtype=torch.complex64, device="cuda")
    at = torch.from_numpy(synth.identity_aterms(1, 2, 16)).cuda()
    tp = torch.ones((16, 16), device="cuda")
    g = torch.ones((4, 64, 64), dtype=torch.complex64, device="cuda")
    idg.idg_grid(plan, uvw, vis, at, tp, g)
    idg.idg_degrid(plan, uvw, g, at, tp, vis)
    torch.cuda.synchronize()
    assert torch.all(g == 1) and torch.all(vis == 0)


def test_everything_skipped_plan():
    """All samples fall off a tiny grid: the planner emits nothing and counts them."""
    w = synth.make_workload("tiny")
    prm = dataclasses.replace(w.params, grid_size=24)
    plan, wc, meta = _plan_both(w, prm)
    assert plan.size()[1] + plan.size()[2] == w.B * w.T * w.C


# ---------------------------------------------------------------------------------------------
# the host-buffer entry points (what bench.py's e2e leg times)
# ---------------------------------------------------------------------------------------------

def test_host_entry_points_match_device_entry_points(tiny_case):
    c = tiny_case
    L = c["prm"].grid_size
    d = c["d"]
    g_dev = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    idg.idg_grid(c["plan"], c["wc"].uvw, c["wc"].vis, c["wc"].aterms, c["wc"].taper, g_dev)
    g_host = np.zeros((4, L, L), dtype=np.complex64)
    idg.idg_grid_host(c["plan"], d["uvw"], d["vis"], d["aterms"], d["taper"], g_host)
    assert H.rel_l2(g_host, g_dev.cpu().numpy()) < 1e-6
    v_dev = torch.zeros(c["wc"].vis.shape, dtype=torch.complex64, device="cuda")
    idg.idg_degrid(c["plan"], c["wc"].uvw, g_dev, c["wc"].aterms, c["wc"].taper, v_dev)
    v_host = np.zeros(d["vis"].shape, dtype=np.complex64)
    idg.idg_degrid_host(c["plan"], d["uvw"], g_dev.cpu().numpy(), d["aterms"], d["taper"], v_host)
    torch.cuda.synchronize()
    assert np.array_equal(v_host, v_dev.cpu().numpy())


def test_fused_host_cycle_matches_the_two_calls(tiny_case):
    """idg_grid_degrid_host (grid resident on the device) = idg_grid_host into a zero grid, then idg_degrid_host of
    that grid: the same kernels in the same order; the adder's atomics are the only difference (FP32 sums in another
    order), hence 1e-6 instead of equality.  With grid=None the visibilities are the same and nothing else is written."""
    c = tiny_case
    L = c["prm"].grid_size
    d = c["d"]
    g_ref = np.zeros((4, L, L), dtype=np.complex64)
    idg.idg_grid_host(c["plan"], d["uvw"], d["vis"], d["aterms"], d["taper"], g_ref)
    v_ref = np.zeros(d["vis"].shape, dtype=np.complex64)
    idg.idg_degrid_host(c["plan"], d["uvw"], g_ref, d["aterms"], d["taper"], v_ref)
    g = np.full((4, L, L), 7 + 7j, dtype=np.complex64)            # overwritten, not accumulated into
    v = np.zeros(d["vis"].shape, dtype=np.complex64)
    idg.idg_grid_degrid_host(c["plan"], d["uvw"], d["vis"], d["aterms"], d["taper"], g, v)
    assert H.rel_l2(g, g_ref) < 1e-6
    assert H.rel_l2(v, v_ref) < 1e-6
    v2 = np.zeros(d["vis"].shape, dtype=np.complex64)
    idg.idg_grid_degrid_host(c["plan"], d["uvw"], d["vis"], d["aterms"], d["taper"], None, v2)
    assert H.rel_l2(v2, v_ref) < 1e-6
    # in place: the predicted visibilities may replace the measured ones
    v3 = d["vis"].copy()
    idg.idg_grid_degrid_host(c["plan"], d["uvw"], v3, d["aterms"], d["taper"], None, v3)
    assert H.rel_l2(v3, v_ref) < 1e-6


# ---------------------------------------------------------------------------------------------
# full-size configurations in the launch configuration bench.py times: sampled subgrids / samples
# ---------------------------------------------------------------------------------------------

def _sampled_full_size_check(w, n_sample, seed):
    plan, wc, meta = _plan_both(w)
    d = _np(w)
    P = len(meta)
    N, L = w.params.subgrid_size, w.params.grid_size
    rng = np.random.default_rng(seed)
    pick = np.sort(rng.choice(P, size=min(n_sample, P), replace=False))
    sample = np.ascontiguousarray(meta[pick])
    # gridder + FFT on the full plan, compared on the sampled subgrids
    sub = plan.subgrids()
    idg.idg_gridder(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, sub)
    idg.idg_subgrid_fft(plan, sub, -1)
    torch.cuda.synchronize()
    got = sub[torch.from_numpy(pick).cuda()].cpu().numpy()
    ref = orc.subgrid_fft(orc.gridder(w.params, sample, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"]), -1)
    worst = max(H.rel_l2(got[i], ref[i]) for i in range(len(pick)))
    assert worst < TOL, worst
    # adder at full size: property -- the grid total equals the total of all subgrids (per polarisation)
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    idg.idg_adder(plan, sub, g)
    torch.cuda.synchronize()
    tot_sub = sub.to(torch.complex128).sum(dim=(0, 2, 3)).cpu().numpy()
    tot_grid = g.to(torch.complex128).sum(dim=(1, 2)).cpu().numpy()
    scale = float(sub.abs().to(torch.float64).sum().item())
    assert np.max(np.abs(tot_sub - tot_grid)) < 1e-6 * scale
    # ... and sampled grid windows against the oracle adder restricted to the subgrids that touch them
    g_np = g.cpu().numpy()
    sub_np_needed = {}
    for p in pick[:8]:
        x0, y0 = int(meta[p]["x0"]), int(meta[p]["y0"])
        touch = np.nonzero((np.abs(meta["x0"] - x0) < N) & (np.abs(meta["y0"] - y0) < N))[0]
        acc = np.zeros((4, N, N), dtype=np.complex128)
        subs = sub[torch.from_numpy(touch).cuda()].cpu().numpy().astype(np.complex128)
        for s_img, q in zip(subs, touch):
            dx, dy = int(meta[q]["x0"]) - x0, int(meta[q]["y0"]) - y0
            xs, ys = max(0, dx), max(0, dy)
            xe, ye = min(N, N + dx), min(N, N + dy)
            acc[:, ys:ye, xs:xe] += s_img[:, ys - dy:ye - dy, xs - dx:xe - dx]
        assert H.rel_l2(g_np[:, y0:y0 + N, x0:x0 + N], acc) < 1e-5
    # degrid direction: splitter (bit-exact on the sample), then IFFT + degridder on sampled blocks
    rng2 = np.random.default_rng(seed + 1)
    model = torch.view_as_complex(torch.randn((4, L, L, 2), device="cuda", generator=torch.Generator("cuda").manual_seed(seed)))
    out = torch.zeros_like(wc.vis)
    idg.idg_degrid(plan, wc.uvw, model, wc.aterms, wc.taper, out)
    torch.cuda.synchronize()
    model_np = model.cpu().numpy()
    refv = orc.degrid(w.params, sample, d["uvw"], d["freqs"], model_np.astype(np.complex128), d["aterms"], d["taper"], w.B)
    got_v = out.cpu().numpy()
    for r in sample:
        sl = (int(r["baseline"]), slice(int(r["time_begin"]), int(r["time_begin"] + r["n_time"])),
              slice(int(r["chan_begin"]), int(r["chan_begin"] + r["n_chan"])))
        assert H.rel_l2(got_v[sl], refv[sl]) < TOL
    return P


def test_lofar_full_size_sampled():
    """BASELINE.json configs[1], exactly what bench.py times; 48 sampled subgrids against the oracle."""
    w = synth.make_workload("lofar")
    assert _sampled_full_size_check(w, 48, 5) > 4000


def test_ska_slice_sampled():
    """A 600-baseline slice of configs[2]/[3] (long baselines: channel halving, w layers, A-term slots up to
    31, grid 8192^2): 32 sampled subgrids against the oracle."""
    w = synth.make_workload("ska", n_baselines=600, baseline_offset=7500)
    assert _sampled_full_size_check(w, 32, 9) > 15000


# ---------------------------------------------------------------------------------------------
# BASELINE.json configs[4]: corners of the kernel sweep (forced blocks), sampled against the oracle
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("N,max_c,max_t,a_int", [(16, 1, 32, 8), (32, 1, 64, 16), (24, 4, 64, 32), (32, 16, 512, 64), (48, 64, 512, 256),
                                                 # long blocks: many staging batches per CTA; N = 24 above 4096 visibilities per
                                                 # block takes the 64-thread gridder instance; (32, 16, 512, 32) the degridder
                                                 # with 8 channels per thread and two pixel groups
                                                 (16, 64, 512, 128), (24, 16, 256, 256), (24, 16, 512, 512), (32, 16, 512, 32),
                                                 # round 2: single-channel plans tile four timesteps per thread (split and
                                                 # unsplit instances); 8 channels per thread with eight pixel groups and the
                                                 # reduction in rounds (N = 24) or at once (N = 48)
                                                 (16, 1, 512, 512), (24, 1, 128, 256), (48, 1, 32, 512), (24, 16, 512, 8), (48, 16, 512, 8),
                                                 (16, 16, 512, 8)])
def test_sweep_corners_sampled(N, max_c, max_t, a_int):
    w = synth.make_workload("sweep", n_baselines=12, n_time=512, subgrid_size=N, max_channels=max_c,
                            max_timesteps=max_t, aterm_interval=a_int)
    P = _sampled_full_size_check(w, 6, 100 + N)
    eff_t = min(max_t, a_int)
    assert P == 12 * (512 // eff_t) * (64 // max_c)


@pytest.mark.parametrize("N", [16, 32])
def test_maximum_channels_per_subgrid(N):
    """256 channels in one subgrid (the ABI's maximum): the gridder stages two timesteps per batch (N = 32, 16) and the
    degridder runs 32 channel groups of 8 per timestep."""
    w = synth.make_workload("tiny", subgrid_size=N, max_channels=256, max_timesteps=16)
    rng = np.random.default_rng(256 + N)
    freqs = 150e6 + 10e3 * np.arange(256, dtype=np.float64)
    vis = torch.from_numpy((rng.standard_normal((w.B, w.T, 256, 4)) + 1j * rng.standard_normal((w.B, w.T, 256, 4)))
                           .astype(np.complex64))
    w = dataclasses.replace(w, freqs=freqs, vis=vis)
    _, _, meta = _plan_both(w)
    assert int(meta["n_chan"].max()) == 256
    _sampled_full_size_check(w, 8, 300 + N)


def test_mixed_channel_groups_paper_shape_sampled():
    """A slice of the paper-shaped workload (20 channels cut into groups of 16 + 4, N = 48): the degridder runs as two
    launches, 8 channels per thread on the 16-channel subgrids and 4 per thread on the 4-channel ones."""
    w = synth.make_workload("paper", n_baselines=10, n_time=512, baseline_offset=700)
    _, _, meta = _plan_both(w)
    assert set(np.unique(meta["n_chan"]).tolist()) >= {4, 16}
    assert int(meta["n_time"].max()) * 2 >= 128          # the condition for 8 channels per thread
    assert _sampled_full_size_check(w, 12, 77) == len(meta)


# ---------------------------------------------------------------------------------------------
# NEXT-1: image-plane wrap with W-stacking (paper_1909_07226_b200.imaging) against the oracle
# ---------------------------------------------------------------------------------------------

def test_w_stacked_dirty_image_and_prediction():
    from paper_1909_07226_b200 import imaging
    w = synth.make_workload("tiny")
    prm = dataclasses.replace(w.params, w_step=150.0)
    wc = _cuda(w)
    d = _np(w)
    meta, _, _ = orc.plan(prm, d["uvw"], d["freqs"], w.baselines)
    assert len(orc.w_layers(meta)) >= 3
    ref_img = orc.dirty_image(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])
    img = imaging.dirty_image(prm, wc.uvw, w.freqs, w.baselines, w.n_stations, wc.vis, wc.aterms, wc.taper)
    L = prm.grid_size
    inner = slice(L // 8, 7 * L // 8)                     # c-bar is tiny at the very edge: compare where it is not
    assert H.rel_l2(img.cpu().numpy()[:, inner, inner], ref_img[:, inner, inner]) < TOL
    # c-bar itself
    cb = imaging.image_taper(wc.taper, L).cpu().numpy()
    assert H.rel_l2(cb, orc.image_taper(d["taper"], L)) < 1e-6
    # prediction from a model image of a few sources
    rng = np.random.default_rng(3)
    model = np.zeros((4, L, L), dtype=np.complex64)
    for _ in range(5):
        x, y = rng.integers(L // 4, 3 * L // 4, 2)
        model[0, y, x] = model[3, y, x] = rng.uniform(0.5, 2.0)
    ref_vis = orc.predict(prm, meta, d["uvw"], d["freqs"], model.astype(np.complex128), d["aterms"], d["taper"], w.B)
    got = imaging.predict(prm, wc.uvw, w.freqs, w.baselines, w.n_stations, torch.from_numpy(model).cuda(),
                          wc.aterms, wc.taper, w.C)
    assert H.rel_l2(got.cpu().numpy(), ref_vis) < TOL


# ---------------------------------------------------------------------------------------------
# NEXT-3: scalar (one polarisation) variant = XX plane of the 4-polarisation oracle with Jones matrices g I_2
# ---------------------------------------------------------------------------------------------

def _scalar_inputs(w, rng):
    """Scalar visibilities and gains, and the 4-polarisation arrays that embed them."""
    N = w.params.subgrid_size
    vis_s = w.vis.numpy()[..., 0].copy()                                   # [B][T][C]
    n_slots = w.aterms.shape[0]
    g = (1.0 + 0.1 * (rng.standard_normal((n_slots, w.n_stations, N, N)) +
                      1j * rng.standard_normal((n_slots, w.n_stations, N, N)))).astype(np.complex64)
    vis4 = np.zeros(w.vis.shape, dtype=np.complex64)
    vis4[..., 0] = vis_s
    at4 = np.zeros((n_slots, w.n_stations, N, N, 4), dtype=np.complex64)
    at4[..., 0] = g
    at4[..., 3] = g
    return vis_s, g, vis4, at4


@pytest.mark.parametrize("name,kw,uneven", [("tiny", {}, False), ("tiny", {}, True),
                                            ("lofar", dict(n_baselines=40, baseline_offset=600, n_time=128), False)])
def test_scalar_variant_matches_xx_plane_of_the_oracle(name, kw, uneven):
    """Equally spaced channels take the phase-recurrence kernels (sin/cos every 4th channel), unevenly spaced
    ones the direct kernels."""
    w = synth.make_workload(name, **kw)
    if uneven:
        w.freqs = w.freqs + np.array([0.0, 30e3, -20e3, 50e3])[: len(w.freqs)]
    prm = dataclasses.replace(w.params, w_step=150.0) if name == "tiny" else w.params
    rng = np.random.default_rng(17)
    vis_s, g, vis4, at4 = _scalar_inputs(w, rng)
    uvw, taper = w.uvw.numpy(), w.taper.numpy()
    d_uvw = w.uvw.cuda()
    plan = idg.idg_plan_create(prm, d_uvw, w.freqs, w.baselines, w.n_stations)
    meta, _, _ = orc.plan(prm, uvw, w.freqs, w.baselines)
    assert plan.metadata().tobytes() == meta.tobytes()
    L, N, P = prm.grid_size, prm.subgrid_size, len(meta)
    d_vis, d_g, d_tp = torch.from_numpy(vis_s).cuda(), torch.from_numpy(g).cuda(), w.taper.cuda()
    # stage: gridder
    ref_img = orc.gridder(prm, meta, uvw, w.freqs, vis4, at4, taper)[:, 0]
    sub = torch.zeros((P, N, N), dtype=torch.complex64, device="cuda")
    idg.idg_gridder_scalar(plan, d_uvw, d_vis, d_g, d_tp, sub)
    torch.cuda.synchronize()
    got = sub.cpu().numpy()
    assert max(H.rel_l2(got[p], ref_img[p]) for p in range(P)) < TOL
    # Alg. 1
    ref_grid = orc.grid(prm, meta, uvw, w.freqs, vis4, at4, taper)[0]
    grid = torch.zeros((L, L), dtype=torch.complex64, device="cuda")
    idg.idg_grid_scalar(plan, d_uvw, d_vis, d_g, d_tp, grid)
    torch.cuda.synchronize()
    assert H.rel_l2(grid.cpu().numpy(), ref_grid) < TOL
    # Alg. 2 on a random model grid (XX plane only: the other planes of the embedding are zero)
    model = (rng.standard_normal((L, L)) + 1j * rng.standard_normal((L, L))).astype(np.complex64)
    model4 = np.zeros((4, L, L), dtype=np.complex128)
    model4[0] = model
    ref_vis = orc.degrid(prm, meta, uvw, w.freqs, model4, at4, taper, w.B)[..., 0]
    out = torch.full(d_vis.shape, 5.0, dtype=torch.complex64, device="cuda")
    idg.idg_degrid_scalar(plan, d_uvw, torch.from_numpy(model).cuda(), d_g, d_tp, out)
    torch.cuda.synchronize()
    assert H.rel_l2(out.cpu().numpy(), ref_vis) < TOL


# ---------------------------------------------------------------------------------------------
# NEXT-4: per-sample c_pk -- blocks that span A-term slots (IDG_PLAN_SPAN_ATERMS)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("a_int", [1, 5])
def test_spanning_blocks_per_sample_aterms(a_int):
    w = synth.make_workload("tiny", aterm_interval=a_int)
    prm = dataclasses.replace(w.params, flags=synth.FLAG_SPAN_ATERMS, w_step=150.0)
    plan, wc, meta = _plan_both(w, prm)                                  # plan bit-exact with the flag
    last = (meta["time_begin"] + meta["n_time"] - 1) // a_int
    assert np.any(last > meta["aterm_slot"])
    d = _np(w)
    L = prm.grid_size
    ref = orc.grid(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    idg.idg_grid(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, g)
    torch.cuda.synchronize()
    assert H.rel_l2(g.cpu().numpy(), ref) < TOL
    ref_sub = orc.gridder(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])
    sub = torch.zeros(ref_sub.shape, dtype=torch.complex64, device="cuda")
    idg.idg_gridder(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, sub)
    torch.cuda.synchronize()
    got = sub.cpu().numpy()
    assert max(H.rel_l2(got[p], ref_sub[p]) for p in range(len(meta))) < TOL
    model = ref.astype(np.complex64)
    refv = orc.degrid(prm, meta, d["uvw"], d["freqs"], model.astype(np.complex128), d["aterms"], d["taper"], w.B)
    out = torch.zeros_like(wc.vis)
    idg.idg_degrid(plan, wc.uvw, torch.from_numpy(model).cuda(), wc.aterms, wc.taper, out)
    torch.cuda.synchronize()
    assert H.rel_l2(out.cpu().numpy(), refv) < TOL
    # the scalar kernels know per-block gains only and must refuse such a plan
    with pytest.raises(idg.IdgError):
        idg.idg_grid_scalar(plan, wc.uvw, wc.vis[..., 0].contiguous(), wc.aterms[..., 0].contiguous(), wc.taper,
                            torch.zeros((L, L), dtype=torch.complex64, device="cuda"))


def test_calls_run_on_the_callers_stream(tiny_case):
    """The library is asynchronous on the stream it is given and never synchronises it: work queued on a side
    stream behind a long-running kernel must not have run until that stream is waited on, and must be right then."""
    c = tiny_case
    L = c["prm"].grid_size
    side = torch.cuda.Stream()
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    ref = torch.zeros_like(g)
    idg.idg_grid(c["plan"], c["wc"].uvw, c["wc"].vis, c["wc"].aterms, c["wc"].taper, ref)      # default stream
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        torch.cuda._sleep(200_000_000)                                   # ~0.1 s of spinning on the side stream
        idg.idg_grid(c["plan"], c["wc"].uvw, c["wc"].vis, c["wc"].aterms, c["wc"].taper, g, stream=side)
        done = torch.cuda.Event()
        done.record(side)
    assert not done.query()                                              # the call returned without waiting
    side.synchronize()
    # the adder's per-tile reductions land in any order, so equal up to FP32 summation order only
    assert H.rel_l2(g.cpu().numpy(), ref.cpu().numpy()) < 1e-6


def test_error_paths_with_a_device(tiny_case):
    """Bad arguments come back as status codes (IdgError in the binding), never as a crash."""
    c = tiny_case
    w, prm = c["w"], c["prm"]
    # metadata that does not fit the arrays or the grid
    bad = c["meta"].copy()
    bad["x0"][0] = prm.grid_size                      # subgrid outside the grid
    with pytest.raises(idg.IdgError, match="metadata does not match"):
        idg.idg_plan_from_metadata(prm, bad, w.freqs, w.B, w.T, w.n_stations)
    bad = c["meta"].copy()
    bad["time_begin"][0] = w.T                        # block beyond the last timestep
    with pytest.raises(idg.IdgError, match="metadata does not match"):
        idg.idg_plan_from_metadata(prm, bad, w.freqs, w.B, w.T, w.n_stations)
    # unsupported subgrid size and bad parameters
    with pytest.raises(idg.IdgError, match="subgrid size"):
        idg.idg_plan_create(dataclasses.replace(prm, subgrid_size=20), c["wc"].uvw, w.freqs, w.baselines, w.n_stations)
    with pytest.raises(idg.IdgError, match="invalid argument"):
        idg.idg_plan_create(dataclasses.replace(prm, max_channels=3), c["wc"].uvw, w.freqs, w.baselines, w.n_stations)
    with pytest.raises(idg.IdgError, match="invalid argument"):
        idg.idg_plan_create(dataclasses.replace(prm, flags=8), c["wc"].uvw, w.freqs, w.baselines, w.n_stations)
    # too few A-term slots, wrong shapes, host tensors where device tensors are expected
    L = prm.grid_size
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    with pytest.raises(idg.IdgError, match="does not match"):     # refused by the C library (IDG_ERR_PLAN_MISMATCH)
        idg.idg_grid(c["plan"], c["wc"].uvw, c["wc"].vis, c["wc"].aterms[:1].contiguous(), c["wc"].taper, g)
    with pytest.raises(idg.IdgError, match="grid shape"):
        idg.idg_grid(c["plan"], c["wc"].uvw, c["wc"].vis, c["wc"].aterms, c["wc"].taper, g[:, :-1].contiguous())
    with pytest.raises(idg.IdgError, match="CUDA tensor"):
        idg.idg_grid(c["plan"], c["wc"].uvw.cpu(), c["wc"].vis, c["wc"].aterms, c["wc"].taper, g)
    # the C ABI itself rejects too few slots on the host path
    with pytest.raises(idg.IdgError):
        idg.idg_subgrid_fft(c["plan"], c["plan"].subgrids(), 0)           # direction must be -1 or +1
    assert torch.all(g == 0)


# ---------------------------------------------------------------------------------------------
# tensor-core gridder (csrc/gridder_tc.cu): N = 32, >= 8 channels per block
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("uneven,spread", [(False, False), (True, False), (False, True)])
def test_tensor_core_gridder_ragged_blocks(uneven, spread):
    """Blocks of 8 / 12 / 16 channels (12 is padded to 16 inside the kernel) and odd timestep counts through the
    tcgen05 gridder: equally spaced channels take the rotation recurrence, unevenly spaced ones sin/cos per channel;
    `spread` gives the visibilities of a block twelve orders of magnitude of dynamic range (the kernel scales every
    block by a power of two into the fp16 range and splits hi + lo)."""
    w = synth.make_workload("lofar", n_baselines=24, baseline_offset=300, n_time=96)
    rng = np.random.default_rng(5)
    if uneven:
        w.freqs = w.freqs + rng.uniform(-40e3, 40e3, len(w.freqs))
    if spread:
        v = w.vis.numpy().copy()
        v *= (10.0 ** rng.uniform(-6, 6, v.shape[:3]))[..., None].astype(np.float32)
        w = dataclasses.replace(w, vis=torch.from_numpy(v))
    d = _np(w)
    meta, _, _ = orc.plan(w.params, d["uvw"], d["freqs"], w.baselines)
    meta = meta.copy()
    meta["n_chan"] = rng.choice([8, 12, 16], len(meta))
    meta["chan_begin"] = 0
    meta["n_time"] = np.minimum(meta["n_time"], rng.choice([13, 21, 33, 64, 64], len(meta)))
    plan = idg.idg_plan_from_metadata(w.params, meta, w.freqs, w.B, w.T, w.n_stations)
    assert plan.uses_tensor_cores()
    wc = _cuda(w)
    ref = orc.gridder(w.params, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])
    sub = torch.zeros(ref.shape, dtype=torch.complex64, device="cuda")
    idg.idg_gridder(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, sub)
    torch.cuda.synchronize()
    got = sub.cpu().numpy()
    err = np.array([H.rel_l2(got[p], ref[p]) for p in range(len(meta))])
    print("tensor-core gridder worst / median rel-L2: %.2e / %.2e" % (err.max(), np.median(err)))
    assert err.max() < TOL, (int(err.argmax()), float(err.max()))


def test_fp32_gridder_flag_and_wide_blocks_leave_the_tensor_cores():
    """IDG_PLAN_FP32_GRIDDER keeps row a1 on the FP32 kernel (closer to float64 than the 22-bit tensor-core operands);
    a block with more channels than a staging batch of the tensor-core kernel holds (128) also takes the FP32 kernel.
    Both against the oracle, and the flag's result against the tensor-core one."""
    w = synth.make_workload("lofar", n_baselines=16, baseline_offset=300, n_time=64)
    d = _np(w)
    meta, _, _ = orc.plan(w.params, d["uvw"], d["freqs"], w.baselines)
    plan_tc = idg.idg_plan_from_metadata(w.params, meta, w.freqs, w.B, w.T, w.n_stations)
    prm32 = dataclasses.replace(w.params, flags=w.params.flags | synth.FLAG_FP32_GRIDDER)
    plan32 = idg.idg_plan_from_metadata(prm32, meta, w.freqs, w.B, w.T, w.n_stations)
    assert plan_tc.uses_tensor_cores() and not plan32.uses_tensor_cores()
    wc = _cuda(w)
    ref = orc.gridder(w.params, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])
    out = {}
    for name, plan in (("tc", plan_tc), ("fp32", plan32)):
        sub = torch.zeros(ref.shape, dtype=torch.complex64, device="cuda")
        idg.idg_gridder(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, sub)
        torch.cuda.synchronize()
        out[name] = sub.cpu().numpy()
        assert H.rel_l2(out[name], ref) < TOL
    assert H.rel_l2(out["tc"], out["fp32"]) < TOL
    # 160 channels in one block: N = 32, per-block A-terms, long blocks -- and still not eligible
    base = synth.make_workload("lofar", n_baselines=4, baseline_offset=300, n_time=32)
    rng = np.random.default_rng(11)
    f = base.freqs
    freqs = np.linspace(f[0], f[-1], 160)                       # the same band in ten times as many channels
    vis = (rng.standard_normal((base.B, base.T, 160, 4)) + 1j * rng.standard_normal((base.B, base.T, 160, 4))).astype(np.complex64)
    wide = dataclasses.replace(base, freqs=freqs, vis=torch.from_numpy(vis))
    dw = _np(wide)
    mw, _, _ = orc.plan(wide.params, dw["uvw"], dw["freqs"], wide.baselines)
    mw = mw.copy()
    mw["chan_begin"] = 0
    mw["n_chan"] = 160
    plan_w = idg.idg_plan_from_metadata(wide.params, mw, wide.freqs, wide.B, wide.T, wide.n_stations)
    assert not plan_w.uses_tensor_cores()
    wcw = _cuda(wide)
    refw = orc.gridder(wide.params, mw, dw["uvw"], dw["freqs"], dw["vis"], dw["aterms"], dw["taper"])
    subw = torch.zeros(refw.shape, dtype=torch.complex64, device="cuda")
    idg.idg_gridder(plan_w, wcw.uvw, wcw.vis, wcw.aterms, wcw.taper, subw)
    torch.cuda.synchronize()
    assert H.rel_l2(subw.cpu().numpy(), refw) < TOL


# ---------------------------------------------------------------------------------------------
# tensor-core degridder (csrc/degridder_tc.cu): N = 32, mean block >= 384 visibilities
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("spread", [False, True])
def test_tensor_core_degridder_ragged_blocks(spread):
    """Blocks of 45 to 1920 visibilities through the tcgen05 degridder: one tile of 128 visibilities with its pixels
    split over four thread groups, two tiles over two each, three and four tiles, and more than four (several rounds
    that stage the B tiles again), channel counts 5 / 9 / 16 so that tiles do not end on timestep boundaries, ragged
    last tiles.  Every visibility against the float64 oracle, per block; `spread` gives the subgrid images of a plan
    twelve orders of magnitude of dynamic range (the kernel scales every subgrid by a power of two into the fp16
    range and splits hi + lo), judged per block like the others."""
    w = synth.make_workload("lofar", n_baselines=24, baseline_offset=300, n_time=128)
    rng = np.random.default_rng(6)
    d = _np(w)
    meta, _, _ = orc.plan(w.params, d["uvw"], d["freqs"], w.baselines)
    meta = meta.copy()
    meta["n_chan"] = rng.choice([5, 9, 16, 16], len(meta))
    meta["chan_begin"] = 0
    meta["n_time"] = np.minimum(meta["n_time"], rng.choice([9, 15, 23, 40, 64, 120, 120], len(meta)))
    plan = idg.idg_plan_from_metadata(w.params, meta, w.freqs, w.B, w.T, w.n_stations)
    assert plan.degridder_uses_tensor_cores()
    nv = meta["n_time"].astype(np.int64) * meta["n_chan"]
    assert nv.min() <= 128 and ((nv > 128) & (nv <= 256)).any() and ((nv > 256) & (nv <= 512)).any() and nv.max() > 512
    N = w.params.subgrid_size
    P = len(meta)
    img = (rng.standard_normal((P, 4, N, N)) + 1j * rng.standard_normal((P, 4, N, N))).astype(np.complex64)
    if spread:
        img *= (10.0 ** rng.uniform(-6, 6, P))[:, None, None, None].astype(np.float32)
    ref = orc.degridder(w.params, meta, d["uvw"], d["freqs"], img.astype(np.complex128), d["aterms"], d["taper"], w.B)
    wc = _cuda(w)
    out = torch.zeros(wc.vis.shape, dtype=torch.complex64, device="cuda")
    idg.idg_degridder(plan, wc.uvw, torch.from_numpy(img).cuda(), wc.aterms, wc.taper, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    # blocks of one baseline overlap in (time, channel) after the edits above: the last writer wins in both
    # implementations only if they run in the same order, so judge the blocks nobody overwrites
    owner = -np.ones((w.B, w.T, len(w.freqs)), dtype=np.int64)
    for p in range(P):
        mm = meta[p]
        owner[mm["baseline"], mm["time_begin"]:mm["time_begin"] + mm["n_time"], 0:mm["n_chan"]] = p
    err = []
    for p in range(P):
        mm = meta[p]
        sl = (mm["baseline"], slice(mm["time_begin"], mm["time_begin"] + mm["n_time"]), slice(0, mm["n_chan"]))
        if (owner[sl] == p).all():
            err.append(H.rel_l2(got[sl], ref[sl]))
    err = np.array(err)
    assert len(err) > P // 2
    print("tensor-core degridder worst / median rel-L2 over %d blocks: %.2e / %.2e" % (len(err), err.max(), np.median(err)))
    assert err.max() < TOL


def test_fp32_flag_keeps_the_degridder_off_the_tensor_cores():
    w = synth.make_workload("lofar", n_baselines=8, baseline_offset=300, n_time=128)
    d = _np(w)
    meta, _, _ = orc.plan(w.params, d["uvw"], d["freqs"], w.baselines)
    plan_tc = idg.idg_plan_from_metadata(w.params, meta, w.freqs, w.B, w.T, w.n_stations)
    prm32 = dataclasses.replace(w.params, flags=w.params.flags | synth.FLAG_FP32_GRIDDER)
    plan32 = idg.idg_plan_from_metadata(prm32, meta, w.freqs, w.B, w.T, w.n_stations)
    assert plan_tc.degridder_uses_tensor_cores() and not plan32.degridder_uses_tensor_cores()
    rng = np.random.default_rng(8)
    N, P = w.params.subgrid_size, len(meta)
    img = (rng.standard_normal((P, 4, N, N)) + 1j * rng.standard_normal((P, 4, N, N))).astype(np.complex64)
    ref = orc.degridder(w.params, meta, d["uvw"], d["freqs"], img.astype(np.complex128), d["aterms"], d["taper"], w.B)
    wc = _cuda(w)
    res = {}
    for name, plan in (("tc", plan_tc), ("fp32", plan32)):
        out = torch.zeros(wc.vis.shape, dtype=torch.complex64, device="cuda")
        idg.idg_degridder(plan, wc.uvw, torch.from_numpy(img).cuda(), wc.aterms, wc.taper, out)
        torch.cuda.synchronize()
        res[name] = out.cpu().numpy()
        assert H.rel_l2(res[name], ref) < TOL
    assert H.rel_l2(res["tc"], res["fp32"]) < TOL
