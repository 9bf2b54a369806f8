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
