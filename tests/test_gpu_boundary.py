"""-m gpu: the C-ABI boundary itself -- error paths a C caller can hit (called through ctypes without the
binding's own checks), caller-made metadata in any order, and guard bands around every output buffer (stands in
for compute-sanitizer, which the GPU pool refuses to run)."""
import ctypes
import dataclasses

import numpy as np
import pytest
import torch

from oracle import idg_oracle as orc
from paper_1909_07226_b200 import binding as idg
from paper_1909_07226_b200 import synth
from tests import helpers as H
from tests.test_gpu_parity import _ragged_case

pytestmark = pytest.mark.gpu
IDG_ERR_INVALID_ARG, IDG_ERR_PLAN_MISMATCH = -1, -4


def _p(t):
    return ctypes.c_void_p(t.data_ptr())


@pytest.fixture(scope="module")
def tiny():
    w = synth.make_workload("tiny")
    wc = w.to("cuda")
    plan = idg.idg_plan_create(w.params, wc.uvw, w.freqs, w.baselines, w.n_stations)
    return w, wc, plan


def test_c_callers_short_aterm_array_is_refused(tiny):
    """Every device compute entry takes n_slots and refuses a plan that indexes beyond it (no out-of-bounds read)."""
    w, wc, plan = tiny
    lib = idg.lib()
    L = w.params.grid_size
    need = plan.slots_needed()
    assert need == 2
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    out = torch.zeros_like(wc.vis)
    sub = plan.subgrids()
    s = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    short = ctypes.c_int32(need - 1)
    assert lib.idg_grid(plan.handle, _p(wc.uvw), _p(wc.vis), _p(wc.aterms), short, _p(wc.taper), _p(g), s) == IDG_ERR_PLAN_MISMATCH
    assert lib.idg_degrid(plan.handle, _p(wc.uvw), _p(g), _p(wc.aterms), short, _p(wc.taper), _p(out), s) == IDG_ERR_PLAN_MISMATCH
    assert lib.idg_gridder(plan.handle, _p(wc.uvw), _p(wc.vis), _p(wc.aterms), short, _p(wc.taper), _p(sub), s) == IDG_ERR_PLAN_MISMATCH
    assert lib.idg_degridder(plan.handle, _p(wc.uvw), _p(sub), _p(wc.aterms), short, _p(wc.taper), _p(out), s) == IDG_ERR_PLAN_MISMATCH
    vs, gs = wc.vis[..., 0].contiguous(), wc.aterms[..., 0].contiguous()
    g1 = torch.zeros((L, L), dtype=torch.complex64, device="cuda")
    assert lib.idg_grid_scalar(plan.handle, _p(wc.uvw), _p(vs), _p(gs), short, _p(wc.taper), _p(g1), s) == IDG_ERR_PLAN_MISMATCH
    assert lib.idg_degrid_scalar(plan.handle, _p(wc.uvw), _p(g1), _p(gs), short, _p(wc.taper), _p(vs), s) == IDG_ERR_PLAN_MISMATCH
    torch.cuda.synchronize()
    assert torch.all(g == 0) and torch.all(out == 0)          # nothing was launched
    # with the right count the same raw call works
    assert lib.idg_grid(plan.handle, _p(wc.uvw), _p(wc.vis), _p(wc.aterms), ctypes.c_int32(need), _p(wc.taper), _p(g), s) == 0
    torch.cuda.synchronize()
    assert float(g.abs().sum()) > 0


def test_misaligned_vector_operands_are_refused(tiny):
    """vis / aterms / subgrids are read as 16-byte vectors: an 8-byte-aligned view comes back as an error, and an
    8-byte-aligned GRID (allowed) takes the 8-byte gather path of the fused splitter + inverse FFT."""
    w, wc, plan = tiny
    lib = idg.lib()
    L = w.params.grid_size
    s = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    g = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    flat = torch.zeros(wc.vis.numel() + 1, dtype=torch.complex64, device="cuda")
    off = flat[1:]                                                       # data_ptr() is 8 mod 16
    assert off.data_ptr() % 16 == 8
    n = ctypes.c_int32(int(wc.aterms.shape[0]))
    assert lib.idg_grid(plan.handle, _p(wc.uvw), _p(off), _p(wc.aterms), n, _p(wc.taper), _p(g), s) == IDG_ERR_INVALID_ARG
    assert lib.idg_degrid(plan.handle, _p(wc.uvw), _p(g), _p(wc.aterms), n, _p(wc.taper), _p(off), s) == IDG_ERR_INVALID_ARG
    # odd-offset grid view: legal, must give the same subgrids as the aligned grid
    model = torch.view_as_complex(torch.randn((4 * L * L + 1, 2), device="cuda", generator=torch.Generator("cuda").manual_seed(1)))
    mis = model[1:].view(4, L, L)
    assert mis.data_ptr() % 16 == 8
    ali = mis.clone()
    sub = plan.subgrids()
    assert lib.idg_splitter_ifft(plan.handle, _p(mis), _p(sub), s) == 0
    torch.cuda.synchronize()
    a = sub.clone()
    idg.idg_splitter_ifft(plan, ali, sub)
    torch.cuda.synchronize()
    assert torch.equal(a, sub)


def test_caller_metadata_checks(tiny):
    w, wc, plan = tiny
    meta = plan.metadata()
    # int32 sums that would wrap past the <= T / <= C checks
    bad = meta.copy()
    bad["time_begin"][0] = 2 ** 31 - 1
    with pytest.raises(idg.IdgError, match="does not match"):
        idg.idg_plan_from_metadata(w.params, bad, w.freqs, w.B, w.T, w.n_stations)
    bad = meta.copy()
    bad["chan_begin"][0] = 2 ** 31 - 2
    with pytest.raises(idg.IdgError, match="does not match"):
        idg.idg_plan_from_metadata(w.params, bad, w.freqs, w.B, w.T, w.n_stations)
    # IDG_PLAN_SPAN_ATERMS: aterm_slot must be the slot of the first timestep
    prm = dataclasses.replace(w.params, flags=synth.FLAG_SPAN_ATERMS)
    ok = meta.copy()
    ok["aterm_slot"] = ok["time_begin"] // prm.aterm_interval
    idg.idg_plan_from_metadata(prm, ok, w.freqs, w.B, w.T, w.n_stations).destroy()
    bad = ok.copy()
    bad["aterm_slot"][-1] += 1
    with pytest.raises(idg.IdgError, match="does not match"):
        idg.idg_plan_from_metadata(prm, bad, w.freqs, w.B, w.T, w.n_stations)


def test_overlapping_caller_metadata_still_zeroes_uncovered_samples(tiny):
    """Two blocks covering the same samples make 'B T C - planned' non-positive although samples are uncovered:
    idg_degrid must still return 0 there (caller-made plans are always zeroed first)."""
    w, wc, plan = tiny
    meta = plan.metadata()
    dup = np.concatenate([meta, meta])                   # every block twice: planned = 2 B T C
    dup = dup[: len(meta) + len(meta) // 2]
    keep = np.ones(len(dup), dtype=bool)
    keep[3] = False                                      # ... and one block (and its duplicate, if any) missing
    if 3 + len(meta) < len(dup):
        keep[3 + len(meta)] = False
    sel = np.ascontiguousarray(dup[keep])
    p2 = idg.idg_plan_from_metadata(w.params, sel, w.freqs, w.B, w.T, w.n_stations)
    L = w.params.grid_size
    model = torch.view_as_complex(torch.randn((4, L, L, 2), device="cuda", generator=torch.Generator("cuda").manual_seed(2)))
    out = torch.full(wc.vis.shape, 9.0, dtype=torch.complex64, device="cuda")
    idg.idg_degrid(p2, wc.uvw, model, wc.aterms, wc.taper, out)
    torch.cuda.synchronize()
    r = meta[3]
    hole = out[int(r["baseline"]), int(r["time_begin"]):int(r["time_begin"] + r["n_time"]),
               int(r["chan_begin"]):int(r["chan_begin"] + r["n_chan"])]
    assert torch.all(hole == 0)


def test_host_entry_points_on_shuffled_caller_metadata():
    """idg_grid_host / idg_degrid_host chunk the work by baseline; metadata that is not sorted by baseline
    (idg_plan_from_metadata accepts any order) must still give the device entry points' result."""
    w = synth.make_workload("lofar", n_baselines=40, baseline_offset=500, n_time=128)
    wc = w.to("cuda")
    meta, _, _ = orc.plan(w.params, w.uvw.numpy(), w.freqs, w.baselines)
    rng = np.random.default_rng(11)
    shuffled = np.ascontiguousarray(meta[rng.permutation(len(meta))])
    assert np.any(np.diff(shuffled["baseline"]) < 0)
    plan = idg.idg_plan_from_metadata(w.params, shuffled, w.freqs, w.B, w.T, w.n_stations)
    L = w.params.grid_size
    d = dict(uvw=w.uvw.numpy(), vis=w.vis.numpy(), aterms=w.aterms.numpy(), taper=w.taper.numpy())
    ref = orc.grid(w.params, meta, d["uvw"], w.freqs, d["vis"], d["aterms"], d["taper"])
    g_host = np.zeros((4, L, L), dtype=np.complex64)
    idg.idg_grid_host(plan, d["uvw"], d["vis"], d["aterms"], d["taper"], g_host)
    assert H.rel_l2(g_host, ref) < 1e-4
    model = ref.astype(np.complex64)
    refv = orc.degrid(w.params, meta, d["uvw"], w.freqs, model.astype(np.complex128), d["aterms"], d["taper"], w.B)
    v_host = np.full(d["vis"].shape, 5.0, dtype=np.complex64)
    idg.idg_degrid_host(plan, d["uvw"], model, d["aterms"], d["taper"], v_host)
    assert H.rel_l2(v_host, refv) < 1e-4


def test_image_taper_and_w_offset_behind_the_abi(tiny):
    """c-bar (Alg. 1's divisor) and the layer offsets w0 come from the library."""
    w, wc, plan = tiny
    for N, L in ((24, 256), (16, 96), (32, 100), (48, 64)):
        tp = synth.prolate_taper(N)
        cb = idg.idg_image_taper(torch.from_numpy(tp).cuda(), L).cpu().numpy()
        ref = orc.image_taper(tp, L)
        assert np.max(np.abs(cb - ref)) < 2e-7 * np.max(np.abs(ref))
    prm = dataclasses.replace(w.params, w_step=150.0)
    p2 = idg.idg_plan_create(prm, wc.uvw, w.freqs, w.baselines, w.n_stations)
    assert p2.w_offset(-2) == -225.0 and p2.w_offset(0) == 75.0
    assert plan.w_offset(3) == 0.0                          # w_step = 0 -> every w0 is 0
    with pytest.raises(idg.IdgError):
        idg.idg_image_taper(torch.ones((20, 20), device="cuda"), 64)


# ---------------------------------------------------------------------------------------------
# guard bands: every output buffer sits between canary-filled bands that must come back untouched
# ---------------------------------------------------------------------------------------------

GUARD = 4096          # elements on each side
CANARY = 12345.0


def _guarded(shape, dtype, fill=0.0):
    n = int(np.prod(shape))
    # keep the payload 16-byte aligned: the band is a multiple of 16 bytes in both dtypes
    buf = torch.full((n + 2 * GUARD,), CANARY, dtype=dtype, device="cuda")
    view = buf[GUARD:GUARD + n].view(*shape)
    view.fill_(fill)
    return buf, view


def _bands_intact(buf):
    return bool(torch.all(buf[:GUARD] == CANARY)) and bool(torch.all(buf[-GUARD:] == CANARY))


@pytest.mark.parametrize("N", [16, 24, 32, 48])
def test_guard_bands_every_stage_ragged_plan(N):
    """Ragged hand-made plan (odd block sizes, subgrids in the grid corners): run every stage and both composite
    calls on outputs surrounded by canaries; the bands must be untouched and the payloads must still be right."""
    prm, meta, uvw, freqs, vis, aterms, taper, B, T, n_st = _ragged_case(N, 7 + N)
    plan = idg.idg_plan_from_metadata(prm, meta, freqs, B, T, n_st)
    P, L = len(meta), prm.grid_size
    d_uvw, d_vis = torch.from_numpy(uvw).cuda(), torch.from_numpy(vis).cuda()
    d_at, d_tp = torch.from_numpy(aterms).cuda(), torch.from_numpy(taper).cuda()
    sub_buf, sub = _guarded((P, 4, N, N), torch.complex64)
    grid_buf, g = _guarded((4, L, L), torch.complex64)
    vis_buf, out = _guarded(tuple(d_vis.shape), torch.complex64, fill=3.0)
    assert sub.data_ptr() % 16 == 0 and out.data_ptr() % 16 == 0

    idg.idg_gridder(plan, d_uvw, d_vis, d_at, d_tp, sub)
    torch.cuda.synchronize()
    assert _bands_intact(sub_buf)
    idg.idg_subgrid_fft(plan, sub, -1)
    torch.cuda.synchronize()
    assert _bands_intact(sub_buf)
    idg.idg_adder(plan, sub, g)
    torch.cuda.synchronize()
    assert _bands_intact(grid_buf) and _bands_intact(sub_buf)
    ref_grid = orc.grid(prm, meta, uvw, freqs, vis, aterms, taper)
    assert H.rel_l2(g.cpu().numpy(), ref_grid) < 1e-4
    idg.idg_splitter(plan, g, sub)
    torch.cuda.synchronize()
    assert _bands_intact(sub_buf) and _bands_intact(grid_buf)
    idg.idg_subgrid_fft(plan, sub, +1)
    idg.idg_splitter_ifft(plan, g, sub)
    torch.cuda.synchronize()
    assert _bands_intact(sub_buf) and _bands_intact(grid_buf)
    idg.idg_degridder(plan, d_uvw, sub, d_at, d_tp, out)
    torch.cuda.synchronize()
    assert _bands_intact(vis_buf) and _bands_intact(sub_buf)
    # composite calls on guarded grid / visibilities (their subgrid scratch is plan-owned)
    g.zero_()
    idg.idg_grid(plan, d_uvw, d_vis, d_at, d_tp, g)
    out.fill_(3.0)
    idg.idg_degrid(plan, d_uvw, g, d_at, d_tp, out)
    torch.cuda.synchronize()
    assert _bands_intact(grid_buf) and _bands_intact(vis_buf)
    ref_vis = orc.degrid(prm, meta, uvw, freqs, g.cpu().numpy().astype(np.complex128), aterms, taper, B)
    assert H.rel_l2(out.cpu().numpy(), ref_vis) < 1e-4


def test_guard_bands_planner_made_plan_with_skips():
    """Planner-made plan on a grid so small that long baselines are skipped: subgrids hug the grid border."""
    w = synth.make_workload("lofar", n_baselines=60, baseline_offset=1060, n_time=128)
    prm = dataclasses.replace(w.params, grid_size=1024)
    wc = w.to("cuda")
    plan = idg.idg_plan_create(prm, wc.uvw, w.freqs, w.baselines, w.n_stations)
    P, planned, skipped = plan.size()
    assert skipped > 0 and P > 0
    L = prm.grid_size
    grid_buf, g = _guarded((4, L, L), torch.complex64)
    vis_buf, out = _guarded(tuple(wc.vis.shape), torch.complex64, fill=3.0)
    idg.idg_grid(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, g)
    idg.idg_degrid(plan, wc.uvw, g, wc.aterms, wc.taper, out)
    torch.cuda.synchronize()
    assert _bands_intact(grid_buf) and _bands_intact(vis_buf)
    meta = plan.metadata()
    covered = np.zeros(tuple(wc.vis.shape[:3]), dtype=bool)
    for r in meta:
        covered[r["baseline"], r["time_begin"]:r["time_begin"] + r["n_time"], r["chan_begin"]:r["chan_begin"] + r["n_chan"]] = True
    assert np.all(out.cpu().numpy()[~covered] == 0)


def test_host_entry_points_with_the_tensor_core_gridder_in_chunks():
    """A planner-made N = 32 plan that takes the tensor-core gridder and degridder, through the chunked host-buffer calls (24
    baseline ranges, each a launch on a sub-range of the subgrids) against the one-launch device calls."""
    w = synth.make_workload("lofar", n_baselines=96, baseline_offset=200, n_time=128)
    wc = w.to("cuda")
    plan = idg.idg_plan_create(w.params, wc.uvw, w.freqs, w.baselines, w.n_stations)
    assert plan.uses_tensor_cores() and plan.degridder_uses_tensor_cores()
    L = w.params.grid_size
    g_dev = torch.zeros((4, L, L), dtype=torch.complex64, device="cuda")
    idg.idg_grid(plan, wc.uvw, wc.vis, wc.aterms, wc.taper, g_dev)
    g_host = np.zeros((4, L, L), dtype=np.complex64)
    idg.idg_grid_host(plan, w.uvw.numpy(), w.vis.numpy(), w.aterms.numpy(), w.taper.numpy(), g_host)
    assert H.rel_l2(g_host, g_dev.cpu().numpy()) < 1e-6
    v_dev = torch.zeros_like(wc.vis)
    idg.idg_degrid(plan, wc.uvw, g_dev, wc.aterms, wc.taper, v_dev)
    v_host = np.zeros(tuple(w.vis.shape), dtype=np.complex64)
    idg.idg_degrid_host(plan, w.uvw.numpy(), g_dev.cpu().numpy(), w.aterms.numpy(), w.taper.numpy(), v_host)
    torch.cuda.synchronize()
    assert np.array_equal(v_host, v_dev.cpu().numpy())
