"""P5: the oracle planner (section 3.2; readings R10-R12) against the
invariants any valid partition has, and against hand-worked tracks whose partition can be
read off without running anything."""
import dataclasses

import re

import numpy as np
import pytest

from oracle import idg_oracle as orc
from paper_1909_07226_b200 import synth
from tests import helpers as H


def check_invariants(prm, meta, planned, skipped, uvw, freqs, baselines):
    """Exact cover, box bounds, one slot / one w layer per block, ordering."""
    B, T, _ = uvw.shape
    C = len(freqs)
    N, L, ks = prm.subgrid_size, prm.grid_size, prm.kernel_size
    cover = np.zeros((B, T, C), dtype=np.int32)
    k = np.asarray(freqs, dtype=np.float64) / H.C0
    force = bool(prm.flags & synth.FLAG_FORCE_BLOCKS)
    for row in meta:
        b, t0, nt, c0, nc = (int(row[f]) for f in ("baseline", "time_begin", "n_time", "chan_begin", "n_chan"))
        cover[b, t0:t0 + nt, c0:c0 + nc] += 1
        assert 1 <= nt <= prm.max_timesteps and 1 <= nc <= prm.max_channels
        assert (row["station1"], row["station2"]) == tuple(baselines[b])
        assert t0 // prm.aterm_interval == (t0 + nt - 1) // prm.aterm_interval == row["aterm_slot"]
        assert 0 <= row["x0"] and row["x0"] + N <= L and 0 <= row["y0"] and row["y0"] + N <= L
        assert row["reserved"] == 0
        u = uvw[b, t0:t0 + nt, 0].astype(np.float64)[:, None] * k[None, c0:c0 + nc] * prm.image_size + L // 2
        v = uvw[b, t0:t0 + nt, 1].astype(np.float64)[:, None] * k[None, c0:c0 + nc] * prm.image_size + L // 2
        if not force and nt > 1:
            # all samples inside the box minus half the kernel on each side (+- the rounding of the centre)
            assert u.min() >= row["x0"] + ks / 2 - 0.5 - 1e-9 and u.max() <= row["x0"] + N - ks / 2 + 0.5 + 1e-9
            assert v.min() >= row["y0"] + ks / 2 - 0.5 - 1e-9 and v.max() <= row["y0"] + N - ks / 2 + 0.5 + 1e-9
        if prm.w_step > 0:
            kmid = 0.5 * (freqs[c0] + freqs[c0 + nc - 1]) / H.C0
            wi = np.floor(uvw[b, t0:t0 + nt, 2].astype(np.float64) * kmid / prm.w_step)
            assert np.all(wi == row["w_index"])
        else:
            assert row["w_index"] == 0
    assert cover.max() <= 1
    assert int(cover.sum()) == planned
    assert planned + skipped == B * T * C
    key = np.stack([meta["baseline"], meta["chan_begin"], meta["time_begin"]], axis=1)
    assert np.array_equal(key, key[np.lexsort((key[:, 2], key[:, 1], key[:, 0]))])
    assert len(np.unique(key, axis=0)) == len(key)


@pytest.mark.parametrize("w_step", [0.0, 150.0])
def test_P5_invariants_tiny(w_step):
    w = synth.make_workload("tiny")
    prm = dataclasses.replace(w.params, w_step=w_step)
    uvw = w.uvw.numpy()
    meta, planned, skipped = orc.plan(prm, uvw, w.freqs, w.baselines)
    check_invariants(prm, meta, planned, skipped, uvw, w.freqs, w.baselines)
    assert skipped == 0


def test_P5_invariants_lofar_slice_and_channel_halving():
    """Long baselines of the LOFAR-like layout over a wide band: the channel group must be
    halved (R11) and time blocks must end on the box budget, not only on max_timesteps."""
    w = synth.make_workload("lofar", n_baselines=60, baseline_offset=1060, n_time=128)
    freqs = 140e6 + 3e6 * np.arange(16)                     # 32 % bandwidth
    prm = dataclasses.replace(w.params, grid_size=4096)
    uvw = w.uvw.numpy()
    meta, planned, skipped = orc.plan(prm, uvw, freqs, w.baselines)
    check_invariants(prm, meta, planned, skipped, uvw, freqs, w.baselines)
    assert meta["n_chan"].min() < 16 and meta["n_time"].min() < 64


def test_P5_force_blocks_are_regular():
    w = synth.make_workload("sweep", n_baselines=5, n_time=96, max_timesteps=32, max_channels=16,
                            aterm_interval=24)
    uvw = w.uvw.numpy()
    meta, planned, skipped = orc.plan(w.params, uvw, w.freqs, w.baselines)
    check_invariants(w.params, meta, planned, skipped, uvw, w.freqs, w.baselines)
    assert np.all(meta["n_time"] == 24) and np.all(meta["n_chan"] == 16)   # min(32, slot of 24)
    assert len(meta) == 5 * 4 * 4 - skipped // (24 * 16)


def _track(u_px, v_px, prm, freq):
    """uvw metres (float64 -> float32) that land on the given pixel coordinates at `freq`."""
    lam = H.C0 / freq
    u = np.asarray(u_px, dtype=np.float64) / prm.image_size * lam
    v = np.asarray(v_px, dtype=np.float64) / prm.image_size * lam
    return np.stack([u, v, np.zeros_like(u)], axis=-1)[None].astype(np.float32)


def test_hand_worked_tracks():
    """Single channel, budget = N - kernel = 12 pixels."""
    prm = synth.PlanParams(grid_size=128, subgrid_size=16, kernel_size=4, max_timesteps=100,
                           max_channels=1, aterm_interval=1000, flags=0, image_size=0.01, w_step=0.0)
    f = np.array([150e6])
    bl = np.array([[0, 1]], dtype=np.int32)
    # (a) a stationary sample at (10.3, -20.6): one block; centre = round-half-up -> (10, -21)
    meta, planned, skipped = orc.plan(prm, _track([10.3] * 7, [-20.6] * 7, prm, f[0]), f, bl)
    assert len(meta) == 1 and planned == 7 and skipped == 0
    assert (meta[0]["x0"], meta[0]["y0"]) == (10 + 64 - 8, -21 + 64 - 8)
    assert (meta[0]["time_begin"], meta[0]["n_time"]) == (0, 7)
    # (b) u moves 0.9 pixel per step: extent of k+1 samples is 0.9 k, > 12 first at k = 14,
    #     so blocks hold 14 samples: [0,14) [14,28) [28,30)
    u = 0.9 * np.arange(30) - 13.0
    meta, planned, _ = orc.plan(prm, _track(u, np.zeros(30), prm, f[0]), f, bl)
    assert [(int(r["time_begin"]), int(r["n_time"])) for r in meta] == [(0, 14), (14, 14), (28, 2)]
    # box midpoint of the first block = -13 + 0.9*13/2 = -7.15 -> centre pixel -7
    assert meta[0]["x0"] == -7 + 64 - 8 and meta[0]["y0"] == 0 + 64 - 8
    # (c) max_timesteps and the A-term interval cut a stationary track
    prm_c = dataclasses.replace(prm, max_timesteps=8, aterm_interval=12)
    meta, _, _ = orc.plan(prm_c, _track([1.0] * 30, [1.0] * 30, prm, f[0]), f, bl)
    assert [(int(r["time_begin"]), int(r["n_time"]), int(r["aterm_slot"])) for r in meta] == \
        [(0, 8, 0), (8, 4, 0), (12, 8, 1), (20, 4, 1), (24, 6, 2)]
    # (d) a sample whose subgrid would leave the grid is skipped and counted
    meta, planned, skipped = orc.plan(prm, _track([60.0] * 3 + [0.0] * 2, [0.0] * 5, prm, f[0]), f, bl)
    assert skipped == 3 and planned == 2 and len(meta) == 1 and meta[0]["time_begin"] == 3
    # (e) w layers: w = 10.2, 10.9, 11.1 wavelengths with w_step 1 -> layers 10, 10, 11
    prm_e = dataclasses.replace(prm, w_step=1.0)
    tr = _track([0.0] * 3, [0.0] * 3, prm, f[0])
    tr[0, :, 2] = np.array([10.2, 10.9, 11.1]) * (H.C0 / f[0])
    meta, _, _ = orc.plan(prm_e, tr, f, bl)
    assert [(int(r["n_time"]), int(r["w_index"])) for r in meta] == [(2, 10), (1, 11)]
    tr[0, :, 2] *= -1.0                                     # floor, not truncation: -10.2 -> -11
    meta, _, _ = orc.plan(prm_e, tr, f, bl)
    assert [(int(r["n_time"]), int(r["w_index"])) for r in meta] == [(2, -11), (1, -12)]


def test_hand_worked_channel_halving():
    """u = 1000 px at the lowest of 8 channels spaced 1 % apart: the spread over n channels is
    10 (n - 1) px, budget 12 -> groups of 2 channels (spread 10), not 4 (spread 30)."""
    prm = synth.PlanParams(grid_size=4096, subgrid_size=16, kernel_size=4, max_timesteps=4,
                           max_channels=8, aterm_interval=4, flags=0, image_size=0.01, w_step=0.0)
    f = 100e6 * (1.0 + 0.01 * np.arange(8))
    bl = np.array([[3, 5]], dtype=np.int32)
    meta, planned, skipped = orc.plan(prm, _track([1000.0] * 4, [0.0] * 4, prm, f[0]), f, bl)
    assert planned == 32 and skipped == 0
    assert [(int(r["chan_begin"]), int(r["n_chan"])) for r in meta] == [(0, 2), (2, 2), (4, 2), (6, 2)]
    assert all((r["station1"], r["station2"]) == (3, 5) for r in meta)
    # centre of the first group: midpoint of 1000 and 1010 px
    assert meta[0]["x0"] == 1005 + 2048 - 8


# ---------------------------------------------------------------------------------------------
# golden fixture: tests/golden/plan_hand_worked.txt (derived by hand from the rule text)
# ---------------------------------------------------------------------------------------------

def _expand(spec):
    """'10.3*7' -> 7 copies; '-13+0.9*30' -> arithmetic progression; '60.0*3,0.0*2' -> concatenation;
    '10.2,10.9' -> literal list."""
    out = []
    for part in spec.split(","):
        part = part.strip()
        m = re.fullmatch(r"(-?[0-9.]+)\+([0-9.]+)\*(\d+)", part)
        if m:
            out += [float(m.group(1)) + float(m.group(2)) * i for i in range(int(m.group(3)))]
            continue
        m = re.fullmatch(r"(-?[0-9.]+)\*(\d+)", part)
        if m:
            out += [float(m.group(1))] * int(m.group(2))
            continue
        out.append(float(part))
    return np.array(out, dtype=np.float64)


def load_golden_plans():
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "plan_hand_worked.txt")
    cases = []
    for line in open(path):
        line = line.strip()
        if not line.startswith("case "):
            continue
        name, over, u, v, w, blocks, planned, skipped = [x.strip() for x in line[5:].split("|")]
        prm = synth.PlanParams(grid_size=128, subgrid_size=16, kernel_size=4, max_timesteps=100,
                               max_channels=1, aterm_interval=1000, flags=0, image_size=0.01, w_step=0.0)
        for kv in over.split():
            k, val = kv.split("=")
            prm = dataclasses.replace(prm, **{k: type(getattr(prm, k))(float(val))})
        f = np.array([150e6])
        lam = H.C0 / f[0]
        uvw = np.stack([_expand(u) / prm.image_size * lam, _expand(v) / prm.image_size * lam,
                        _expand(w) * lam], axis=-1)[None].astype(np.float32)
        exp = [tuple(int(x) for x in b.strip().split(":")) for b in blocks.split(";")]
        cases.append((name, prm, uvw, f, exp, int(planned), int(skipped)))
    return cases


def check_golden_plan(meta, planned, skipped, exp, exp_planned, exp_skipped):
    got = [tuple(int(r[k]) for k in ("time_begin", "n_time", "chan_begin", "n_chan", "aterm_slot", "x0", "y0",
                                     "w_index")) for r in meta]
    assert got == exp
    assert (planned, skipped) == (exp_planned, exp_skipped)
    assert all(int(r["baseline"]) == 0 and (int(r["station1"]), int(r["station2"])) == (0, 1) for r in meta)


@pytest.mark.parametrize("case", load_golden_plans(), ids=lambda c: c[0])
def test_golden_hand_worked_plans(case):
    name, prm, uvw, f, exp, exp_planned, exp_skipped = case
    meta, planned, skipped = orc.plan(prm, uvw, f, np.array([[0, 1]], dtype=np.int32))
    check_golden_plan(meta, planned, skipped, exp, exp_planned, exp_skipped)
