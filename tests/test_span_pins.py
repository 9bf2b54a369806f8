"""NEXT-4: per-sample c_pk (IDG_PLAN_SPAN_ATERMS).  Section 3.4 allows the A-term to change inside a
block; Alg. 1 has c*_pk inside the visibility sum and Alg. 2 c_pk per sample.  The
oracle's spanning path is pinned against the defining sums (Eq. 11, with per-sample Jones matrices),
the adjoint identity, and the constant-A-term special case."""
import dataclasses

import numpy as np

from oracle import idg_oracle as orc
from paper_1909_07226_b200 import synth
from tests import helpers as H
from tests.test_oracle_pins import _lattice, _np

SPAN = synth.FLAG_SPAN_ATERMS


def _case(a_int=5):
    w = synth.make_workload("tiny", aterm_interval=a_int)             # 32 timesteps -> 7 slots of 5
    prm = dataclasses.replace(w.params, flags=SPAN, w_step=150.0)
    d = _np(w)
    meta, planned, skipped = orc.plan(prm, d["uvw"], d["freqs"], w.baselines)
    assert skipped == 0 and planned == w.B * w.T * w.C
    return w, prm, d, meta


def test_span_plan_ignores_slot_boundaries():
    """Hand-worked: a stationary track of 30 timesteps, max_timesteps 8, aterm_interval 12.  Without the flag the
    blocks are cut at t = 12 and 24 (tests/golden/plan_hand_worked.txt, case `cuts`); with it they are
    [0,8) [8,16) [16,24) [24,30) and aterm_slot is the slot of the first timestep: 0, 0, 1, 2."""
    prm = synth.PlanParams(grid_size=128, subgrid_size=16, kernel_size=4, max_timesteps=8, max_channels=1,
                           aterm_interval=12, flags=SPAN, image_size=0.01, w_step=0.0)
    f = np.array([150e6])
    lam = H.C0 / f[0]
    uvw = np.zeros((1, 30, 3), dtype=np.float32)
    uvw[0, :, 0] = 1.0 / prm.image_size * lam
    uvw[0, :, 1] = 1.0 / prm.image_size * lam
    meta, planned, skipped = orc.plan(prm, uvw, f, np.array([[0, 1]], dtype=np.int32))
    assert [(int(r["time_begin"]), int(r["n_time"]), int(r["aterm_slot"])) for r in meta] == \
        [(0, 8, 0), (8, 8, 0), (16, 8, 1), (24, 6, 2)]
    assert (planned, skipped) == (30, 0)


def test_span_blocks_really_span_slots():
    w, prm, d, meta = _case()
    last = (meta["time_begin"] + meta["n_time"] - 1) // prm.aterm_interval
    assert np.any(last > meta["aterm_slot"])


def test_constant_aterms_reduce_to_the_per_block_variant():
    """With the same Jones matrices in every slot the per-sample path must equal the per-block path on the SAME
    metadata (the NEXT-4 row's pin: "reduces to (a) when c_pk is constant")."""
    w, prm, d, meta = _case()
    at = d["aterms"].copy()
    at[:] = at[0:1]
    a = orc.gridder(prm, meta, d["uvw"], d["freqs"], d["vis"], at, d["taper"])
    b = orc.gridder(dataclasses.replace(prm, flags=0), meta, d["uvw"], d["freqs"], d["vis"], at, d["taper"])
    assert H.rel_l2(a, b) < 1e-13
    rng = np.random.default_rng(2)
    img = rng.standard_normal(a.shape) + 1j * rng.standard_normal(a.shape)
    va = orc.degridder(prm, meta, d["uvw"], d["freqs"], img, at, d["taper"], w.B)
    vb = orc.degridder(dataclasses.replace(prm, flags=0), meta, d["uvw"], d["freqs"], img, at, d["taper"], w.B)
    assert H.rel_l2(va, vb) < 1e-13


def test_lattice_identity_with_per_sample_jones_matrices():
    """Eq. 11 with g_k per sample: on the lattice the image is taper sum_k A1_k^H Y_k A2_k exp(2 pi i (...)) to
    round-off, A_k = Jones matrices of the slot of timestep k."""
    w, prm, d, meta = _case()
    grid = orc.grid(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])
    image = H.image_from_grid(grid)
    L, N, S = prm.grid_size, prm.subgrid_size, prm.image_size
    idx, xs = _lattice(L, N)
    l = H.lm_of_pixels(idx, N, S)
    ll, mm = np.meshgrid(l, l)
    expected = np.zeros((len(idx), len(idx), 2, 2), dtype=np.complex128)
    for row in meta:
        for t in range(int(row["time_begin"]), int(row["time_begin"] + row["n_time"])):
            one = row.copy()
            one["time_begin"], one["n_time"] = t, 1
            D = H.die_per_subgrid(one, H.w_offset(row, prm.w_step), d["uvw"], d["freqs"], d["vis"], ll, mm)
            slot = t // prm.aterm_interval
            A1 = H.jones(d["aterms"], slot, row["station1"])[np.ix_(idx, idx)]
            A2 = H.jones(d["aterms"], slot, row["station2"])[np.ix_(idx, idx)]
            expected += np.conj(np.swapaxes(A1, -1, -2)) @ D @ A2
    expected *= d["taper"].astype(np.float64)[np.ix_(idx, idx)][..., None, None]
    got = np.moveaxis(image[:, xs[:, None], xs[None, :]], 0, -1).reshape(len(idx), len(idx), 2, 2)
    assert H.rel_l2(got, expected) < 1e-12
    # the per-block reading on the same metadata is a different (wrong) answer here:
    wrong = orc.grid(dataclasses.replace(prm, flags=0), meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])
    assert H.rel_l2(H.image_from_grid(wrong)[:, xs[:, None], xs[None, :]], image[:, xs[:, None], xs[None, :]]) > 1e-3


def test_adjoint_identity_with_spanning_blocks():
    w, prm, d, meta = _case()
    rng = np.random.default_rng(12)
    L = prm.grid_size
    x = rng.standard_normal((4, L, L)) + 1j * rng.standard_normal((4, L, L))
    v = (rng.standard_normal(d["vis"].shape) + 1j * rng.standard_normal(d["vis"].shape)).astype(np.complex64)
    Dx = orc.degrid(prm, meta, d["uvw"], d["freqs"], x, d["aterms"], d["taper"], w.B)
    Gv = orc.grid(prm, meta, d["uvw"], d["freqs"], v, d["aterms"], d["taper"])
    lhs, rhs = np.vdot(Dx, v.astype(np.complex128)), np.vdot(x, Gv)
    assert abs(lhs - rhs) / abs(lhs) < 1e-10
