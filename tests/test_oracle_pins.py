"""Pins for the float64 oracle (oracle/idg_oracle.c) against what the paper and the
mathematics fix -- none of them re-types the oracle's own formulae:

  P1  lattice identity: at image pixels that coincide with subgrid-image pixels the IDG
      image equals the brute-force direct imaging equation (Eq. 11) to
      round-off, because the effective window is a sinc interpolation of the discrete
      taper and is exact at the sample points (section 4.2).
  P2  point source: degridding a model image with one pixel on that lattice gives the closed
      form of the measurement equation (Eq. 3); and with L = N degridding equals
      the discrete measurement equation (Eq. 6) for ANY image.
  P3  gridding is the Hermitian adjoint of degridding (Eq. 7/10).
  P4  off the lattice IDG agrees with Eq. 11 to the taper's side-lobe level (Table 1,
      PAPER.md:255-266; Fig. 6).
  FFT the subgrid transform equals numpy.fft with the centring shifts (library routine).
plus the degenerate cases (single visibility at the subgrid centre, adder / splitter
against numpy slicing).  P5 (plan invariants) is in test_plan.py.
"""
import dataclasses

import numpy as np
import pytest

from oracle import idg_oracle as orc
from paper_1909_07226_b200 import synth
from tests import helpers as H


@pytest.fixture(scope="module")
def tiny():
    return synth.make_workload("tiny")


def _np(w):
    return dict(uvw=w.uvw.numpy(), freqs=w.freqs, vis=w.vis.numpy(), aterms=w.aterms.numpy(),
                taper=w.taper.numpy())


def _lattice(L, N):
    """Subgrid pixels i whose direction coincides with an image pixel x (R1, R3)."""
    idx = [i for i in range(N) if ((i - N // 2) * L) % N == 0]
    xs = [L // 2 + (i - N // 2) * L // N for i in idx]
    return np.array(idx), np.array(xs)


@pytest.mark.parametrize("w_step", [0.0, 150.0])
def test_P1_lattice_identity_vs_direct_imaging(tiny, w_step):
    prm = dataclasses.replace(tiny.params, w_step=w_step)
    d = _np(tiny)
    meta, planned, skipped = orc.plan(prm, d["uvw"], d["freqs"], tiny.baselines)
    assert planned == tiny.B * tiny.T * tiny.C and skipped == 0
    if w_step > 0:
        assert len(np.unique(meta["w_index"])) > 2          # the w layers are exercised
    grid = orc.grid(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])
    image = H.image_from_grid(grid)                          # [4][L][L]
    L, N, S = prm.grid_size, prm.subgrid_size, prm.image_size
    idx, xs = _lattice(L, N)
    assert len(idx) == 8
    l = H.lm_of_pixels(idx, N, S)
    ll, mm = np.meshgrid(l, l)                               # [j][i]: l varies along x
    expected = np.zeros((len(idx), len(idx), 2, 2), dtype=np.complex128)
    for row in meta:
        D = H.die_per_subgrid(row, H.w_offset(row, w_step), d["uvw"], d["freqs"], d["vis"], ll, mm)
        A1 = H.jones(d["aterms"], row["aterm_slot"], row["station1"])[np.ix_(idx, idx)]
        A2 = H.jones(d["aterms"], row["aterm_slot"], row["station2"])[np.ix_(idx, idx)]
        expected += np.conj(np.swapaxes(A1, -1, -2)) @ D @ A2
    expected *= d["taper"].astype(np.float64)[np.ix_(idx, idx)][..., None, None]
    got = image[:, xs[:, None], xs[None, :]]                 # [4][j][i]  (y index first)
    got = np.moveaxis(got, 0, -1).reshape(len(idx), len(idx), 2, 2)
    assert H.rel_l2(got, expected) < 1e-12


@pytest.mark.parametrize("w_step", [0.0, 150.0])
def test_P2_point_source_closed_form(tiny, w_step):
    prm = dataclasses.replace(tiny.params, w_step=w_step)
    d = _np(tiny)
    meta, _, _ = orc.plan(prm, d["uvw"], d["freqs"], tiny.baselines)
    L, N, S = prm.grid_size, prm.subgrid_size, prm.image_size
    idx, xs = _lattice(L, N)
    i, j = idx[5], idx[2]
    x, y = xs[5], xs[2]
    Bm = np.array([[1.0 + 0.2j, 0.3 - 0.1j], [-0.2 + 0.4j, 0.7 + 0.0j]])
    img = np.zeros((4, L, L), dtype=np.complex128)
    img[:, y, x] = Bm.ravel() / np.float64(d["taper"][j, i])
    model = H.grid_from_image(img)
    got = orc.degrid(prm, meta, d["uvw"], d["freqs"], model, d["aterms"], d["taper"], tiny.B)
    l0 = H.lm_of_pixels(i, N, S)
    m0 = H.lm_of_pixels(j, N, S)
    n0 = H.nprime(l0, m0)
    expected = np.zeros_like(got)
    for row in meta:
        b = row["baseline"]
        A1 = H.jones(d["aterms"], row["aterm_slot"], row["station1"])[j, i]
        A2 = H.jones(d["aterms"], row["aterm_slot"], row["station2"])[j, i]
        M = A1 @ Bm @ np.conj(A2.T)
        w0 = H.w_offset(row, w_step)
        for t in range(row["time_begin"], row["time_begin"] + row["n_time"]):
            for c in range(row["chan_begin"], row["chan_begin"] + row["n_chan"]):
                k = d["freqs"][c] / H.C0
                u, v, w = (np.float64(q) * k for q in d["uvw"][b, t])
                ph = -2.0 * np.pi * (u * l0 + v * m0 + (w - w0) * n0)
                expected[b, t, c] = (M * np.exp(1j * ph)).ravel()
    assert H.rel_l2(got, expected) < 1e-12


def test_P2_full_grid_subgrid_equals_discrete_measurement_equation():
    """L = N: one subgrid is the whole grid, so Alg. 2 must reproduce Eq. 6 for any image."""
    rng = np.random.default_rng(7)
    N, S, n_st, T, C = 16, 0.1, 3, 5, 3
    prm = synth.PlanParams(grid_size=N, subgrid_size=N, kernel_size=4, max_timesteps=T,
                           max_channels=C, aterm_interval=T, flags=0, image_size=S, w_step=0.0)
    freqs = 100e6 + 1e6 * np.arange(C)
    uvw = (rng.standard_normal((1, T, 3)) * 40.0).astype(np.float32)
    aterms = synth.random_aterms(rng, 1, n_st, N)
    taper = synth.prolate_taper(N)
    meta = np.zeros(1, dtype=orc.META_DTYPE)
    meta[0] = (0, 2, 1, 0, T, 0, C, 0, 0, 0, 0, 0)
    img = rng.standard_normal((4, N, N)) + 1j * rng.standard_normal((4, N, N))
    got = orc.degrid(prm, meta, uvw, freqs, H.grid_from_image(img), aterms, taper, 1)
    l = H.lm_of_pixels(np.arange(N), N, S)
    ll, mm = np.meshgrid(l, l)
    nn = H.nprime(ll, mm)
    A1 = H.jones(aterms, 0, 2)
    A2 = H.jones(aterms, 0, 1)
    I22 = np.moveaxis(img, 0, -1).reshape(N, N, 2, 2) * taper.astype(np.float64)[..., None, None]
    gI = A1 @ I22 @ np.conj(np.swapaxes(A2, -1, -2))          # g_k(l,m) I[i,j] of Eq. 6
    expected = np.zeros((1, T, C, 4), dtype=np.complex128)
    for t in range(T):
        for c in range(C):
            k = freqs[c] / H.C0
            u, v, w = (np.float64(q) * k for q in uvw[0, t])
            ph = np.exp(-2j * np.pi * (u * ll + v * mm + w * nn))
            expected[0, t, c] = (gI * ph[..., None, None]).sum(axis=(0, 1)).ravel()
    assert H.rel_l2(got, expected) < 1e-12


def test_P3_gridding_is_adjoint_of_degridding(tiny):
    prm = dataclasses.replace(tiny.params, w_step=150.0)
    d = _np(tiny)
    meta, _, _ = orc.plan(prm, d["uvw"], d["freqs"], tiny.baselines)
    rng = np.random.default_rng(11)
    L = prm.grid_size
    x = rng.standard_normal((4, L, L)) + 1j * rng.standard_normal((4, L, L))
    v = (rng.standard_normal(d["vis"].shape) + 1j * rng.standard_normal(d["vis"].shape)).astype(np.complex64)
    Dx = orc.degrid(prm, meta, d["uvw"], d["freqs"], x, d["aterms"], d["taper"], tiny.B)
    Gv = orc.grid(prm, meta, d["uvw"], d["freqs"], v, d["aterms"], d["taper"])
    lhs = np.vdot(Dx, v.astype(np.complex128))
    rhs = np.vdot(x, Gv)
    assert abs(lhs - rhs) / abs(lhs) < 1e-10


def test_P4_off_lattice_agreement_with_direct_imaging():
    """Whole image (inner half) against Eq. 11 -- this is what sees a planner that lets
    samples leave the box, which the lattice identity cannot."""
    w = synth.make_workload("tiny", identity_a=True)
    d = _np(w)
    prm = w.params
    meta, planned, _ = orc.plan(prm, d["uvw"], d["freqs"], w.baselines)
    grid = orc.grid(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])
    L, N, S = prm.grid_size, prm.subgrid_size, prm.image_size
    image = H.image_from_grid(grid)[0]
    # effective window of a centred sample = trigonometric interpolation of the taper (4.2)
    a = synth.prolate_taper_1d(N)
    k = np.arange(N) - N // 2
    A = np.array([np.sum(a * np.exp(-2j * np.pi * kk * k / N)) for kk in k]) / N
    xx = np.arange(L) - L // 2
    c1d = np.real(np.exp(2j * np.pi * np.outer(xx, k) / L) @ A)
    inner = slice(L // 4, 3 * L // 4)
    corrected = image[inner, inner] / np.outer(c1d[inner], c1d[inner])
    lv = H.lm_of_pixels(np.arange(L)[inner], L, S)
    ll, mm = np.meshgrid(lv, lv)
    nn = H.nprime(ll, mm)
    die = np.zeros(ll.shape, dtype=np.complex128)
    kf = d["freqs"] / H.C0
    for b in range(w.B):
        for t in range(w.T):
            u, v, ww = (np.float64(q) for q in d["uvw"][b, t])
            for c in range(w.C):
                ph = 2.0 * np.pi * kf[c] * (u * ll + v * mm + ww * nn)
                die += np.exp(1j * ph) * np.complex128(d["vis"][b, t, c, 0])
    err = H.rel_l2(corrected, die)
    assert err < 1e-3, err
    assert err > 1e-9      # it IS an approximation off the lattice; exact equality would mean the test is vacuous


@pytest.mark.parametrize("N", [16, 24, 32, 48])
def test_subgrid_fft_equals_library_fft(N):
    rng = np.random.default_rng(N)
    x = rng.standard_normal((3, 4, N, N)) + 1j * rng.standard_normal((3, 4, N, N))
    fwd = orc.subgrid_fft(x, -1)
    ref = np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(x, axes=(-2, -1))), axes=(-2, -1)) / (N * N)
    assert H.rel_l2(fwd, ref) < 1e-13
    inv = orc.subgrid_fft(x, +1)
    ref = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(x, axes=(-2, -1))), axes=(-2, -1))
    assert H.rel_l2(inv, ref) < 1e-13
    # a delta at the centre pixel transforms to a constant 1/N^2 (fixes centring and scale)
    dlt = np.zeros((1, 4, N, N), dtype=np.complex128)
    dlt[:, :, N // 2, N // 2] = 1.0
    assert np.allclose(orc.subgrid_fft(dlt, -1), 1.0 / (N * N), atol=1e-15)


def test_single_visibility_at_subgrid_centre():
    """Delta = 0: every phasor is 1, so the subgrid image is taper * A1^H Y A2 exactly."""
    rng = np.random.default_rng(3)
    N, L, S = 16, 64, 0.02
    prm = synth.PlanParams(L, N, 4, 1, 1, 1, 0, S, 0.0)
    freqs = np.array([150e6])
    x0, y0 = 30, 11
    u0 = (x0 + N // 2 - L // 2) / S
    v0 = (y0 + N // 2 - L // 2) / S
    lam = H.C0 / freqs[0]
    uvw = np.array([[[u0 * lam, v0 * lam, 0.0]]], dtype=np.float64)
    # pick metres that are exactly representable so that u*f/c - u0 cancels to ~1e-13
    uvw32 = uvw.astype(np.float32)
    aterms = synth.random_aterms(rng, 1, 2, N)
    taper = synth.prolate_taper(N)
    vis = (rng.standard_normal((1, 1, 1, 4)) + 1j * rng.standard_normal((1, 1, 1, 4))).astype(np.complex64)
    meta = np.zeros(1, dtype=orc.META_DTYPE)
    meta[0] = (0, 0, 1, 0, 1, 0, 1, 0, x0, y0, 0, 0)
    img = orc.gridder(prm, meta, uvw32, freqs, vis, aterms, taper)[0]
    # residual offset from float32 rounding of the metres, as a phase gradient bound
    du = float(uvw32[0, 0, 0]) * freqs[0] / H.C0 - u0
    dv = float(uvw32[0, 0, 1]) * freqs[0] / H.C0 - v0
    bound = 2 * np.pi * (abs(du) + abs(dv)) * S / 2 + 1e-12
    Y = vis[0, 0, 0].astype(np.complex128).reshape(2, 2)
    A1 = H.jones(aterms, 0, 0)
    A2 = H.jones(aterms, 0, 1)
    expected = np.conj(np.swapaxes(A1, -1, -2)) @ Y @ A2 * taper.astype(np.float64)[..., None, None]
    got = np.moveaxis(img, 0, -1).reshape(N, N, 2, 2)
    assert H.rel_l2(got, expected) < 4 * bound


def test_adder_and_splitter_against_slicing():
    rng = np.random.default_rng(5)
    N, L, P = 16, 80, 9
    meta = np.zeros(P, dtype=orc.META_DTYPE)
    meta["x0"] = rng.integers(0, L - N + 1, P)
    meta["y0"] = rng.integers(0, L - N + 1, P)
    meta["x0"][:3] = [0, L - N, 20]
    meta["y0"][:3] = [L - N, 0, 20]
    meta["x0"][3], meta["y0"][3] = 25, 17          # overlaps subgrid 2
    sub = rng.standard_normal((P, 4, N, N)) + 1j * rng.standard_normal((P, 4, N, N))
    grid0 = rng.standard_normal((4, L, L)) + 1j * rng.standard_normal((4, L, L))
    ref = grid0.copy()
    for p in range(P):
        ref[:, meta["y0"][p]:meta["y0"][p] + N, meta["x0"][p]:meta["x0"][p] + N] += sub[p]
    got = orc.adder(meta, sub, grid0.copy())
    assert np.array_equal(got, ref)                # accumulates on top of what was there
    sp = orc.splitter(meta, grid0, N)
    for p in range(P):
        assert np.array_equal(sp[p], grid0[:, meta["y0"][p]:meta["y0"][p] + N, meta["x0"][p]:meta["x0"][p] + N])
