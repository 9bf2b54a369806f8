"""Pins of the W-stacked image-plane wrap of the oracle (NEXT-1): against the paper's defining sums, not
against itself.  Direct imaging equation, Eq. 11, and discrete measurement equation, Eq. 6
(PAPER.md:84), with the FULL w term -- the w layers must cancel exactly."""
import dataclasses

import numpy as np

from oracle import idg_oracle as orc
from paper_1909_07226_b200 import synth
from tests import helpers as H


def _case(w_step):
    w = synth.make_workload("tiny", identity_a=True)
    prm = dataclasses.replace(w.params, w_step=w_step)
    d = dict(uvw=w.uvw.numpy(), freqs=w.freqs, vis=w.vis.numpy(), aterms=w.aterms.numpy(), taper=w.taper.numpy())
    meta, planned, skipped = orc.plan(prm, d["uvw"], d["freqs"], w.baselines)
    assert skipped == 0
    return w, prm, d, meta


def _die(d, w, ll, mm):
    """Eq. 11 on XX for directions (ll, mm): sum_k Y_k exp(+2 pi i (u l + v m + w n'))."""
    nn = H.nprime(ll, mm)
    out = np.zeros(ll.shape, dtype=np.complex128)
    kf = d["freqs"] / H.C0
    for b in range(w.B):
        for t in range(w.T):
            u, v, ww = (np.float64(q) for q in d["uvw"][b, t])
            for c in range(w.C):
                out += np.exp(2j * np.pi * kf[c] * (u * ll + v * mm + ww * nn)) * np.complex128(d["vis"][b, t, c, 0])
    return out


def test_image_taper_reproduces_the_taper_on_the_lattice():
    N, L = 24, 96
    t = synth.prolate_taper(N).astype(np.float64)
    cb = orc.image_taper(t, L)
    idx = L // 2 + (np.arange(N) - N // 2) * (L // N)
    assert np.allclose(cb[np.ix_(idx, idx)], t, atol=1e-12)


def test_w_stacked_image_equals_direct_imaging_on_the_lattice():
    """Several w layers (w_step 150 wavelengths): at the lattice pixels the corrected image is Eq. 11 with the
    full w n' phase, to round-off; in between it agrees to the taper's side-lobe level."""
    w, prm, d, meta = _case(150.0)
    assert len(orc.w_layers(meta)) >= 3
    L, N, S = prm.grid_size, prm.subgrid_size, prm.image_size
    img = orc.dirty_image(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"])[0]
    step = L // np.gcd(L, N)
    idx = np.arange(L // 2 % step, L, step)
    idx = idx[(idx > L // 4) & (idx < 3 * L // 4)]
    lv = H.lm_of_pixels(idx, L, S)
    ll, mm = np.meshgrid(lv, lv)
    ref = _die(d, w, ll, mm)
    assert H.rel_l2(img[np.ix_(idx, idx)], ref) < 1e-11
    # a dropped or wrongly signed layer factor is a gross error:
    bad = orc.dirty_image(dataclasses.replace(prm, w_step=prm.w_step), meta, d["uvw"], d["freqs"], d["vis"],
                          d["aterms"], d["taper"])[0] * np.exp(-4j * np.pi * 75.0 * orc.image_nprime(L, S))
    assert H.rel_l2(bad[np.ix_(idx, idx)], ref) > 1e-3
    # off the lattice: approximation at the side-lobe level
    inner = np.arange(L // 4, 3 * L // 4, 5)
    lv = H.lm_of_pixels(inner, L, S)
    ll, mm = np.meshgrid(lv, lv)
    err = H.rel_l2(img[np.ix_(inner, inner)], _die(d, w, ll, mm))
    assert 1e-9 < err < 1e-3, err


def test_w_stacked_prediction_of_a_point_source_is_the_measurement_equation():
    """One source on the lattice: every predicted visibility is B exp(-2 pi i (u l0 + v m0 + w n'0)) (Eq. 6),
    with the full w, to round-off."""
    w, prm, d, meta = _case(150.0)
    L, N, S = prm.grid_size, prm.subgrid_size, prm.image_size
    step = L // np.gcd(L, N)
    x0, y0 = L // 2 + 2 * step, L // 2 - step
    flux = 2.5
    img = np.zeros((4, L, L), dtype=np.complex128)
    img[0, y0, x0] = flux
    img[3, y0, x0] = flux
    pred = orc.predict(prm, meta, d["uvw"], d["freqs"], img, d["aterms"], d["taper"], w.B)
    l0, m0 = H.lm_of_pixels(np.array([x0, y0]), L, S)
    n0 = H.nprime(l0, m0)
    kf = d["freqs"] / H.C0
    u, v, ww = (d["uvw"][..., i].astype(np.float64)[:, :, None] * kf[None, None, :] for i in range(3))
    ref = flux * np.exp(-2j * np.pi * (u * l0 + v * m0 + ww * n0))
    assert H.rel_l2(pred[..., 0], ref) < 1e-11
    assert H.rel_l2(pred[..., 3], ref) < 1e-11
    assert np.abs(pred[..., 1]).max() < 1e-12 and np.abs(pred[..., 2]).max() < 1e-12
