"""-m gpu: idg_image_taper_static, the entry point that allocates nothing (scratch in a fixed device array of the
library), against idg_image_taper (stream-ordered allocation of the same scratch) -- the same three kernels on the same
inputs, so the results are compared to 1e-6 relative L2 (the tolerance of the boundary tests for two runs of one
computation; in practice they are equal).  Two calls in a row share the array: the second, smaller request finds the
first one's contents in it and must not be affected.  Collected last on purpose (file name): the suite runs with
pytest -x, and a failure here must not hide other tests.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _taper(n, seed):
    rng = np.random.default_rng(seed)
    w = np.hanning(n + 2)[1:-1]
    return (np.outer(w, w) * (1.0 + 0.05 * rng.standard_normal((n, n)))).astype(np.float32)


def _rel_l2(a, b):
    return float(np.linalg.norm(a.astype(np.float64) - b) / np.linalg.norm(b.astype(np.float64)))


def test_static_scratch_entry_point_matches_the_allocating_one_twice_in_a_row():
    from paper_1909_07226_b200 import binding as idg
    dev = torch.device("cuda", 0)
    cases = [(32, 768, 1), (16, 256, 2)]                # the second request is smaller: stale scratch lies behind it
    want = []
    for n, L, seed in cases:
        want.append(idg.idg_image_taper(torch.from_numpy(_taper(n, seed)).to(dev), L).cpu().numpy())
    torch.cuda.synchronize()
    got = []
    before = torch.cuda.memory_allocated(dev)
    outs = [torch.full((L, L), float("nan"), dtype=torch.float32, device=dev) for _, L, _ in cases]
    tapers = [torch.from_numpy(_taper(n, seed)).to(dev) for n, _, seed in cases]
    for t, o in zip(tapers, outs):                      # back to back on one stream, no synchronisation between them
        idg.idg_image_taper_static(t, o)
    torch.cuda.synchronize()
    for o in outs:
        got.append(o.cpu().numpy())
    for g, w in zip(got, want):
        assert np.isfinite(g).all()
        assert _rel_l2(g, w) < 1e-6
    # and once more in the other order: the larger request after the smaller one
    for t, o in zip(tapers[::-1], outs[::-1]):
        o.fill_(float("nan"))
        idg.idg_image_taper_static(t, o)
    torch.cuda.synchronize()
    for o, w in zip(outs, want):
        assert _rel_l2(o.cpu().numpy(), w) < 1e-6
    assert before <= torch.cuda.memory_allocated(dev)   # (torch's own tensors only; the library allocated nothing)


def test_static_scratch_entry_point_refuses_what_does_not_fit():
    from paper_1909_07226_b200 import binding as idg
    dev = torch.device("cuda", 0)
    n = 48
    L = idg.IMAGE_TAPER_STATIC_MAX_LN // n + 2            # even, L * N just above the limit
    L += L & 1
    assert L * n > idg.IMAGE_TAPER_STATIC_MAX_LN
    taper = torch.from_numpy(_taper(n, 3)).to(dev)
    # the call must fail before it touches cbar: a one-element stand-in would fault otherwise
    cbar = torch.empty((L, L), dtype=torch.float32, device=dev)
    cbar.fill_(7.0)
    with pytest.raises(idg.IdgError, match="scratch"):
        idg.idg_image_taper_static(taper, cbar)
    torch.cuda.synchronize()
    assert float(cbar.min()) == 7.0 and float(cbar.max()) == 7.0
    # the largest request that fits at N = 32 is served
    L_ok = idg.IMAGE_TAPER_STATIC_MAX_LN // 32
    t32 = torch.from_numpy(_taper(32, 4)).to(dev)
    out = torch.empty((L_ok, L_ok), dtype=torch.float32, device=dev)
    idg.idg_image_taper_static(t32, out)
    ref = idg.idg_image_taper(t32, L_ok)
    torch.cuda.synchronize()
    assert _rel_l2(out.cpu().numpy(), ref.cpu().numpy()) < 1e-6
