"""Test-side ground truth written from the paper's *defining* equations (not from
Alg. 1/2): the direct imaging equation (Eq. 11), the discrete
measurement equation (Eq. 6) and the large centred transforms that
sit outside the hot path (Alg. 1 last line PAPER.md:308, Alg. 2 first lines
PAPER.md:319-322).  numpy only; shares nothing with oracle/ or the CUDA code."""
from __future__ import annotations

import numpy as np

C0 = 299792458.0


def rel_l2(a, b) -> float:
    a = np.asarray(a)
    b = np.asarray(b)
    den = np.linalg.norm(b.ravel())
    return float(np.linalg.norm((a - b).ravel()) / (den if den > 0 else 1.0))


def image_from_grid(grid: np.ndarray) -> np.ndarray:
    """R8: image[y][x] = sum_{q,r} grid[r][q] exp(+2 pi i((q-L/2)(x-L/2)+(r-L/2)(y-L/2))/L),
    unnormalised, per polarisation plane.  Library FFT with the centring shifts."""
    L = grid.shape[-1]
    return np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(grid, axes=(-2, -1))), axes=(-2, -1)) * (L * L)


def grid_from_image(img: np.ndarray) -> np.ndarray:
    """Model grid = sum_{x,y} img[y][x] exp(-2 pi i(...)/L), unnormalised (Alg. 2)."""
    return np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(img, axes=(-2, -1))), axes=(-2, -1))


def lm_of_pixels(idx: np.ndarray, n_pix: int, S: float) -> np.ndarray:
    """Eq. 5 centred on the DC pixel n_pix/2."""
    return (np.asarray(idx, dtype=np.float64) - n_pix // 2) * S / n_pix


def nprime(l, m):
    return np.sqrt(1.0 - l * l - m * m) - 1.0


def jones(aterms: np.ndarray, slot: int, station: int) -> np.ndarray:
    """[N][N][2][2] complex128."""
    a = np.asarray(aterms[slot, station], dtype=np.complex128)
    return a.reshape(a.shape[0], a.shape[1], 2, 2)


def die_per_subgrid(meta_row, w0: float, uvw, freqs, vis, l, m):
    """Eq. 11 restricted to the samples of one block: sum_k Y_k exp(+2 pi i (u_k l + v_k m +
    (w_k - w0) n')) for directions (l, m) (arrays of equal shape).  -> [..., 2, 2]."""
    b = int(meta_row["baseline"])
    t0, nt = int(meta_row["time_begin"]), int(meta_row["n_time"])
    c0, nc = int(meta_row["chan_begin"]), int(meta_row["n_chan"])
    n = nprime(l, m)
    out = np.zeros(l.shape + (4,), dtype=np.complex128)
    k = np.asarray(freqs[c0:c0 + nc], dtype=np.float64) / C0
    for t in range(t0, t0 + nt):
        u, v, w = (np.float64(x) for x in uvw[b, t])
        for ci in range(nc):
            ph = 2.0 * np.pi * (u * k[ci] * l + v * k[ci] * m + (w * k[ci] - w0) * n)
            out += np.exp(1j * ph)[..., None] * np.asarray(vis[b, t, c0 + ci], dtype=np.complex128)
    return out.reshape(l.shape + (2, 2))


def w_offset(meta_row, w_step: float) -> float:
    return (int(meta_row["w_index"]) + 0.5) * w_step if w_step > 0 else 0.0
