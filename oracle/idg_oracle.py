"""numpy/ctypes front end of the float64 CPU oracle (oracle/idg_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  It imports nothing from the
product package and the product never imports it.  The arithmetic of the hot path lives in
idg_oracle.c; this file marshals numpy arrays and composes the stages in
the order of Alg. 1 / Alg. 2.  The image-plane wrap with
W-stacking at the end of the file (NEXT-1, outside the timed path) is plain numpy.
Pins of that part: tests/test_imaging_pins.py (Eq. 11 and Eq. 6 with the full w term).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "idg_oracle.c")
_LIB = os.path.join(_HERE, "libidg_oracle.so")

META_DTYPE = np.dtype([(n, "<i4") for n in (
    "baseline", "station1", "station2", "time_begin", "n_time", "chan_begin", "n_chan",
    "aterm_slot", "x0", "y0", "w_index", "reserved")])
assert META_DTYPE.itemsize == 48


class Params(ctypes.Structure):
    _fields_ = [("grid_size", ctypes.c_int32), ("subgrid_size", ctypes.c_int32),
                ("kernel_size", ctypes.c_int32), ("max_timesteps", ctypes.c_int32),
                ("max_channels", ctypes.c_int32), ("aterm_interval", ctypes.c_int32),
                ("flags", ctypes.c_int32), ("reserved", ctypes.c_int32),
                ("image_size", ctypes.c_double), ("w_step", ctypes.c_double)]


def build(force: bool = False) -> str:
    """Compile idg_oracle.c with gcc (no FMA contraction, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c11",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_plan.restype = ctypes.c_int64
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _params(p) -> Params:
    """Accept any object with the idg_plan_params field names (e.g. synth.PlanParams)."""
    return Params(int(p.grid_size), int(p.subgrid_size), int(p.kernel_size), int(p.max_timesteps),
                  int(p.max_channels), int(p.aterm_interval), int(p.flags), 0,
                  float(p.image_size), float(p.w_step))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a), dtype=np.float32)


def _c64_as_f32(a) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(a), dtype=np.complex64)
    return a.view(np.float32)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def plan(params, uvw, freqs, baselines) -> Tuple[np.ndarray, int, int]:
    """-> (meta[P] structured array, n_planned_vis, n_skipped_vis)."""
    prm = _params(params)
    uvw = _f32(uvw)
    B, T, _ = uvw.shape
    freqs = np.ascontiguousarray(freqs, dtype=np.float64)
    bl = np.ascontiguousarray(baselines, dtype=np.int32)
    planned, skipped = ctypes.c_int64(0), ctypes.c_int64(0)
    args = (ctypes.byref(prm), _ptr(uvw), _ptr(freqs), _ptr(bl), ctypes.c_int32(B),
            ctypes.c_int32(T), ctypes.c_int32(len(freqs)))
    n = lib().oracle_plan(*args, None, ctypes.c_int64(0), ctypes.byref(planned), ctypes.byref(skipped))
    meta = np.zeros(n, dtype=META_DTYPE)
    lib().oracle_plan(*args, _ptr(meta), ctypes.c_int64(n), ctypes.byref(planned), ctypes.byref(skipped))
    return meta, int(planned.value), int(skipped.value)


def gridder(params, meta, uvw, freqs, vis, aterms, taper) -> np.ndarray:
    """Subgrid images [P][4][N][N] complex128 (Eq. 25 + A-terms + taper)."""
    prm = _params(params)
    uvw = _f32(uvw)
    _, T, _ = uvw.shape
    freqs = np.ascontiguousarray(freqs, dtype=np.float64)
    visf = _c64_as_f32(vis)
    at = _c64_as_f32(aterms)
    n_stations = np.asarray(aterms).shape[1]
    tp = _f32(taper)
    meta = np.ascontiguousarray(meta)
    N = prm.subgrid_size
    out = np.zeros((len(meta), 4, N, N), dtype=np.complex128)
    lib().oracle_gridder(ctypes.byref(prm), _ptr(meta), ctypes.c_int64(len(meta)), _ptr(uvw),
                         _ptr(freqs), _ptr(visf), _ptr(at), _ptr(tp), ctypes.c_int32(T),
                         ctypes.c_int32(len(freqs)), ctypes.c_int32(n_stations), _ptr(out))
    return out


def subgrid_fft(subgrids: np.ndarray, sign: int) -> np.ndarray:
    """Centred 2-D DFT of every [N][N] plane, scaled 1/N^2; sign=-1 forward, +1 inverse."""
    s = np.array(subgrids, dtype=np.complex128, order="C", copy=True)
    P, four, N, _ = s.shape
    assert four == 4
    lib().oracle_subgrid_fft(_ptr(s), ctypes.c_int64(P), ctypes.c_int32(N), ctypes.c_int32(sign))
    return s


def adder(meta, subgrids, grid: np.ndarray) -> np.ndarray:
    """grid[4][L][L] complex128 += subgrids at their (x0, y0); returns grid (in place)."""
    assert grid.dtype == np.complex128 and grid.flags.c_contiguous
    s = np.ascontiguousarray(subgrids, dtype=np.complex128)
    meta = np.ascontiguousarray(meta)
    lib().oracle_adder(_ptr(meta), ctypes.c_int64(len(meta)), _ptr(s), ctypes.c_int32(s.shape[-1]),
                       ctypes.c_int32(grid.shape[-1]), _ptr(grid))
    return grid


def splitter(meta, grid, N: int) -> np.ndarray:
    g = np.ascontiguousarray(grid, dtype=np.complex128)
    meta = np.ascontiguousarray(meta)
    out = np.zeros((len(meta), 4, N, N), dtype=np.complex128)
    lib().oracle_splitter(_ptr(meta), ctypes.c_int64(len(meta)), _ptr(g), ctypes.c_int32(N),
                          ctypes.c_int32(g.shape[-1]), _ptr(out))
    return out


def degridder(params, meta, uvw, freqs, subgrid_images, aterms, taper, n_baselines: int) -> np.ndarray:
    """Predicted visibilities [B][T][C][4] complex128 (0 where the plan covers nothing)."""
    prm = _params(params)
    uvw = _f32(uvw)
    _, T, _ = uvw.shape
    freqs = np.ascontiguousarray(freqs, dtype=np.float64)
    at = _c64_as_f32(aterms)
    n_stations = np.asarray(aterms).shape[1]
    tp = _f32(taper)
    s = np.ascontiguousarray(subgrid_images, dtype=np.complex128)
    meta = np.ascontiguousarray(meta)
    out = np.zeros((n_baselines, T, len(freqs), 4), dtype=np.complex128)
    lib().oracle_degridder(ctypes.byref(prm), _ptr(meta), ctypes.c_int64(len(meta)), _ptr(uvw),
                           _ptr(freqs), _ptr(s), _ptr(at), _ptr(tp), ctypes.c_int32(T),
                           ctypes.c_int32(len(freqs)), ctypes.c_int32(n_stations), _ptr(out))
    return out


# ---- the two directions, stage after stage (Alg. 1 / Alg. 2) ------------------------------

def grid(params, meta, uvw, freqs, vis, aterms, taper, grid_out: Optional[np.ndarray] = None) -> np.ndarray:
    """Alg. 1 without its last line: gridder -> subgrid FFT -> adder.  complex128 [4][L][L]."""
    L = int(params.grid_size)
    if grid_out is None:
        grid_out = np.zeros((4, L, L), dtype=np.complex128)
    img = gridder(params, meta, uvw, freqs, vis, aterms, taper)
    sub = subgrid_fft(img, -1)
    return adder(meta, sub, grid_out)


def degrid(params, meta, uvw, freqs, grid_in, aterms, taper, n_baselines: int) -> np.ndarray:
    """Alg. 2 after its first two lines: splitter -> subgrid IFFT -> degridder."""
    sub = splitter(meta, grid_in, int(params.subgrid_size))
    img = subgrid_fft(sub, +1)
    return degridder(params, meta, uvw, freqs, img, aterms, taper, n_baselines)


# ---- image-plane wrap with W-stacking (outside the timed path) --------------
# Alg. 1 last line "I <- FFT(V)/c-bar" (reading R8: inverse-sign centred DFT, unnormalised),
# Alg. 2 first lines "I <- I/c-bar; V <- FFT(I)", the per-subgrid w offset of Alg. 1
# (R4) resolved per w layer (W-stacking).  Plain numpy, float64; the library FFT
# with its centring shifts is the step, everything else is written out.

def _centred_ifft2_unnormalised(grid: np.ndarray) -> np.ndarray:
    L = grid.shape[-1]
    return np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(grid, axes=(-2, -1))), axes=(-2, -1)) * (L * L)


def _centred_fft2(img: np.ndarray) -> np.ndarray:
    return np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(img, axes=(-2, -1))), axes=(-2, -1))


def image_nprime(L: int, image_size: float) -> np.ndarray:
    """n'(l_x, m_y) on the image raster, l_x = (x - L/2) S / L (Eq. 5; R2)."""
    l = (np.arange(L, dtype=np.float64) - L // 2) * image_size / L
    ll, mm = np.meshgrid(l, l)
    r2 = ll * ll + mm * mm
    return -r2 / (1.0 + np.sqrt(1.0 - r2))


def image_taper(taper: np.ndarray, L: int) -> np.ndarray:
    """c-bar [L][L]: the subgrid taper [N][N] carried to the image raster.  Section 4.2: the
    effective window is the trigonometric interpolation of the discrete one, i.e. its centred DFT
    coefficients evaluated on the finer raster."""
    t = np.asarray(taper, dtype=np.float64)
    N = t.shape[0]
    k = np.arange(N) - N // 2
    F = np.exp(-2j * np.pi * np.outer(k, k) / N) / N            # centred DFT, scale 1/N per axis
    coef = F @ t @ F.T                                          # [N][N] coefficients
    x = np.arange(L) - L // 2
    E = np.exp(2j * np.pi * np.outer(x, k) / L)                 # evaluate on the L-raster
    return np.real(E @ coef @ E.T)


def w_layers(meta: np.ndarray):
    return [int(w) for w in np.unique(meta["w_index"])]


def dirty_image(params, meta, uvw, freqs, vis, aterms, taper) -> np.ndarray:
    """Alg. 1 complete, one grid per w layer: image[pol][y][x] = (sum_layers IDFT(grid_layer) e^{+2 pi i w0 n'}) / c-bar."""
    L, S = int(params.grid_size), float(params.image_size)
    n = image_nprime(L, S)
    img = np.zeros((4, L, L), dtype=np.complex128)
    for wi in w_layers(meta):
        sel = np.ascontiguousarray(meta[meta["w_index"] == wi])
        g = grid(params, sel, uvw, freqs, vis, aterms, taper)
        w0 = (wi + 0.5) * params.w_step if params.w_step > 0 else 0.0
        img += _centred_ifft2_unnormalised(g) * np.exp(2j * np.pi * w0 * n)
    return img / image_taper(taper, L)


def predict(params, meta, uvw, freqs, image, aterms, taper, n_baselines: int) -> np.ndarray:
    """Alg. 2 complete: per w layer, V = FFT((I / c-bar) e^{-2 pi i w0 n'}), then splitter -> IFFT -> degridder."""
    L, S = int(params.grid_size), float(params.image_size)
    n = image_nprime(L, S)
    base = np.asarray(image, dtype=np.complex128) / image_taper(taper, L)
    out = np.zeros((n_baselines, np.asarray(uvw).shape[1], len(freqs), 4), dtype=np.complex128)
    for wi in w_layers(meta):
        sel = np.ascontiguousarray(meta[meta["w_index"] == wi])
        w0 = (wi + 0.5) * params.w_step if params.w_step > 0 else 0.0
        g = _centred_fft2(base * np.exp(-2j * np.pi * w0 * n))
        out += degrid(params, sel, uvw, freqs, g, aterms, taper, n_baselines)   # layers cover disjoint samples
    return out
