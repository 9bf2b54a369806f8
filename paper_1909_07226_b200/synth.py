"""Seeded synthetic IDG workloads (input generators only).

This module serves BOTH the CUDA path and the CPU oracle with identical input
arrays.  It holds none of the method's arithmetic (no planner, gridder, FFT,
adder, splitter, degridder): it only builds the *inputs* the paper's Algorithm 1
and 2 take -- station layouts, uvw tracks by
textbook earth-rotation synthesis, frequencies, point-source visibilities from
the measurement equation (Eq. 1-3), random A-terms and a
prolate-spheroidal taper -- for the shapes BASELINE.json:configs names.  The
synthetic data stand in for the LOFAR "Toothbrush" measurement set the paper
used, which is not available here.  It imports nothing from the
rest of the package and nothing from ``oracle/``.

Recipe (also stated in DESIGN.md):
  * RNG: ``numpy.random.default_rng(1000 + config index)``, fixed draw order
    stations -> sources -> A-terms; the visibility noise uses a
    ``torch.Generator`` seeded with the same number on the device the
    visibilities are produced on (CPU for the small configs, CUDA for the big
    ones), so a given (config, device type) pair is reproducible.
  * uvw in metres, float32; frequencies float64; visibilities complex64
    [B][T][C][4] (XX, XY, YX, YY); A-terms complex64
    [slots][stations][N][N][4]; taper float32 [N][N].
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np
import torch

SPEED_OF_LIGHT = 299792458.0
EARTH_ROTATION_RAD_S = 7.2921150e-5

FLAG_FORCE_BLOCKS = 1
FLAG_SPAN_ATERMS = 2
FLAG_FP32_GRIDDER = 4


@dataclasses.dataclass
class PlanParams:
    """Mirror of ``idg_plan_params`` (include/idg_b200.h); plain numbers only."""

    grid_size: int
    subgrid_size: int
    kernel_size: int
    max_timesteps: int
    max_channels: int
    aterm_interval: int
    flags: int
    image_size: float
    w_step: float


@dataclasses.dataclass
class Workload:
    name: str
    seed: int
    n_stations: int
    baselines: np.ndarray      # [B][2] int32
    uvw: torch.Tensor          # [B][T][3] float32 (metres)
    freqs: np.ndarray          # [C] float64 (Hz)
    vis: torch.Tensor          # [B][T][C][4] complex64
    aterms: torch.Tensor       # [slots][stations][N][N][4] complex64
    taper: torch.Tensor        # [N][N] float32
    params: PlanParams
    sources: np.ndarray        # [S][3] (l, m, flux) -- what the visibilities contain

    @property
    def B(self) -> int:
        return int(self.baselines.shape[0])

    @property
    def T(self) -> int:
        return int(self.uvw.shape[1])

    @property
    def C(self) -> int:
        return int(self.freqs.shape[0])

    def to(self, device) -> "Workload":
        return dataclasses.replace(
            self,
            uvw=self.uvw.to(device),
            vis=self.vis.to(device),
            aterms=self.aterms.to(device),
            taper=self.taper.to(device),
        )


# ----------------------------------------------------------------------------
# geometry
# ----------------------------------------------------------------------------

def all_baselines(n_stations: int) -> np.ndarray:
    """All station pairs i<j in lexicographic order, int32 [B][2]."""
    i, j = np.triu_indices(n_stations, k=1)
    return np.stack([i, j], axis=1).astype(np.int32)


def layout_disk(rng, n: int, radius_m: float) -> np.ndarray:
    """n stations uniform in a disk; ENU with up = 0."""
    r = radius_m * np.sqrt(rng.random(n))
    az = 2.0 * math.pi * rng.random(n)
    return np.stack([r * np.sin(az), r * np.cos(az), np.zeros(n)], axis=1)


def layout_core_plus_outliers(rng, n_core: int, core_radius_m: float,
                              n_out: int, r_min_m: float, r_max_m: float) -> np.ndarray:
    core = layout_disk(rng, n_core, core_radius_m)
    r = r_min_m + (r_max_m - r_min_m) * rng.random(n_out)
    az = 2.0 * math.pi * rng.random(n_out)
    out = np.stack([r * np.sin(az), r * np.cos(az), np.zeros(n_out)], axis=1)
    return np.concatenate([core, out], axis=0)


def layout_log_radial(rng, n: int, r_min_m: float, r_max_m: float) -> np.ndarray:
    r = r_min_m * (r_max_m / r_min_m) ** rng.random(n)
    az = 2.0 * math.pi * rng.random(n)
    return np.stack([r * np.sin(az), r * np.cos(az), np.zeros(n)], axis=1)


def earth_rotation_uvw(enu: np.ndarray, baselines: np.ndarray, latitude_deg: float,
                       declination_deg: float, hour_angle0_deg: float,
                       integration_s: float, n_time: int) -> np.ndarray:
    """Textbook earth-rotation synthesis -> uvw [B][T][3] float32 metres.

    ENU -> equatorial (X,Y,Z) at the array latitude, then the usual rotation by
    hour angle H and declination (Thompson, Moran & Swenson eq. 4.1).
    """
    lat = math.radians(latitude_deg)
    dec = math.radians(declination_deg)
    e, n, u = enu[:, 0], enu[:, 1], enu[:, 2]
    X = -math.sin(lat) * n + math.cos(lat) * u
    Y = e
    Z = math.cos(lat) * n + math.sin(lat) * u
    d = np.stack([X, Y, Z], axis=1)
    dxyz = d[baselines[:, 1]] - d[baselines[:, 0]]                    # [B][3]
    H = math.radians(hour_angle0_deg) + EARTH_ROTATION_RAD_S * integration_s * np.arange(n_time)
    sH, cH = np.sin(H)[None, :], np.cos(H)[None, :]
    bx, by, bz = dxyz[:, 0:1], dxyz[:, 1:2], dxyz[:, 2:3]
    uu = sH * bx + cH * by
    vv = -math.sin(dec) * cH * bx + math.sin(dec) * sH * by + math.cos(dec) * bz
    ww = math.cos(dec) * cH * bx - math.cos(dec) * sH * by + math.sin(dec) * bz
    return np.stack([uu, vv, ww], axis=2).astype(np.float32)


# ----------------------------------------------------------------------------
# sky, visibilities, A-terms, taper
# ----------------------------------------------------------------------------

def random_sources(rng, n: int, image_size: float, inner_fraction: float,
                   flux_min: Optional[float], flux_max: Optional[float]) -> np.ndarray:
    """n point sources uniform in the inner part of the field; flux from a power law
    of index -2 on [flux_min, flux_max] (inverse-CDF sampling), or 1 Jy if None."""
    half = 0.5 * inner_fraction * image_size
    l = (2.0 * rng.random(n) - 1.0) * half
    m = (2.0 * rng.random(n) - 1.0) * half
    if flux_min is None:
        flux = np.ones(n)
    else:
        q = rng.random(n)
        flux = 1.0 / (1.0 / flux_min - q * (1.0 / flux_min - 1.0 / flux_max))
    return np.stack([l, m, flux], axis=1)


def point_source_visibilities(uvw: torch.Tensor, freqs: np.ndarray, sources: np.ndarray,
                              noise_sigma: float, seed: int, device,
                              baseline_chunk: int = 64) -> torch.Tensor:
    """Measurement equation for unpolarised point sources (Eq. 1-3):
    Y = sum_s F_s exp(-2 pi i (u l_s + v m_s + w n'_s)) on XX and YY, 0 on XY/YX,
    plus complex Gaussian noise on all four.  complex64 [B][T][C][4]."""
    dev = torch.device(device)
    B, T, _ = uvw.shape
    C = len(freqs)
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed)
    vis = torch.empty((B, T, C, 4), dtype=torch.complex64, device=dev)
    k = torch.as_tensor(freqs / SPEED_OF_LIGHT, dtype=torch.float64, device=dev)      # [C] 1/m
    src = torch.as_tensor(sources, dtype=torch.float64, device=dev)
    ls, ms, fs = src[:, 0], src[:, 1], src[:, 2]
    ns = torch.sqrt(1.0 - ls * ls - ms * ms) - 1.0
    for b0 in range(0, B, baseline_chunk):
        b1 = min(B, b0 + baseline_chunk)
        uvw_c = uvw[b0:b1].to(dev, torch.float64)                                      # [b][T][3]
        # path length difference in metres per (b, t, source)
        d = (uvw_c[..., 0:1] * ls + uvw_c[..., 1:2] * ms + uvw_c[..., 2:3] * ns)       # [b][T][S]
        acc = torch.zeros((b1 - b0, T, C), dtype=torch.complex128, device=dev)
        for s in range(src.shape[0]):
            ph = (-2.0 * math.pi) * d[..., s:s + 1] * k                                # [b][T][C]
            acc += fs[s] * torch.polar(torch.ones_like(ph), ph)
        acc = acc.to(torch.complex64)
        noise = torch.randn((b1 - b0, T, C, 4, 2), generator=gen, device=dev,
                            dtype=torch.float32) * noise_sigma
        blk = torch.view_as_complex(noise)
        blk[..., 0] += acc
        blk[..., 3] += acc
        vis[b0:b1] = blk
    return vis


def random_aterms(rng, n_slots: int, n_stations: int, N: int, sigma: float = 0.1) -> np.ndarray:
    """A = I_2 + sigma (N(0,1) + i N(0,1)) per slot, station, pixel, element; complex64
    [slots][stations][N][N][4] (row-major 2x2)."""
    shape = (n_slots, n_stations, N, N, 4)
    a = rng.standard_normal(shape, dtype=np.float32) + 1j * rng.standard_normal(shape, dtype=np.float32)
    a = (sigma * a).astype(np.complex64)
    a[..., 0] += 1.0
    a[..., 3] += 1.0
    return a


def identity_aterms(n_slots: int, n_stations: int, N: int) -> np.ndarray:
    a = np.zeros((n_slots, n_stations, N, N, 4), dtype=np.complex64)
    a[..., 0] = 1.0
    a[..., 3] = 1.0
    return a


def prolate_taper_1d(N: int, NW: float = 3.0) -> np.ndarray:
    """Discrete prolate-spheroidal sequence of length N, periodic form (symmetric about
    index N/2, the centre pixel of the subgrid image), peak 1.  float64."""
    from scipy.signal.windows import dpss
    w = dpss(N, NW, sym=False)
    return w / w.max()


def prolate_taper(N: int, NW: float = 3.0) -> np.ndarray:
    a = prolate_taper_1d(N, NW)
    return np.outer(a, a).astype(np.float32)


# ----------------------------------------------------------------------------
# the configurations of BASELINE.json
# ----------------------------------------------------------------------------

_CONFIG_TABLE = {
    # name: layout, (lat, dec), T, dt, f0, df, C, N, L, S, max_t, max_c, aterm_interval, w_step, n_src, flux, NW
    "tiny": dict(idx=0, lat=52.9, dec=50.0, T=32, dt=10.0, f0=150e6, df=200e3, C=4, N=24, L=256,
                 S=0.06, max_t=16, max_c=4, a_int=16, w_step=0.0, n_src=3, flux=None, inner=0.6),
    "lofar": dict(idx=1, lat=52.9, dec=50.0, T=256, dt=2.0, f0=140e6, df=195e3, C=16, N=32, L=2048,
                  S=0.05, max_t=128, max_c=16, a_int=64, w_step=0.0, n_src=100, flux=(0.01, 10.0), inner=0.6),
    "ska": dict(idx=2, lat=-26.8, dec=-40.0, T=1024, dt=1.0, f0=100e6, df=100e3, C=16, N=32, L=8192,
                S=0.16, max_t=256, max_c=16, a_int=32, w_step=256.0, n_src=100, flux=(0.01, 10.0), inner=0.6),
    # context only: the shape of the paper's simulation (section 5.1/5.3): 55 stations,
    # baselines out to 84 km, 3122 x 10 s, 20 channels 130-132 MHz, 2048^2 image with 1" cells, 48 x 48 subgrids
    "paper": dict(idx=5, lat=52.9, dec=50.0, T=3122, dt=10.0, f0=130e6, df=100e3, C=20, N=48, L=2048,
                  S=2048 * math.pi / (180.0 * 3600.0), max_t=256, max_c=32, a_int=256, w_step=0.0, n_src=1,
                  flux=None, inner=0.2),
    "sweep": dict(idx=4, lat=52.9, dec=50.0, T=1024, dt=2.0, f0=140e6, df=195e3, C=64, N=32, L=2048,
                  S=0.05, max_t=128, max_c=16, a_int=64, w_step=0.0, n_src=100, flux=(0.01, 10.0), inner=0.6),
}

CONFIG_NAMES = tuple(_CONFIG_TABLE.keys())


def _stations(name: str, rng) -> np.ndarray:
    if name == "tiny":
        return layout_disk(rng, 8, 1500.0)
    if name in ("lofar", "sweep"):
        return layout_core_plus_outliers(rng, 36, 2500.0, 12, 2500.0, 20000.0)
    if name == "ska":
        return layout_log_radial(rng, 128, 50.0, 35000.0)
    if name == "paper":
        return layout_log_radial(rng, 55, 60.0, 42000.0)
    raise KeyError(name)


def n_stations_of(name: str) -> int:
    """Number of stations of a named workload (its baselines are all pairs, lexicographic)."""
    return {"tiny": 8, "lofar": 48, "sweep": 48, "ska": 128, "paper": 55}[name]


def make_workload(name: str, device="cpu", *, n_baselines: Optional[int] = None,
                  n_time: Optional[int] = None, subgrid_size: Optional[int] = None,
                  max_timesteps: Optional[int] = None, max_channels: Optional[int] = None,
                  aterm_interval: Optional[int] = None, flags: Optional[int] = None,
                  identity_a: bool = False, seed_offset: int = 0,
                  baseline_offset: int = 0, baseline_stride: int = 1) -> Workload:
    """Build one of BASELINE.json's workloads ("tiny", "lofar", "ska", "sweep").

    Optional overrides shrink it (first ``n_baselines`` baselines starting at
    ``baseline_offset``, every ``baseline_stride``-th of those, first ``n_time`` timesteps) or change the plan
    parameters (the sweep of config 4).  ``seed_offset`` gives another
    realisation of the same shape (used to hand every rank of a weak-scaling
    run its own data).
    """
    c = _CONFIG_TABLE[name]
    seed = 1000 + c["idx"] + 7919 * seed_offset
    rng = np.random.default_rng(seed)
    enu = _stations(name, rng)
    n_st = enu.shape[0]
    bl = all_baselines(n_st)
    if name == "sweep":
        bl = bl[:1024]
    if n_baselines is not None or baseline_offset:
        end = len(bl) if n_baselines is None else baseline_offset + n_baselines
        bl = bl[baseline_offset:end]
    if baseline_stride > 1:
        bl = np.ascontiguousarray(bl[::baseline_stride])
    T = c["T"] if n_time is None else n_time
    uvw_np = earth_rotation_uvw(enu, bl, c["lat"], c["dec"], -30.0, c["dt"], T)
    freqs = c["f0"] + c["df"] * np.arange(c["C"], dtype=np.float64)
    N = c["N"] if subgrid_size is None else subgrid_size
    fl = c["flux"]
    sources = random_sources(rng, c["n_src"], c["S"], c["inner"],
                             None if fl is None else fl[0], None if fl is None else fl[1])
    a_int = c["a_int"] if aterm_interval is None else aterm_interval
    n_slots = (T + a_int - 1) // a_int
    if identity_a:
        aterms_np = identity_aterms(n_slots, n_st, N)
    else:
        aterms_np = random_aterms(rng, n_slots, n_st, N)
    taper_np = prolate_taper(N)
    dev = torch.device(device)
    uvw = torch.from_numpy(uvw_np)
    vis = point_source_visibilities(uvw, freqs, sources, 0.1, seed, dev)
    params = PlanParams(
        grid_size=c["L"], subgrid_size=N, kernel_size=N // 4,
        max_timesteps=c["max_t"] if max_timesteps is None else max_timesteps,
        max_channels=c["max_c"] if max_channels is None else max_channels,
        aterm_interval=a_int,
        flags=(FLAG_FORCE_BLOCKS if name == "sweep" else 0) if flags is None else flags,
        image_size=c["S"], w_step=c["w_step"])
    return Workload(name=name, seed=seed, n_stations=n_st, baselines=bl,
                    uvw=uvw.to(dev), freqs=freqs, vis=vis,
                    aterms=torch.from_numpy(aterms_np).to(dev),
                    taper=torch.from_numpy(taper_np).to(dev), params=params, sources=sources)


def model_grid_from_sources(grid_size: int, n_sources: int, seed: int, device,
                            inner_fraction: float = 0.8) -> torch.Tensor:
    """Config 3's model grid: n unpolarised sources (flux power law, index -2, on
    [0.01, 10]) at integer pixels of a grid_size^2 image, transformed with a centred
    forward FFT per polarisation plane (library FFT; outside the timed path,
    Alg. 2).  complex64 [4][L][L]."""
    rng = np.random.default_rng(seed)
    L = grid_size
    half = int(0.5 * inner_fraction * L)
    x = rng.integers(L // 2 - half, L // 2 + half, n_sources)
    y = rng.integers(L // 2 - half, L // 2 + half, n_sources)
    q = rng.random(n_sources)
    flux = 1.0 / (1.0 / 0.01 - q * (1.0 / 0.01 - 1.0 / 10.0))
    dev = torch.device(device)
    img = torch.zeros((L, L), dtype=torch.complex64, device=dev)
    img.index_put_((torch.as_tensor(y, device=dev), torch.as_tensor(x, device=dev)),
                   torch.as_tensor(flux, dtype=torch.complex64, device=dev), accumulate=True)
    plane = torch.fft.fftshift(torch.fft.fft2(torch.fft.ifftshift(img)))
    grid = torch.zeros((4, L, L), dtype=torch.complex64, device=dev)
    grid[0] = plane
    grid[3] = plane
    return grid
