"""Image-plane wrap around the hot path with W-stacking: a science-valid dirty
image and model prediction.  Outside the timed path (BASELINE.json: "the large-grid FFT is outside the timed
path").

Alg. 1 last line "I <- FFT(V)/c-bar" (R8) and Alg. 2 first lines "I <- I/c-bar; V <- FFT(I)"
(PAPER.md:319-322); the per-subgrid w offset (R4) is resolved by W-stacking: one
w layer at a time is gridded onto a scratch grid, transformed with the LIBRARY FFT (cuFFT through
torch.fft -- the one library step, as SURVEY.md allows for this row), multiplied by exp(+2 pi i w0 n') and
accumulated by this package's CUDA kernels (csrc/image.cu); the sum is divided by the image-domain taper.
Only one [4][L][L] grid and one image are resident, whatever the number of layers.

Everything numerical except the FFT runs in libidg_b200.so; this module sequences the calls.
"""
from __future__ import annotations

import dataclasses
from typing import List, Tuple

import numpy as np
import torch

from . import binding as idg


def _centred_ifft2_unnormalised(grid: torch.Tensor) -> torch.Tensor:
    L = grid.shape[-1]
    return torch.fft.fftshift(torch.fft.ifft2(torch.fft.ifftshift(grid, dim=(-2, -1)), norm="forward"), dim=(-2, -1))


def _centred_fft2(img: torch.Tensor) -> torch.Tensor:
    return torch.fft.fftshift(torch.fft.fft2(torch.fft.ifftshift(img, dim=(-2, -1))), dim=(-2, -1))


def image_taper(taper: torch.Tensor, L: int) -> torch.Tensor:
    """c-bar [L][L] float32 (idg_image_taper: the subgrid taper on the image raster)."""
    return idg.idg_image_taper(taper, L)


def layer_plans(params, uvw: torch.Tensor, freqs, baselines, n_stations: int) -> List[Tuple[int, float, "idg.Plan"]]:
    """Plan once, then one plan per w layer (idg_plan_from_metadata on the rows with that w_index)."""
    full = idg.idg_plan_create(params, uvw, freqs, baselines, n_stations)
    meta = full.metadata()
    B, T = int(uvw.shape[0]), int(uvw.shape[1])
    full.destroy()
    out = []
    for wi in np.unique(meta["w_index"]):
        sel = np.ascontiguousarray(meta[meta["w_index"] == wi])
        layer = idg.idg_plan_from_metadata(params, sel, freqs, B, T, n_stations)
        out.append((int(wi), layer.w_offset(int(wi)), layer))
    return out


def dirty_image(params, uvw, freqs, baselines, n_stations, vis, aterms, taper) -> torch.Tensor:
    """Alg. 1 complete -> image [4][L][L] complex64 on the device of the inputs."""
    L, S = int(params.grid_size), float(params.image_size)
    dev = uvw.device
    image = torch.zeros((4, L, L), dtype=torch.complex64, device=dev)
    grid = torch.empty((4, L, L), dtype=torch.complex64, device=dev)
    for wi, w0, plan in layer_plans(params, uvw, freqs, baselines, n_stations):
        grid.zero_()
        idg.idg_grid(plan, uvw, vis, aterms, taper, grid)
        layer = _centred_ifft2_unnormalised(grid).contiguous()
        idg.idg_image_w_accumulate(image, layer, S, w0, +1)
        torch.cuda.synchronize(dev)
        plan.destroy()
    idg.idg_image_divide(image, image_taper(taper, L))
    return image


def predict(params, uvw, freqs, baselines, n_stations, image, aterms, taper, n_channels: int) -> torch.Tensor:
    """Alg. 2 complete -> visibilities [B][T][C][4] complex64 (0 where the plan covers nothing)."""
    L, S = int(params.grid_size), float(params.image_size)
    dev = uvw.device
    B, T = int(uvw.shape[0]), int(uvw.shape[1])
    base = image.clone()
    idg.idg_image_divide(base, image_taper(taper, L))
    vis = torch.zeros((B, T, n_channels, 4), dtype=torch.complex64, device=dev)
    tmp = torch.empty_like(base)
    for wi, w0, plan in layer_plans(params, uvw, freqs, baselines, n_stations):
        idg.idg_image_w_apply(tmp, base, S, w0, -1)
        grid = _centred_fft2(tmp).contiguous()
        sub = plan.subgrids()
        # stage calls, not idg_degrid: the layers fill disjoint samples of one output array
        idg.idg_splitter(plan, grid, sub)
        idg.idg_subgrid_fft(plan, sub, +1)
        idg.idg_degridder(plan, uvw, sub, aterms, taper, vis)
        torch.cuda.synchronize(dev)
        del sub
        plan.destroy()
    return vis
