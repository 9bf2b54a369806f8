"""Thin ctypes binding of libidg_b200.so (include/idg_b200.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device
memory and streams.  There is NO CPU fallback: loading fails loudly when the library is
missing, and every call raises ``IdgError`` on a non-zero status.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libidg_b200.so")

META_DTYPE = np.dtype([(n, "<i4") for n in (
    "baseline", "station1", "station2", "time_begin", "n_time", "chan_begin", "n_chan",
    "aterm_slot", "x0", "y0", "w_index", "reserved")])
assert META_DTYPE.itemsize == 48

EXPORTS = (
    "idg_strerror", "idg_last_cuda_error", "idg_kernel_launches", "idg_bench_instruction_mix", "idg_bench_mma_rate", "idg_plan_create", "idg_plan_from_metadata",
    "idg_plan_size", "idg_plan_metadata", "idg_plan_subgrids", "idg_plan_aterm_slots", "idg_plan_w_offset", "idg_plan_uses_tensor_cores",
    "idg_plan_destroy", "idg_grid",
    "idg_degrid", "idg_grid_host", "idg_degrid_host", "idg_grid_degrid_host", "idg_gridder", "idg_subgrid_fft",
    "idg_adder", "idg_splitter", "idg_splitter_ifft", "idg_degridder", "idg_image_w_accumulate", "idg_image_w_apply",
    "idg_image_divide", "idg_image_taper", "idg_image_taper_static", "idg_taper_optimal", "idg_grid_scalar", "idg_degrid_scalar", "idg_gridder_scalar", "idg_degridder_scalar")


class IdgError(RuntimeError):
    pass


class PlanParams(ctypes.Structure):
    """idg_plan_params"""
    _fields_ = [("grid_size", ctypes.c_int32), ("subgrid_size", ctypes.c_int32),
                ("kernel_size", ctypes.c_int32), ("max_timesteps", ctypes.c_int32),
                ("max_channels", ctypes.c_int32), ("aterm_interval", ctypes.c_int32),
                ("flags", ctypes.c_int32), ("reserved", ctypes.c_int32),
                ("image_size", ctypes.c_double), ("w_step", ctypes.c_double)]


_lib = None


def lib() -> ctypes.CDLL:
    """The loaded C-ABI library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise IdgError("libidg_b200.so is missing: run `python -m paper_1909_07226_b200.build` "
                           "(needs nvcc); there is no CPU fallback")
        _lib = ctypes.CDLL(LIB_PATH)
        _lib.idg_strerror.restype = ctypes.c_char_p
        _lib.idg_kernel_launches.restype = ctypes.c_longlong
        _lib.idg_kernel_launches.argtypes = []
        _lib.idg_strerror.argtypes = [ctypes.c_int]
        _lib.idg_plan_destroy.restype = None
        _lib.idg_plan_destroy.argtypes = [ctypes.c_void_p]
        for name in EXPORTS:
            getattr(_lib, name)          # AttributeError if a declared symbol is not exported
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        l = lib()
        msg = l.idg_strerror(rc).decode()
        raise IdgError("%s failed: %s (status %d, cudaError %d)" % (what, msg, rc, l.idg_last_cuda_error()))


def _params(p) -> PlanParams:
    return PlanParams(int(p.grid_size), int(p.subgrid_size), int(p.kernel_size), int(p.max_timesteps),
                      int(p.max_channels), int(p.aterm_interval), int(p.flags), 0,
                      float(p.image_size), float(p.w_step))


def _dev(t: torch.Tensor, dtype, what: str) -> ctypes.c_void_p:
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise IdgError("%s must be a CUDA tensor" % what)
    if t.dtype != dtype or not t.is_contiguous():
        raise IdgError("%s must be contiguous %s" % (what, dtype))
    return ctypes.c_void_p(t.data_ptr())


def _host(a, dtype, what: str) -> Tuple[ctypes.c_void_p, object]:
    """Host pointer of a numpy array or CPU tensor (kept alive by the returned object)."""
    if isinstance(a, torch.Tensor):
        if a.is_cuda or not a.is_contiguous():
            raise IdgError("%s must be a contiguous host tensor" % what)
        return ctypes.c_void_p(a.data_ptr()), a
    arr = np.ascontiguousarray(a, dtype=dtype)
    return ctypes.c_void_p(arr.ctypes.data), arr


def _stream(stream) -> ctypes.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


class Plan:
    """Owner of an ``idg_plan*``."""

    def __init__(self, handle: ctypes.c_void_p, params, B: int, T: int, C: int, n_stations: int):
        self._h = handle
        self.params = params
        self.B, self.T, self.C, self.n_stations = B, T, C, n_stations

    @property
    def handle(self) -> ctypes.c_void_p:
        if not self._h:
            raise IdgError("plan was destroyed")
        return self._h

    def size(self) -> Tuple[int, int, int]:
        """(n_subgrids, n_planned_vis, n_skipped_vis)"""
        a, b, c = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        _check(lib().idg_plan_size(self.handle, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), "idg_plan_size")
        return int(a.value), int(b.value), int(c.value)

    def metadata(self) -> np.ndarray:
        P = self.size()[0]
        out = np.zeros(P, dtype=META_DTYPE)
        _check(lib().idg_plan_metadata(self.handle, ctypes.c_void_p(out.ctypes.data), ctypes.c_int64(P)),
               "idg_plan_metadata")
        return out

    def slots_needed(self) -> int:
        """Number of A-term slots the plan indexes (idg_plan_aterm_slots)."""
        n = ctypes.c_int32()
        _check(lib().idg_plan_aterm_slots(self.handle, ctypes.byref(n)), "idg_plan_aterm_slots")
        return int(n.value)

    def uses_tensor_cores(self) -> bool:
        """True if the gridder runs this plan on the tcgen05 path (idg_plan_uses_tensor_cores)."""
        f = ctypes.c_int32()
        _check(lib().idg_plan_uses_tensor_cores(self.handle, ctypes.byref(f)), "idg_plan_uses_tensor_cores")
        return bool(f.value & 1)

    def degridder_uses_tensor_cores(self) -> bool:
        """True if the degridder runs this plan on the tcgen05 path (bit 1 of idg_plan_uses_tensor_cores)."""
        f = ctypes.c_int32()
        _check(lib().idg_plan_uses_tensor_cores(self.handle, ctypes.byref(f)), "idg_plan_uses_tensor_cores")
        return bool(f.value & 2)

    def w_offset(self, w_index: int) -> float:
        """w0 of a w layer (idg_plan_w_offset; Alg. 1, R4)."""
        w0 = ctypes.c_double()
        _check(lib().idg_plan_w_offset(self.handle, ctypes.c_int32(int(w_index)), ctypes.byref(w0)), "idg_plan_w_offset")
        return float(w0.value)

    def subgrids(self) -> torch.Tensor:
        """The plan-owned [P][4][N][N] complex64 scratch as a tensor view (not owned by torch)."""
        P = self.size()[0]
        N = int(self.params.subgrid_size)
        ptr = ctypes.c_void_p()
        _check(lib().idg_plan_subgrids(self.handle, ctypes.byref(ptr)), "idg_plan_subgrids")
        if P == 0:
            return torch.empty((0, 4, N, N), dtype=torch.complex64, device="cuda")
        holder = _DevView(ptr.value, (P, 4, N, N, 2), self)
        return torch.view_as_complex(torch.as_tensor(holder, device="cuda"))

    def destroy(self) -> None:
        if self._h:
            lib().idg_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class _DevView:
    """__cuda_array_interface__ carrier for plan-owned float32 device memory."""

    def __init__(self, ptr: int, shape, owner):
        self._owner = owner
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": "<f4", "data": (int(ptr), False),
                                         "version": 2, "strides": None}


def idg_kernel_launches() -> int:
    """Kernels launched by the library in this process so far (host-side counter)."""
    return int(lib().idg_kernel_launches())


def idg_bench_instruction_mix(iters: int = 4096, variant: int = 0, stream=None) -> float:
    """TFLOP-equivalents/s of the bare gridder instruction mix on this device (csrc/mixbench.cu)."""
    out = ctypes.c_double()
    _check(lib().idg_bench_instruction_mix(ctypes.c_int32(int(iters)), ctypes.c_int32(int(variant)), ctypes.byref(out),
                                           _stream(stream)),
           "idg_bench_instruction_mix")
    return float(out.value)


def idg_bench_mma_rate(n: int = 16, ctas_per_sm: int = 1, n_mma: int = 8000, stream=None) -> float:
    """SM cycles per tcgen05.mma (kind::f16, M128 x N x K16, A in tensor memory) and SM (csrc/mmabench.cu)."""
    out = ctypes.c_double()
    _check(lib().idg_bench_mma_rate(ctypes.c_int32(int(n)), ctypes.c_int32(int(ctas_per_sm)), ctypes.c_int32(int(n_mma)),
                                    ctypes.byref(out), _stream(stream)), "idg_bench_mma_rate")
    return float(out.value)


def idg_plan_create(params, uvw: torch.Tensor, freqs, baselines, n_stations: int, stream=None) -> Plan:
    """Planner (a0): uvw is a CUDA float32 [B][T][3] tensor; freqs / baselines are host arrays."""
    prm = _params(params)
    B, T, three = uvw.shape
    assert three == 3
    fp, fk = _host(freqs, np.float64, "freqs")
    bp, bk = _host(np.asarray(baselines, dtype=np.int32), np.int32, "baselines")
    C = int(np.asarray(fk).shape[0])
    h = ctypes.c_void_p()
    rc = lib().idg_plan_create(ctypes.byref(h), ctypes.byref(prm), _dev(uvw, torch.float32, "uvw"), fp, bp,
                               ctypes.c_int32(B), ctypes.c_int32(T), ctypes.c_int32(C),
                               ctypes.c_int32(int(n_stations)), _stream(stream))
    _check(rc, "idg_plan_create")
    return Plan(h, params, int(B), int(T), C, int(n_stations))


def idg_plan_from_metadata(params, meta: np.ndarray, freqs, B: int, T: int, n_stations: int, stream=None) -> Plan:
    prm = _params(params)
    meta = np.ascontiguousarray(meta, dtype=META_DTYPE)
    fp, fk = _host(freqs, np.float64, "freqs")
    C = int(np.asarray(fk).shape[0])
    h = ctypes.c_void_p()
    rc = lib().idg_plan_from_metadata(ctypes.byref(h), ctypes.byref(prm), ctypes.c_void_p(meta.ctypes.data),
                                      ctypes.c_int64(len(meta)), fp, ctypes.c_int32(B), ctypes.c_int32(T),
                                      ctypes.c_int32(C), ctypes.c_int32(int(n_stations)), _stream(stream))
    _check(rc, "idg_plan_from_metadata")
    return Plan(h, params, int(B), int(T), C, int(n_stations))


def _shape_check(plan: Plan, uvw=None, vis=None, aterms=None, taper=None, grid=None, subgrids=None):
    N, L = int(plan.params.subgrid_size), int(plan.params.grid_size)
    if uvw is not None and tuple(uvw.shape) != (plan.B, plan.T, 3):
        raise IdgError("uvw shape %s != %s" % (tuple(uvw.shape), (plan.B, plan.T, 3)))
    if vis is not None and tuple(vis.shape) != (plan.B, plan.T, plan.C, 4):
        raise IdgError("vis shape %s != %s" % (tuple(vis.shape), (plan.B, plan.T, plan.C, 4)))
    if aterms is not None:
        s = tuple(aterms.shape)
        if len(s) != 5 or s[1:] != (plan.n_stations, N, N, 4):
            raise IdgError("aterms shape %s != [slots][%d][%d][%d][4]" % (s, plan.n_stations, N, N))
    if taper is not None and tuple(taper.shape) != (N, N):
        raise IdgError("taper shape %s != (%d, %d)" % (tuple(taper.shape), N, N))
    if grid is not None and tuple(grid.shape) != (4, L, L):
        raise IdgError("grid shape %s != (4, %d, %d)" % (tuple(grid.shape), L, L))
    if subgrids is not None and tuple(subgrids.shape) != (plan.size()[0], 4, N, N):
        raise IdgError("subgrids shape %s != (%d, 4, %d, %d)" % (tuple(subgrids.shape), plan.size()[0], N, N))


_C64, _F32 = torch.complex64, torch.float32


def idg_grid(plan: Plan, uvw, vis, aterms, taper, grid, stream=None) -> None:
    """Alg. 1: gridder -> subgrid FFT -> adder; accumulates into ``grid``."""
    _shape_check(plan, uvw=uvw, vis=vis, aterms=aterms, taper=taper, grid=grid)
    _check(lib().idg_grid(plan.handle, _dev(uvw, _F32, "uvw"), _dev(vis, _C64, "vis"),
                          _dev(aterms, _C64, "aterms"), ctypes.c_int32(int(aterms.shape[0])), _dev(taper, _F32, "taper"),
                          _dev(grid, _C64, "grid"), _stream(stream)), "idg_grid")


def idg_degrid(plan: Plan, uvw, grid, aterms, taper, vis_out, stream=None) -> None:
    """Alg. 2: splitter -> subgrid IFFT -> degridder; writes ``vis_out``."""
    _shape_check(plan, uvw=uvw, vis=vis_out, aterms=aterms, taper=taper, grid=grid)
    _check(lib().idg_degrid(plan.handle, _dev(uvw, _F32, "uvw"), _dev(grid, _C64, "grid"),
                            _dev(aterms, _C64, "aterms"), ctypes.c_int32(int(aterms.shape[0])), _dev(taper, _F32, "taper"),
                            _dev(vis_out, _C64, "vis_out"), _stream(stream)), "idg_degrid")


def idg_gridder(plan: Plan, uvw, vis, aterms, taper, subgrids, stream=None) -> None:
    _shape_check(plan, uvw=uvw, vis=vis, aterms=aterms, taper=taper, subgrids=subgrids)
    _check(lib().idg_gridder(plan.handle, _dev(uvw, _F32, "uvw"), _dev(vis, _C64, "vis"),
                             _dev(aterms, _C64, "aterms"), ctypes.c_int32(int(aterms.shape[0])), _dev(taper, _F32, "taper"),
                             _dev(subgrids, _C64, "subgrids"), _stream(stream)), "idg_gridder")


def idg_subgrid_fft(plan: Plan, subgrids, direction: int, stream=None) -> None:
    _shape_check(plan, subgrids=subgrids)
    _check(lib().idg_subgrid_fft(plan.handle, _dev(subgrids, _C64, "subgrids"), ctypes.c_int32(direction),
                                 _stream(stream)), "idg_subgrid_fft")


def idg_adder(plan: Plan, subgrids, grid, stream=None) -> None:
    _shape_check(plan, subgrids=subgrids, grid=grid)
    _check(lib().idg_adder(plan.handle, _dev(subgrids, _C64, "subgrids"), _dev(grid, _C64, "grid"),
                           _stream(stream)), "idg_adder")


def idg_splitter(plan: Plan, grid, subgrids, stream=None) -> None:
    _shape_check(plan, subgrids=subgrids, grid=grid)
    _check(lib().idg_splitter(plan.handle, _dev(grid, _C64, "grid"), _dev(subgrids, _C64, "subgrids"),
                              _stream(stream)), "idg_splitter")


def idg_splitter_ifft(plan: Plan, grid, subgrids, stream=None) -> None:
    """Rows a4 + a5 in one kernel: subgrids = IFFT of the grid windows."""
    _shape_check(plan, subgrids=subgrids, grid=grid)
    _check(lib().idg_splitter_ifft(plan.handle, _dev(grid, _C64, "grid"), _dev(subgrids, _C64, "subgrids"),
                              _stream(stream)), "idg_splitter_ifft")


def idg_degridder(plan: Plan, uvw, subgrids, aterms, taper, vis_out, stream=None) -> None:
    _shape_check(plan, uvw=uvw, vis=vis_out, aterms=aterms, taper=taper, subgrids=subgrids)
    _check(lib().idg_degridder(plan.handle, _dev(uvw, _F32, "uvw"), _dev(subgrids, _C64, "subgrids"),
                               _dev(aterms, _C64, "aterms"), ctypes.c_int32(int(aterms.shape[0])), _dev(taper, _F32, "taper"),
                               _dev(vis_out, _C64, "vis_out"), _stream(stream)), "idg_degridder")


def _host_c64(t, what):
    if isinstance(t, torch.Tensor):
        if t.dtype != _C64:
            raise IdgError("%s must be complex64" % what)
        return _host(t, None, what)
    return _host(t, np.complex64, what)


def idg_grid_host(plan: Plan, uvw, vis, aterms, taper, grid, stream=None) -> None:
    """idg_grid on HOST buffers (numpy arrays or CPU tensors, ideally pinned); grid is updated in place."""
    _shape_check(plan, uvw=uvw, vis=vis, aterms=aterms, taper=taper, grid=grid)
    up, k1 = _host(uvw, np.float32, "uvw"); vp, k2 = _host_c64(vis, "vis"); ap, k3 = _host_c64(aterms, "aterms")
    tp, k4 = _host(taper, np.float32, "taper"); gp, k5 = _host_c64(grid, "grid")
    if isinstance(grid, np.ndarray) and k5 is not grid:
        raise IdgError("grid must be a contiguous complex64 array (it is written in place)")
    _check(lib().idg_grid_host(plan.handle, up, vp, ap, ctypes.c_int32(int(aterms.shape[0])), tp, gp,
                               _stream(stream)), "idg_grid_host")


def idg_degrid_host(plan: Plan, uvw, grid, aterms, taper, vis_out, stream=None) -> None:
    _shape_check(plan, uvw=uvw, vis=vis_out, aterms=aterms, taper=taper, grid=grid)
    up, k1 = _host(uvw, np.float32, "uvw"); gp, k2 = _host_c64(grid, "grid"); ap, k3 = _host_c64(aterms, "aterms")
    tp, k4 = _host(taper, np.float32, "taper"); vp, k5 = _host_c64(vis_out, "vis_out")
    if isinstance(vis_out, np.ndarray) and k5 is not vis_out:
        raise IdgError("vis_out must be a contiguous complex64 array (it is written in place)")
    _check(lib().idg_degrid_host(plan.handle, up, gp, ap, ctypes.c_int32(int(aterms.shape[0])), tp, vp,
                                 _stream(stream)), "idg_degrid_host")


def idg_grid_degrid_host(plan: Plan, uvw, vis, aterms, taper, grid, vis_out, stream=None) -> None:
    """Alg. 1 then Alg. 2 on HOST buffers with the grid resident on the device; grid may be None (not copied back),
    otherwise it is overwritten with the grid of `vis`; vis_out receives the predicted visibilities."""
    _shape_check(plan, uvw=uvw, vis=vis, aterms=aterms, taper=taper)
    _shape_check(plan, vis=vis_out)
    up, k1 = _host(uvw, np.float32, "uvw"); vp, k2 = _host_c64(vis, "vis"); ap, k3 = _host_c64(aterms, "aterms")
    tp, k4 = _host(taper, np.float32, "taper"); op, k5 = _host_c64(vis_out, "vis_out")
    if isinstance(vis_out, np.ndarray) and k5 is not vis_out:
        raise IdgError("vis_out must be a contiguous complex64 array (it is written in place)")
    gp, k6 = None, None
    if grid is not None:
        _shape_check(plan, grid=grid)
        gp, k6 = _host_c64(grid, "grid")
        if isinstance(grid, np.ndarray) and k6 is not grid:
            raise IdgError("grid must be a contiguous complex64 array (it is written in place)")
    _check(lib().idg_grid_degrid_host(plan.handle, up, vp, ap, ctypes.c_int32(int(aterms.shape[0])), tp, gp, op,
                                      _stream(stream)), "idg_grid_degrid_host")


def idg_image_w_accumulate(acc, layer, image_size: float, w0: float, sign: int = 1, stream=None) -> None:
    """acc += layer * exp(sign 2 pi i w0 n'(l, m)); [4][L][L] complex64 device tensors (W-stacking)."""
    L = int(acc.shape[-1])
    if tuple(acc.shape) != (4, L, L) or tuple(layer.shape) != (4, L, L):
        raise IdgError("images must be [4][L][L]")
    _check(lib().idg_image_w_accumulate(_dev(acc, _C64, "acc"), _dev(layer, _C64, "layer"), ctypes.c_int32(L),
                                        ctypes.c_double(image_size), ctypes.c_double(w0), ctypes.c_int32(sign),
                                        _stream(stream)), "idg_image_w_accumulate")


def idg_image_w_apply(out, inp, image_size: float, w0: float, sign: int, stream=None) -> None:
    L = int(out.shape[-1])
    if tuple(out.shape) != (4, L, L) or tuple(inp.shape) != (4, L, L):
        raise IdgError("images must be [4][L][L]")
    _check(lib().idg_image_w_apply(_dev(out, _C64, "out"), _dev(inp, _C64, "in"), ctypes.c_int32(L),
                                   ctypes.c_double(image_size), ctypes.c_double(w0), ctypes.c_int32(sign),
                                   _stream(stream)), "idg_image_w_apply")


def idg_image_divide(image, cbar, stream=None) -> None:
    L = int(image.shape[-1])
    if tuple(image.shape) != (4, L, L) or tuple(cbar.shape) != (L, L):
        raise IdgError("image must be [4][L][L] and cbar [L][L]")
    _check(lib().idg_image_divide(_dev(image, _C64, "image"), _dev(cbar, _F32, "cbar"), ctypes.c_int32(L),
                                  _stream(stream)), "idg_image_divide")


def idg_image_taper(taper, L: int, stream=None) -> torch.Tensor:
    """c-bar [L][L] float32 from the [N][N] subgrid taper (idg_image_taper; section 4.2)."""
    N = int(taper.shape[0])
    if tuple(taper.shape) != (N, N):
        raise IdgError("taper must be [N][N]")
    out = torch.empty((int(L), int(L)), dtype=_F32, device=taper.device)
    _check(lib().idg_image_taper(_dev(taper, _F32, "taper"), ctypes.c_int32(N), _dev(out, _F32, "cbar"),
                                 ctypes.c_int32(int(L)), _stream(stream)), "idg_image_taper")
    return out


IMAGE_TAPER_STATIC_MAX_LN = 262144      # IDG_IMAGE_TAPER_STATIC_MAX_LN of include/idg_b200.h


def idg_image_taper_static(taper, cbar, stream=None) -> None:
    """idg_image_taper without any allocation: writes c-bar into the caller's [L][L] float32 device tensor; the scratch
    is a fixed 8 MiB device array of the library (L * N <= IMAGE_TAPER_STATIC_MAX_LN), shared by every call."""
    N, L = int(taper.shape[0]), int(cbar.shape[0])
    if tuple(taper.shape) != (N, N) or tuple(cbar.shape) != (L, L):
        raise IdgError("taper must be [N][N] and cbar [L][L]")
    _check(lib().idg_image_taper_static(_dev(taper, _F32, "taper"), ctypes.c_int32(N), _dev(cbar, _F32, "cbar"),
                                        ctypes.c_int32(L), _stream(stream)), "idg_image_taper_static")


def idg_taper_optimal(N: int, beta: float, device="cuda", stream=None):
    """Optimal IDG taper (NEXT-2, section 4.3 / Appendix A): -> (taper [N][N] float32 on `device`, a [N] float64
    numpy, epsilon)."""
    taper = torch.empty((int(N), int(N)), dtype=_F32, device=device)
    a = np.zeros(int(N), dtype=np.float64)
    eps = ctypes.c_double()
    _check(lib().idg_taper_optimal(ctypes.c_int32(int(N)), ctypes.c_double(float(beta)), _dev(taper, _F32, "taper"),
                                   ctypes.c_void_p(a.ctypes.data), ctypes.byref(eps), _stream(stream)),
           "idg_taper_optimal")
    return taper, a, float(eps.value)


def _scalar_check(plan: Plan, uvw, vis, gains, taper, grid=None, subgrids=None):
    N, L = int(plan.params.subgrid_size), int(plan.params.grid_size)
    if tuple(uvw.shape) != (plan.B, plan.T, 3) or tuple(vis.shape) != (plan.B, plan.T, plan.C):
        raise IdgError("scalar variant: uvw must be [B][T][3] and vis [B][T][C]")
    g = tuple(gains.shape)
    if len(g) != 4 or g[1:] != (plan.n_stations, N, N):
        raise IdgError("scalar variant: gains must be [slots][%d][%d][%d]" % (plan.n_stations, N, N))
    if tuple(taper.shape) != (N, N):
        raise IdgError("taper shape")
    if grid is not None and tuple(grid.shape) != (L, L):
        raise IdgError("scalar variant: grid must be [L][L]")
    if subgrids is not None and tuple(subgrids.shape) != (plan.size()[0], N, N):
        raise IdgError("scalar variant: subgrids must be [P][N][N]")


def idg_grid_scalar(plan: Plan, uvw, vis, gains, taper, grid, stream=None) -> None:
    """Scalar (one polarisation) Alg. 1; accumulates into grid [L][L] (NEXT-3)."""
    _scalar_check(plan, uvw, vis, gains, taper, grid=grid)
    _check(lib().idg_grid_scalar(plan.handle, _dev(uvw, _F32, "uvw"), _dev(vis, _C64, "vis"), _dev(gains, _C64, "gains"), ctypes.c_int32(int(gains.shape[0])),
                                 _dev(taper, _F32, "taper"), _dev(grid, _C64, "grid"), _stream(stream)), "idg_grid_scalar")


def idg_degrid_scalar(plan: Plan, uvw, grid, gains, taper, vis_out, stream=None) -> None:
    _scalar_check(plan, uvw, vis_out, gains, taper, grid=grid)
    _check(lib().idg_degrid_scalar(plan.handle, _dev(uvw, _F32, "uvw"), _dev(grid, _C64, "grid"), _dev(gains, _C64, "gains"), ctypes.c_int32(int(gains.shape[0])),
                                   _dev(taper, _F32, "taper"), _dev(vis_out, _C64, "vis_out"), _stream(stream)),
           "idg_degrid_scalar")


def idg_gridder_scalar(plan: Plan, uvw, vis, gains, taper, subgrids, stream=None) -> None:
    _scalar_check(plan, uvw, vis, gains, taper, subgrids=subgrids)
    _check(lib().idg_gridder_scalar(plan.handle, _dev(uvw, _F32, "uvw"), _dev(vis, _C64, "vis"), _dev(gains, _C64, "gains"), ctypes.c_int32(int(gains.shape[0])),
                                    _dev(taper, _F32, "taper"), _dev(subgrids, _C64, "subgrids"), _stream(stream)),
           "idg_gridder_scalar")


def idg_degridder_scalar(plan: Plan, uvw, subgrids, gains, taper, vis_out, stream=None) -> None:
    _scalar_check(plan, uvw, vis_out, gains, taper, subgrids=subgrids)
    _check(lib().idg_degridder_scalar(plan.handle, _dev(uvw, _F32, "uvw"), _dev(subgrids, _C64, "subgrids"),
                                      _dev(gains, _C64, "gains"), ctypes.c_int32(int(gains.shape[0])), _dev(taper, _F32, "taper"),
                                      _dev(vis_out, _C64, "vis_out"), _stream(stream)), "idg_degridder_scalar")
