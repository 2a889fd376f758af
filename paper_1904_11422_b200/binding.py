"""ctypes binding of libepic.so (include/epic.h).  Argument marshalling only: every step of the
EPIC path (unpack, gridding, transform, products, accumulation) runs in the
library's CUDA kernels.  PyTorch is used for device memory and streams.  There is no CPU
fallback: a missing library raises."""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libepic.so")

EPIC_OK = 0
EPIC_ERR_ARG, EPIC_ERR_RANGE, EPIC_ERR_CUDA, EPIC_ERR_NOMEM, EPIC_ERR_SCRATCH = -1, -2, -3, -4, -5
EPIC_PATH_AUTO, EPIC_PATH_TWOPASS, EPIC_PATH_FUSED, EPIC_PATH_TILED, EPIC_PATH_TENSOR, EPIC_PATH_STREAM = 0, 1, 2, 3, 4, 5
EPIC_ORDER_TCPA, EPIC_ORDER_TCAP = 0, 1

# every symbol include/epic.h declares: name -> (restype, argtypes)
_vp, _i, _l = ctypes.c_void_p, ctypes.c_int, ctypes.c_long
SYMBOLS = {
    "epic_plan_create": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _vp, _vp, _i]),
    "epic_plan_create_per_channel": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _i, _vp, _vp, _i]),
    "epic_plan_get_n_layouts": (_i, [_vp]),
    "epic_plan_destroy": (_i, [_vp]),
    "epic_plan_set_products": (_i, [_vp, _i]),
    "epic_plan_set_path": (_i, [_vp, _i]),
    "epic_plan_set_scratch_limit": (_i, [_vp, ctypes.c_longlong]),
    "epic_plan_set_input_order": (_i, [_vp, _i]),
    "epic_plan_set_delay_phasors": (_i, [_vp, _i, _i, _vp]),
    "epic_image": (_i, [_vp, _vp, _i, _i, _i, _vp, _vp]),
    "epic_image_cf32": (_i, [_vp, _vp, _i, _i, _i, _vp, _vp]),
    "epic_image_host": (_i, [_vp, _vp, _i, _i, _i, _vp, _i, _i]),
    "epic_image_noalloc": (_i, [_vp, _vp, _i, _i, _i, _vp, _vp]),
    "epic_noalloc_scratch_bytes": (ctypes.c_longlong, []),
    "epic_autocorr_remove": (_i, [_vp, _vp, _i, _i, _i, _vp, _vp]),
    "epic_plan_get_n": (_i, [_vp]),
    "epic_plan_get_n_planes": (_i, [_vp, _i]),
    "epic_plan_get_cells": (_i, [_vp, _vp]),
    "epic_plan_get_support": (_i, [_vp, _vp]),
    "epic_plan_get_path": (_i, [_vp, _i]),
    "epic_plan_last_launches": (_i, [_vp]),
    "epic_debug_unpack": (_i, [_vp, _l, _vp, _vp]),
    "epic_debug_grid": (_i, [_vp, _vp, _i, _i, _vp, _vp]),
    "epic_debug_grid_layout": (_i, [_vp, _i, _vp, _i, _i, _vp, _vp]),
    "epic_fp32_peak_probe": (_i, [_i, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_double)]),
    "epic_status_string": (ctypes.c_char_p, [_i]),
    "epic_last_cuda_error": (_i, []),
}

_lib = None


class EpicError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().epic_status_string(status).decode()
        if status == EPIC_ERR_CUDA:
            msg += f" (cudaError {lib().epic_last_cuda_error()})"
        super().__init__(f"{where}: {msg}")


def lib() -> ctypes.CDLL:
    """The loaded libepic.so.  Raises if it has not been built (python -m paper_1904_11422_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1904_11422_b200.build` "
                "(there is no CPU fallback)")
        handle = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(handle, name)
            fn.restype = res
            fn.argtypes = args
        _lib = handle
    return _lib


def _check(status: int, where: str) -> int:
    if status < 0:
        raise EpicError(status, where)
    return status


def _ptr(x) -> int:
    """Device/host address of a torch tensor, numpy array or raw integer."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    raise TypeError(type(x))


def _check_tensor(x, what: str, dtype_name: str, min_numel: int, device_index: Optional[int]) -> None:
    """Shape/placement checks for a torch tensor handed to a DEVICE-pointer argument (raw integer
    addresses are the caller's responsibility, as in C): CUDA, contiguous, the dtype the ABI reads,
    at least the elements the call will touch, on the plan's device."""
    if x is None or isinstance(x, int) or not hasattr(x, "data_ptr"):
        return
    if not getattr(x, "is_cuda", False):
        raise ValueError(f"{what}: expected a CUDA tensor (DEVICE pointer)")
    if not x.is_contiguous():
        raise ValueError(f"{what}: tensor must be contiguous")
    if str(x.dtype) != f"torch.{dtype_name}":
        raise ValueError(f"{what}: dtype {x.dtype}, expected torch.{dtype_name}")
    if x.numel() < min_numel:
        raise ValueError(f"{what}: {x.numel()} elements, the call needs {min_numel}")
    if device_index is not None and x.device.index is not None and x.device.index != device_index:
        raise ValueError(f"{what}: on cuda:{x.device.index}, the plan lives on cuda:{device_index}")


def _current_device() -> Optional[int]:
    try:
        import torch
        return torch.cuda.current_device() if torch.cuda.is_available() else None
    except Exception:
        return None


def _stream(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


class Plan:
    """Owns an epic_plan* (include/epic.h).  ant_uv float32 [A][2] in cell units, kernel_taps
    float32 [A][K][K][2] or None for the delta kernel; both HOST arrays, copied by the library."""

    def __init__(self, grid_n: int, pad: int, ant_uv: np.ndarray,
                 kernel_taps: Optional[np.ndarray] = None, kernel_k: int = 1):
        uv = np.ascontiguousarray(ant_uv, dtype=np.float32)
        if uv.ndim not in (2, 3) or uv.shape[-1] != 2:
            raise ValueError("ant_uv must be [n_ant][2], or [n_chan][n_ant][2] for one layout per channel")
        per_channel = uv.ndim == 3
        taps = None
        if kernel_taps is not None:
            taps = np.ascontiguousarray(kernel_taps, dtype=np.float32)
            if taps.shape != uv.shape[:-1] + (kernel_k, kernel_k, 2):
                raise ValueError(f"kernel_taps shape {taps.shape}")
        self._h = _vp()
        self.n_ant = int(uv.shape[-2])
        self.kernel_k = int(kernel_k)
        if per_channel:  # epic_plan_create_per_channel: channel c of every call uses ant_uv[c], kernel_taps[c]
            _check(lib().epic_plan_create_per_channel(ctypes.byref(self._h), grid_n, pad, self.n_ant, int(uv.shape[0]),
                                                      _ptr(uv), _ptr(taps), kernel_k), "epic_plan_create_per_channel")
        else:
            _check(lib().epic_plan_create(ctypes.byref(self._h), grid_n, pad, self.n_ant,
                                          _ptr(uv), _ptr(taps), kernel_k), "epic_plan_create")
        self.N = lib().epic_plan_get_n(self._h)
        self.device_index = _current_device()   # the plan's tables live on the device current at creation
        self.n_layouts = _check(lib().epic_plan_get_n_layouts(self._h), "epic_plan_get_n_layouts")

    # -- lifetime
    def destroy(self) -> None:
        if self._h:
            h, self._h = self._h, _vp()
            _check(lib().epic_plan_destroy(h), "epic_plan_destroy")

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    # -- configuration / queries
    def set_products(self, n_products: int) -> None:
        _check(lib().epic_plan_set_products(self._h, n_products), "epic_plan_set_products")

    def set_input_order(self, order: int) -> None:
        """EPIC_ORDER_TCPA (default) or EPIC_ORDER_TCAP: voltages in [T][C][A][Np] order."""
        _check(lib().epic_plan_set_input_order(self._h, int(order)), "epic_plan_set_input_order")

    def set_delay_phasors(self, phasors: Optional[np.ndarray]) -> None:
        """HOST complex multipliers [n_chan][n_pol][n_ant] (complex64, or float32 [...][2]); None clears."""
        if phasors is None:
            _check(lib().epic_plan_set_delay_phasors(self._h, 0, 0, 0), "epic_plan_set_delay_phasors")
            return
        ph = np.asarray(phasors)
        if np.iscomplexobj(ph):
            ph = np.stack([ph.real, ph.imag], axis=-1)
        ph = np.ascontiguousarray(ph, dtype=np.float32)
        if ph.ndim != 4 or ph.shape[2] != self.n_ant or ph.shape[3] != 2:
            raise ValueError(f"phasors shape {ph.shape}")
        _check(lib().epic_plan_set_delay_phasors(self._h, ph.shape[0], ph.shape[1], _ptr(ph)),
               "epic_plan_set_delay_phasors")

    def set_scratch_limit(self, n_bytes: int):
        _check(lib().epic_plan_set_scratch_limit(self._h, int(n_bytes)), "epic_plan_set_scratch_limit")

    def set_path(self, path: int) -> None:
        _check(lib().epic_plan_set_path(self._h, path), "epic_plan_set_path")

    def n_planes(self, n_pol: int) -> int:
        return _check(lib().epic_plan_get_n_planes(self._h, n_pol), "epic_plan_get_n_planes")

    def path(self, n_pol: int) -> int:
        return _check(lib().epic_plan_get_path(self._h, n_pol), "epic_plan_get_path")

    def last_launches(self) -> int:
        return _check(lib().epic_plan_last_launches(self._h), "epic_plan_last_launches")

    def cells(self) -> np.ndarray:
        """int32 [n_ant][K][K] ([n_layouts][n_ant][K][K] for a per-channel plan): y*N + x of every tap."""
        out = np.empty((self.n_layouts, self.n_ant, self.kernel_k, self.kernel_k), dtype=np.int32)
        _check(lib().epic_plan_get_cells(self._h, _ptr(out)), "epic_plan_get_cells")
        return out if self.n_layouts > 1 else out[0]

    def support(self) -> tuple:
        out = np.empty(4, dtype=np.int32)
        _check(lib().epic_plan_get_support(self._h, _ptr(out)), "epic_plan_get_support")
        return tuple(int(v) for v in out)

    # -- device work
    def _check_call(self, voltages, vdtype: str, per_sample: int, n_t: int, n_chan: int, n_pol: int, out_accum) -> None:
        if n_t <= 0 or n_chan <= 0 or n_pol not in (1, 2):
            return  # empty calls are no-ops; bad n_pol is the library's error to report
        _check_tensor(voltages, "voltages", vdtype, n_t * n_chan * n_pol * self.n_ant * per_sample, self.device_index)
        planes = lib().epic_plan_get_n_planes(self._h, n_pol)
        if planes > 0:
            _check_tensor(out_accum, "out_accum", "float32", n_chan * planes * self.N * self.N, self.device_index)

    def image(self, voltages, n_t: int, n_chan: int, n_pol: int, out_accum, stream=None) -> None:
        """epic_image: voltages DEVICE uint8 [T][C][Np][A]; ADDS into out_accum DEVICE float32
        [C][planes][N][N]."""
        self._check_call(voltages, "uint8", 1, n_t, n_chan, n_pol, out_accum)
        _check(lib().epic_image(self._h, _ptr(voltages), n_t, n_chan, n_pol, _ptr(out_accum),
                                _stream(stream)), "epic_image")

    def image_noalloc(self, voltages, n_t: int, n_chan: int, n_pol: int, out_accum, stream=None) -> None:
        """epic_image_noalloc: epic_image for callers that must not allocate -- the fused kernel with its scratch in
        the library's static 80 MiB device array (one-layout plans with N = 64 / 128 and a 32 x 32 support); calls that
        overlap on the GPU race on that array."""
        self._check_call(voltages, "uint8", 1, n_t, n_chan, n_pol, out_accum)
        _check(lib().epic_image_noalloc(self._h, _ptr(voltages), n_t, n_chan, n_pol, _ptr(out_accum),
                                        _stream(stream)), "epic_image_noalloc")

    def image_host(self, voltages_host, n_t: int, n_chan: int, n_pol: int, out_accum_host, accumulate: bool = True,
                   n_chunks: int = 0) -> None:
        """epic_image_host: the same gulp from HOST memory (numpy arrays or CPU torch tensors, pinned or not): the
        library pipelines the host->device copies with the kernels and copies the images back; synchronous."""
        for x, what, dt, need in ((voltages_host, "voltages_host", "uint8", n_t * n_chan * n_pol * self.n_ant),
                                  (out_accum_host, "out_accum_host", "float32",
                                   n_chan * max(lib().epic_plan_get_n_planes(self._h, n_pol), 0) * self.N * self.N)):
            if isinstance(x, np.ndarray):
                if x.dtype != np.dtype(dt) or not x.flags["C_CONTIGUOUS"] or x.size < need:
                    raise ValueError(f"{what}: need a C-contiguous {dt} array of at least {need} elements")
            elif hasattr(x, "data_ptr"):
                if getattr(x, "is_cuda", False) or not x.is_contiguous() or str(x.dtype) != f"torch.{dt}" or x.numel() < need:
                    raise ValueError(f"{what}: need a contiguous CPU {dt} tensor of at least {need} elements")
            elif x is not None and not isinstance(x, int):
                raise TypeError(type(x))
        _check(lib().epic_image_host(self._h, _ptr(voltages_host), n_t, n_chan, n_pol, _ptr(out_accum_host),
                                     int(bool(accumulate)), int(n_chunks)), "epic_image_host")

    def image_cf32(self, voltages, n_t: int, n_chan: int, n_pol: int, out_accum, stream=None) -> None:
        """epic_image_cf32: voltages DEVICE float32 [T][C][Np][A][2]."""
        self._check_call(voltages, "float32", 2, n_t, n_chan, n_pol, out_accum)
        _check(lib().epic_image_cf32(self._h, _ptr(voltages), n_t, n_chan, n_pol, _ptr(out_accum),
                                     _stream(stream)), "epic_image_cf32")

    def autocorr_remove(self, voltages, n_t: int, n_chan: int, n_pol: int, out_accum, stream=None) -> None:
        """epic_autocorr_remove: subtract the a = b (zero-spacing) part of the same gulp."""
        self._check_call(voltages, "uint8", 1, n_t, n_chan, n_pol, out_accum)
        _check(lib().epic_autocorr_remove(self._h, _ptr(voltages), n_t, n_chan, n_pol, _ptr(out_accum),
                                          _stream(stream)), "epic_autocorr_remove")

    def debug_grid(self, voltages, is_cf32: bool, n_pol: int, out_plane, stream=None, layout: int = 0) -> None:
        if n_pol in (1, 2):
            _check_tensor(voltages, "voltages", "float32" if is_cf32 else "uint8",
                          n_pol * self.n_ant * (2 if is_cf32 else 1), self.device_index)
            _check_tensor(out_plane, "out_plane", "float32", n_pol * self.N * self.N * 2, self.device_index)
        _check(lib().epic_debug_grid_layout(self._h, int(layout), _ptr(voltages), int(bool(is_cf32)), n_pol,
                                            _ptr(out_plane), _stream(stream)), "epic_debug_grid_layout")


# free functions with the names of include/epic.h
def epic_plan_create(grid_n, pad, n_ant, ant_uv, kernel_taps, kernel_k=1) -> Plan:
    uv = np.asarray(ant_uv, dtype=np.float32).reshape(n_ant, 2)
    return Plan(grid_n, pad, uv, kernel_taps, kernel_k)


def epic_plan_create_per_channel(grid_n, pad, n_ant, n_layout, ant_uv, kernel_taps, kernel_k=1) -> Plan:
    uv = np.asarray(ant_uv, dtype=np.float32).reshape(n_layout, n_ant, 2)
    return Plan(grid_n, pad, uv, kernel_taps, kernel_k)


def epic_plan_destroy(plan: Optional[Plan]) -> None:
    if plan is not None:
        plan.destroy()


def epic_image(plan: Plan, voltages, n_t, n_chan, n_pol, out_accum, stream=None) -> None:
    plan.image(voltages, n_t, n_chan, n_pol, out_accum, stream)


def epic_image_noalloc(plan: Plan, voltages, n_t, n_chan, n_pol, out_accum, stream=None) -> None:
    plan.image_noalloc(voltages, n_t, n_chan, n_pol, out_accum, stream)


def epic_noalloc_scratch_bytes() -> int:
    return int(lib().epic_noalloc_scratch_bytes())


def epic_image_host(plan: Plan, voltages_host, n_t, n_chan, n_pol, out_accum_host, accumulate=True, n_chunks=0) -> None:
    plan.image_host(voltages_host, n_t, n_chan, n_pol, out_accum_host, accumulate, n_chunks)


def epic_image_cf32(plan: Plan, voltages, n_t, n_chan, n_pol, out_accum, stream=None) -> None:
    plan.image_cf32(voltages, n_t, n_chan, n_pol, out_accum, stream)


def epic_autocorr_remove(plan: Plan, voltages, n_t, n_chan, n_pol, out_accum, stream=None) -> None:
    plan.autocorr_remove(voltages, n_t, n_chan, n_pol, out_accum, stream)


def epic_debug_unpack(bytes_dev, n: int, out_dev, stream=None) -> None:
    _check(lib().epic_debug_unpack(_ptr(bytes_dev), n, _ptr(out_dev), _stream(stream)), "epic_debug_unpack")


def epic_fp32_peak_probe(iters: int = 4096) -> dict:
    """Measured FP32 FMA rate of the device (roofline denominator): {"ms", "flops", "tflops"}."""
    ms = ctypes.c_float()
    fl = ctypes.c_double()
    _check(lib().epic_fp32_peak_probe(iters, ctypes.byref(ms), ctypes.byref(fl)), "epic_fp32_peak_probe")
    return {"ms": ms.value, "flops": fl.value, "tflops": fl.value / (ms.value * 1e-3) / 1e12}
