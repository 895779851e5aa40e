"""Thin Python binding of the f1 entry points of libpwfs.so (include/pwfs_atmo.h):
propagation through phase screens.  Argument marshalling only; no CPU fallback."""
from __future__ import annotations

import ctypes as C

import numpy as np

from .pwfs import PWFS_OK, PwfsError, load_library, strerror

EXPORTS = ("pwfs_atmo_create", "pwfs_atmo_frames_per_step", "pwfs_atmo_propagate", "pwfs_atmo_destroy")


class pwfs_atmo_params(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("screen_px", C.c_int32), ("screens", C.POINTER(C.c_float)),
                ("pitch", C.c_double), ("wind_vxy", C.POINTER(C.c_double)), ("heights", C.POINTER(C.c_double)),
                ("n_dirs", C.c_int32), ("dirs_tan", C.POINTER(C.c_double)), ("n_wl", C.c_int32),
                ("wl_scale", C.POINTER(C.c_double)), ("n_pupil", C.c_int32), ("device", C.c_int32)]


_declared = False


def _lib():
    global _declared
    lib = load_library()
    if not _declared:
        vp = C.c_void_p
        lib.pwfs_atmo_create.argtypes = [C.POINTER(pwfs_atmo_params), C.POINTER(vp)]
        lib.pwfs_atmo_create.restype = C.c_int
        lib.pwfs_atmo_frames_per_step.argtypes = [vp, C.POINTER(C.c_int32)]
        lib.pwfs_atmo_frames_per_step.restype = C.c_int
        lib.pwfs_atmo_propagate.argtypes = [vp, C.c_int64, C.c_int32, C.c_double, vp, vp]
        lib.pwfs_atmo_propagate.restype = C.c_int
        lib.pwfs_atmo_destroy.argtypes = [vp]
        lib.pwfs_atmo_destroy.restype = None
        _declared = True
    return lib


class Atmosphere:
    """Frozen-flow layers resident on one GPU: pwfs_atmo_create / _propagate / _destroy."""

    def __init__(self, screens, pitch, wind_vxy, heights, dirs_tan, wl_scale, n_pupil, device: int = 0, **_ignored):
        self._h = None
        self._lib = _lib()
        scr = np.ascontiguousarray(screens, dtype=np.float32)
        if scr.ndim != 3 or scr.shape[1] != scr.shape[2]:
            raise ValueError("screens must be [L][G][G]")
        f64 = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        wind, hts, dirs, wls = f64(wind_vxy), f64(heights), f64(dirs_tan), f64(wl_scale)
        if wind.shape != (scr.shape[0], 2) or hts.shape != (scr.shape[0],) or dirs.ndim != 2 or dirs.shape[1] != 2:
            raise ValueError("wind_vxy [L][2], heights [L], dirs_tan [S][2] expected")
        dp = C.POINTER(C.c_double)
        prm = pwfs_atmo_params(scr.shape[0], scr.shape[1], scr.ctypes.data_as(C.POINTER(C.c_float)), float(pitch),
                               wind.ctypes.data_as(dp), hts.ctypes.data_as(dp), dirs.shape[0],
                               dirs.ctypes.data_as(dp), wls.size, wls.ctypes.data_as(dp), int(n_pupil), device)
        h = C.c_void_p()
        rc = self._lib.pwfs_atmo_create(C.byref(prm), C.byref(h))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_atmo_create", strerror(rc))
        self._h = h
        self.device, self.n_pupil = device, int(n_pupil)
        self.frames_per_step = dirs.shape[0] * wls.size

    def close(self):
        if getattr(self, "_h", None):
            self._lib.pwfs_atmo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def propagate(self, first_step: int, n_steps: int, dt: float, out=None, stream=None):
        """-> CUDA float32 tensor [n_steps * frames_per_step, N, N], asynchronous on `stream`."""
        import torch
        N, B = self.n_pupil, n_steps * self.frames_per_step
        dev = torch.device("cuda", self.device)
        if out is None:
            out = torch.empty((B, N, N), dtype=torch.float32, device=dev)
        if not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.numel() == B * N * N):
            raise ValueError(f"out must be a contiguous CUDA float32 tensor of {B}x{N}x{N}")
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        rc = self._lib.pwfs_atmo_propagate(self._h, int(first_step), int(n_steps), float(dt),
                                           C.c_void_p(out.data_ptr()), C.c_void_p(st.cuda_stream))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_atmo_propagate", strerror(rc))
        return out
