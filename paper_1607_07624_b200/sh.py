"""Thin Python binding of the f4 Shack-Hartmann entry points of libpwfs.so (include/pwfs_sh.h).
Argument marshalling only; no CPU fallback."""
from __future__ import annotations

import ctypes as C

import numpy as np

from .pwfs import PWFS_OK, PwfsError, load_library, strerror

EXPORTS = ("pwfs_sh_create", "pwfs_sh_info", "pwfs_sh_valid_mask", "pwfs_sh_run", "pwfs_sh_destroy")


class pwfs_sh_params(C.Structure):
    _fields_ = [("n_pupil", C.c_int32), ("n_subap", C.c_int32), ("pupil_amp", C.POINTER(C.c_float)),
                ("fft_px", C.c_int32), ("n_px", C.c_int32), ("bin", C.c_int32), ("illum_thresh", C.c_float),
                ("phase_scale", C.c_float), ("device", C.c_int32)]


_declared = False


def _lib():
    global _declared
    lib = load_library()
    if not _declared:
        vp, i32 = C.c_void_p, C.c_int32
        lib.pwfs_sh_create.argtypes = [C.POINTER(pwfs_sh_params), C.POINTER(vp)]
        lib.pwfs_sh_info.argtypes = [vp, C.POINTER(i32), C.POINTER(i32)]
        lib.pwfs_sh_valid_mask.argtypes = [vp, vp]
        lib.pwfs_sh_run.argtypes = [vp, vp, i32, vp, vp, vp]
        for n in ("pwfs_sh_create", "pwfs_sh_info", "pwfs_sh_valid_mask", "pwfs_sh_run"):
            getattr(lib, n).restype = C.c_int
        lib.pwfs_sh_destroy.argtypes = [vp]
        lib.pwfs_sh_destroy.restype = None
        _declared = True
    return lib


class ShackHartmann:
    """pwfs_sh_create / _run / _destroy: wavefronts -> spot frames and centre-of-gravity slopes."""

    def __init__(self, pupil_amp, n_subap: int, fft_px: int, n_px: int, bin: int = 1, illum_thresh: float = 0.5,
                 phase_scale: float = 1.0, device: int = 0):
        self._h, self._lib = None, _lib()
        A = np.ascontiguousarray(pupil_amp, dtype=np.float32)
        if A.ndim != 2 or A.shape[0] != A.shape[1]:
            raise ValueError("pupil_amp must be [N][N]")
        prm = pwfs_sh_params(A.shape[0], int(n_subap), A.ctypes.data_as(C.POINTER(C.c_float)), int(fft_px), int(n_px),
                             int(bin), float(illum_thresh), float(phase_scale), device)
        h = C.c_void_p()
        rc = self._lib.pwfs_sh_create(C.byref(prm), C.byref(h))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_sh_create", strerror(rc))
        self._h, self.device, self.n_pupil, self.n_subap = h, device, A.shape[0], int(n_subap)
        d, nv = C.c_int32(), C.c_int32()
        self._lib.pwfs_sh_info(h, C.byref(d), C.byref(nv))
        self.det_size, self.n_valid = d.value, nv.value

    def close(self):
        if getattr(self, "_h", None):
            self._lib.pwfs_sh_destroy(self._h)
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

    def valid_mask(self) -> np.ndarray:
        m = np.empty((self.n_subap, self.n_subap), dtype=np.uint8)
        rc = self._lib.pwfs_sh_valid_mask(self._h, C.c_void_p(m.ctypes.data))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_sh_valid_mask", strerror(rc))
        return m

    def run(self, phase, want_slopes: bool = True, stream=None):
        """phase: CUDA float32 [B, N, N] -> (frames [B, D, D], slopes [B, 2 n_valid] or None)."""
        import torch
        N, D = self.n_pupil, self.det_size
        if not (phase.is_cuda and phase.dtype == torch.float32 and phase.is_contiguous() and tuple(phase.shape[1:]) == (N, N)):
            raise ValueError(f"phase must be a contiguous CUDA float32 tensor [B, {N}, {N}]")
        B = phase.shape[0]
        frames = torch.empty((B, D, D), dtype=torch.float32, device=phase.device)
        slopes = torch.empty((B, 2 * self.n_valid), dtype=torch.float32, device=phase.device) if want_slopes else None
        st = stream if stream is not None else torch.cuda.current_stream(phase.device)
        rc = self._lib.pwfs_sh_run(self._h, C.c_void_p(phase.data_ptr()), B, C.c_void_p(frames.data_ptr()),
                                   C.c_void_p(slopes.data_ptr()) if want_slopes else None, C.c_void_p(st.cuda_stream))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_sh_run", strerror(rc))
        return frames, slopes
