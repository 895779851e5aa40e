"""Thin Python binding of the f4 PSF-camera entry points of libpwfs.so (include/pwfs_psf.h).
Argument marshalling only; no CPU fallback."""
from __future__ import annotations

import ctypes as C

import numpy as np

from .pwfs import PWFS_OK, PwfsError, load_library, strerror

EXPORTS = ("pwfs_psf_create", "pwfs_psf_accumulate", "pwfs_psf_read", "pwfs_psf_reset", "pwfs_psf_destroy")


class pwfs_psf_params(C.Structure):
    _fields_ = [("n_pupil", C.c_int32), ("m_grid", C.c_int32), ("pupil_amp", C.POINTER(C.c_float)),
                ("phase_scale", C.c_float), ("device", C.c_int32)]


_declared = False


def _lib():
    global _declared
    lib = load_library()
    if not _declared:
        vp = C.c_void_p
        lib.pwfs_psf_create.argtypes = [C.POINTER(pwfs_psf_params), C.POINTER(vp)]
        lib.pwfs_psf_accumulate.argtypes = [vp, vp, C.c_int32, vp, vp]
        lib.pwfs_psf_read.argtypes = [vp, vp, C.POINTER(C.c_int64), vp]
        lib.pwfs_psf_reset.argtypes = [vp, vp]
        for n in ("pwfs_psf_create", "pwfs_psf_accumulate", "pwfs_psf_read", "pwfs_psf_reset"):
            getattr(lib, n).restype = C.c_int
        lib.pwfs_psf_destroy.argtypes = [vp]
        lib.pwfs_psf_destroy.restype = None
        _declared = True
    return lib


class PsfCamera:
    """pwfs_psf_create / _accumulate / _read / _reset / _destroy."""

    def __init__(self, pupil_amp, m_grid: int, phase_scale: float = 1.0, device: int = 0):
        self._h, self._lib = None, _lib()
        A = np.ascontiguousarray(pupil_amp, dtype=np.float32)
        if A.ndim != 2 or A.shape[0] != A.shape[1]:
            raise ValueError("pupil_amp must be [N][N]")
        prm = pwfs_psf_params(A.shape[0], int(m_grid), A.ctypes.data_as(C.POINTER(C.c_float)), float(phase_scale), device)
        h = C.c_void_p()
        rc = self._lib.pwfs_psf_create(C.byref(prm), C.byref(h))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_psf_create", strerror(rc))
        self._h, self.device, self.n_pupil, self.m_grid = h, device, A.shape[0], int(m_grid)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.pwfs_psf_destroy(self._h)
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

    def _stream(self, stream):
        import torch
        st = stream if stream is not None else torch.cuda.current_stream(torch.device("cuda", self.device))
        return C.c_void_p(st.cuda_stream)

    def accumulate(self, phase, want_sr: bool = True, stream=None):
        """Add the frames of `phase` (CUDA float32 [B, N, N]) to the long exposure; -> Strehl ratios [B]."""
        import torch
        N = self.n_pupil
        if not (phase.is_cuda and phase.dtype == torch.float32 and phase.is_contiguous() and tuple(phase.shape[1:]) == (N, N)):
            raise ValueError(f"phase must be a contiguous CUDA float32 tensor [B, {N}, {N}]")
        B = phase.shape[0]
        sr = torch.empty(B, dtype=torch.float32, device=phase.device) if want_sr else None
        rc = self._lib.pwfs_psf_accumulate(self._h, C.c_void_p(phase.data_ptr()), B,
                                           C.c_void_p(sr.data_ptr()) if (want_sr and B) else None, self._stream(stream))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_psf_accumulate", strerror(rc))
        return sr

    def read(self, out=None, stream=None):
        """-> (long-exposure PSF, CUDA float32 [M, M], zero frequency at [M/2, M/2]; frames accumulated)."""
        import torch
        M = self.m_grid
        if out is None:
            out = torch.empty((M, M), dtype=torch.float32, device=torch.device("cuda", self.device))
        if not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and tuple(out.shape) == (M, M)):
            raise ValueError(f"out must be a contiguous CUDA float32 tensor [{M}, {M}]")
        n = C.c_int64()
        rc = self._lib.pwfs_psf_read(self._h, C.c_void_p(out.data_ptr()), C.byref(n), self._stream(stream))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_psf_read", strerror(rc))
        return out, n.value

    def reset(self, stream=None):
        rc = self._lib.pwfs_psf_reset(self._h, self._stream(stream))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_psf_reset", strerror(rc))
