"""Thin Python binding of the DM / integrator entry points of libpwfs.so (include/pwfs_dm.h).
Argument marshalling only; no CPU fallback."""
from __future__ import annotations

import ctypes as C

import numpy as np

from .chain import _Handle, _check
from .pwfs import load_library

EXPORTS = ("pwfs_dm_create", "pwfs_dm_apply", "pwfs_dm_destroy",
           "pwfs_int_create", "pwfs_int_step", "pwfs_int_reset", "pwfs_int_destroy")

_declared = False


def _lib():
    global _declared
    lib = load_library()
    if not _declared:
        vp, i32 = C.c_void_p, C.c_int32
        lib.pwfs_dm_create.argtypes = [i32, i32, i32, vp, vp, i32, C.POINTER(vp)]
        lib.pwfs_dm_apply.argtypes = [vp, vp, i32, vp, C.c_float, C.c_float, vp]
        lib.pwfs_int_create.argtypes = [i32, vp, i32, i32, C.POINTER(vp)]
        lib.pwfs_int_step.argtypes = [vp, vp, vp, vp]
        lib.pwfs_int_reset.argtypes = [vp, vp]
        for n in ("pwfs_dm_create", "pwfs_dm_apply", "pwfs_int_create", "pwfs_int_step", "pwfs_int_reset"):
            getattr(lib, n).restype = C.c_int
        for n in ("pwfs_dm_destroy", "pwfs_int_destroy"):
            getattr(lib, n).argtypes = [vp]
            getattr(lib, n).restype = None
        _declared = True
    return lib


class DeformableMirror(_Handle):
    """pwfs_dm_*: commands x influence functions -> phase layer, scaled and added to a phase batch."""
    _destroy = "pwfs_dm_destroy"

    def __init__(self, ifs, pix, n_pupil: int, device: int = 0):
        self._h, self._lib = None, _lib()
        ifs = np.ascontiguousarray(ifs, dtype=np.float32)
        pix = np.ascontiguousarray(pix, dtype=np.int32)
        if ifs.ndim != 2 or pix.shape != (ifs.shape[1],):
            raise ValueError("ifs must be [n_act][n_pix] and pix [n_pix]")
        self.n_act, self.n_pix, self.n_pupil, self.device = ifs.shape[0], ifs.shape[1], int(n_pupil), device
        h = C.c_void_p()
        _check(self._lib.pwfs_dm_create(self.n_act, self.n_pupil, self.n_pix, C.c_void_p(pix.ctypes.data),
                                        C.c_void_p(ifs.ctypes.data), device, C.byref(h)), "pwfs_dm_create")
        self._h = h

    def apply(self, cmd, phase=None, alpha: float = 1.0, beta: float = 0.0, stream=None):
        """phase = beta * phase + alpha * layer(cmd), in place on `phase` ([B,N,N]; allocated when None and beta = 0)."""
        cmd = self._in(cmd, (self.n_act,), "cmd")
        N = self.n_pupil
        if phase is None and beta != 0.0:
            raise ValueError("beta != 0 needs a phase batch to add to")
        phase = self._out(phase, (cmd.shape[0], N, N))
        _check(self._lib.pwfs_dm_apply(self._h, C.c_void_p(cmd.data_ptr()), cmd.shape[0], C.c_void_p(phase.data_ptr()),
                                       float(alpha), float(beta), self._stream(stream)), "pwfs_dm_apply")
        return phase


class Integrator(_Handle):
    """pwfs_int_*: c_t = c_{t-1} + gain * delta_t, output delayed by `delay` frames."""
    _destroy = "pwfs_int_destroy"

    def __init__(self, gain, delay: int = 0, device: int = 0):
        self._h, self._lib = None, _lib()
        g = np.ascontiguousarray(gain, dtype=np.float32).ravel()
        self.n_modes, self.delay, self.device = g.size, int(delay), device
        h = C.c_void_p()
        _check(self._lib.pwfs_int_create(g.size, C.c_void_p(g.ctypes.data), int(delay), device, C.byref(h)), "pwfs_int_create")
        self._h = h

    def step(self, delta, out=None, stream=None):
        import torch
        if not (isinstance(delta, torch.Tensor) and delta.is_cuda and delta.dtype == torch.float32
                and delta.is_contiguous() and delta.numel() == self.n_modes):
            raise ValueError(f"delta must be a contiguous CUDA float32 tensor of {self.n_modes} numbers")
        out = self._out(out, (self.n_modes,)) if out is None or out.dim() == 1 else self._out(out, (1, self.n_modes))
        _check(self._lib.pwfs_int_step(self._h, C.c_void_p(delta.data_ptr()), C.c_void_p(out.data_ptr()),
                                       self._stream(stream)), "pwfs_int_step")
        return out

    def reset(self, stream=None):
        _check(self._lib.pwfs_int_reset(self._h, self._stream(stream)), "pwfs_int_reset")
