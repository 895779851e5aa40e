"""Thin Python binding of the f2 entry points of libpwfs.so (include/pwfs_chain.h):
CCD detector, slope computer with reference vector, modal reconstructor.
Argument marshalling only; no CPU fallback."""
from __future__ import annotations

import ctypes as C

import numpy as np

from .pwfs import PWFS_OK, PwfsError, load_library, strerror

EXPORTS = ("pwfs_ccd_create", "pwfs_ccd_run", "pwfs_ccd_destroy",
           "pwfs_slopec_create", "pwfs_slopec_set_reference", "pwfs_slopec_n_slopes", "pwfs_slopec_run",
           "pwfs_slopec_destroy", "pwfs_rec_create", "pwfs_rec_run", "pwfs_rec_reserve", "pwfs_rec_destroy")


class pwfs_ccd_params(C.Structure):
    _fields_ = [("det_size", C.c_int32), ("n_inst", C.c_int32), ("n_int", C.c_int32), ("gain", C.c_double),
                ("quantum_eff", C.c_double), ("photon_noise", C.c_int32), ("readout_noise", C.c_int32),
                ("readout_level", C.c_double), ("seed", C.c_uint64), ("device", C.c_int32)]


_declared = False


def _lib():
    global _declared
    lib = load_library()
    if not _declared:
        vp, i32 = C.c_void_p, C.c_int32
        lib.pwfs_ccd_create.argtypes = [C.POINTER(pwfs_ccd_params), C.POINTER(vp)]
        lib.pwfs_ccd_run.argtypes = [vp, vp, i32, C.c_int64, vp, vp]
        lib.pwfs_slopec_create.argtypes = [i32, vp, i32, vp, i32, C.POINTER(vp)]
        lib.pwfs_slopec_set_reference.argtypes = [vp, vp]
        lib.pwfs_slopec_n_slopes.argtypes = [vp, C.POINTER(i32)]
        lib.pwfs_slopec_run.argtypes = [vp, vp, i32, vp, vp]
        lib.pwfs_rec_create.argtypes = [i32, i32, vp, i32, C.POINTER(vp)]
        lib.pwfs_rec_run.argtypes = [vp, vp, i32, vp, vp]
        lib.pwfs_rec_reserve.argtypes = [vp, i32]
        for n in ("pwfs_ccd_create", "pwfs_ccd_run", "pwfs_slopec_create", "pwfs_slopec_set_reference",
                  "pwfs_slopec_n_slopes", "pwfs_slopec_run", "pwfs_rec_create", "pwfs_rec_run", "pwfs_rec_reserve"):
            getattr(lib, n).restype = C.c_int
        for n in ("pwfs_ccd_destroy", "pwfs_slopec_destroy", "pwfs_rec_destroy"):
            getattr(lib, n).argtypes = [vp]
            getattr(lib, n).restype = None
        _declared = True
    return lib


def _check(rc, what):
    if rc != PWFS_OK:
        raise PwfsError(rc, what, strerror(rc))


class _Handle:
    _destroy = ""

    def close(self):
        if getattr(self, "_h", None):
            getattr(self._lib, self._destroy)(self._h)
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

    def _out(self, out, shape):
        import torch
        if out is None:
            return torch.empty(shape, dtype=torch.float32, device=torch.device("cuda", self.device))
        if not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and tuple(out.shape) == tuple(shape)):
            raise ValueError(f"out must be a contiguous CUDA float32 tensor of shape {tuple(shape)}")
        return out

    @staticmethod
    def _in(x, shape_tail, what):
        import torch
        if not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous() and tuple(x.shape[1:]) == tuple(shape_tail)):
            raise ValueError(f"{what} must be a contiguous CUDA float32 tensor [B]{list(shape_tail)}")
        return x


class CCD(_Handle):
    """pwfs_ccd_create / _run / _destroy: intensity frames -> detector pixels [e-]."""
    _destroy = "pwfs_ccd_destroy"

    def __init__(self, det_size, n_inst=1, n_int=1, gain=1.0, quantum_eff=1.0, photon_noise=False,
                 readout_noise=False, readout_level=0.0, seed=0, device: int = 0):
        self._h, self._lib = None, _lib()
        prm = pwfs_ccd_params(int(det_size), int(n_inst), int(n_int), float(gain), float(quantum_eff),
                              int(bool(photon_noise)), int(bool(readout_noise)), float(readout_level),
                              int(seed) & 0xFFFFFFFFFFFFFFFF, device)
        h = C.c_void_p()
        _check(self._lib.pwfs_ccd_create(C.byref(prm), C.byref(h)), "pwfs_ccd_create")
        self._h, self.device = h, device
        self.det_size, self.n_inst, self.n_int = int(det_size), int(n_inst), int(n_int)

    def run(self, frames, first_out_frame: int = 0, out=None, stream=None):
        D = self.det_size
        frames = self._in(frames, (D, D), "frames")
        B = frames.shape[0]
        if B % self.n_inst:
            raise ValueError("frame count must be a multiple of n_inst")
        n_steps = B // self.n_inst
        out = self._out(out, (n_steps // self.n_int * self.n_inst, D, D))
        _check(self._lib.pwfs_ccd_run(self._h, C.c_void_p(frames.data_ptr()), n_steps, int(first_out_frame),
                                      C.c_void_p(out.data_ptr()), self._stream(stream)), "pwfs_ccd_run")
        return out


class SlopeComputer(_Handle):
    """pwfs_slopec_*: detector pixels -> slopes minus the reference vector."""
    _destroy = "pwfs_slopec_destroy"

    def __init__(self, valid_mask, slope_norm: int = 0, sn=None, device: int = 0):
        self._h, self._lib = None, _lib()
        v = np.ascontiguousarray(valid_mask, dtype=np.uint8)
        if v.ndim != 2 or v.shape[0] != v.shape[1]:
            raise ValueError("valid_mask must be [n_sub][n_sub]")
        self.n_sub, self.n_slopes, self.device = v.shape[0], 2 * int(np.count_nonzero(v)), device
        sn_arr = None if sn is None else self._sn(sn)
        h = C.c_void_p()
        _check(self._lib.pwfs_slopec_create(v.shape[0], C.c_void_p(v.ctypes.data), int(slope_norm),
                                            None if sn_arr is None else C.c_void_p(sn_arr.ctypes.data),
                                            device, C.byref(h)), "pwfs_slopec_create")
        self._h = h

    def _sn(self, sn):
        a = np.ascontiguousarray(sn, dtype=np.float32)
        if a.shape != (self.n_slopes,):
            raise ValueError(f"sn must hold {self.n_slopes} numbers")
        return a

    def set_reference(self, sn):
        a = None if sn is None else self._sn(sn)
        _check(self._lib.pwfs_slopec_set_reference(self._h, None if a is None else C.c_void_p(a.ctypes.data)),
               "pwfs_slopec_set_reference")

    def run(self, pixels, out=None, stream=None):
        D = 2 * self.n_sub
        pixels = self._in(pixels, (D, D), "pixels")
        out = self._out(out, (pixels.shape[0], self.n_slopes))
        _check(self._lib.pwfs_slopec_run(self._h, C.c_void_p(pixels.data_ptr()), pixels.shape[0],
                                         C.c_void_p(out.data_ptr()), self._stream(stream)), "pwfs_slopec_run")
        return out


class Reconstructor(_Handle):
    """pwfs_rec_*: slopes -> modes = recmat @ slopes."""
    _destroy = "pwfs_rec_destroy"

    def __init__(self, recmat, device: int = 0):
        self._h, self._lib = None, _lib()
        R = np.ascontiguousarray(recmat, dtype=np.float32)
        if R.ndim != 2:
            raise ValueError("recmat must be [n_modes][n_slopes]")
        self.n_modes, self.n_slopes, self.device = R.shape[0], R.shape[1], device
        h = C.c_void_p()
        _check(self._lib.pwfs_rec_create(R.shape[0], R.shape[1], C.c_void_p(R.ctypes.data), device, C.byref(h)),
               "pwfs_rec_create")
        self._h = h

    def reserve(self, batch: int):
        """Size the batched (tensor-core) path's scratch so that run() neither allocates nor synchronises."""
        _check(self._lib.pwfs_rec_reserve(self._h, int(batch)), "pwfs_rec_reserve")

    def run(self, slopes, out=None, stream=None):
        slopes = self._in(slopes, (self.n_slopes,), "slopes")
        out = self._out(out, (slopes.shape[0], self.n_modes))
        _check(self._lib.pwfs_rec_run(self._h, C.c_void_p(slopes.data_ptr()), slopes.shape[0],
                                      C.c_void_p(out.data_ptr()), self._stream(stream)), "pwfs_rec_run")
        return out
