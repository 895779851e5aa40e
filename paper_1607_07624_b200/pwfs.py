"""Thin Python binding of libpwfs.so (include/pwfs.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is
used for device memory and streams.  There is no CPU fallback: if the library
has not been built (python -m paper_1607_07624_b200.build) or no CUDA device is
present, construction raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("PWFS_LIB_PATH") or os.path.join(_HERE, "libpwfs.so")

PWFS_OK, PWFS_EINVAL, PWFS_ENOMEM, PWFS_ECUDA, PWFS_EUNSUPPORTED, PWFS_ELIMIT = 0, -1, -2, -3, -4, -5
NOALLOC_MAX_FRAMES, NOALLOC_MAX_PART_FLOATS = 64, 1 << 20     # PWFS_NOALLOC_* of include/pwfs.h
NUM_KERNEL_CLASSES = 5
KERNEL_CLASSES = ("xpass", "ypass", "xrebin", "slopes", "fused")

EXPORTS = ("pwfs_create", "pwfs_create_ex", "pwfs_info", "pwfs_valid_mask", "pwfs_run", "pwfs_run_host",
           "pwfs_destroy", "pwfs_strerror", "pwfs_last_cuda_error", "pwfs_supported_grid",
           "pwfs_set_schedule", "pwfs_set_timing", "pwfs_get_timing", "pwfs_geometry", "pwfs_reserve",
           "pwfs_last_failed_kernel", "pwfs_debug_create", "pwfs_debug_intensity",
           "pwfs_run_noalloc")


class pwfs_params(C.Structure):
    _fields_ = [("n_pupil", C.c_int32), ("m_grid", C.c_int32), ("pupil_amp", C.POINTER(C.c_float)),
                ("mask_shift_px", C.c_int32), ("mod_radius", C.c_float), ("mod_points", C.c_int32),
                ("mod_angle0", C.c_float), ("n_subap", C.c_int32), ("illum_thresh", C.c_float),
                ("slope_norm", C.c_int32), ("device", C.c_int32)]


class pwfs_ext(C.Structure):
    _fields_ = [("n_tilts", C.c_int32), ("tilt_x", C.POINTER(C.c_float)), ("tilt_y", C.POINTER(C.c_float)),
                ("tilt_w", C.POINTER(C.c_float)), ("field_stop_px", C.c_float)]


class PwfsError(RuntimeError):
    def __init__(self, code: int, what: str, detail: str = ""):
        self.code = code
        super().__init__(f"{what}: {detail or code}")


_lib = None


def load_library() -> C.CDLL:
    """dlopen libpwfs.so and declare every prototype of include/pwfs.h."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} is missing: build it with `python -m paper_1607_07624_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32 = C.c_void_p, C.c_int32
    lib.pwfs_create.argtypes = [C.POINTER(pwfs_params), C.POINTER(vp)]
    lib.pwfs_create.restype = C.c_int
    lib.pwfs_create_ex.argtypes = [C.POINTER(pwfs_params), C.POINTER(pwfs_ext), C.POINTER(vp)]
    lib.pwfs_create_ex.restype = C.c_int
    lib.pwfs_info.argtypes = [vp, C.POINTER(i32), C.POINTER(i32)]
    lib.pwfs_info.restype = C.c_int
    lib.pwfs_valid_mask.argtypes = [vp, vp]
    lib.pwfs_valid_mask.restype = C.c_int
    lib.pwfs_run.argtypes = [vp, vp, i32, vp, vp, vp]
    lib.pwfs_run.restype = C.c_int
    lib.pwfs_run_noalloc.argtypes = [vp, vp, i32, vp, vp, vp]
    lib.pwfs_run_noalloc.restype = C.c_int
    lib.pwfs_run_host.argtypes = [vp, vp, i32, vp, vp]
    lib.pwfs_run_host.restype = C.c_int
    lib.pwfs_destroy.argtypes = [vp]
    lib.pwfs_destroy.restype = None
    lib.pwfs_strerror.argtypes = [C.c_int]
    lib.pwfs_strerror.restype = C.c_char_p
    lib.pwfs_last_cuda_error.argtypes = [vp]
    lib.pwfs_last_cuda_error.restype = C.c_int
    lib.pwfs_reserve.argtypes = [vp, i32]
    lib.pwfs_reserve.restype = C.c_int
    lib.pwfs_last_failed_kernel.argtypes = [vp]
    lib.pwfs_last_failed_kernel.restype = C.c_int
    lib.pwfs_debug_create.argtypes = [C.POINTER(pwfs_params), C.POINTER(pwfs_ext), i32, C.POINTER(vp)]
    lib.pwfs_debug_create.restype = C.c_int
    lib.pwfs_debug_intensity.argtypes = [vp, vp, i32, vp, vp]
    lib.pwfs_debug_intensity.restype = C.c_int
    lib.pwfs_supported_grid.argtypes = [i32]
    lib.pwfs_supported_grid.restype = C.c_int
    lib.pwfs_set_schedule.argtypes = [vp, i32, i32]
    lib.pwfs_set_schedule.restype = C.c_int
    lib.pwfs_set_timing.argtypes = [vp, i32]
    lib.pwfs_set_timing.restype = C.c_int
    lib.pwfs_get_timing.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_int64)]
    lib.pwfs_get_timing.restype = C.c_int
    lib.pwfs_geometry.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]
    lib.pwfs_geometry.restype = C.c_int
    _lib = lib
    return lib


def strerror(code: int) -> str:
    return load_library().pwfs_strerror(code).decode()


def supported_grid(m_grid: int) -> bool:
    return bool(load_library().pwfs_supported_grid(m_grid))


class PWFS:
    """One pyramid sensor on one GPU: pwfs_create / pwfs_run / pwfs_destroy."""

    def __init__(self, pupil_amp: np.ndarray, m_grid: int, mod_radius: float, mod_points: int,
                 n_subap: int, mask_shift_px: int = 0, mod_angle0: float = 0.0,
                 illum_thresh: float = 0.5, slope_norm: int = 0, device: int = 0,
                 tilt_list=None, field_stop_px: float = -1.0, debug_shift_px: Optional[int] = None):
        """tilt_list = (x, y[, w]) arrays in lambda/D replaces the modulation circle;
        field_stop_px >= 0 adds the square focal-plane stop (include/pwfs.h, pwfs_ext).
        debug_shift_px (tests only): pwfs_debug_create with this mask shift, window checks off."""
        self._h = None
        self._lib = load_library()
        amp = np.ascontiguousarray(pupil_amp, dtype=np.float32)
        if amp.ndim != 2 or amp.shape[0] != amp.shape[1]:
            raise ValueError("pupil_amp must be a square 2-D array")
        prm = pwfs_params(amp.shape[0], m_grid, amp.ctypes.data_as(C.POINTER(C.c_float)),
                          mask_shift_px, mod_radius, mod_points, mod_angle0, n_subap, illum_thresh,
                          slope_norm, device)
        h = C.c_void_p()
        if debug_shift_px is not None and tilt_list is None:
            ext = pwfs_ext(0, None, None, None, field_stop_px)
            rc = self._lib.pwfs_debug_create(C.byref(prm), C.byref(ext), int(debug_shift_px), C.byref(h))
        elif tilt_list is None and field_stop_px < 0:
            rc = self._lib.pwfs_create(C.byref(prm), C.byref(h))
        else:
            fp = C.POINTER(C.c_float)
            ext = pwfs_ext(0, None, None, None, field_stop_px)
            if tilt_list is not None:
                tl = [np.ascontiguousarray(a, dtype=np.float32).ravel() for a in tilt_list]
                if len(tl) not in (2, 3) or any(a.size != tl[0].size for a in tl):
                    raise ValueError("tilt_list must be (x, y) or (x, y, w) arrays of one length")
                ext.n_tilts = tl[0].size
                ext.tilt_x, ext.tilt_y = tl[0].ctypes.data_as(fp), tl[1].ctypes.data_as(fp)
                ext.tilt_w = tl[2].ctypes.data_as(fp) if len(tl) == 3 else None
                mod_points = tl[0].size
            rc = self._lib.pwfs_create_ex(C.byref(prm), C.byref(ext), C.byref(h))
        if rc != PWFS_OK:
            raise PwfsError(rc, "pwfs_create", strerror(rc))
        self._h = h
        self.device = device
        self.n_pupil = amp.shape[0]
        self.m_grid = m_grid
        self.mod_points = mod_points
        det, nv = C.c_int32(), C.c_int32()
        self._check(self._lib.pwfs_info(self._h, C.byref(det), C.byref(nv)), "pwfs_info")
        self.det_size, self.n_valid = det.value, nv.value

    # -- plumbing ---------------------------------------------------------
    def _check(self, rc: int, what: str):
        if rc != PWFS_OK:
            detail = strerror(rc)
            if rc == PWFS_ECUDA and self._h:
                detail += f" (cudaError {self._lib.pwfs_last_cuda_error(self._h)})"
            raise PwfsError(rc, what, detail)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.pwfs_destroy(self._h)
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

    # -- queries ----------------------------------------------------------
    def valid_mask(self) -> np.ndarray:
        ns = self.det_size // 2
        out = np.empty((ns, ns), dtype=np.uint8)
        self._check(self._lib.pwfs_valid_mask(self._h, out.ctypes.data_as(C.c_void_p)), "pwfs_valid_mask")
        return out

    def geometry(self, batch: int) -> dict:
        a, b, c, d = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32()
        self._check(self._lib.pwfs_geometry(self._h, batch, C.byref(a), C.byref(b), C.byref(c), C.byref(d)),
                    "pwfs_geometry")
        return dict(n_cols=a.value, k_unique=b.value, frames_per_chunk=c.value, k_split=d.value)

    def set_schedule(self, frames_per_chunk: int = 0, k_split: int = 0):
        self._check(self._lib.pwfs_set_schedule(self._h, frames_per_chunk, k_split), "pwfs_set_schedule")

    def set_timing(self, enable: bool):
        self._check(self._lib.pwfs_set_timing(self._h, int(enable)), "pwfs_set_timing")

    def get_timing(self) -> Tuple[dict, dict]:
        ms = (C.c_float * NUM_KERNEL_CLASSES)()
        n = (C.c_int64 * NUM_KERNEL_CLASSES)()
        self._check(self._lib.pwfs_get_timing(self._h, ms, n), "pwfs_get_timing")
        return ({k: float(ms[i]) for i, k in enumerate(KERNEL_CLASSES)},
                {k: int(n[i]) for i, k in enumerate(KERNEL_CLASSES)})

    # -- the hot path -----------------------------------------------------
    def _dev_out(self, t, shape, what):
        """A caller-supplied output: exactly `shape`, float32, contiguous, on this sensor's device."""
        import torch
        if not isinstance(t, torch.Tensor):
            raise TypeError(f"{what} must be a torch tensor")
        if not t.is_cuda or t.device.index != self.device:
            raise ValueError(f"{what} must live on cuda:{self.device}")
        if t.dtype != torch.float32:
            raise TypeError(f"{what} must be float32, got {t.dtype}")
        if tuple(t.shape) != tuple(shape) or not t.is_contiguous():
            raise ValueError(f"{what} must be a contiguous tensor of shape {tuple(shape)}, got {tuple(t.shape)}")
        return t

    def debug_intensity(self, phase):
        """Tests only: full-resolution I[B,M,M] = mean_k |E_k|^2 from the hot path's own row and column kernels
        (pwfs_debug_intensity), in the placement of the definition."""
        import torch
        if phase.dim() == 2:
            phase = phase.unsqueeze(0)
        phase = phase.contiguous()
        B, N, M = phase.shape[0], self.n_pupil, self.m_grid
        if not (phase.is_cuda and phase.dtype == torch.float32 and tuple(phase.shape[1:]) == (N, N)):
            raise ValueError(f"phase must be a CUDA float32 tensor [B,{N},{N}]")
        out = torch.empty((B, M, M), dtype=torch.float32, device=phase.device)
        st = torch.cuda.current_stream(phase.device)
        self._check(self._lib.pwfs_debug_intensity(self._h, C.c_void_p(phase.data_ptr()), B, C.c_void_p(out.data_ptr()),
                                                   C.c_void_p(st.cuda_stream)), "pwfs_debug_intensity")
        return out

    def reserve(self, batch: int):
        """Size scratch for batches of up to `batch` frames (needed before capturing run() in a CUDA graph)."""
        self._check(self._lib.pwfs_reserve(self._h, int(batch)), "pwfs_reserve")

    def run(self, phase, frames=None, slopes=None, want_slopes: bool = True, stream=None):
        """phase: CUDA float32 tensor [B,N,N] (or [N,N]).  Returns (frames, slopes)
        CUDA tensors [B,2n_sub,2n_sub], [B,2 n_valid]; asynchronous on `stream`
        (default: torch's current stream)."""
        import torch
        if not (isinstance(phase, torch.Tensor) and phase.is_cuda and phase.dtype == torch.float32):
            raise TypeError("phase must be a CUDA float32 tensor")
        if phase.device.index != self.device:
            raise ValueError("phase lives on another device than the sensor")
        if phase.dim() == 2:
            phase = phase.unsqueeze(0)
        B, N = phase.shape[0], self.n_pupil
        if phase.dim() != 3 or tuple(phase.shape[1:]) != (N, N):
            raise ValueError(f"phase must be [B,{N},{N}]")
        st = stream if stream is not None else torch.cuda.current_stream(phase.device)
        if not phase.is_contiguous():
            with torch.cuda.stream(st):              # the copy is made, used and freed in stream order on `st`
                phase = phase.contiguous()
        D = self.det_size
        if frames is None:
            frames = torch.empty((B, D, D), dtype=torch.float32, device=phase.device)
        else:
            self._dev_out(frames, (B, D, D), "frames")
        if slopes is None:
            if want_slopes:
                slopes = torch.empty((B, 2 * self.n_valid), dtype=torch.float32, device=phase.device)
        else:
            self._dev_out(slopes, (B, 2 * self.n_valid), "slopes")
        rc = self._lib.pwfs_run(self._h, C.c_void_p(phase.data_ptr()), B, C.c_void_p(frames.data_ptr()),
                                C.c_void_p(slopes.data_ptr()) if slopes is not None else None,
                                C.c_void_p(st.cuda_stream))
        self._check(rc, "pwfs_run")
        if stream is not None:                       # buffers allocated on torch's current stream, used on another one
            for t in (phase, frames, slopes):
                if t is not None:
                    t.record_stream(st)
        return frames, slopes

    def run_noalloc(self, phase, frames, slopes=None, stream=None):
        """pwfs_run_noalloc: run() for callers that may not allocate device memory -- a control loop that cannot
        afford cudaMalloc's device-wide stall, or a process whose GPU memory belongs to another allocator.  The
        kernel's working memory is a fixed array inside libpwfs.so instead of heap scratch, so nothing is allocated
        here either: `phase` [B,N,N] must already be contiguous and `frames` [B,2n_sub,2n_sub] (and `slopes`
        [B,2 n_valid], optional) must be passed in; nothing is returned.  M = 128 sensors only, B <= 64 and
        B * K * det_size^2 <= 2^20 (PwfsError PWFS_EUNSUPPORTED / PWFS_ELIMIT otherwise).  One array per GPU is shared
        by all sensors: calls that could run at the same time on one GPU must be serialised by the caller.  Make the
        first call on each GPU at start-up (it looks the array up)."""
        import torch
        N, D = self.n_pupil, self.det_size
        if not (isinstance(phase, torch.Tensor) and phase.is_cuda and phase.dtype == torch.float32):
            raise TypeError("phase must be a CUDA float32 tensor")
        if phase.device.index != self.device:
            raise ValueError("phase lives on another device than the sensor")
        if phase.dim() != 3 or tuple(phase.shape[1:]) != (N, N) or not phase.is_contiguous():
            raise ValueError(f"phase must be a contiguous [B,{N},{N}] tensor (a copy would allocate)")
        B = phase.shape[0]
        self._dev_out(frames, (B, D, D), "frames")
        if slopes is not None:
            self._dev_out(slopes, (B, 2 * self.n_valid), "slopes")
        st = stream if stream is not None else torch.cuda.current_stream(phase.device)
        rc = self._lib.pwfs_run_noalloc(self._h, C.c_void_p(phase.data_ptr()), B, C.c_void_p(frames.data_ptr()),
                                        C.c_void_p(slopes.data_ptr()) if slopes is not None else None,
                                        C.c_void_p(st.cuda_stream))
        self._check(rc, "pwfs_run_noalloc")

    @staticmethod
    def _host_buf(a, shape, what):
        """Pointer of a HOST float32 C-contiguous buffer (numpy array or CPU torch tensor) of exactly `shape`."""
        if isinstance(a, np.ndarray):
            if a.dtype != np.float32:
                raise TypeError(f"{what} must be float32, got {a.dtype}")
            if not a.flags.c_contiguous or tuple(a.shape) != tuple(shape):
                raise ValueError(f"{what} must be a C-contiguous array of shape {tuple(shape)}, got {a.shape}")
            return a.ctypes.data
        import torch
        if not isinstance(a, torch.Tensor):
            raise TypeError(f"{what} must be a numpy array or a CPU torch tensor")
        if a.is_cuda:
            raise ValueError(f"{what} must be host memory (use run() for device tensors)")
        if a.dtype != torch.float32:
            raise TypeError(f"{what} must be float32, got {a.dtype}")
        if not a.is_contiguous() or tuple(a.shape) != tuple(shape):
            raise ValueError(f"{what} must be a contiguous tensor of shape {tuple(shape)}, got {tuple(a.shape)}")
        return a.data_ptr()

    def run_host(self, phase, frames=None, slopes=None, want_slopes: bool = True):
        """Same with HOST buffers (numpy arrays or CPU torch tensors, float32,
        ideally pinned): host->device, run, device->host inside the call."""
        N, D = self.n_pupil, self.det_size
        shp = tuple(phase.shape)
        if len(shp) == 2:
            shp = (1,) + shp
        if len(shp) != 3 or shp[1:] != (N, N):
            raise ValueError(f"phase must be [B,{N},{N}], got {tuple(phase.shape)}")
        B = shp[0]
        p = self._host_buf(phase, tuple(phase.shape), "phase")
        if frames is None:
            frames = np.empty((B, D, D), dtype=np.float32)
        if slopes is None and want_slopes:
            slopes = np.empty((B, 2 * self.n_valid), dtype=np.float32)
        fp = self._host_buf(frames, (B, D, D), "frames")
        sp = self._host_buf(slopes, (B, 2 * self.n_valid), "slopes") if slopes is not None else None
        rc = self._lib.pwfs_run_host(self._h, C.c_void_p(p), B, C.c_void_p(fp),
                                     C.c_void_p(sp) if sp is not None else None)
        self._check(rc, "pwfs_run_host")
        return frames, slopes


def from_config(cfg, device: int = 0, **overrides) -> PWFS:
    """Build the sensor of a workloads.WfsConfig."""
    from . import workloads
    kw = dict(pupil_amp=workloads.make_pupil(cfg), m_grid=cfg.m_grid, mod_radius=cfg.mod_radius,
              mod_points=cfg.mod_points, n_subap=cfg.n_subap, device=device)
    kw.update(overrides)
    return PWFS(**kw)
