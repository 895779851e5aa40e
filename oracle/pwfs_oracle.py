"""ctypes front-end of the CPU ORACLE (oracle/pwfs_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this module; the
product package paper_1607_07624_b200 never does (it fails loudly when its CUDA
library is missing instead of falling back here).  This module holds argument
marshalling only -- every number comes from the C file, whose functions cite
the passage they follow (SURVEY.md 8(c) O0..O9 / BASELINE.json north_star /
PAPER.md:L19, L119-136, L261-262, L317-318, L342).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pwfs_oracle.c")
_LIB = os.path.join(_HERE, "libpwfs_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (double precision, OpenMP).  -O2, no
    fast-math: the oracle is never tuned.

    PWFS_ORACLE_SANITIZE=1 builds and loads a second library, libpwfs_oracle_san.so,
    with -fsanitize=address,undefined (host-side sanitizer pass
    over the oracle pins).  Python is not an ASan binary, so the runtime must be
    preloaded:
        LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
        PWFS_ORACLE_SANITIZE=1 python -m pytest tests -m "not gpu" -k oracle
    Same source, same arithmetic; only the instrumentation differs."""
    san = os.environ.get("PWFS_ORACLE_SANITIZE") == "1"
    lib = _LIB.replace(".so", "_san.so") if san else _LIB
    with _lock:
        if (not force and os.path.exists(lib)
                and os.path.getmtime(lib) >= os.path.getmtime(_SRC)):
            return lib
        tmp = lib + f".tmp{os.getpid()}"
        opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
               "-fno-sanitize-recover=undefined"] if san else ["-O2"]
        cmd = ["gcc"] + opt + ["-std=c11", "-fopenmp", "-fPIC", "-shared",
                               "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, lib)
        return lib


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        i, d, p = C.c_int, C.c_double, C.c_void_p
        lib.orc_num_threads.restype = i
        lib.orc_dft_naive.argtypes = [i, p, p, i]
        lib.orc_dft_naive.restype = None
        lib.orc_fft.argtypes = [i, p, p, i]
        lib.orc_fft.restype = i
        lib.orc_fft2.argtypes = [i, p, i, i]
        lib.orc_fft2.restype = i
        lib.orc_mod_offsets.argtypes = [i, d, d, p, p]
        lib.orc_mod_offsets.restype = None
        lib.orc_phasor.argtypes = [i, p, p, d, d, p]
        lib.orc_phasor.restype = None
        lib.orc_embed.argtypes = [i, i, p, p]
        lib.orc_embed.restype = None
        lib.orc_pyramid_mask.argtypes = [i, d, p]
        lib.orc_pyramid_mask.restype = None
        lib.orc_field.argtypes = [i, i, p, p, d, d, p, p, p, i]
        lib.orc_field.restype = i
        lib.orc_intensity.argtypes = [i, i, p, p, i, d, d, p, p, i]
        lib.orc_intensity.restype = i
        lib.orc_rebin_weights.argtypes = [i, i, p]
        lib.orc_rebin_weights.restype = None
        lib.orc_frame.argtypes = [i, i, i, i, p, p]
        lib.orc_frame.restype = i
        lib.orc_valid_mask.argtypes = [i, i, p, d, p]
        lib.orc_valid_mask.restype = i
        lib.orc_slopes.argtypes = [i, p, p, i, p]
        lib.orc_slopes.restype = i
        lib.orc_pwfs_run.argtypes = [i, i, p, i, d, i, d, i, d, i, i, p, p, p]
        lib.orc_pwfs_run.restype = i
        lib.orc_field_stop.argtypes = [i, d, p]
        lib.orc_field_stop.restype = None
        lib.orc_intensity_list.argtypes = [i, i, p, p, i, p, p, p, p, p, i]
        lib.orc_intensity_list.restype = i
        lib.orc_pwfs_run_list.argtypes = [i, i, p, i, i, p, p, p, d, i, d, i, i, p, p, p]
        lib.orc_pwfs_run_list.restype = i
        _lib = lib
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _check(rc, what):
    if rc < 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")
    return rc


def num_threads() -> int:
    return int(_load().orc_num_threads())


def dft_naive(x, sign=-1):
    x = _c128(x)
    out = np.empty_like(x)
    _load().orc_dft_naive(x.size, _ptr(x), _ptr(out), sign)
    return out


def fft(x, sign=-1):
    x = _c128(x)
    out = np.empty_like(x)
    _check(_load().orc_fft(x.size, _ptr(x), _ptr(out), sign), "fft")
    return out


def fft2(a, sign=-1, naive=False):
    a = _c128(a).copy()
    assert a.ndim == 2 and a.shape[0] == a.shape[1]
    _check(_load().orc_fft2(a.shape[0], _ptr(a), sign, int(naive)), "fft2")
    return a


def mod_offsets(K, r, theta0=0.0):
    dx = np.empty(K)
    dy = np.empty(K)
    _load().orc_mod_offsets(K, float(r), float(theta0), _ptr(dx), _ptr(dy))
    return dx, dy


def phasor(A, phi, dx, dy):
    A, phi = _f32(A), _f32(phi)
    N = A.shape[0]
    P = np.empty((N, N), dtype=np.complex128)
    _load().orc_phasor(N, _ptr(A), _ptr(phi), float(dx), float(dy), _ptr(P))
    return P


def embed(P, M):
    P = _c128(P)
    G = np.empty((M, M), dtype=np.complex128)
    _load().orc_embed(P.shape[0], M, _ptr(P), _ptr(G))
    return G


def pyramid_mask(M, s):
    m = np.empty((M, M), dtype=np.complex128)
    _load().orc_pyramid_mask(M, float(s), _ptr(m))
    return m


def field(A, phi, M, dx, dy, mask, naive=False, want_focal=False):
    """E (and optionally the unnormalised focal-plane F) for one tilt."""
    A, phi, mask = _f32(A), _f32(phi), _c128(mask)
    N = A.shape[0]
    E = np.empty((M, M), dtype=np.complex128)
    F = np.empty((M, M), dtype=np.complex128) if want_focal else None
    _check(_load().orc_field(N, M, _ptr(A), _ptr(phi), float(dx), float(dy), _ptr(mask),
                             _ptr(E), _ptr(F) if want_focal else None, int(naive)), "field")
    return (E, F) if want_focal else E


def intensity(A, phi, M, K, r, theta0=0.0, mask=None, s=None, naive=False):
    """Full-resolution I = mean_k |E_k|^2 on the M x M grid."""
    A, phi = _f32(A), _f32(phi)
    N = A.shape[0]
    if mask is None:
        mask = pyramid_mask(M, M // 4 if s is None else s)
    mask = _c128(mask)
    out = np.empty((M, M), dtype=np.float64)
    _check(_load().orc_intensity(N, M, _ptr(A), _ptr(phi), K, float(r), float(theta0),
                                 _ptr(mask), _ptr(out), int(naive)), "intensity")
    return out


def rebin_weights(N, n_sub):
    W = np.empty((n_sub, N), dtype=np.float64)
    _load().orc_rebin_weights(N, n_sub, _ptr(W))
    return W


def frame(I, N, s, n_sub):
    I = np.ascontiguousarray(I, dtype=np.float64)
    M = I.shape[0]
    out = np.empty((2 * n_sub, 2 * n_sub), dtype=np.float64)
    _check(_load().orc_frame(N, M, int(s), n_sub, _ptr(I), _ptr(out)), "frame")
    return out


def valid_mask(A, n_sub, thresh=0.5):
    A = _f32(A)
    v = np.empty((n_sub, n_sub), dtype=np.uint8)
    n = _check(_load().orc_valid_mask(A.shape[0], n_sub, _ptr(A), float(thresh), _ptr(v)),
               "valid_mask")
    return v, n


def slopes(frm, valid, norm_mode=0):
    frm = np.ascontiguousarray(frm, dtype=np.float64)
    valid = np.ascontiguousarray(valid, dtype=np.uint8)
    n_sub = valid.shape[0]
    nv = int(valid.sum())
    out = np.empty(2 * nv, dtype=np.float64)
    _check(_load().orc_slopes(n_sub, _ptr(frm), _ptr(valid), norm_mode, _ptr(out)), "slopes")
    return out


def pwfs_run(A, M, r, K, n_sub, phase, s=0, theta0=0.0, thresh=0.5, norm_mode=0):
    """Whole path for a batch: returns (frames [B,2n,2n] f64, slopes [B,2nv] f64)."""
    A = _f32(A)
    phase = _f32(phase)
    N = A.shape[0]
    if phase.ndim == 2:
        phase = phase[None]
    B = phase.shape[0]
    assert phase.shape[1:] == (N, N)
    _, nv = valid_mask(A, n_sub, thresh)
    frames = np.empty((B, 2 * n_sub, 2 * n_sub), dtype=np.float64)
    slp = np.empty((B, 2 * nv), dtype=np.float64)
    rc = _load().orc_pwfs_run(N, M, _ptr(A), int(s), float(r), K, float(theta0), n_sub,
                              float(thresh), norm_mode, B, _ptr(phase), _ptr(frames), _ptr(slp))
    _check(rc, "pwfs_run")
    assert rc == nv
    return frames, slp


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def field_stop(mask, h):
    """mask * (square stop |u~|,|v~| <= h bins); h < 0: unchanged."""
    m = _c128(mask).copy()
    _load().orc_field_stop(m.shape[0], float(h), _ptr(m))
    return m


def intensity_list(A, phi, M, dx, dy, w, mask=None, s=None, naive=False):
    """Full-resolution I = sum_k w_k |E_k|^2 / sum_k w_k for a list of tilts."""
    A, phi = _f32(A), _f32(phi)
    dx, dy, w = _f64(dx), _f64(dy), _f64(w)
    N = A.shape[0]
    if mask is None:
        mask = pyramid_mask(M, M // 4 if s is None else s)
    mask = _c128(mask)
    out = np.empty((M, M), dtype=np.float64)
    _check(_load().orc_intensity_list(N, M, _ptr(A), _ptr(phi), dx.size, _ptr(dx), _ptr(dy), _ptr(w),
                                      _ptr(mask), _ptr(out), int(naive)), "intensity_list")
    return out


def pwfs_run_list(A, M, dx, dy, w, n_sub, phase, s=0, stop_h=-1.0, thresh=0.5, norm_mode=0):
    """Whole path with a weighted tilt list and an optional square field stop."""
    A, phase = _f32(A), _f32(phase)
    dx, dy, w = _f64(dx), _f64(dy), _f64(w)
    N = A.shape[0]
    if phase.ndim == 2:
        phase = phase[None]
    B = phase.shape[0]
    _, nv = valid_mask(A, n_sub, thresh)
    frames = np.empty((B, 2 * n_sub, 2 * n_sub), dtype=np.float64)
    slp = np.empty((B, 2 * nv), dtype=np.float64)
    rc = _load().orc_pwfs_run_list(N, M, _ptr(A), int(s), dx.size, _ptr(dx), _ptr(dy), _ptr(w),
                                   float(stop_h), n_sub, float(thresh), norm_mode, B, _ptr(phase),
                                   _ptr(frames), _ptr(slp))
    _check(rc, "pwfs_run_list")
    return frames, slp
