"""ORACLE (test infrastructure, NOT the product) for SURVEY.md 8(f) row f4, second
part: Shack-Hartmann propagation (wavefront -> spots on the detector) and its
centre-of-gravity slopes.

Plain numpy, float64, one subaperture at a time, numpy.fft.fft2 as the one
library step; shares nothing with the CUDA path
(paper_1607_07624_b200/csrc/sh_api.cu) and is imported only by tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline leg.

What it follows.  The paper names the routine only: PASSATA simulates
"Shack-Hartmann" sensors (PAPER.md:L9 abstract) and "Pyramid and Shack
Hartmann propagation (from wavefront to detector plane)" is GPU-accelerated
(section 6); the example of section 4 uses the pyramid, so no
SH parameter set is printed.  Readings taken:

  F4e  the N x N pupil is cut into n_sub x n_sub square subapertures of
       b = N / n_sub pixels (b an integer); subaperture (j, i) holds pupil
       pixels [j b, (j+1) b) x [i b, (i+1) b).
  F4f  spot of one subaperture: g = A exp(i c phi) on its b x b pixels,
       zero-padded to P x P, multiplied by the half-pixel centring phase
       exp(-i pi (x + y) / P), forward DFT2 (sign -, unnormalised), fftshift,
       |.|^2 / P^2.  The centring phase puts the spot of a flat wavefront on the
       geometric centre of the P x P array (between the four middle pixels), so
       that an even detector window is symmetric about it.  With the full P x P
       kept, the spot's total is sum |g|^2 (Parseval); FFT pixel = lambda / (d P / b).
  F4g  detector: the central (n_px bin) x (n_px bin) FFT pixels of each spot are
       summed in bin x bin blocks into n_px x n_px detector pixels; the frame is
       the mosaic [n_sub n_px][n_sub n_px], subaperture (j, i) at rows
       [j n_px, (j+1) n_px), columns [i n_px, (i+1) n_px).
  F4h  valid subapertures: sum A^2 over the subaperture >= thresh * b^2 * max A^2
       (the pyramid path's rule A11 applied to b x b blocks).
  F4i  slopes by centre of gravity, in detector pixels from the window centre:
       Sx = sum (px - (n_px-1)/2) I / sum I (Sy likewise with py), output
       [Sx(valid, row-major) ..., Sy ...] as for the pyramid.  +x tilt => Sx > 0.
"""
from __future__ import annotations

import numpy as np


def valid_mask(A, n_sub, thresh=0.5):
    """F4h -> (uint8 [n_sub][n_sub], n_valid)."""
    A = np.asarray(A, dtype=np.float64)
    N = A.shape[0]
    if N % n_sub:
        raise ValueError("n_sub must divide N")
    b = N // n_sub
    lit = (A ** 2).reshape(n_sub, b, n_sub, b).sum(axis=(1, 3))
    v = lit >= thresh * b * b * (A ** 2).max()
    return v.astype(np.uint8), int(v.sum())


def spot(g, P):
    """F4f: b x b complex field -> P x P spot image."""
    b = g.shape[0]
    pad = np.zeros((P, P), dtype=np.complex128)
    x = np.arange(b)
    ramp = np.exp(-1j * np.pi * x / P)
    pad[:b, :b] = g * ramp[None, :] * ramp[:, None]
    X = np.fft.fftshift(np.fft.fft2(pad))
    return (X.real ** 2 + X.imag ** 2) / float(P * P)


def detector_window(S, n_px, bin_):
    """F4g for one spot: central crop, bin x bin sums."""
    P = S.shape[0]
    Pc = n_px * bin_
    if Pc > P or (P - Pc) % 2:
        raise ValueError("n_px * bin must be <= P with the same parity")
    o = (P - Pc) // 2
    return S[o:o + Pc, o:o + Pc].reshape(n_px, bin_, n_px, bin_).sum(axis=(1, 3))


def sh_frame(A, phi, n_sub, P, n_px, bin_, phase_scale=1.0):
    """F4e-F4g: one wavefront -> detector frame [n_sub n_px][n_sub n_px]."""
    A = np.asarray(A, dtype=np.float64)
    phi = np.asarray(phi, dtype=np.float64)
    N = A.shape[0]
    b = N // n_sub
    G = A * np.exp(1j * phase_scale * phi)
    out = np.zeros((n_sub * n_px, n_sub * n_px))
    for j in range(n_sub):
        for i in range(n_sub):
            g = G[j * b:(j + 1) * b, i * b:(i + 1) * b]
            out[j * n_px:(j + 1) * n_px, i * n_px:(i + 1) * n_px] = detector_window(spot(g, P), n_px, bin_)
    return out


def cog_slopes(frame, valid, n_px):
    """F4i: centre of gravity of every valid subaperture's window."""
    valid = np.asarray(valid).astype(bool)
    n_sub = valid.shape[0]
    c = np.arange(n_px) - (n_px - 1) / 2.0
    sx, sy = [], []
    for j in range(n_sub):
        for i in range(n_sub):
            if valid[j, i]:
                w = frame[j * n_px:(j + 1) * n_px, i * n_px:(i + 1) * n_px]
                tot = w.sum()
                sx.append((w.sum(axis=0) * c).sum() / tot)
                sy.append((w.sum(axis=1) * c).sum() / tot)
    return np.array(sx + sy)


def sh_run(A, phase, n_sub, P, n_px, bin_, thresh=0.5, phase_scale=1.0):
    """Whole SH path for a batch -> (frames [B][D][D], slopes [B][2 n_valid])."""
    phase = np.asarray(phase)
    if phase.ndim == 2:
        phase = phase[None]
    valid, _ = valid_mask(A, n_sub, thresh)
    frames = np.stack([sh_frame(A, p, n_sub, P, n_px, bin_, phase_scale) for p in phase])
    slopes = np.stack([cog_slopes(f, valid, n_px) for f in frames])
    return frames, slopes
