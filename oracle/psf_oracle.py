"""ORACLE (test infrastructure, NOT the product) for SURVEY.md 8(f) row f4, first
part: the PSF camera ("PSF generation from residual wavefront").

Plain numpy, float64, the definition written out with numpy.fft.fft2 as the one
library step; shares nothing with the CUDA path
(paper_1607_07624_b200/csrc/psf_api.cu) and is imported only by tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline leg.

What it follows.  The paper names the object and its parameters only:
"generating a PSF at a given wavelength based on an input wavefront"
(section 2); Table 1 `camera`:
wavelengthInNm "[nm] Imaging wavelength", nd "padding coefficient for PSF
computation", start_time "PSF integration start time";
`psf = factory.get_psf(params.camera)` (L247-248), `store.add, psf.out_sr,
name='sr'` (L270-271); "PSF generation from residual wavefront" is one of the
GPU routines (L344, section 6).  No formula is given; the readings taken
(DESIGN.md "f4"):

  F4a  field: G = A exp(i c phi) on the N x N pupil, c = lambda_phase /
       lambda_camera rescales the phase (given in radians at the wavelength it
       was generated for) to the imaging wavelength; zero-padded to M x M with
       M = nd * N (nd need not be an integer; M is what the caller fixes).
  F4b  instantaneous PSF = |DFT2(G)|^2 / (M^2 sum A^2): forward transform, sign
       -, unnormalised; the divisor makes sum(PSF) = 1 (Parseval).  Displayed
       with the zero frequency at pixel [M/2][M/2] (fftshift); pixel scale
       lambda / (nd D).  Where the pupil sits in the padded grid only changes
       the phase of the transform, not the PSF.
  F4c  Strehl ratio of a frame = PSF[centre] / PSF_flat[centre]
       = |sum A exp(i c phi)|^2 / (sum A)^2 (on-axis value against the
       diffraction limit of the same pupil).
  F4d  long exposure = mean of the instantaneous PSFs of the frames handed in
       (integration "from start_time" is the caller starting to hand frames in
       at that time; the loop control object is out of scope).
"""
from __future__ import annotations

import numpy as np


def field(A, phi, M, phase_scale=1.0):
    """F4a: A exp(i c phi) in the corner of an M x M grid of zeros."""
    A = np.asarray(A, dtype=np.float64)
    phi = np.asarray(phi, dtype=np.float64)
    N = A.shape[0]
    if M < N:
        raise ValueError("M must be >= N")
    G = np.zeros((M, M), dtype=np.complex128)
    G[:N, :N] = A * np.exp(1j * phase_scale * phi)
    return G


def psf_frame(A, phi, M, phase_scale=1.0):
    """F4b, F4c: (PSF [M][M] with the zero frequency at [M/2][M/2], Strehl ratio)."""
    A = np.asarray(A, dtype=np.float64)
    X = np.fft.fft2(field(A, phi, M, phase_scale))
    P = (X.real ** 2 + X.imag ** 2) / (float(M) ** 2 * (A ** 2).sum())
    sr = (X[0, 0].real ** 2 + X[0, 0].imag ** 2) / A.sum() ** 2
    return np.roll(P, (M // 2, M // 2), axis=(0, 1)), sr


def psf_long_exposure(A, phase, M, phase_scale=1.0):
    """F4d: (mean PSF over the frames, per-frame Strehl ratios)."""
    phase = np.asarray(phase)
    acc = np.zeros((M, M))
    sr = np.empty(phase.shape[0])
    for b in range(phase.shape[0]):
        P, sr[b] = psf_frame(A, phase[b], M, phase_scale)
        acc += P
    return acc / max(phase.shape[0], 1), sr
