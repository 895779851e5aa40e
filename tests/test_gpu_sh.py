"""GPU parity of the f4 Shack-Hartmann sensor against oracle/sh_oracle.py on the same seeded
inputs.

Bars: detector frames element by element, max|dI| <= 1e-4 * max I per frame
(the hot path's intensity bar; direct FP32 sums of <= 16 terms give ~1e-6); slopes
|dS| <= 1e-4 detector pixels (centre of gravity = ratio of two FP32 sums of <= 256 terms)."""
import numpy as np
import pytest

from paper_1607_07624_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _disc(N, obs=0.0):
    yy, xx = (np.mgrid[0:N, 0:N] - (N - 1) / 2.0) / (N / 2.0)
    r = np.hypot(xx, yy)
    return ((r <= 1.0) & (r >= obs)).astype(np.float32)


def _phase(rng, B, N, rms):
    k = np.fft.fftfreq(N)[:, None] ** 2 + np.fft.fftfreq(N)[None, :] ** 2
    filt = 1.0 / (k + (1.0 / N) ** 2) ** (11.0 / 12.0)
    out = np.empty((B, N, N), np.float32)
    for b in range(B):
        s = np.fft.ifft2(np.fft.fft2(rng.standard_normal((N, N))) * filt).real
        out[b] = rms * s / s.std()
    return out


def _check(torch, A, phase, n_sub, P, n_px, bin_, thresh=0.5, scale=1.0):
    from oracle import sh_oracle as so
    from paper_1607_07624_b200.sh import ShackHartmann
    with ShackHartmann(A, n_sub, P, n_px, bin_, illum_thresh=thresh, phase_scale=scale) as sh:
        fr, sl = sh.run(torch.from_numpy(phase).to("cuda:0"))
        torch.cuda.synchronize()
        valid, nv = sh.valid_mask(), sh.n_valid
        D = sh.det_size
    fr, sl = fr.cpu().numpy().astype(np.float64), sl.cpu().numpy().astype(np.float64)
    want_valid, want_nv = so.valid_mask(A, n_sub, thresh)
    assert nv == want_nv and np.array_equal(valid, want_valid) and D == n_sub * n_px
    fr_ref, sl_ref = so.sh_run(A, phase, n_sub, P, n_px, bin_, thresh, scale)
    assert fr.shape == fr_ref.shape and sl.shape == sl_ref.shape and np.isfinite(fr).all() and np.isfinite(sl).all()
    for b in range(fr.shape[0]):
        assert np.abs(fr[b] - fr_ref[b]).max() <= 1e-4 * fr_ref[b].max(), b
    assert np.abs(sl - sl_ref).max() <= 1e-4, np.abs(sl - sl_ref).max()
    return fr, sl


@pytest.mark.parametrize("N,n_sub,P,n_px,bin_,B", [
    (32, 4, 16, 8, 2, 3),        # b = 8
    (30, 6, 10, 4, 2, 2),        # b = 5, P not a power of two, crop 8 of 10
    (48, 16, 8, 8, 1, 2),        # b = 3, full window
    (64, 4, 64, 16, 4, 2),       # b = 16, P = 64: the largest subaperture
    (70, 7, 20, 6, 3, 2),        # b = 10, ragged subaperture count per CTA (49 = 12*4 + 1)
    (40, 40, 2, 2, 1, 2),        # b = 1: one pixel per subaperture, quad cell
    (160, 40, 8, 4, 2, 2),       # cfg2-like geometry
    (96, 12, 32, 2, 8, 2),       # quad-cell detector from a finely sampled spot
])
def test_sh_matches_oracle(torch_cuda, N, n_sub, P, n_px, bin_, B):
    rng = np.random.default_rng(N + 13 * P)
    _check(torch_cuda, _disc(N, 0.2), _phase(rng, B, N, 3.0), n_sub, P, n_px, bin_)


def test_flat_and_tilted_wavefront(torch_cuda):
    N, n_sub, P, n_px, bin_ = 64, 8, 32, 16, 2
    A = np.ones((N, N), np.float32)
    x = (np.arange(N) - (N - 1) / 2.0)
    flat = np.zeros((1, N, N), np.float32)
    tilt = np.tile(2 * np.pi * 0.1 * x / 8.0, (N, 1)).astype(np.float32)[None]        # 0.1 lambda/d in +x
    _, s0 = _check(torch_cuda, A, flat, n_sub, P, n_px, bin_)
    _, s1 = _check(torch_cuda, A, tilt, n_sub, P, n_px, bin_)
    nv = 64
    assert np.abs(s0).max() < 1e-5
    assert np.allclose(s1[0, :nv], 0.2, rtol=0.05) and np.abs(s1[0, nv:]).max() < 1e-5


def test_non_binary_amplitude_phase_scale_threshold_and_large_phase(torch_cuda):
    rng = np.random.default_rng(8)
    N = 48
    A = (_disc(N, 0.3) * (0.3 + 0.7 * rng.random((N, N)))).astype(np.float32)
    ph = _phase(rng, 2, N, 8.0) + 300.0
    _check(torch_cuda, A, ph.astype(np.float32), 8, 12, 6, 2, thresh=0.3, scale=0.45)


def test_empty_batch_and_frames_only(torch_cuda):
    from paper_1607_07624_b200.sh import ShackHartmann
    torch = torch_cuda
    A = _disc(32)
    ph = torch.zeros((2, 32, 32), dtype=torch.float32, device="cuda:0")
    with ShackHartmann(A, 4, 16, 8, 2) as sh:
        fr0, sl0 = sh.run(ph[:0])
        assert fr0.shape == (0, 32, 32) and sl0.shape == (0, 2 * sh.n_valid)
        fr, none = sh.run(ph, want_slopes=False)
        fr2, _ = sh.run(ph)
        assert none is None and torch.equal(fr, fr2)
        assert torch.equal(fr[0], fr[1])


def test_sh_at_bench_size(torch_cuda):
    """cfg4 pupil: 480 px, 96 x 96 subapertures of 5 px, P = 16, 8 x 8 detector pixels per
    subaperture (768^2 detector), 2 frames of its turbulence: the geometry bench.py times."""
    cfg = wl.CONFIGS["cfg4_elt"]
    A = wl.make_pupil(cfg)
    phase = wl.phase_batch(cfg, steps=2)
    _check(torch_cuda, A, phase, 96, 16, 8, 2, scale=0.5)
