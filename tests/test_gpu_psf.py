"""GPU parity of the f4 PSF camera against oracle/psf_oracle.py on the same seeded inputs.

Bars: the long-exposure PSF is compared element by element on the whole
M x M grid, max|dP| <= 1e-4 * max P (the hot path's intensity bar; FP32 FFT error is ~1e-6);
Strehl ratios |dSR| <= 1e-5 sqrt(SR) + 1e-9 (an amplitude error of 5e-6 of the coherent sum)."""
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


def _smooth_phase(rng, B, N, rms):
    """Band-limited random phase (a few cycles across the pupil) plus white noise."""
    k = np.fft.fftfreq(N)[:, None] ** 2 + np.fft.fftfreq(N)[None, :] ** 2
    filt = 1.0 / (k + (2.0 / N) ** 2) ** (11.0 / 12.0)
    out = np.empty((B, N, N), np.float32)
    for b in range(B):
        s = np.fft.ifft2(np.fft.fft2(rng.standard_normal((N, N))) * filt).real
        out[b] = rms * s / s.std() + 0.05 * rng.standard_normal((N, N))
    return out


def _check(torch, A, phase, M, scale=1.0):
    from oracle import psf_oracle as po
    from paper_1607_07624_b200.psf import PsfCamera
    with PsfCamera(A, M, phase_scale=scale) as cam:
        sr = cam.accumulate(torch.from_numpy(phase).to("cuda:0"))
        psf, n = cam.read()
        torch.cuda.synchronize()
    psf, sr = psf.cpu().numpy().astype(np.float64), sr.cpu().numpy().astype(np.float64)
    want, sr_want = po.psf_long_exposure(A, phase, M, scale)
    assert n == phase.shape[0] and psf.shape == (M, M) and np.isfinite(psf).all()
    assert np.abs(psf - want).max() <= 1e-4 * want.max(), np.abs(psf - want).max() / want.max()
    assert (np.abs(sr - sr_want) <= 1e-5 * np.sqrt(sr_want) + 1e-9).all(), (sr, sr_want)
    assert abs(psf.sum() - 1.0) < 1e-4
    return psf, sr


@pytest.mark.parametrize("N,M,B,rms", [(64, 128, 3, 1.0), (37, 128, 2, 0.5), (100, 256, 3, 2.0), (160, 320, 3, 3.0),
                                       (150, 320, 2, 1.0), (240, 480, 2, 2.0), (120, 512, 2, 1.0), (256, 512, 2, 4.0),
                                       (60, 640, 1, 1.0), (320, 640, 2, 2.0), (400, 800, 2, 3.0), (480, 1024, 2, 5.0),
                                       (500, 1024, 1, 1.0),
                                       (80, 160, 2, 1.0), (96, 192, 2, 2.0), (140, 288, 2, 1.0), (192, 384, 2, 3.0),
                                       (288, 576, 2, 2.0), (384, 768, 1, 2.0), (430, 864, 1, 1.0), (480, 960, 1, 3.0),
                                       # R1 > 32: two rounds of size-32 transforms per warp, no register prefetch
                                       (570, 1152, 1, 1.0), (600, 1280, 2, 2.0), (720, 1440, 1, 1.0), (768, 1536, 1, 2.0),
                                       (790, 1600, 1, 1.0), (860, 1728, 1, 1.0), (960, 1920, 1, 2.0), (1000, 2048, 2, 3.0)])
def test_psf_matches_oracle_on_every_grid(torch_cuda, N, M, B, rms):
    rng = np.random.default_rng(N * 7 + M)
    _check(torch_cuda, _disc(N, 0.15), _smooth_phase(rng, B, N, rms), M)


def test_phase_scale_and_non_binary_amplitude(torch_cuda):
    rng = np.random.default_rng(5)
    N, M = 96, 256
    A = (_disc(N) * (0.5 + 0.5 * rng.random((N, N)))).astype(np.float32)
    ph = _smooth_phase(rng, 2, N, 6.0)
    _, sr_a = _check(torch_cuda, A, ph, M, scale=750.0 / 1650.0)
    _, sr_b = _check(torch_cuda, A, ph, M, scale=1.0)
    assert (sr_a > sr_b).all()


def test_flat_and_tilted_wavefronts(torch_cuda):
    N, M = 64, 256
    A = _disc(N)
    x = (np.arange(N) - (N - 1) / 2.0).astype(np.float64)
    flat = np.zeros((1, N, N), np.float32)
    tilt = np.tile(2 * np.pi * 3.0 * x / N, (N, 1)).astype(np.float32)[None]       # +3 lambda/D in x
    p0, sr0 = _check(torch_cuda, A, flat, M)
    p1, sr1 = _check(torch_cuda, A, tilt, M)
    c = M // 2
    assert abs(sr0[0] - 1.0) < 1e-5 and p0.argmax() == c * M + c
    assert p1.argmax() == c * M + c + 12 and sr1[0] < 5e-3


def test_large_phase_values_keep_their_accuracy(torch_cuda):
    """|phi| of several hundred radians: the range reduction must not lose the fraction."""
    rng = np.random.default_rng(9)
    N, M = 64, 128
    ph = (_smooth_phase(rng, 2, N, 1.0) + 400.0).astype(np.float32)
    _check(torch_cuda, _disc(N), ph, M)


def test_accumulate_in_pieces_reset_and_empty(torch_cuda):
    from paper_1607_07624_b200.psf import PsfCamera
    torch = torch_cuda
    rng = np.random.default_rng(2)
    N, M = 80, 320
    A = _disc(N, 0.2)
    ph = torch.from_numpy(_smooth_phase(rng, 7, N, 2.0)).to("cuda:0")
    with PsfCamera(A, M) as cam:
        zero, n0 = cam.read()
        assert n0 == 0 and float(zero.abs().max()) == 0.0
        sr_all = cam.accumulate(ph)
        whole, n = cam.read()
        whole = whole.clone()
        assert n == 7
        cam.reset()
        sr_a = cam.accumulate(ph[:3])
        sr_b = cam.accumulate(ph[3:])
        cam.accumulate(ph[:0])
        parts, n2 = cam.read()
        assert n2 == 7
        assert torch.equal(torch.cat([sr_a, sr_b]), sr_all)
        assert float((parts - whole).abs().max()) <= 1e-6 * float(whole.max())
        cam.reset()
        cam.accumulate(ph[:1], want_sr=False)
        one, n3 = cam.read()
        assert n3 == 1 and abs(float(one.sum()) - 1.0) < 1e-4


def test_psf_at_bench_size_and_batch(torch_cuda):
    """cfg4 pupil (480 px, obstruction and spiders) on the 1024 grid, 24 frames of its turbulence
    rescaled to the H band: the launch configuration bench.py times (frame split > 1)."""
    cfg = wl.CONFIGS["cfg4_elt"]
    A = wl.make_pupil(cfg)
    phase = wl.phase_batch(cfg, steps=24)
    _check(torch_cuda, A, phase, 1024, scale=0.2)
