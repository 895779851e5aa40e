"""Pins of the f4 PSF-camera oracle (oracle/psf_oracle.py): the definition by brute force,
Parseval, the diffraction limit (Airy pattern via scipy.special.j1), shift theorem, Marechal."""
import numpy as np
import pytest
from scipy.special import j1

from oracle import psf_oracle as po


def _disc(N, obs=0.0):
    yy, xx = (np.mgrid[0:N, 0:N] - (N - 1) / 2.0) / (N / 2.0)
    r = np.hypot(xx, yy)
    return ((r <= 1.0) & (r >= obs)).astype(np.float64)


def test_psf_is_the_dft_definition_by_brute_force():
    rng = np.random.default_rng(0)
    N, M = 6, 14
    A, phi = rng.random((N, N)), rng.standard_normal((N, N))
    P, sr = po.psf_frame(A, phi, M, phase_scale=0.7)
    G = np.zeros((M, M), complex)
    G[:N, :N] = A * (np.cos(0.7 * phi) + 1j * np.sin(0.7 * phi))
    want = np.empty((M, M))
    for v in range(M):
        for u in range(M):
            s = 0j
            for y in range(N):
                for x in range(N):
                    s += G[y, x] * np.exp(-2j * np.pi * (u * x + v * y) / M)
            want[(v + M // 2) % M, (u + M // 2) % M] = abs(s) ** 2 / (M * M * (A ** 2).sum())
    assert np.abs(P - want).max() < 1e-14
    assert sr == pytest.approx(abs((A * np.exp(0.7j * phi)).sum()) ** 2 / A.sum() ** 2, rel=1e-13)


@pytest.mark.parametrize("N,M", [(16, 32), (20, 64), (15, 40)])
def test_unit_energy_flat_strehl_and_symmetry(N, M):
    A = _disc(N, 0.2)
    rng = np.random.default_rng(N)
    P, sr = po.psf_frame(A, rng.standard_normal((N, N)), M)
    assert P.sum() == pytest.approx(1.0, rel=1e-13) and 0.0 < sr < 1.0
    P0, sr0 = po.psf_frame(A, np.zeros((N, N)), M)
    c = M // 2
    assert sr0 == pytest.approx(1.0, rel=1e-14)
    assert P0.argmax() == c * M + c
    assert P0[c, c] == pytest.approx(A.sum() ** 2 / (M * M * (A ** 2).sum()), rel=1e-13)
    # real symmetric aperture: point-symmetric PSF about the centre pixel
    assert np.abs(P0[1:, 1:] - P0[1:, 1:][::-1, ::-1]).max() < 1e-15
    # a piston changes nothing
    P1, sr1 = po.psf_frame(A, np.full((N, N), 1.234), M)
    assert np.abs(P1 - P0).max() < 1e-15 and sr1 == pytest.approx(1.0, rel=1e-13)


def test_tilt_shifts_the_psf_by_nd_pixels_per_lambda_over_d():
    N, M = 16, 64                                    # nd = 4 px per lambda/D
    A = _disc(N)
    x = np.arange(N) - (N - 1) / 2.0
    P0, _ = po.psf_frame(A, np.zeros((N, N)), M)
    Px, srx = po.psf_frame(A, np.tile(2 * np.pi * 2.0 * x / N, (N, 1)), M)          # +2 lambda/D along x
    Py, _ = po.psf_frame(A, np.tile(-2 * np.pi * 1.0 * x / N, (N, 1)).T, M)         # -1 lambda/D along y
    assert np.abs(Px - np.roll(P0, 8, axis=1)).max() < 1e-14                        # +x tilt -> +u
    assert np.abs(Py - np.roll(P0, -4, axis=0)).max() < 1e-14
    assert srx < 0.01                                                               # on-axis light is gone


def test_airy_pattern_of_a_circular_aperture():
    N, nd = 256, 4
    M = nd * N
    P, _ = po.psf_frame(_disc(N), np.zeros((N, N)), M)
    c = M // 2
    cut = P[c, c:c + 6 * nd + 1] / P[c, c]
    rho = np.arange(cut.size) / nd                   # lambda/D
    arg = np.pi * rho
    airy = np.ones_like(rho)
    airy[1:] = (2 * j1(arg[1:]) / arg[1:]) ** 2
    assert np.abs(cut - airy).max() < 2e-3           # pixelated disc vs the continuous one
    # first dark ring at 1.22 lambda/D: between the samples at 1.0 and 1.5 the cut dips below 1e-3
    fine, _ = po.psf_frame(_disc(128), np.zeros((128, 128)), 128 * 16)
    cf = 128 * 8
    ring = fine[cf, cf:cf + 33] / fine[cf, cf]
    assert abs(ring[8:].argmin() + 8 - 1.22 * 16) <= 1 and ring[8:].min() < 1e-3


def test_marechal_and_phase_scale():
    N, M = 64, 128
    A = _disc(N, 0.1)
    rng = np.random.default_rng(3)
    phi = 0.1 * rng.standard_normal((N, N))
    _, sr = po.psf_frame(A, phi, M)
    var = np.average((phi - np.average(phi, weights=A)) ** 2, weights=A)
    assert sr == pytest.approx(np.exp(-var), abs=3e-4)
    Pa, sra = po.psf_frame(A, phi, M, phase_scale=750.0 / 1650.0)
    Pb, srb = po.psf_frame(A, phi * (750.0 / 1650.0), M)
    assert np.abs(Pa - Pb).max() < 1e-16 and sra == pytest.approx(srb, rel=1e-14)
    assert sra > sr                                  # longer wavelength, smaller phase, higher Strehl


def test_long_exposure_is_the_mean_of_the_frames():
    N, M = 12, 32
    A = _disc(N)
    rng = np.random.default_rng(4)
    ph = rng.standard_normal((5, N, N))
    L, sr = po.psf_long_exposure(A, ph, M)
    each = [po.psf_frame(A, p, M) for p in ph]
    assert np.abs(L - np.mean([e[0] for e in each], axis=0)).max() < 1e-16
    assert np.array_equal(sr, [e[1] for e in each])
    assert L.sum() == pytest.approx(1.0, rel=1e-13)
    # the long exposure is broader than the diffraction limit: lower peak
    assert L.max() < po.psf_frame(A, np.zeros((N, N)), M)[0].max()
