"""Pins of the f4 Shack-Hartmann oracle (oracle/sh_oracle.py): brute-force definition, the
Dirichlet-kernel closed form of a square subaperture, Parseval, symmetry, the shift theorem,
centre-of-gravity response, window/mosaic placement, and the valid mask against the pyramid
oracle's independent implementation of the same rule."""
import numpy as np
import pytest

from oracle import pwfs_oracle as orc
from oracle import sh_oracle as so
from paper_1607_07624_b200 import workloads as wl


def test_spot_is_the_definition_by_brute_force():
    rng = np.random.default_rng(0)
    b, P = 3, 8
    g = rng.standard_normal((b, b)) + 1j * rng.standard_normal((b, b))
    S = so.spot(g, P)
    want = np.empty((P, P))
    for v in range(P):
        for u in range(P):
            fu, fv = (u - P / 2 + 0.5) / P, (v - P / 2 + 0.5) / P
            s = sum(g[y, x] * np.exp(-2j * np.pi * (fu * x + fv * y)) for y in range(b) for x in range(b))
            want[v, u] = abs(s) ** 2 / P ** 2
    assert np.abs(S - want).max() < 1e-14


@pytest.mark.parametrize("b,P", [(4, 8), (5, 16), (8, 32), (6, 12)])
def test_flat_square_subaperture_is_a_dirichlet_kernel(b, P):
    S = so.spot(np.ones((b, b), complex), P)
    f = (np.arange(P) - P / 2 + 0.5) / P
    d = (np.sin(np.pi * b * f) / np.sin(np.pi * f)) ** 2          # |sum_x e^{-2 pi i f x}|^2
    assert np.abs(S - np.outer(d, d) / P ** 2).max() < 1e-12 * b ** 4
    assert S.sum() == pytest.approx(b * b, rel=1e-13)             # Parseval
    assert np.abs(S - S[::-1, :]).max() < 1e-12 and np.abs(S - S[:, ::-1]).max() < 1e-12 and np.abs(S - S.T).max() < 1e-12
    assert S.argmax() in (P // 2 * P + P // 2, (P // 2 - 1) * P + P // 2 - 1, (P // 2 - 1) * P + P // 2, P // 2 * P + P // 2 - 1)


def test_integer_pixel_tilt_rolls_the_spot():
    b, P = 4, 16                                                   # 1 lambda/d of tilt = P/b = 4 FFT pixels
    x = np.arange(b)
    S0 = so.spot(np.ones((b, b), complex), P)
    Sx = so.spot(np.exp(2j * np.pi * 0.5 * x / b)[None, :] * np.ones((b, 1)), P)      # +0.5 lambda/d along x
    Sy = so.spot(np.exp(-2j * np.pi * 0.75 * x / b)[:, None] * np.ones((1, b)), P)    # -0.75 lambda/d along y
    assert np.abs(Sx - np.roll(S0, 2, axis=1)).max() < 1e-12
    assert np.abs(Sy - np.roll(S0, -3, axis=0)).max() < 1e-12


def test_detector_window_worked_example():
    S = np.arange(64, dtype=float).reshape(8, 8)
    w = so.detector_window(S, 2, 2)                                # central 4 x 4, 2 x 2 blocks
    assert np.array_equal(w, [[18 + 19 + 26 + 27, 20 + 21 + 28 + 29], [34 + 35 + 42 + 43, 36 + 37 + 44 + 45]])
    assert np.array_equal(so.detector_window(S, 8, 1), S)
    assert so.detector_window(S, 1, 8)[0, 0] == S.sum()
    with pytest.raises(ValueError):
        so.detector_window(S, 3, 3)


def test_mosaic_placement_and_flux():
    N, n_sub, P, n_px, bin_ = 12, 3, 8, 8, 1
    A = np.zeros((N, N))
    A[4:8, 8:12] = 2.0                                              # only subaperture (j=1, i=2) is lit
    fr = so.sh_frame(A, np.zeros((N, N)), n_sub, P, n_px, bin_)
    assert fr.shape == (24, 24)
    assert fr[8:16, 16:24].sum() == pytest.approx(4.0 * 16, rel=1e-13)
    fr[8:16, 16:24] = 0.0
    assert np.abs(fr).max() == 0.0


def test_cog_slopes_zero_sign_axis_and_gain():
    N, n_sub, P, n_px, bin_ = 32, 4, 32, 16, 2                      # b = 8, 4 FFT px per lambda/d, 2 per detector px
    A = np.ones((N, N))
    valid, nv = so.valid_mask(A, n_sub)
    assert nv == 16
    x = np.arange(N) - (N - 1) / 2.0
    _, s0 = so.sh_run(A, np.zeros((N, N)), n_sub, P, n_px, bin_)
    assert np.abs(s0).max() < 1e-13
    t = 0.1                                                         # lambda/d of tilt per subaperture
    _, sx = so.sh_run(A, np.tile(2 * np.pi * t * x / 8.0, (N, 1)), n_sub, P, n_px, bin_)
    _, sy = so.sh_run(A, np.tile(2 * np.pi * t * x / 8.0, (N, 1)).T, n_sub, P, n_px, bin_)
    assert (sx[0, :nv] > 0).all() and np.abs(sx[0, nv:]).max() < 1e-13
    assert np.allclose(sy[0, nv:], sx[0, :nv], atol=1e-13) and np.abs(sy[0, :nv]).max() < 1e-13
    _, sm = so.sh_run(A, np.tile(-2 * np.pi * t * x / 8.0, (N, 1)), n_sub, P, n_px, bin_)
    assert np.allclose(sm, -sx, atol=1e-13)
    # geometric value t * (P / b) / bin = 0.2 detector px; a window of +-2 lambda/d keeps the
    # centre-of-gravity gain within a few per cent of it
    assert sx[0, 0] == pytest.approx(0.2, rel=0.05)
    # doubling the tilt doubles the response to first order
    _, s2 = so.sh_run(A, np.tile(2 * np.pi * 2 * t * x / 8.0, (N, 1)), n_sub, P, n_px, bin_)
    assert np.allclose(s2[0, :nv] / sx[0, :nv], 2.0, rtol=0.05)


def test_whole_window_centre_of_gravity_recovers_the_mean_gradient():
    # with the full P x P kept the first moment of |G(f)|^2 is the intensity-weighted mean phase
    # gradient (moment theorem), up to the wrap of the discrete grid: exact for a band-limited field
    b, P = 8, 64
    x = np.arange(b)
    for t in (0.05, 0.3):
        g = np.exp(2j * np.pi * t * x / b)[None, :] * np.ones((b, 1))
        S = so.spot(g, P)
        c = np.arange(P) - (P - 1) / 2.0
        cog = (S.sum(axis=0) * c).sum() / S.sum()
        # discrete moment: sum_f f |G|^2 over a full period is not the continuous one because f |G|^2
        # is not periodic; the dominant term is still t P / b, within the 1/f^2 wings' contribution
        assert abs(cog - t * P / b) < 0.35 * t * P / b


@pytest.mark.parametrize("name,n_sub", [("cfg1_tiny", 16), ("cfg2_flao", 40), ("cfg5_multi", 80), ("cfg4_elt", 96)])
def test_valid_mask_agrees_with_the_pyramid_oracles_rule(name, n_sub):
    A = wl.make_pupil(wl.CONFIGS[name])
    v, nv = so.valid_mask(A, n_sub)
    v2, nv2 = orc.valid_mask(A, n_sub)
    assert nv == nv2 and np.array_equal(v, v2)
    assert np.array_equal(v, v[::-1, :]) and np.array_equal(v, v[:, ::-1])


def test_phase_scale_is_a_multiplication_of_the_phase():
    rng = np.random.default_rng(3)
    N = 16
    A, phi = np.ones((N, N)), rng.standard_normal((N, N))
    a = so.sh_frame(A, phi, 4, 8, 4, 2, phase_scale=0.4)
    b = so.sh_frame(A, 0.4 * phi, 4, 8, 4, 2)
    assert np.abs(a - b).max() < 1e-15
