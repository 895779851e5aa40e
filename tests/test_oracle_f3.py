"""Pins of the oracle's f3 generalisations: weighted tilt
list in place of the modulation circle, square focal-plane field stop.

Each pin compares against something other than the function under test: the
already-pinned circle path (orc_intensity), numpy.fft (library routine), closed
forms, or the physics (a source offset is a tilt of the wavefront)."""
import math

import numpy as np
import pytest

from oracle import pwfs_oracle as orc
from paper_1607_07624_b200 import workloads as wl


def _pupil(N, obs=0.2):
    c = np.arange(N) - (N - 1) / 2.0
    X, Y = np.meshgrid(c, c)
    rho = np.hypot(X, Y)
    return ((rho <= N / 2.0) & (rho >= obs * N / 2.0)).astype(np.float32)


def _phase(N, seed, amp=1.5):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal((N, N)) * amp).astype(np.float32)


N, M = 16, 48


def test_uniform_circle_list_reproduces_the_circle():
    A, phi = _pupil(N), _phase(N, 1)
    K, r, th0 = 8, 2.5, 0.3
    dx, dy = orc.mod_offsets(K, r, th0)
    I_list = orc.intensity_list(A, phi, M, dx, dy, np.ones(K))
    I_circ = orc.intensity(A, phi, M, K, r, th0)
    assert np.abs(I_list - I_circ).max() <= 1e-13 * I_circ.max()


def test_weighted_list_is_the_weighted_mean_of_single_point_images():
    A, phi = _pupil(N), _phase(N, 2)
    pts = [(0.7, -1.1, 0.5), (-2.0, 0.4, 2.0), (0.0, 0.0, 1.25), (1.5, 1.5, 0.25)]
    dx, dy, w = map(np.array, zip(*pts))
    I_list = orc.intensity_list(A, phi, M, dx, dy, w)
    acc = np.zeros((M, M))
    for x, y, wk in pts:   # one modulation "circle" of a single point at (r, theta0) = polar(x, y)
        acc += wk * orc.intensity(A, phi, M, 1, math.hypot(x, y), math.atan2(y, x))
    acc /= w.sum()
    assert np.abs(I_list - acc).max() <= 1e-12 * acc.max()
    # only the ratios of the weights matter
    I_scaled = orc.intensity_list(A, phi, M, dx, dy, 3.0 * w)
    assert np.abs(I_scaled - I_list).max() <= 1e-13 * I_list.max()
    # a zero-weight point contributes nothing
    I_zero = orc.intensity_list(A, phi, M, np.append(dx, 5.0), np.append(dy, -3.0), np.append(w, 0.0))
    assert np.abs(I_zero - I_list).max() <= 1e-13 * I_list.max()


def test_list_point_offset_equals_wavefront_tilt():
    """A source at (dx, dy) lambda/D is a tilt 2 pi (dx (x-c) + dy (y-c)) / N of the
    wavefront (A1-A3): pins sign, units and centre of the list tilts."""
    A = _pupil(N)
    ax, ay = 0.75, -0.5
    I_pt = orc.intensity_list(A, np.zeros((N, N), np.float32), M, [ax], [ay], [1.0])
    I_ph = orc.intensity_list(A, wl.tilt_phase(N, ax, ay), M, [0.0], [0.0], [1.0])
    assert np.abs(I_pt - I_ph).max() <= 2e-6 * I_ph.max()      # tilt_phase is float32


def test_negative_or_all_zero_weights_are_rejected():
    A, phi = _pupil(N), _phase(N, 3)
    with pytest.raises(RuntimeError):
        orc.intensity_list(A, phi, M, [0.0, 1.0], [0.0, 0.0], [1.0, -0.5])
    with pytest.raises(RuntimeError):
        orc.intensity_list(A, phi, M, [0.0], [0.0], [0.0])


def test_field_stop_wider_than_the_grid_changes_nothing():
    A, phi = _pupil(N), _phase(N, 4)
    m0 = orc.pyramid_mask(M, M // 4)
    assert np.array_equal(orc.field_stop(m0, -1.0), m0)
    assert np.array_equal(orc.field_stop(m0, M / 2), m0)       # |u~| <= M/2 always
    I0 = orc.intensity(A, phi, M, 4, 1.0)
    I1 = orc.intensity(A, phi, M, 4, 1.0, mask=orc.field_stop(m0, M / 2))
    assert np.array_equal(I0, I1)


@pytest.mark.parametrize("h", [0.0, 3.0, 7.5, 11.0])
def test_field_stop_geometry_against_numpy_fft(h):
    """Parseval through the stop: sum I = (1/M^2) sum_{|u~|,|v~| <= h} |F|^2 with F
    from numpy.fft.fft2 of the padded phasor (library routine, test-only)."""
    A, phi = _pupil(N), _phase(N, 5)
    G = np.zeros((M, M), complex)
    o = M // 2 - N // 2
    G[o:o + N, o:o + N] = A * np.exp(1j * phi.astype(np.float64))
    F = np.fft.fft2(G)
    f = np.fft.fftfreq(M, 1.0 / M)                            # signed integer bins
    inside = (np.abs(f)[None, :] <= h) & (np.abs(f)[:, None] <= h)
    want = (np.abs(F) ** 2 * inside).sum() / (M * M)
    mask = orc.field_stop(orc.pyramid_mask(M, M // 4), h)
    assert np.count_nonzero(mask) == inside.sum()
    assert np.array_equal(mask != 0, inside)
    I = orc.intensity_list(A, phi, M, [0.0], [0.0], [1.0], mask=mask)
    assert abs(I.sum() - want) <= 1e-12 * want


def test_pinhole_stop_gives_a_uniform_plane():
    """h = 0 passes the DC bin only: E = sum(P) / M^2 everywhere (closed form)."""
    A, phi = _pupil(N), _phase(N, 6, amp=0.3)
    P = A * np.exp(1j * phi.astype(np.float64))
    mask = orc.field_stop(orc.pyramid_mask(M, M // 4), 0.0)
    I = orc.intensity_list(A, phi, M, [0.0], [0.0], [1.0], mask=mask)
    want = abs(P.sum()) ** 2 / M ** 4
    assert np.abs(I - want).max() <= 1e-13 * want


def test_whole_path_list_entry_matches_the_circle_entry_and_keeps_flat_slopes_zero():
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    phase = wl.phase_batch(cfg, steps=1)
    dx, dy = orc.mod_offsets(cfg.mod_points, cfg.mod_radius)
    f_l, s_l = orc.pwfs_run_list(A, cfg.m_grid, dx, dy, np.ones(cfg.mod_points), cfg.n_subap, phase)
    f_c, s_c = orc.pwfs_run(A, cfg.m_grid, cfg.mod_radius, cfg.mod_points, cfg.n_subap, phase)
    assert np.abs(f_l - f_c).max() <= 1e-12 * f_c.max() and np.abs(s_l - s_c).max() <= 1e-12
    # symmetric weighted list + symmetric stop + flat phase: the slopes vanish (P4 generalised)
    pts_x = np.array([1.0, -1.0, 0.0, 0.0, 2.0, -2.0])
    pts_y = np.array([0.0, 0.0, 1.0, -1.0, 2.0, -2.0])
    pts_w = np.array([1.0, 1.0, 1.0, 1.0, 0.5, 0.5])
    # (2,2)/(-2,-2) alone would break x<->-x symmetry of the list: add their mirrors
    pts_x = np.concatenate([pts_x, [2.0, -2.0]]); pts_y = np.concatenate([pts_y, [-2.0, 2.0]])
    pts_w = np.concatenate([pts_w, [0.5, 0.5]])
    flat = np.zeros((1, cfg.n_pupil, cfg.n_pupil), np.float32)
    fr, sl = orc.pwfs_run_list(A, cfg.m_grid, pts_x, pts_y, pts_w, cfg.n_subap, flat, stop_h=40.0)
    assert np.abs(sl).max() <= 1e-12
    assert fr.sum() < (A.astype(np.float64) ** 2).sum()        # the stop removes light
