"""Pins of the f1 oracle (oracle/atmo_oracle.py): propagation through phase screens.

Closed forms and library routines the definition must reduce to, plus agreement with
the independently written frozen-flow sampler of the input generator."""
import numpy as np
import pytest

from oracle import atmo_oracle as ao
from paper_1607_07624_b200 import workloads as wl


def _screens(L, G, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((L, G, G)).astype(np.float32)


def test_integer_shift_is_a_roll():
    G, N = 24, 10
    scr = _screens(1, G, 1)
    # wind (3, -2) px per unit time, pitch 1, t = 1: pixel (x, y) sees screen (x - 3, y + 2)
    out = ao.propagate(scr, 1.0, [[3.0, -2.0]], [0.0], [[0.0, 0.0]], [1.0], 1, 1, 1.0, N, scalar=True)[0]
    want = np.roll(scr[0].astype(np.float64), (-2, 3), axis=(0, 1))[:N, :N]
    assert np.array_equal(out, want)


def test_height_times_direction_shifts_the_other_way():
    G, N = 24, 10
    scr = _screens(1, G, 2)
    # h * tan = (+4, +1) px: pixel (x, y) sees screen (x + 4, y + 1)
    out = ao.propagate(scr, 0.5, [[0.0, 0.0]], [1000.0], [[2e-3, 0.5e-3]], [1.0], 0, 1, 1.0, N, scalar=True)[0]
    want = np.roll(scr[0].astype(np.float64), (-1, -4), axis=(0, 1))[:N, :N]
    assert np.allclose(out, want, rtol=0, atol=1e-12)


def test_linear_ramp_is_reproduced_exactly_away_from_the_wrap():
    G, N = 64, 12
    yy, xx = np.mgrid[0:G, 0:G]
    scr = (0.25 * xx - 0.5 * yy + 3.0).astype(np.float32)[None]          # exact in float32
    sx, sy = 7.3125, 11.71875                                           # exact binary fractions
    out = ao.propagate(scr, 1.0, [[-sx, -sy]], [0.0], [[0.0, 0.0]], [1.0], 1, 1, 1.0, N, scalar=True)[0]
    want = 0.25 * (xx[:N, :N] + sx) - 0.5 * (yy[:N, :N] + sy) + 3.0
    assert np.abs(out - want).max() <= 1e-12


def test_half_pixel_shift_is_the_neighbour_average_and_wraps():
    G = 8
    scr = _screens(1, G, 3)
    out = ao.propagate(scr, 1.0, [[-0.5, 0.0]], [0.0], [[0.0, 0.0]], [1.0], 1, 1, 1.0, G, scalar=True)[0]
    s = scr[0].astype(np.float64)
    want = 0.5 * (s + np.roll(s, -1, axis=1))                           # last column wraps to column 0
    assert np.abs(out - want).max() <= 1e-15
    out = ao.propagate(scr, 1.0, [[0.0, -0.25]], [0.0], [[0.0, 0.0]], [1.0], 1, 1, 1.0, G, scalar=True)[0]
    want = 0.75 * s + 0.25 * np.roll(s, -1, axis=0)
    assert np.abs(out - want).max() <= 1e-15


def test_layers_add_and_wavelengths_scale_and_frames_are_ordered_step_dir_wavelength():
    G, N, L = 32, 9, 3
    scr = _screens(L, G, 4)
    wind = [[1.25, -0.5], [-2.0, 0.75], [0.3, 0.2]]
    heights = [0.0, 4000.0, 9000.0]
    dirs = [[0.0, 0.0], [1e-4, -2e-4]]
    wls = [1.0, 0.75, 0.3]
    out = ao.propagate(scr, 0.5, wind, heights, dirs, wls, 2, 3, 0.1, N, scalar=True)
    assert out.shape == (3 * 2 * 3, N, N)
    for i in range(3):
        for d in range(2):
            single = sum(ao.propagate(scr[l:l + 1], 0.5, wind[l:l + 1], heights[l:l + 1], [dirs[d]], [1.0],
                                      2 + i, 1, 0.1, N, scalar=True)[0] for l in range(L))
            for w in range(3):
                got = out[(i * 2 + d) * 3 + w]
                assert np.abs(got - wls[w] * single).max() <= 1e-13


def test_row_vectorised_variant_equals_the_scalar_definition():
    G, N = 40, 17
    scr = _screens(2, G, 5)
    args = (scr, 0.7, [[3.3, -1.7], [-0.9, 2.1]], [0.0, 7000.0], [[2e-4, 1e-4]], [0.6], 5, 2, 0.01, N)
    a = ao.propagate(*args, scalar=True)
    b = ao.propagate(*args, scalar=False)
    assert np.array_equal(a, b)


@pytest.mark.parametrize("name,steps,first", [("cfg2_flao", 2, 0), ("cfg4_elt", 1, 37), ("cfg5_multi", 1, 3)])
def test_agrees_with_the_input_generators_frozen_flow(name, steps, first):
    """workloads.phase_batch (written earlier, for the hot path's inputs) samples the same
    layers with its own bilinear code in float64; the oracle works from the float32 copy of
    the screens, so they agree to float32 rounding of ~100 rad values."""
    cfg = wl.CONFIGS[name]
    atm = wl.atmosphere(cfg)
    got = ao.propagate(atm["screens"], atm["pitch"], atm["wind_vxy"], atm["heights"], atm["dirs_tan"],
                       atm["wl_scale"], first, steps, atm["dt"], cfg.n_pupil)
    want = wl.phase_batch(cfg, steps=steps, first_step=first).astype(np.float64)
    assert got.shape == want.shape
    assert np.abs(got - want).max() <= 3e-5
    assert np.abs(want).max() > 1.0
