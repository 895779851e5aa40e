"""GPU parity of f1 (propagation through phase screens) against oracle/atmo_oracle.py,
element by element on the same seeded float32 screens.

Tolerance: the kernel interpolates and sums in float32; with L layers the
rounding error is bounded by about (4 + L + 2) ulp of the largest partial sum, so
    |d phi| <= 4e-6 * max|phi|   per frame
(a wrong neighbour, weight or shift sign gives errors of order 0.1-10 rad)."""
import numpy as np
import pytest

from paper_1607_07624_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL_REL = 4e-6


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _both(torch, atm, first, steps, dt=None):
    from oracle import atmo_oracle as ao
    from paper_1607_07624_b200.atmo import Atmosphere
    dt = atm["dt"] if dt is None else dt
    with Atmosphere(**atm) as a:
        got = a.propagate(first, steps, dt)
        torch.cuda.synchronize()
        got = got.cpu().numpy().astype(np.float64)
    want = ao.propagate(atm["screens"], atm["pitch"], atm["wind_vxy"], atm["heights"], atm["dirs_tan"],
                        atm["wl_scale"], first, steps, dt, atm["n_pupil"])
    assert got.shape == want.shape and np.isfinite(got).all()
    for b in range(want.shape[0]):
        scale = max(np.abs(want[b]).max(), 1e-30)
        err = np.abs(got[b] - want[b]).max()
        assert err <= TOL_REL * scale, f"frame {b}: {err:.3e} vs max {scale:.3e}"
    return got, want


def _random_atm(L, G, N, S, W, seed, pitch=0.25):
    rng = np.random.default_rng(seed)
    return dict(screens=(rng.standard_normal((L, G, G)) * 10).astype(np.float32), pitch=pitch,
                wind_vxy=rng.uniform(-30, 30, (L, 2)), heights=rng.uniform(0, 15000, L),
                dirs_tan=rng.uniform(-3e-4, 3e-4, (S, 2)), wl_scale=rng.uniform(0.2, 1.0, W), dt=1e-3, n_pupil=N)


@pytest.mark.parametrize("L,G,N,S,W", [
    (1, 16, 16, 1, 1),        # N == G: every row and column wraps
    (3, 64, 50, 2, 2),        # ragged N (scalar stores), several tiles in y
    (4, 300, 257, 3, 1),      # non power-of-two G, N % 4 == 1, three tiles in x
    (2, 256, 128, 1, 3),      # exactly one x tile
    (16, 32, 20, 1, 1),       # maximum layer count
])
def test_random_geometries(torch_cuda, L, G, N, S, W):
    atm = _random_atm(L, G, N, S, W, seed=L * 1000 + N)
    _both(torch_cuda, atm, first=3, steps=4)


def test_negative_time_large_time_and_zero_steps(torch_cuda):
    from paper_1607_07624_b200.atmo import Atmosphere
    atm = _random_atm(2, 128, 96, 2, 1, seed=7)
    _both(torch_cuda, atm, first=-250, steps=2)
    _both(torch_cuda, atm, first=10_000_000, steps=2)          # shifts of ~1e6 px: needs the double-precision split
    with Atmosphere(**atm) as a:
        out = a.propagate(0, 0, 1e-3)
        assert out.shape == (0, 96, 96)


@pytest.mark.parametrize("name,first,steps", [("cfg2_flao", 0, 6), ("cfg3_npot", 100, 3), ("cfg4_elt", 50, 4),
                                               ("cfg5_multi", 7, 2)])
def test_full_size_atmospheres(torch_cuda, name, first, steps):
    cfg = wl.CONFIGS[name]
    got, _ = _both(torch_cuda, wl.atmosphere(cfg), first, steps)
    # and it is the batch the hot path was fed all along (independent float64 sampler of the input generator)
    ref = wl.phase_batch(cfg, steps=steps, first_step=first)
    assert np.abs(got - ref).max() <= 5e-5


def test_device_pipeline_atmosphere_to_slopes_matches_the_oracle_chain(torch_cuda):
    """f1 -> a1..a8 without leaving the device, against oracle f1 -> oracle O0..O9."""
    from oracle import atmo_oracle as ao
    from oracle import pwfs_oracle as orc
    from paper_1607_07624_b200.atmo import Atmosphere
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg2_flao"]
    atm = wl.atmosphere(cfg)
    with Atmosphere(**atm) as a, from_config(cfg) as sensor:
        phase = a.propagate(10, 3, atm["dt"])
        fr, sl = sensor.run(phase)
        torch.cuda.synchronize()
    ph_ref = ao.propagate(atm["screens"], atm["pitch"], atm["wind_vxy"], atm["heights"], atm["dirs_tan"],
                          atm["wl_scale"], 10, 3, atm["dt"], cfg.n_pupil).astype(np.float32)
    fr_ref, sl_ref = orc.pwfs_run(wl.make_pupil(cfg), cfg.m_grid, cfg.mod_radius, cfg.mod_points, cfg.n_subap, ph_ref)
    fr, sl = fr.cpu().numpy().astype(np.float64), sl.cpu().numpy().astype(np.float64)
    for b in range(3):
        assert np.abs(fr[b] - fr_ref[b]).max() / fr_ref[b].max() <= 1e-4
        assert np.abs(sl[b] - sl_ref[b]).max() <= 1e-4
