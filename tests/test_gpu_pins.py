"""Pins on the CUDA path that need NO oracle: what the physics and SURVEY.md's stated
values fix, checked directly on the output of pwfs_run (SURVEY.md 8(c) pins P2-P6,
P10; values in tests/golden/survey_scratch_values.json, each cited there).

These would catch a mistake that the oracle and the kernels happened to share (a
reading taken the same wrong way on both sides), which element-wise parity cannot.
FP32 bars: 1e-5 relative on flux, 2e-5 absolute on slopes (the parity bar is 1e-4).
"""
import math

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


def _run(torch, cfg, phase, **kw):
    from paper_1607_07624_b200.pwfs import from_config
    with from_config(cfg, **kw) as sensor:
        fr, sl = sensor.run(torch.from_numpy(np.ascontiguousarray(phase, dtype=np.float32)).cuda())
        torch.cuda.synchronize()
        return (fr.cpu().numpy().astype(np.float64), sl.cpu().numpy().astype(np.float64),
                sensor.valid_mask().astype(bool), sensor.n_valid)


def _to2d(vec, valid):
    g = np.zeros(valid.shape)
    g[valid] = vec
    return g


# P2: for M = 2N the four windows tile the grid, so the detector frame holds all the light: sum = sum A^2
@pytest.mark.parametrize("name", ["cfg1_tiny", "cfg2_flao", "cfg3_npot", "cfg5_multi"])
def test_parseval_total_flux_on_the_detector(torch_cuda, golden, name):
    cfg = wl.CONFIGS[name]
    assert cfg.m_grid == 2 * cfg.n_pupil
    lit = float((wl.make_pupil(cfg).astype(np.float64) ** 2).sum())
    assert lit == golden["configs"][name]["lit_px"]
    steps = 2 if cfg.instances == 1 else 1
    phase = wl.phase_batch(cfg, steps=steps)[:2]
    fr, _, _, nv = _run(torch_cuda, cfg, phase)
    assert nv == golden["configs"][name]["n_valid"]
    for b in range(fr.shape[0]):
        assert abs(fr[b].sum() / lit - 1.0) < 1e-5, (name, b, fr[b].sum(), lit)


# P3 / P4: flat wavefront -> the four pupil images are mirror copies with equal flux, slopes vanish
@pytest.mark.parametrize("name", ["cfg1_tiny", "cfg3_npot", "cfg4_elt"])
def test_flat_wavefront_mirror_images_and_zero_slopes(torch_cuda, golden, name):
    cfg = wl.CONFIGS[name]
    N, ns = cfg.n_pupil, cfg.n_subap
    fr, sl, _, _ = _run(torch_cuda, cfg, np.zeros((1, N, N), np.float32))
    f = fr[0]
    a, b, c, d = f[:ns, :ns], f[:ns, ns:], f[ns:, :ns], f[ns:, ns:]
    scale = f.max()
    assert np.abs(b - a[:, ::-1]).max() < 1e-5 * scale
    assert np.abs(c - a[::-1, :]).max() < 1e-5 * scale
    assert np.abs(d - a[::-1, ::-1]).max() < 1e-5 * scale
    assert np.abs(sl).max() < 2e-5
    if name == "cfg1_tiny":
        for t in (a, b, c, d):
            assert abs(t.sum() - golden["P3_cfg1_flat_flux_per_pupil_image"]) < 799.0 * 1e-5
        assert np.abs(a - a.T).max() < 1e-5 * scale                       # pupil symmetric under x <-> y, K % 4 == 0
    if name == "cfg4_elt":                                                # 16-px margins drop 1.97 % of the light
        lit = float(wl.make_pupil(cfg).sum())
        assert abs(f.sum() / lit - golden["P3_cfg4_flat_fraction_inside_windows"]) < 1e-4


# P5: +-tilt antisymmetry, sign convention (+x tilt => Sx > 0, +y tilt => Sy > 0), x <-> y exchange
def test_tilt_sign_and_antisymmetry(torch_cuda):
    cfg = wl.CONFIGS["cfg1_tiny"]
    N = cfg.n_pupil
    phase = np.stack([wl.tilt_phase(N, +0.1), wl.tilt_phase(N, -0.1), wl.tilt_phase(N, 0.0, +0.1)])
    _, sl, valid, nv = _run(torch_cuda, cfg, phase)
    sxp, syp, sxm = sl[0, :nv], sl[0, nv:], sl[1, :nv]
    assert sxp.mean() > 0.01 and abs(syp.mean()) < 2e-6
    assert np.abs(_to2d(sxp, valid) + _to2d(sxm, valid)[:, ::-1]).max() < 2e-5
    assert sl[2, nv:].mean() > 0.01 and abs(sl[2, :nv].mean()) < 2e-6
    assert np.abs(_to2d(sl[2, nv:], valid) - _to2d(sxp, valid).T).max() < 2e-5


# P6: small-tilt linearity and the three values SURVEY.md states for cfg1
def test_small_tilt_response_values_from_survey(torch_cuda, golden):
    cfg = wl.CONFIGS["cfg1_tiny"]
    N = cfg.n_pupil
    alphas = [0.05, 0.1, 0.2]
    _, sl, _, nv = _run(torch_cuda, cfg, np.stack([wl.tilt_phase(N, a) for a in alphas]))
    got = {a: sl[i, :nv].mean() for i, a in enumerate(alphas)}
    for key, val in golden["P6_cfg1_mean_sx_vs_alpha"].items():
        assert abs(got[float(key)] - val) < 5e-6, (key, got[float(key)], val)
    assert abs(got[0.1] / got[0.05] - 2.0) < 0.03
    assert got[0.2] / got[0.1] < 2.0


# P10: geometric-optics gain (2/pi) asin(alpha/r) with well-sampled modulation; the full cfg4 geometry value
def test_geometric_gain(torch_cuda, golden):
    g = golden["P10_geometric_gain"]
    cfg = wl.CONFIGS["cfg1_tiny"]
    _, sl, _, nv = _run(torch_cuda, cfg, wl.tilt_phase(cfg.n_pupil, 0.1)[None], mod_points=48)
    ratio = sl[0, :nv].mean() / (2.0 / math.pi * math.asin(0.1 / cfg.mod_radius))
    assert abs(ratio - g["ratio_N64_M128_K48_r3"]) < 2e-3
    cfg4 = wl.CONFIGS["cfg4_elt"]
    _, sl4, _, nv4 = _run(torch_cuda, cfg4, wl.tilt_phase(cfg4.n_pupil, 0.1)[None])
    assert abs(sl4[0, :nv4].mean() - g["cfg4_alpha0.1_mean_sx"]) < 5e-6


# Non-finite phase values propagate (include/pwfs.h): the frame that holds one comes out non-finite, its neighbours do not
def test_non_finite_phase_propagates_to_its_own_frame_only(torch_cuda):
    cfg = wl.CONFIGS["cfg1_tiny"]
    phase = wl.phase_batch(cfg, steps=3)
    phase[1, 20, 30] = np.nan
    fr, sl, _, _ = _run(torch_cuda, cfg, phase)
    assert not np.isfinite(fr[1]).all() and not np.isfinite(sl[1]).all()
    assert np.isfinite(fr[0]).all() and np.isfinite(fr[2]).all()
    assert np.isfinite(sl[0]).all() and np.isfinite(sl[2]).all()


# ---- full-resolution intensity through the test-only export (pins P2, P3, P7 on the CUDA path) -------
def test_identity_mask_returns_the_embedded_pupil(torch_cuda):
    """P7: s = 0 (mask == 1), r = 0, K = 1: IDFT2(DFT2(G)) = G, so I is A^2 at offset o = M/2 - N/2 whatever the phase.
    Checks padding offset, both transform scalings and the window/column bookkeeping of the kernels."""
    from paper_1607_07624_b200.pwfs import PWFS
    torch = torch_cuda
    for N, M in [(64, 128), (60, 128), (160, 320), (100, 256)]:
        rng = np.random.default_rng(N + M)
        A = (rng.random((N, N)) > 0.2).astype(np.float32) * (0.5 + rng.random((N, N))).astype(np.float32)
        phase = (rng.standard_normal((2, N, N)) * 5.0).astype(np.float32)
        with PWFS(A, M, 0.0, 1, N // 4, debug_shift_px=0) as sensor:
            I = sensor.debug_intensity(torch.from_numpy(phase).cuda()).cpu().numpy().astype(np.float64)
            with pytest.raises(Exception):
                sensor.run(torch.from_numpy(phase).cuda())                   # a debug handle does not serve the hot path
        o = M // 2 - N // 2
        want = np.zeros((M, M))
        want[o:o + N, o:o + N] = A.astype(np.float64) ** 2
        for b in range(2):
            assert np.abs(I[b] - want).max() < 2e-6 * want.max(), (N, M, b, np.abs(I[b] - want).max())


def test_full_resolution_flux_and_flat_wavefront_symmetry(torch_cuda, golden):
    """P2: sum I = sum A^2 over the whole grid (Parseval through both transforms, unit-modulus mask, mean over k);
    P3: flat wavefront -> I mirror-symmetric in x and y and under transposition (cfg1: symmetric pupil, K % 4 == 0)."""
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    N, M = cfg.n_pupil, cfg.m_grid
    phase = np.concatenate([np.zeros((1, N, N), np.float32), wl.phase_batch(cfg, steps=1)])
    with from_config(cfg) as sensor:
        I = sensor.debug_intensity(torch.from_numpy(phase).cuda()).cpu().numpy().astype(np.float64)
    lit = golden["P2_cfg1_total_flux"]
    for b in range(2):
        assert abs(I[b].sum() / lit - 1.0) < 1e-5
    flat = I[0]
    assert np.abs(flat - flat[:, ::-1]).max() < 1e-5 * flat.max()
    assert np.abs(flat - flat[::-1, :]).max() < 1e-5 * flat.max()
    assert np.abs(flat - flat.T).max() < 1e-5 * flat.max()
