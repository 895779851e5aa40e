"""The seeded input generators (shared by oracle-side and CUDA-side tests)."""
import numpy as np
import pytest

from paper_1607_07624_b200 import workloads as wl


def test_configs_match_baseline_json_shapes():
    exp = {"cfg1_tiny": (64, 128, 12, 16, 10), "cfg2_flao": (160, 320, 24, 40, 1000),
           "cfg3_npot": (240, 480, 36, 40, 500), "cfg4_elt": (480, 1024, 48, 92, 100),
           "cfg5_multi": (400, 800, 32, 80, 600)}
    for name, (N, M, K, ns, B) in exp.items():
        c = wl.CONFIGS[name]
        assert (c.n_pupil, c.m_grid, c.mod_points, c.n_subap, c.batch) == (N, M, K, ns, B)
        assert c.m_grid >= 2 * c.n_pupil
    assert wl.CONFIGS["cfg5_multi"].instances == 12


def test_pupils_are_binary_and_symmetric():
    for name in wl.CONFIG_ORDER:
        A = wl.make_pupil(wl.CONFIGS[name])
        assert A.dtype == np.float32 and set(np.unique(A)) <= {0.0, 1.0}
        assert np.array_equal(A, A[::-1]) and np.array_equal(A, A[:, ::-1])
    A4 = wl.make_pupil(wl.CONFIGS["cfg4_elt"])
    N = A4.shape[0]
    assert A4[N // 2, N // 2] == 0 and A4[N // 2, N - 5] == 0     # obstruction; spider along +x
    assert 0.65 < A4.mean() < 0.75


def test_screens_are_seeded_and_have_von_karman_variance():
    a = wl.vk_screen(256, 0.125, 0.244, 25.0, 7)
    b = wl.vk_screen(256, 0.125, 0.244, 25.0, 7)
    c = wl.vk_screen(256, 0.125, 0.244, 25.0, 8)
    assert np.array_equal(a, b) and not np.array_equal(a, c)
    # expected variance = sum of the sampled PSD (~163 rad^2 for this grid)
    f = np.fft.fftfreq(256, 0.125)
    fx, fy = np.meshgrid(f, f)
    psd = 0.0229 * 0.244 ** (-5 / 3) * (fx ** 2 + fy ** 2 + 1 / 25.0 ** 2) ** (-11 / 6)
    psd[0, 0] = 0
    expect = psd.sum() * (1 / (256 * 0.125)) ** 2
    var = np.mean([wl.vk_screen(256, 0.125, 0.244, 25.0, s).var() for s in range(20)])
    assert abs(var / expect - 1) < 0.25


def test_phase_batches_shapes_order_and_frozen_flow():
    c1 = wl.CONFIGS["cfg1_tiny"]
    p = wl.phase_batch(c1, steps=3)
    assert p.shape == (3, 64, 64) and p.dtype == np.float32
    assert np.array_equal(p, wl.phase_batch(c1, steps=3))
    assert np.array_equal(p[2], wl.phase_batch(c1, steps=1, first_step=2)[0])
    c5 = wl.CONFIGS["cfg5_multi"]
    q = wl.phase_batch(c5, steps=1)
    assert q.shape == (12, 400, 400)
    # star-major, wavelength-minor: instance 1 is star 0 at 2200 nm = instance 0 scaled by 1650/2200
    assert np.allclose(q[1], q[0] * (1650.0 / 2200.0), rtol=1e-5, atol=1e-5)
    assert not np.allclose(q[2], q[0])
    c2 = wl.CONFIGS["cfg2_flao"]
    r = wl.phase_batch(c2, steps=2)
    assert 0.0 < np.abs(r[1] - r[0]).max() < 0.5 * np.ptp(r[0])    # frozen flow: small step-to-step change


def test_tilt_phase_and_shard_range():
    t = wl.tilt_phase(8, 1.0)
    assert abs((t[0, -1] - t[0, 0]) - 2 * np.pi * 7 / 8) < 1e-6 and abs(t.mean()) < 1e-6
    for n, w in [(100, 8), (7, 3), (5, 8), (0, 2)]:
        rs = [wl.shard_range(n, r, w) for r in range(w)]
        assert rs[0][0] == 0 and rs[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(rs, rs[1:]))
        sizes = [hi - lo for lo, hi in rs]
        assert max(sizes) - min(sizes) <= 1
