"""Pins of the f2 oracle (oracle/chain_oracle.py): detector, slope reference,
reconstructor.  Each pin is something other than the oracle's own formula: published
known-answer vectors, scipy's distribution functions, moments, closed forms, and the closed
chain through the hot-path oracle."""
import json
import os

import numpy as np
import pytest
from scipy import stats

from oracle import chain_oracle as co
from oracle import pwfs_oracle as orc
from paper_1607_07624_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.json")


def test_philox_known_answer_vectors():
    # Random123 kat_vectors, philox4x32 10 rounds (Salmon et al., SC'11): zeros, all ones, digits of pi
    with open(GOLD) as f:
        kat = json.load(f)["vectors"]
    assert len(kat) == 3
    for v in kat:
        ctr = [int(x, 16) for x in v["counter"]]
        key = [int(x, 16) for x in v["key"]]
        assert [f"{x:08x}" for x in co.philox4x32_10(ctr, key)] == v["out"]


def test_philox_block_is_the_scalar_generator_at_counter_pixel_frame():
    seed = (0x12345678 << 32) | 0x9ABCDEF0
    frame = (3 << 32) | 0xFFFFFFFE
    blk = co.philox_block(37, frame, seed)
    assert blk.dtype == np.uint32 and blk.shape == (37, 4)
    for i in (0, 1, 17, 36):
        want = co.philox4x32_10((i, 0xFFFFFFFE, 3, 0), (0x9ABCDEF0, 0x12345678))
        assert tuple(int(x) for x in blk[i]) == want


def test_philox_words_look_uniform_and_independent():
    blk = co.philox_block(1 << 16, 5, 42)
    u = co.uniform01(blk)
    assert u.min() > 0.0 and u.max() < 1.0
    for c in range(4):
        assert stats.kstest(u[:, c], "uniform").pvalue > 1e-3
    assert np.abs(np.corrcoef(u.T) - np.eye(4)).max() < 0.02
    # another frame or seed: a different stream
    assert (co.philox_block(64, 6, 42) != blk[:64]).any() and (co.philox_block(64, 5, 43) != blk[:64]).any()


def test_uniform01_end_points():
    assert co.uniform01(0) == 0.5 / 2 ** 32 and co.uniform01(0xFFFFFFFF) == 1.0 - 0.5 / 2 ** 32


@pytest.mark.parametrize("lam", [1e-3, 0.3, 1.0, 4.5, 17.0, 60.0, 127.9])
def test_poisson_inversion_is_the_quantile_function(lam):
    rng = np.random.default_rng(int(lam * 1000))
    u = rng.random(400)
    k = np.array([co.poisson_inversion(lam, x) for x in u])
    want = stats.poisson.ppf(u, lam)
    # away from CDF steps (where 1e-13 of rounding could decide) they agree exactly
    cdf = stats.poisson.cdf(np.arange(0, 400), lam)
    near = np.abs(u[:, None] - cdf[None, :]).min(axis=1) < 1e-12
    assert np.array_equal(k[~near], want[~near])
    assert co.poisson_inversion(lam, 1e-300) == 0
    assert co.poisson_inversion(0.0, 0.7) == 0 and co.poisson_inversion(-1.0, 0.7) == 0


def test_poisson_counts_moments_both_branches():
    n = 20000
    u = co.uniform01(co.philox_block(n, 0, 7))
    for lam in (0.05, 2.0, 50.0, 127.0, 128.0, 900.0):
        k = co.poisson_counts(np.full(n, lam), u[:, 0], u[:, 1])
        assert np.array_equal(k, np.round(k)) and k.min() >= 0
        assert abs(k.mean() - lam) < 5 * np.sqrt(lam / n)
        assert abs(k.var() / lam - 1.0) < 0.05
    # small lam: the whole distribution against the pmf
    k = co.poisson_counts(np.full(n, 3.0), u[:, 0], u[:, 1]).astype(int)
    obs = np.bincount(k, minlength=12)[:12]
    exp = stats.poisson.pmf(np.arange(12), 3.0) * n
    assert stats.chisquare(obs[:10], exp[:10] * obs[:10].sum() / exp[:10].sum()).pvalue > 1e-3


def test_normal_branch_is_rounded_gaussian():
    lam, ua, ub = 400.0, 0.3, 0.125
    z = np.sqrt(-2 * np.log(ua)) * np.cos(2 * np.pi * ub)
    assert co.poisson_counts([lam], [ua], [ub])[0] == np.floor(lam + 20.0 * z + 0.5)
    assert co.poisson_counts([128.0], [1e-9], [0.5])[0] >= 0.0          # clipped at 0 (z = -6.4)


def test_box_muller_identity_and_normality():
    u = co.uniform01(co.philox_block(1 << 15, 1, 3))
    z = co.box_muller(u[:, 0], u[:, 1])
    zs = np.sqrt(-2 * np.log(u[:, 0])) * np.sin(2 * np.pi * u[:, 1])
    assert np.allclose(z * z + zs * zs, -2 * np.log(u[:, 0]), rtol=1e-12)
    assert stats.kstest(z, "norm").pvalue > 1e-3
    assert co.box_muller(np.exp(-0.5), 0.0) == pytest.approx(1.0, abs=1e-15)
    assert co.box_muller(np.exp(-0.5), 0.5) == pytest.approx(-1.0, abs=1e-15)


def test_integration_is_a_reshape_sum():
    rng = np.random.default_rng(0)
    n_steps, n_inst, n_int, D = 12, 3, 4, 6
    fr = rng.random((n_steps * n_inst, D, D))
    got = co.integrate(fr, n_inst, n_int)
    want = fr.reshape(n_steps // n_int, n_int, n_inst, D, D).sum(axis=1).reshape(-1, D, D)
    assert np.allclose(got, want, rtol=0, atol=1e-13)
    assert np.array_equal(co.integrate(fr, n_inst, 1), fr)
    with pytest.raises(ValueError):
        co.integrate(fr, n_inst, 5)


def test_ccd_without_noise_is_qe_gain_sum():
    rng = np.random.default_rng(1)
    fr = rng.random((8, 5, 5))
    pix = co.ccd(fr, n_inst=2, n_int=2, gain=1000.0, quantum_eff=0.32)
    assert np.allclose(pix, 320.0 * co.integrate(fr, 2, 2), rtol=1e-15)


def test_ccd_noise_statistics_and_reproducibility():
    D = 64
    fr = np.full((2, D, D), 1.0)
    kw = dict(gain=25.0, quantum_eff=0.8, photon_noise=True, readout_noise=True, readout_level=3.0, seed=11)
    a = co.ccd(fr, **kw)
    assert np.array_equal(a, co.ccd(fr, **kw))                          # same seed, same pixels
    assert not np.array_equal(a[0], a[1])                               # frame index enters the counter
    assert np.array_equal(co.ccd(fr[1:], first_out_frame=1, **kw)[0], a[1])
    assert abs(a.mean() - 20.0) < 5 * np.sqrt(29.0 / a.size)            # mean qe*gain, var lam + sigma^2
    assert abs(a.var() / 29.0 - 1.0) < 0.06
    only_ron = co.ccd(fr, gain=25.0, quantum_eff=0.8, readout_noise=True, readout_level=3.0, seed=11)
    assert abs((only_ron - 20.0).std() / 3.0 - 1.0) < 0.03
    only_phot = co.ccd(fr, gain=25.0, quantum_eff=0.8, photon_noise=True, seed=11)
    assert np.array_equal(only_phot, np.round(only_phot))
    # read noise rides on top of the same photon counts (separate Philox words)
    assert stats.kstest(((a - only_phot) / 3.0).ravel(), "norm").pvalue > 1e-3


def _tiny_sensor():
    N, M, K, r, ns = 32, 64, 8, 3.0, 8
    yy, xx = (np.mgrid[0:N, 0:N] - (N - 1) / 2.0) / (N / 2.0)
    A = ((xx ** 2 + yy ** 2) <= 1.0).astype(np.float32)
    modes = np.stack([xx, yy, 2 * (xx ** 2 + yy ** 2) - 1, xx ** 2 - yy ** 2, 2 * xx * yy]) * A
    return N, M, K, r, ns, A, modes


def test_reference_slopes_cancel_a_static_aberration():
    N, M, K, r, ns, A, modes = _tiny_sensor()
    static = 0.3 * modes[3]
    _, s = orc.pwfs_run(A, M, r, K, ns, np.stack([static, static + 0.05 * modes[0]]))
    sn = s[0]
    out = co.slopes_with_reference(s, sn)
    assert np.abs(out[0]).max() == 0.0
    assert np.array_equal(out[1], s[1] - s[0])
    assert np.array_equal(co.slopes_with_reference(s, None), s)


def test_reconstructor_closes_the_chain_on_small_modal_inputs():
    # interaction matrix by push-pull through the hot-path oracle, recmat = its pseudo-inverse;
    # a small modal vector must come back (the sensor is linear to ~(a/r)^2 under modulation)
    N, M, K, r, ns, A, modes = _tiny_sensor()
    amp = 0.05
    push = np.concatenate([amp * modes, -amp * modes])
    _, s = orc.pwfs_run(A, M, r, K, ns, push)
    D = ((s[:5] - s[5:]) / (2 * amp)).T                                 # [2 nv][5]
    R = np.linalg.pinv(D)                                               # [5][2 nv]
    assert np.linalg.cond(D) < 50
    a = np.array([0.04, -0.03, 0.02, 0.05, -0.01])
    _, s1 = orc.pwfs_run(A, M, r, K, ns, np.tensordot(a, modes, axes=1)[None])
    _, s0 = orc.pwfs_run(A, M, r, K, ns, np.zeros((1, N, N)))
    got = co.reconstruct(R, co.slopes_with_reference(s1, s0[0]))[0]
    assert np.abs(got - a).max() < 2e-3
    # and it is the plain matrix product, row-major [n_modes][n_slopes]
    assert co.reconstruct(np.array([[1.0, 2.0, 3.0], [0.0, -1.0, 0.5]]), np.array([[1.0, 1.0, 2.0]]))[0] \
        == pytest.approx([9.0, 0.0])


def test_photon_noise_propagates_to_slopes_as_expected():
    # total flux n_ph over the valid subapertures, global-mean normalisation: a flat wavefront
    # gives slope noise variance ~ n_valid / n_ph per element (4 pixels of mean n_ph/(4 n_valid))
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    fr, _ = orc.pwfs_run(A, cfg.m_grid, cfg.mod_radius, cfg.mod_points, cfg.n_subap, np.zeros((1, 64, 64)))
    valid, nv = orc.valid_mask(A, cfg.n_subap)
    n_ph = 2.0e5
    frames = np.repeat(fr, 40, axis=0)
    pix = co.ccd(frames, gain=n_ph / fr.sum(), photon_noise=True, seed=5)
    s = np.stack([orc.slopes(p, valid) for p in pix])
    ns = cfg.n_subap
    tiles = fr[0].reshape(2, ns, 2, ns).sum(axis=(0, 2))[valid.astype(bool)]     # a+b+c+d per subap
    nbar = tiles.mean() * n_ph / fr.sum()
    want_var = (tiles * n_ph / fr.sum()).mean() / nbar ** 2
    assert abs(s.var() / want_var - 1.0) < 0.1
    assert abs(s.mean()) < 5 * np.sqrt(want_var / s.size)
