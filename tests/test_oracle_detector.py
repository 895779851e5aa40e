"""Pins P11 (rebin), P12 (valid mask) and a hand-worked slope example for the
oracle's detector side (O7-O9)."""
import numpy as np
import pytest

from oracle import pwfs_oracle as orc
from paper_1607_07624_b200 import workloads as wl


@pytest.mark.parametrize("N,ns", [(64, 16), (160, 40), (240, 40), (480, 92), (400, 80), (10, 3), (7, 7)])
def test_rebin_weights_partition_of_unity(N, ns):
    W = orc.rebin_weights(N, ns)
    assert W.shape == (ns, N)
    assert np.abs(W.sum(axis=0) - 1.0).max() < 1e-14            # every source px is used once
    assert np.abs(W.sum(axis=1) - N / ns).max() < 1e-13          # every bin is b px wide
    assert (W >= 0).all()
    # integer-scaled weights are integers (exact rationals k / n_sub)
    assert np.abs(W * ns - np.round(W * ns)).max() < 1e-12
    # contiguous support, at most ceil(b)+1 px
    for i in range(ns):
        nz = np.nonzero(W[i])[0]
        assert nz.size <= int(np.ceil(N / ns)) + 1 and (np.diff(nz) == 1).all()


def test_rebin_weights_worked_example():
    # N=10 px into 3 bins, b = 10/3: bin 0 = [0, 3.333), bin 1 = [3.333, 6.667), bin 2 = rest
    W = orc.rebin_weights(10, 3)
    third = 1.0 / 3.0
    ref = np.array([[1, 1, 1, third, 0, 0, 0, 0, 0, 0],
                    [0, 0, 0, 2 * third, 1, 1, 2 * third, 0, 0, 0],
                    [0, 0, 0, 0, 0, 0, third, 1, 1, 1]])
    assert np.abs(W - ref).max() < 1e-15


@pytest.mark.parametrize("N,M,ns", [(64, 128, 16), (60, 128, 23), (48, 128, 10)])
def test_frame_constant_image_flux_and_windows(N, M, ns):
    s = M // 4
    b = N / ns
    const = np.full((M, M), 2.5)
    fr = orc.frame(const, N, s, ns)
    assert fr.shape == (2 * ns, 2 * ns)
    assert np.abs(fr - 2.5 * b * b).max() < 1e-12
    rng = np.random.default_rng(N)
    I = rng.random((M, M))
    fr = orc.frame(I, N, s, ns)
    tot = 0.0
    for qy in (0, 1):
        for qx in (0, 1):
            wx = M // 2 + (2 * qx - 1) * s - N // 2
            wy = M // 2 + (2 * qy - 1) * s - N // 2
            win = I[wy:wy + N, wx:wx + N]
            tot += win.sum()
            tile = fr[qy * ns:(qy + 1) * ns, qx * ns:(qx + 1) * ns]
            assert abs(tile.sum() - win.sum()) < 1e-9             # rebin is a SUM
            if N % ns == 0:                                      # integer b == block sums
                bb = N // ns
                ref = win.reshape(ns, bb, ns, bb).sum(axis=(1, 3))
                assert np.abs(tile - ref).max() < 1e-12
    assert abs(fr.sum() - tot) < 1e-9


def test_frame_places_quadrants_by_qx_qy():
    # light only in the (x-, y+) window must land in tile (qx=0, qy=1) = lower-left block
    N, M, ns = 16, 64, 4
    s = M // 4
    I = np.zeros((M, M))
    wx, wy = M // 2 - s - N // 2, M // 2 + s - N // 2
    I[wy + 2, wx + 13] = 1.0                                    # row (y) 2, column (x) 13
    fr = orc.frame(I, N, s, ns)
    assert fr[ns + 0, 0 + 3] == 1.0 and fr.sum() == 1.0


def test_frame_rejects_windows_outside_the_grid():
    with pytest.raises(RuntimeError):
        orc.frame(np.zeros((64, 64)), 40, 16, 4)               # 32 - 16 - 20 < 0


def test_valid_mask_counts_ties_and_symmetry(golden):
    for name, g in golden["configs"].items():
        cfg = wl.CONFIGS[name]
        assert (cfg.n_pupil, cfg.m_grid, cfg.mod_points, cfg.n_subap) == (g["N"], g["M"], g["K"], g["n_sub"])
        A = wl.make_pupil(cfg)
        assert int(A.sum()) == g["lit_px"]
        v, nv = orc.valid_mask(A, cfg.n_subap, 0.5)
        assert nv == g["n_valid"] == int(v.sum())
        assert np.array_equal(v, v[:, ::-1]) and np.array_equal(v, v[::-1, :])
        if "ties_at_half" in g:                                  # `>=` keeps exact 50 % ties
            _, nv_strict = orc.valid_mask(A, cfg.n_subap, 0.5 + 1e-9)
            assert nv - nv_strict == g["ties_at_half"]


def test_valid_mask_against_block_sums_for_integer_binning():
    cfg = wl.CONFIGS["cfg2_flao"]
    A = wl.make_pupil(cfg)
    b = cfg.n_pupil // cfg.n_subap
    ill = (A.astype(np.int64) ** 2).reshape(cfg.n_subap, b, cfg.n_subap, b).sum(axis=(1, 3))
    v, _ = orc.valid_mask(A, cfg.n_subap, 0.5)
    assert np.array_equal(v.astype(bool), 2 * ill >= b * b)


def test_valid_mask_scales_with_amplitude():
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    v1, n1 = orc.valid_mask(A, cfg.n_subap)
    v2, n2 = orc.valid_mask(3.0 * A, cfg.n_subap)
    assert n1 == n2 and np.array_equal(v1, v2)


def test_slopes_hand_worked_example():
    # n_sub = 2; tiles a (top-left), b (top-right), c (bottom-left), d (bottom-right)
    a = np.array([[1.0, 2.0], [3.0, 4.0]])
    b = np.array([[2.0, 2.0], [1.0, 0.0]])
    c = np.array([[0.0, 1.0], [1.0, 2.0]])
    d = np.array([[1.0, 3.0], [3.0, 2.0]])
    fr = np.block([[a, b], [c, d]])
    valid = np.array([[1, 0], [1, 1]], np.uint8)
    # valid subaps (row-major): (0,0), (1,0), (1,1); sums a+b+c+d = 4, 8, 8 -> nbar = 20/3
    nbar = 20.0 / 3.0
    sx = np.array([(1 + 0) - (2 + 1), (3 + 1) - (1 + 3), (4 + 2) - (0 + 2)]) / nbar
    sy = np.array([(1 + 2) - (0 + 1), (3 + 1) - (1 + 3), (4 + 0) - (2 + 2)]) / nbar
    got = orc.slopes(fr, valid, 0)
    assert np.abs(got - np.concatenate([sx, sy])).max() < 1e-15
    got1 = orc.slopes(fr, valid, 1)                              # per-subaperture normalisation
    sums = np.array([4.0, 8.0, 8.0])
    assert np.abs(got1 - np.concatenate([sx * nbar / sums, sy * nbar / sums])).max() < 1e-15


def test_slopes_no_valid_subaperture_is_an_error():
    with pytest.raises(RuntimeError):
        orc.slopes(np.ones((4, 4)), np.zeros((2, 2), np.uint8))
