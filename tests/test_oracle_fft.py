"""Pin P1: the oracle's textbook FFT against the DFT's
definition (brute force) and against an independent library (numpy.fft,
test-only).  A wrong twiddle index, sign, stride or recombination in
oracle/pwfs_oracle.c:fft_rec fails here."""
import numpy as np
import pytest

from oracle import pwfs_oracle as orc

SIZES_1D = [1, 2, 3, 4, 5, 6, 8, 9, 10, 12, 15, 16, 20, 25, 27, 30, 32, 60, 7, 14, 49, 77]


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _definition(x, sign):
    """DFT definition with an explicit exponent matrix (numpy, not the oracle)."""
    n = x.size
    j = np.arange(n)
    W = np.exp(sign * 2j * np.pi * ((j[:, None] * j[None, :]) % n) / n)
    return W @ x


@pytest.mark.parametrize("n", SIZES_1D)
@pytest.mark.parametrize("sign", [-1, 1])
def test_naive_dft_is_the_definition(n, sign):
    rng = np.random.default_rng(n)
    x = _rand(rng, n)
    ref = _definition(x, sign)
    assert np.abs(orc.dft_naive(x, sign) - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())


@pytest.mark.parametrize("n", SIZES_1D)
@pytest.mark.parametrize("sign", [-1, 1])
def test_fft_matches_brute_force(n, sign):
    rng = np.random.default_rng(100 + n)
    x = _rand(rng, n)
    ref = orc.dft_naive(x, sign)
    assert np.abs(orc.fft(x, sign) - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())


def test_fft_delta_and_shift_theorem():
    # delta at j0 -> pure exponential exp(-2 pi i j0 k / n): fixes the sign convention
    n, j0 = 30, 7
    x = np.zeros(n, complex)
    x[j0] = 1.0
    k = np.arange(n)
    assert np.abs(orc.fft(x, -1) - np.exp(-2j * np.pi * j0 * k / n)).max() < 1e-13
    assert np.abs(orc.fft(x, +1) - np.exp(+2j * np.pi * j0 * k / n)).max() < 1e-13


@pytest.mark.parametrize("n", [128, 320, 480, 800, 1024])
def test_fft_1d_against_numpy_at_config_sizes(n):
    rng = np.random.default_rng(n)
    x = _rand(rng, n)
    ref = np.fft.fft(x)
    assert np.abs(orc.fft(x, -1) - ref).max() <= 1e-10 * np.abs(ref).max()
    assert np.abs(orc.fft(x, +1) - np.fft.ifft(x) * n).max() <= 1e-10 * np.abs(ref).max()


@pytest.mark.parametrize("M", [4, 6, 10, 12, 15, 20])
def test_fft2_matches_brute_force_2d(M):
    rng = np.random.default_rng(M)
    a = _rand(rng, M, M)
    j = np.arange(M)
    W = np.exp(-2j * np.pi * ((j[:, None] * j[None, :]) % M) / M)
    ref = W @ a @ W.T                 # F[v][u] = sum_y sum_x a[y][x] w^(ux+vy)
    for naive in (False, True):
        got = orc.fft2(a, -1, naive=naive)
        assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    # a non-symmetric input distinguishes F[v][u] from its transpose
    assert np.abs(ref - ref.T).max() > 1e-3


@pytest.mark.parametrize("M", [128, 320, 480, 800, 1024])
def test_fft2_against_numpy_at_config_sizes(M):
    rng = np.random.default_rng(M)
    a = _rand(rng, M, M)
    ref = np.fft.fft2(a)
    assert np.abs(orc.fft2(a, -1) - ref).max() <= 1e-10 * np.abs(ref).max()
    if M <= 480:
        back = orc.fft2(ref, +1) / (M * M)
        assert np.abs(back - a).max() <= 1e-10 * np.abs(a).max()
