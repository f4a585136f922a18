"""Pins for the oracle's Fourier transforms (SURVEY.md 8(c) "pins", row FFT).

The radix-2 FFT the loop uses is held against: the brute-force O(N^4) DFT (a separate code path in
the oracle), numpy.fft (an independent library; reading A10 makes the conventions equal), and the
identities any correct DFT satisfies."""
import numpy as np
import pytest

from oracle import dft2_naive, fft2


def _rand(N, seed, count=None):
    rng = np.random.default_rng(seed)
    shape = (N, N) if count is None else (count, N, N)
    return rng.normal(size=shape) + 1j * rng.normal(size=shape)


@pytest.mark.parametrize("N", [2, 4, 8, 16])
def test_fft_equals_bruteforce_dft(N):
    a = _rand(N, N)
    assert np.abs(fft2(a, -1) - dft2_naive(a, -1)).max() <= 1e-12 * np.abs(a).sum()
    assert np.abs(fft2(a, +1) - dft2_naive(a, +1)).max() <= 1e-12 * np.abs(a).sum()


def test_bruteforce_dft_is_the_definition():
    # the brute-force routine itself against a hand-evaluated 2x2 case: sum with signs (-1)^(k.x)
    a = np.array([[1 + 2j, 3 - 1j], [-2 + 0.5j, 4j]])
    want = np.array([[a.sum(), a[:, 0].sum() - a[:, 1].sum()],
                     [a[0].sum() - a[1].sum(), a[0, 0] - a[0, 1] - a[1, 0] + a[1, 1]]])
    assert np.allclose(dft2_naive(a, -1), want, atol=1e-14)
    assert np.allclose(dft2_naive(a, +1), want / 4, atol=1e-14)


@pytest.mark.parametrize("N", [16, 64, 128, 512])
def test_fft_equals_numpy(N):
    a = _rand(N, 10 + N, count=2)
    ref = np.fft.fft2(a)
    assert np.abs(fft2(a, -1) - ref).max() <= 1e-12 * np.abs(ref).max()
    refi = np.fft.ifft2(a)
    assert np.abs(fft2(a, +1) - refi).max() <= 1e-12 * np.abs(refi).max()


def test_inverse_of_forward_is_identity_and_parseval():
    a = _rand(64, 3)
    G = fft2(a, -1)
    assert np.abs(fft2(G, +1) - a).max() <= 1e-13
    assert abs((np.abs(a) ** 2).sum() - (np.abs(G) ** 2).sum() / 64 ** 2) <= 1e-10 * (np.abs(a) ** 2).sum()


def test_delta_shift_linearity():
    N = 32
    d = np.zeros((N, N), complex)
    d[0, 0] = 1.0
    assert np.abs(fft2(d) - 1.0).max() <= 1e-14                      # delta -> constant
    d2 = np.zeros((N, N), complex)
    d2[3, 5] = 1.0                                                   # forward sign is e^{-2 pi i k x/N}
    ky, kx = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    assert np.abs(fft2(d2) - np.exp(-2j * np.pi * (3 * ky + 5 * kx) / N)).max() <= 1e-13
    a, b = _rand(N, 1), _rand(N, 2)
    # circular shift theorem: rows are y (first index), columns x
    sh = np.roll(a, (2, 7), axis=(0, 1))
    assert np.abs(fft2(sh) - fft2(a) * np.exp(-2j * np.pi * (2 * ky + 7 * kx) / N)).max() <= 1e-11
    assert np.abs(fft2(2.5 * a - 1j * b) - (2.5 * fft2(a) - 1j * fft2(b))).max() <= 1e-11


def test_rows_and_columns_not_transposed():
    # a pure x-frequency must land in the kx (last) index
    N = 16
    x = np.arange(N)
    img = np.tile(np.exp(2j * np.pi * 3 * x / N), (N, 1))            # varies along x only
    G = fft2(img)
    assert abs(G[0, 3] - N * N) < 1e-9 and np.abs(G).sum() - abs(G[0, 3]) < 1e-8
