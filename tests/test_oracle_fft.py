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


def test_sizes_that_are_not_powers_of_two_against_numpy():
    """The paper's own detector sizes are 160 = 2^5 5 and 700 = 2^2 5^2 7: for such N the
    oracle's transform is the O(N^2)-per-line definition; numpy's FFT is the independent library."""
    from oracle import fft2
    for N in (12, 20, 28, 160):
        rng = np.random.default_rng(N)
        x = rng.normal(size=(2, N, N)) + 1j * rng.normal(size=(2, N, N))
        F = fft2(x, -1)
        assert np.abs(F - np.fft.fft2(x)).max() < 1e-10 * np.abs(F).max()
        assert np.abs(fft2(F, +1) - x).max() < 1e-12
    d = np.zeros((20, 20), complex)
    d[3, 7] = 1.0
    ky, kx = np.meshgrid(np.arange(20), np.arange(20), indexing="ij")
    assert np.abs(fft2(d, -1) - np.exp(-2j * np.pi * (3 * ky + 7 * kx) / 20)).max() < 1e-13


def test_loop_on_a_size_that_is_not_a_power_of_two():
    """The whole iteration at N = 20: the true projections with exact intensities are a fixed point, and one
    HIO iteration equals its definition evaluated with numpy's FFT."""
    from oracle import Oracle
    N, Np = 20, 3
    rng = np.random.default_rng(5)
    P = np.zeros((Np, N, N), complex)
    P[:, 6:14, 5:13] = rng.uniform(0.2, 1.0, size=(Np, 8, 8))
    I_c = np.fft.fftshift(np.abs(np.fft.fft2(P)) ** 2, axes=(-2, -1))
    S = np.zeros((Np, N, N), np.uint8)
    S[:, 5:15, 4:14] = 1
    o = Oracle(N, Np)
    o.set_data(I_c)
    o.set_support(S)
    o.set_carousel([1.0], 1)
    o.set_estimate(P)
    o.iterate(2, 0.9)
    assert np.abs(o.get_projections(0) - P).max() < 1e-12 and o.get_error()[1] < 1e-12
    g0 = rng.normal(size=(Np, N, N)) + 1j * rng.normal(size=(Np, N, N))
    o.set_carousel([0.6, 0.2], 1)
    o.set_estimate(g0)
    o.iterate(1, 0.9)
    gh = 0.6 * g0 + 0.2 * (np.roll(g0, 1, axis=0) + np.roll(g0, -1, axis=0))
    G = np.fft.fft2(gh)
    gp = np.fft.ifft2(np.sqrt(np.fft.ifftshift(I_c, axes=(-2, -1))) * G / np.abs(G))
    want = np.where(S == 1, gp, gh - 0.9 * gp)
    assert np.abs(o.get_projections(0) - want).max() < 1e-12
