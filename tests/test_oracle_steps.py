"""Pins for the oracle's pointwise operators: carousel mix (Eq. (4)), Fourier-modulus
constraint and support/HIO update (P:98 ref [22]).  Each test states a property
that the paper or the mathematics fixes, chosen so that a dropped term, a wrong sign or index, or a
transposed operand fails at least one of them (SURVEY.md 8(c) "pins")."""
import os

import numpy as np

from oracle import Oracle, fft2, hio, mix, modulus

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _stack(Np, N, seed):
    rng = np.random.default_rng(seed)
    return rng.normal(size=(Np, N, N)) + 1j * rng.normal(size=(Np, N, N))


# ---------------------------------------------------------------- mix
def _paper_alpha():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "alpha_example.txt")) if not l.startswith("#")]
    return {int(k): float(v) for k, v in rows}


def test_default_weights_are_the_papers_example():
    # alpha_0 = 0.6, alpha_+-1 = 0.2; a one-hot stack through a default plan shows them, with wrap
    al = _paper_alpha()
    Np, N = 5, 4
    for j in (0, 2, Np - 1):
        g = np.zeros((Np, N, N), complex)
        g[j] = 1.0
        o = Oracle(N, Np)
        # M = 0 everywhere and S = 1 everywhere: one iteration returns exactly the mixed stack
        o.set_data(np.ones((Np, N, N)), np.zeros((Np, N, N), np.uint8))
        o.set_support(np.ones((Np, N, N), np.uint8))
        o.set_estimate(g)
        o.iterate(1, 0.9)
        out = o.get_projections(0)
        for n in range(Np):
            d = (n - j + Np // 2) % Np - Np // 2         # signed distance n - j on the ring
            want = al.get(d, 0.0)
            assert np.abs(out[n] - want).max() < 1e-15, (j, n)


def test_mix_constant_stack_sum_and_onehot_wrap():
    Np, N = 7, 4
    alpha = [0.6, 0.2]
    img = _stack(1, N, 1)[0]
    const = np.repeat(img[None], Np, axis=0)
    assert np.abs(mix(const, alpha) - const).max() < 1e-15           # sum(alpha)=1
    g = _stack(Np, N, 2)
    m = mix(g, alpha)
    assert np.abs(m.sum(axis=0) - g.sum(axis=0)).max() < 1e-13       # sum over n conserved
    for j in (0, Np - 1):
        e = np.zeros((Np, N, N), complex)
        e[j] = img
        me = mix(e, alpha)
        assert np.abs(me[j] - 0.6 * img).max() < 1e-15
        assert np.abs(me[(j - 1) % Np] - 0.2 * img).max() < 1e-15
        assert np.abs(me[(j + 1) % Np] - 0.2 * img).max() < 1e-15
        assert np.abs(me[(j + 3) % Np]).max() == 0.0


def test_mix_circulant_eigenvalues():
    # g_n = e^{2 pi i m n/Np} img  =>  ghat_n = (a0 + 2 a1 cos(2 pi m/Np) + 2 a2 cos(4 pi m/Np)) g_n
    Np, N = 9, 4
    img = _stack(1, N, 3)[0]
    alpha = [0.5, 0.15, 0.1]
    for m_ in (0, 1, 4):
        ph = np.exp(2j * np.pi * m_ * np.arange(Np) / Np)
        g = ph[:, None, None] * img
        lam = alpha[0] + 2 * alpha[1] * np.cos(2 * np.pi * m_ / Np) + 2 * alpha[2] * np.cos(4 * np.pi * m_ / Np)
        assert np.abs(mix(g, alpha) - lam * g).max() < 1e-14


def test_mix_is_jacobi_not_sequential():
    # with a sequential (Gauss-Seidel) sweep image 1 would see the already-mixed image 0
    Np, N = 4, 2
    g = np.zeros((Np, N, N), complex)
    g[0] = 1.0
    m = mix(g, [0.6, 0.2])
    assert abs(m[1, 0, 0] - 0.2) < 1e-16 and abs(m[2, 0, 0]) < 1e-16 and abs(m[3, 0, 0] - 0.2) < 1e-16


# ---------------------------------------------------------------- modulus
def test_modulus_properties():
    N = 16
    rng = np.random.default_rng(5)
    G = _stack(1, N, 4)[0]
    A = rng.uniform(0.1, 3.0, size=(N, N))
    M = (rng.uniform(size=(N, N)) > 0.2).astype(np.uint8)
    G[2, 3] = 0.0                                                    # |G| = 0 on a measured pixel
    M[2, 3] = 1
    Gp, num = modulus(G, A, M)
    meas = M == 1
    assert np.abs(np.abs(Gp[meas]) - A[meas]).max() < 1e-14           # |G'| = A where measured
    nz = meas & (np.abs(G) > 0)
    assert np.abs(np.angle(Gp[nz] * np.conj(G[nz]))).max() < 1e-14    # phase kept
    assert np.array_equal(Gp[~meas], G[~meas])                        # masked: bit-identical
    assert Gp[2, 3] == A[2, 3]                                        # |G|=0: phase 0 (reading A13)
    Gpp, num2 = modulus(Gp, A, M)                                     # idempotent, and then error 0
    assert np.abs(Gpp - Gp).max() < 1e-14 and num2 < 1e-26
    assert abs(num - ((np.abs(G[meas]) - A[meas]) ** 2).sum()) < 1e-10 * num


def test_twin_image_has_the_same_modulus():
    # |F[O(r)]| = |F[O(-r)]| for the (real) projected density
    N = 32
    rng = np.random.default_rng(6)
    g = rng.normal(size=(N, N)).astype(complex)
    twin = np.roll(g[::-1, ::-1], (1, 1), axis=(0, 1))                # g(-r) on the periodic grid
    assert np.abs(np.abs(fft2(g)) - np.abs(fft2(twin))).max() < 1e-11


# ---------------------------------------------------------------- HIO
def test_hio_operator():
    N = 8
    rng = np.random.default_rng(7)
    ghat, gp = _stack(2, N, 8)
    S = (rng.uniform(size=(N, N)) > 0.5).astype(np.uint8)
    out = hio(ghat, gp, S, 0.9)
    assert np.array_equal(out[S == 1], gp[S == 1])
    assert np.abs(out[S == 0] - (ghat[S == 0] - 0.9 * gp[S == 0])).max() < 1e-15
    # projecting twice with the support (beta irrelevant inside) is idempotent inside S
    assert np.array_equal(hio(out, gp, S, 0.9)[S == 1], gp[S == 1])


def test_hio_closed_form_nothing_measured():
    # M = 0 everywhere, no coupling (K=0): g' = ghat, so inside S nothing changes and outside
    # g <- (1 - beta) g each iteration  =>  (1-beta)^k g0 after k iterations.
    Np, N, k, beta = 3, 8, 5, 0.9
    rng = np.random.default_rng(9)
    g0 = _stack(Np, N, 10)
    S = (rng.uniform(size=(Np, N, N)) > 0.5).astype(np.uint8)
    o = Oracle(N, Np)
    o.set_data(np.ones((Np, N, N)), np.zeros((Np, N, N), np.uint8))
    o.set_support(S)
    o.set_carousel([1.0], 1)
    o.set_estimate(g0)
    o.iterate(k, beta)
    out = o.get_projections(0)
    assert np.abs(out[S == 1] - g0[S == 1]).max() < 1e-13
    assert np.abs(out[S == 0] - (1 - beta) ** k * g0[S == 0]).max() < 1e-13


def test_full_support_one_iteration_matches_modulus_then_nothing_changes():
    Np, N = 2, 16
    rng = np.random.default_rng(11)
    g0 = _stack(Np, N, 12)
    I = rng.uniform(0.5, 4.0, size=(Np, N, N))
    o = Oracle(N, Np)
    o.set_data(I)
    o.set_support(np.ones((Np, N, N), np.uint8))
    o.set_carousel([1.0], 1)
    o.set_estimate(g0)
    o.iterate(1, 0.9)
    g1 = o.get_projections(0)
    A_native = np.fft.ifftshift(np.sqrt(I), axes=(-2, -1))
    assert np.abs(np.abs(fft2(g1)) - A_native).max() < 1e-11           # |F[g]| = A exactly
    o.iterate(1, 0.9)
    assert np.abs(o.get_projections(0) - g1).max() < 1e-13             # second iteration: no change
    assert o.get_error()[1] < 1e-13


# ---------------------------------------------------------------- A0: negative intensities
def test_negative_intensity_is_clamped_to_zero_amplitude():
    """I = |E|^2 cannot be negative; reading A14: I < 0 => A = 0.  With everything
    measured and S = 1 everywhere one iteration returns g' itself, whose Fourier modulus (numpy's
    FFT, not the oracle's) is exactly A: 0 on the pixels with I < 0, sqrt(I) elsewhere -- not
    sqrt(|I|).  den_n counts the clamped intensities: a zero estimate has num_n = sum A^2 = den_n."""
    Np, N = 3, 8
    rng = np.random.default_rng(31)
    I_c = rng.gamma(2.0, 3.0, size=(Np, N, N))
    neg = rng.uniform(size=(Np, N, N)) < 0.3
    I_c[neg] *= -1.0
    g0 = _stack(Np, N, 32)
    o = Oracle(N, Np)
    o.set_data(I_c)
    o.set_support(np.ones((Np, N, N), np.uint8))
    o.set_carousel([1.0], 1)
    o.set_estimate(g0)
    o.iterate(1, 0.9)
    mod = np.abs(np.fft.fftshift(np.fft.fft2(o.get_projections(0)), axes=(-2, -1)))     # detector-centred
    assert neg.any() and mod[neg].max() < 1e-12
    assert np.abs(mod[~neg] - np.sqrt(I_c[~neg])).max() < 1e-12
    z = Oracle(N, Np)
    z.set_data(I_c)
    z.set_support(np.ones((Np, N, N), np.uint8))
    z.set_carousel([1.0], 1)
    z.set_estimate(np.zeros((Np, N, N), complex))
    z.iterate(1, 0.9)
    E, Eg = z.get_error()
    assert np.abs(E - 1.0).max() < 1e-14 and abs(Eg - 1.0) < 1e-14
    # and the error of g0 is normalised by the clamped sum, not by sum |I|
    G = np.abs(np.fft.fftshift(np.fft.fft2(g0), axes=(-2, -1)))
    A = np.sqrt(np.maximum(I_c, 0.0))
    want = np.sqrt(((G - A) ** 2).sum(axis=(1, 2)) / np.maximum(I_c, 0.0).sum(axis=(1, 2)))
    o2 = Oracle(N, Np)
    o2.set_data(I_c)
    o2.set_support(np.ones((Np, N, N), np.uint8))
    o2.set_carousel([1.0], 1)
    o2.set_estimate(g0)
    o2.iterate(1, 0.9)
    assert np.abs(o2.get_error()[0] - want).max() < 1e-12
