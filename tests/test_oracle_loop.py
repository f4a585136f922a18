"""Pins for the whole oracle iteration (SURVEY.md 8(c) "pins": whole iteration, error metric,
equivariances, API).  No expected value comes from the oracle itself: each test states a closed
form, an invariant or a symmetry that the paper's definitions fix."""
import numpy as np

import cpra_inputs
from oracle import Oracle, fft2


def _exact_problem(cfg=1, Np=8, N=None):
    """True projections with exact noise-free double-precision intensities (not rounded to fp32)."""
    p = cpra_inputs.make_problem(cfg, Np=Np, N=N, noise=False)
    P = p.projections
    I_native = np.abs(np.fft.fft2(P)) ** 2
    I_c = np.fft.fftshift(I_native, axes=(-2, -1))
    S = (np.abs(P) > 0).astype(np.uint8) | p.support              # S contains the true support
    return p, P, I_c, S


def test_true_object_is_a_fixed_point_without_coupling():
    p, P, I_c, S = _exact_problem()
    o = Oracle(p.N, p.Np)
    o.set_data(I_c, None, p.angles)
    o.set_support(S)
    o.set_carousel([1.0], 1)                                       # K=0
    o.set_estimate(P)
    o.iterate(3, 0.9)
    assert np.abs(o.get_projections(0) - P).max() <= 1e-12 * np.abs(P).max()
    E, Eg = o.get_error()
    assert Eg < 1e-12 and E.max() < 1e-12


def test_coupled_fixed_point_needs_equal_projections():
    # with the default alpha the true stack is a fixed point only if all projections coincide
    # (an object rotationally symmetric about z); in general it is NOT (adjacent projections differ)
    p, P, I_c, S = _exact_problem()
    same = np.repeat(P[:1], p.Np, axis=0)
    I_same = np.repeat(I_c[:1], p.Np, axis=0)
    S_same = np.repeat(S[:1], p.Np, axis=0)
    o = Oracle(p.N, p.Np)
    o.set_data(I_same)
    o.set_support(S_same)
    o.set_estimate(same)
    o.iterate(2, 0.9)
    assert np.abs(o.get_projections(0) - same).max() <= 1e-12 * np.abs(P).max()
    o2 = Oracle(p.N, p.Np)
    o2.set_data(I_c)
    o2.set_support(S)
    o2.set_estimate(P)
    o2.iterate(1, 0.9)
    assert np.abs(o2.get_projections(0) - P).max() > 1e-3 * np.abs(P).max()


def test_error_metric_closed_forms():
    p, P, I_c, S = _exact_problem()
    for c, want in ((1.3 * np.exp(0.7j), 0.3), (0.25, 0.75), (0.0, 1.0), (1.0, 0.0)):
        o = Oracle(p.N, p.Np)
        o.set_data(I_c)
        o.set_support(S)
        o.set_carousel([1.0], 1)
        o.set_estimate(c * P)
        o.iterate(1, 0.9)
        E, Eg = o.get_error()
        assert abs(Eg - want) < 1e-12 and np.abs(E - want).max() < 1e-12, (c, Eg)


def test_error_metric_ignores_masked_pixels_and_uses_mixed_input():
    p, P, I_c, S = _exact_problem()
    mask = np.ones_like(S)
    mask[:, p.N // 2 - 2:p.N // 2 + 3, p.N // 2 - 2:p.N // 2 + 3] = 0
    o = Oracle(p.N, p.Np)
    o.set_data(I_c, mask)
    o.set_support(S)
    o.set_estimate(P)                               # default alpha: error is that of the MIXED stack
    o.iterate(1, 0.9)
    E, Eg = o.get_error()
    mixed = 0.6 * P + 0.2 * (np.roll(P, 1, axis=0) + np.roll(P, -1, axis=0))
    Gm = np.abs(np.fft.fftshift(np.fft.fft2(mixed), axes=(-2, -1)))
    num = (((Gm - np.sqrt(I_c)) ** 2) * mask).sum(axis=(1, 2))
    den = (I_c * mask).sum(axis=(1, 2))
    assert np.abs(E - np.sqrt(num / den)).max() < 1e-12
    assert abs(Eg - np.sqrt(num.sum() / den.sum())) < 1e-12


def _run(p, g0, S=None, I=None, mask="same", alpha=(0.6, 0.2), n_ei=1, k=3, beta=0.9):
    o = Oracle(p.N, p.Np)
    o.set_data(p.intensity if I is None else I, p.mask if isinstance(mask, str) else mask, p.angles)
    o.set_support(p.support if S is None else S)
    o.set_carousel(list(alpha), n_ei)
    o.set_estimate(g0)
    o.iterate(k, beta)
    return o


def test_equivariances():
    p = cpra_inputs.make_problem(2, Np=6, N=32)
    g0 = p.estimate.astype(np.complex128)
    base = _run(p, g0)
    gb, Eb = base.get_projections(0), base.get_error()[1]
    # global phase
    ph = np.exp(1.1j)
    o = _run(p, ph * g0)
    assert np.abs(o.get_projections(0) - ph * gb).max() < 1e-11 * np.abs(gb).max()
    assert abs(o.get_error()[1] - Eb) < 1e-12
    # joint scaling (g, A) -> (c g, c A): error unchanged, state scales
    o = _run(p, 3.0 * g0, I=9.0 * p.intensity.astype(np.float64))
    assert np.abs(o.get_projections(0) - 3.0 * gb).max() < 1e-11 * np.abs(gb).max()
    assert abs(o.get_error()[1] - Eb) < 1e-12
    # joint circular shift of (g, S)
    sh = (3, -5)
    o = _run(p, np.roll(g0, sh, axis=(1, 2)), S=np.roll(p.support, sh, axis=(1, 2)))
    assert np.abs(o.get_projections(0) - np.roll(gb, sh, axis=(1, 2))).max() < 1e-11 * np.abs(gb).max()
    # cyclic roll of the stack in n rolls the output
    r = 2
    o = _run(p, np.roll(g0, r, axis=0), S=np.roll(p.support, r, axis=0),
             I=np.roll(p.intensity, r, axis=0), mask=np.roll(p.mask, r, axis=0))
    assert np.abs(o.get_projections(0) - np.roll(gb, r, axis=0)).max() < 1e-11 * np.abs(gb).max()


def test_uncoupled_projections_are_independent():
    p = cpra_inputs.make_problem(2, Np=5, N=32)
    g0 = p.estimate.astype(np.complex128)
    full = _run(p, g0, alpha=(1.0,)).get_projections(0)
    perm = np.array([3, 0, 4, 1, 2])
    o = _run(p, g0[perm], S=p.support[perm], I=p.intensity[perm], mask=p.mask[perm], alpha=(1.0,))
    assert np.array_equal(o.get_projections(0), full[perm])
    # and with coupling they are NOT independent (the permuted run differs)
    c1 = _run(p, g0).get_projections(0)
    c2 = _run(p, g0[perm], S=p.support[perm], I=p.intensity[perm], mask=p.mask[perm]).get_projections(0)
    assert np.abs(c2 - c1[perm]).max() > 1e-6 * np.abs(c1).max()


def test_api_split_resume_and_nei():
    p = cpra_inputs.make_problem(2, Np=6, N=32)
    g0 = p.estimate.astype(np.complex128)
    a = _run(p, g0, k=5, n_ei=2)
    b = _run(p, g0, k=2, n_ei=2)
    b.iterate(3, 0.9)
    assert np.array_equal(a.get_projections(0), b.get_projections(0))
    assert a.iteration == b.iteration == 5
    # get -> set round trip with the counter restored resumes exactly (n_ei > 1 needs t)
    c = _run(p, g0, k=3, n_ei=2)
    mid = c.get_projections(0)
    d = Oracle(p.N, p.Np).load(p, n_ei=2)
    d.set_estimate(mid)
    d.set_iteration(3)
    d.iterate(2, 0.9)
    assert np.array_equal(d.get_projections(0), a.get_projections(0))
    # n_ei = 2 equals manual alternation: coupled iteration, then uncoupled iteration
    m = Oracle(p.N, p.Np).load(p)
    m.set_estimate(g0)
    for t in range(4):
        m.set_carousel([0.6, 0.2] if t % 2 == 0 else [1.0], 1)
        m.iterate(1, 0.9)
    e = _run(p, g0, k=4, n_ei=2)
    assert np.abs(m.get_projections(0) - e.get_projections(0)).max() < 1e-13 * np.abs(g0).max()


def test_supported_output_and_hio_feedback_region():
    p = cpra_inputs.make_problem(2, Np=4, N=32)
    o = _run(p, p.estimate.astype(np.complex128), k=2)
    g = o.get_projections(0)
    s = o.get_projections(1)
    assert np.array_equal(s, g * p.support)
    # inside the support the state equals the modulus-constrained estimate g' of the last iteration:
    # its Fourier modulus on measured pixels is A for the part ... checked via |F[g']| on full-support
    # case in test_oracle_steps; here only that outside-support energy is non-zero (HIO feedback).
    assert np.abs(g[p.support == 0]).max() > 0


def test_trajectory_error_decreases_on_tiny(tiny_problem):
    # not a parity pin (PARITY UNPINNED for trajectories): a sanity check that the loop, as read
    # from the paper, actually retrieves phases on the noise-free Tiny config
    p = tiny_problem
    o = Oracle(p.N, p.Np).load(p)
    o.iterate(1, 0.9)
    e0 = o.get_error()[1]
    o.iterate(49, 0.9)
    assert o.get_error()[1] < 0.35 * e0


# ------------------------------------------------------------------------------------------------
# the other real-space updates (reading A22): RAAR (PAPER.md:98 ref [38], :104) and ER
# ------------------------------------------------------------------------------------------------
def _one_uncoupled_iteration(rule, beta, S):
    """One iteration with K = 0 on a seeded random stack, and the modulus-constrained estimate g'
    computed here with numpy's FFT (independent of the oracle's transforms)."""
    rng = np.random.default_rng(5)
    N, Np = 16, 3
    g0 = rng.normal(size=(Np, N, N)) + 1j * rng.normal(size=(Np, N, N))
    I_native = rng.gamma(2.0, 3.0, size=(Np, N, N))
    G = np.fft.fft2(g0)
    gp = np.fft.ifft2(np.sqrt(I_native) * G / np.abs(G))
    o = Oracle(N, Np)
    o.set_data(np.fft.fftshift(I_native, axes=(-2, -1)), None, np.zeros(Np))
    o.set_support(S)
    o.set_carousel([1.0], 1)
    o.set_update(rule)
    o.set_estimate(g0)
    o.iterate(1, beta)
    return g0, gp, o.get_projections(0)


def test_raar_and_er_outside_and_inside_the_support():
    S = np.zeros((3, 16, 16), np.uint8)
    S[:, 4:12, 5:11] = 1
    inside = S.astype(bool)
    for beta in (0.9, 0.5, 0.3):
        g0, gp, out = _one_uncoupled_iteration("raar", beta, S)
        assert np.abs(out[inside] - gp[inside]).max() < 1e-12
        assert np.abs(out[~inside] - (beta * g0 + (1 - 2 * beta) * gp)[~inside]).max() < 1e-12
        g0, gp, out = _one_uncoupled_iteration("hio", beta, S)
        assert np.abs(out[~inside] - (g0 - beta * gp)[~inside]).max() < 1e-12
    g0, gp, out = _one_uncoupled_iteration("er", 0.9, S)
    assert np.abs(out[inside] - gp[inside]).max() < 1e-12 and np.all(out[~inside] == 0)


def test_raar_is_the_relaxed_reflection_formula():
    """RAAR as its authors define it: x+ = beta/2 (R_S R_M + I) x + (1 - beta) P_M x with R = 2P - I,
    evaluated with numpy operators on the whole image, against the oracle's pointwise form."""
    beta = 0.9
    S = np.zeros((3, 16, 16), np.uint8)
    S[:, 3:13, 2:9] = 1
    g0, gp, out = _one_uncoupled_iteration("raar", beta, S)
    RM = 2 * gp - g0
    RSRM = 2 * S * RM - RM
    ref = 0.5 * beta * (RSRM + g0) + (1 - beta) * gp
    assert np.abs(out - ref).max() < 1e-12


def test_true_object_is_a_fixed_point_of_raar_and_er():
    p, P, I_c, S = _exact_problem()
    for rule in ("raar", "er"):
        o = Oracle(p.N, p.Np)
        o.set_data(I_c, None, p.angles)
        o.set_support(S)
        o.set_carousel([1.0], 1)
        o.set_update(rule)
        o.set_estimate(P)
        o.iterate(3, 0.9)
        assert np.abs(o.get_projections(0) - P).max() <= 1e-12 * np.abs(P).max()


# ------------------------------------------------------------------------------------------------
# which state feeds the HIO / RAAR feedback term when the carousel fires (SURVEY.md 8(c) step 6:
# ghat, the MIXED stack -- PAPER.md:58-62: the mix forms "the initial guess for each PO" of the
# episode, and the conventional iteration that follows starts from that guess)
# ------------------------------------------------------------------------------------------------
def test_feedback_term_uses_the_mixed_stack_closed_form():
    """Nothing measured (M = 0: G' = G, so g' = ghat), K = 1, a one-hot stack at n = j.  Outside the
    support one iteration leaves (1 - beta) alpha_|n-j| X for HIO (ghat - beta ghat) and for RAAR
    (beta ghat + (1 - 2 beta) ghat); with the pre-mix g_n as the feedback operand it would be
    (delta_nj - beta alpha_|n-j|) X instead.  Inside the support: alpha_|n-j| X."""
    Np, N, beta = 6, 8, 0.9
    al = {0: 0.6, 1: 0.2}
    rng = np.random.default_rng(21)
    X = rng.normal(size=(N, N)) + 1j * rng.normal(size=(N, N))
    S = np.zeros((Np, N, N), np.uint8)
    S[:, 2:6, 1:5] = 1
    inside = S[0].astype(bool)
    for rule in ("hio", "raar"):
        for j in (0, 3, Np - 1):
            g = np.zeros((Np, N, N), complex)
            g[j] = X
            o = Oracle(N, Np)
            o.set_data(np.ones((Np, N, N)), np.zeros((Np, N, N), np.uint8))     # M = 0 everywhere
            o.set_support(S)
            o.set_update(rule)
            o.set_estimate(g)
            o.iterate(1, beta)
            out = o.get_projections(0)
            for n in range(Np):
                d = abs((n - j + Np // 2) % Np - Np // 2)
                a = al.get(d, 0.0)
                assert np.abs(out[n][inside] - a * X[inside]).max() < 1e-14, (rule, j, n)
                assert np.abs(out[n][~inside] - (1 - beta) * a * X[~inside]).max() < 1e-14, (rule, j, n)
            # the two readings differ by O(1) here, so the pin cannot pass by accident
            assert np.abs((1 - beta) * al[0] * X[~inside] - (1 - beta * al[0]) * X[~inside]).max() > 0.1
