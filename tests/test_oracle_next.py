"""Pins for the oracle's SURVEY.md 8(f) functions: the seam of a 180 degree scan and shrink-wrap (f2),
Step A and Step C (f1), the 3D transform of Step D (f3).  No expected value comes from the oracle
itself: each test states a closed form, an identity of the forward model, or an independent library
routine (numpy)."""
import numpy as np

import cpra_inputs
from oracle import Oracle, align_episode, blur, center_of_mass, fft3, fsc, mix, mix_seam, refine_3d, refine_3d_sw


def _stack(Np, N, seed):
    rng = np.random.default_rng(seed)
    return rng.normal(size=(Np, N, N)) + 1j * rng.normal(size=(Np, N, N))


# ---------------------------------------------------------------- f2: seam of a [0, 180) scan
def test_seam_flip_equals_the_full_turn_carousel():
    """one rotation axis, so the projection at theta + 180 degrees is the projection at
    theta mirrored in u.  The first half of a [0, 360) scan of 2 Np angles IS the [0, 180) scan of Np
    angles; mixing the full-turn stack needs no flip (true periodicity), and its first half must equal
    the flipped-seam mix of the half-turn stack -- for the generator's projections exactly."""
    N, Np = 16, 6
    rng = np.random.default_rng(4)
    obj = rng.uniform(size=(8, 8, 8))
    full = cpra_inputs.project(obj, N, 2 * np.pi * np.arange(2 * Np) / (2 * Np))
    half = full[:Np]
    # the forward model's symmetry itself (columns 1..N-1 mirror about N/2; column 0 has no partner)
    assert np.abs(full[Np:, :, 1:] - full[:Np, :, :0:-1]).max() < 1e-12
    for alpha in ([0.6, 0.2], [0.4, 0.2, 0.1]):
        want = mix(full, alpha)[:Np]
        got = mix_seam(half, alpha, 1)
        assert np.abs(got - want).max() < 1e-12
        # and the literal wrap (reading A5) differs at the seam projections only
        lit = mix_seam(half, alpha, 0)
        K = len(alpha) - 1
        assert np.abs(lit[K:Np - K] - want[K:Np - K]).max() < 1e-12
        assert np.abs(lit[0] - want[0]).max() > 1e-3 and np.abs(lit[Np - 1] - want[Np - 1]).max() > 1e-3


def test_seam_flip_index_convention_and_loop_use():
    """One-hot stacks: with the flip, projection 0 receives alpha_1 times projection Np-1 read at column
    (N - x) mod N (column 0 and the centre column N/2 map to themselves), rows untouched; the loop uses the
    same mix (M = 0, S = 1: one iteration returns the mixed stack)."""
    N, Np = 8, 5
    img = _stack(1, N, 7)[0]
    mirrored = img[:, (N - np.arange(N)) % N]
    assert np.array_equal(mirrored[:, 0], img[:, 0]) and np.array_equal(mirrored[:, N // 2], img[:, N // 2])
    for j, tgt in ((Np - 1, 0), (0, Np - 1)):
        g = np.zeros((Np, N, N), complex)
        g[j] = img
        m = mix_seam(g, [0.6, 0.2], 1)
        assert np.abs(m[tgt] - 0.2 * mirrored).max() < 1e-15
        assert np.abs(m[j] - 0.6 * img).max() < 1e-15
        inner = (j + (1 if j == 0 else -1)) % Np
        assert np.abs(m[inner] - 0.2 * img).max() < 1e-15          # the neighbour inside the stack: no flip
        o = Oracle(N, Np)
        o.set_data(np.ones((Np, N, N)), np.zeros((Np, N, N), np.uint8))
        o.set_support(np.ones((Np, N, N), np.uint8))
        o.set_seam(1)
        o.set_estimate(g)
        o.iterate(1, 0.9)
        assert np.abs(o.get_projections(0) - m).max() < 1e-15


# ---------------------------------------------------------------- f2: shrink-wrap
def test_blur_of_a_delta_is_the_periodic_gaussian():
    N, sig = 32, 2.5            # exp(-2 pi^2 sigma^2 / 4) = 4e-14 at Nyquist: the sampled transfer function is exact
    a = np.zeros((N, N))
    a[5, 9] = 2.5
    b = blur(a, sig)
    # closed form: the N-periodic sum of a continuous Gaussian of standard deviation sigma, sampled
    d = N * np.arange(-3, 4)                                        # the periodic images
    g1 = lambda c: np.array([np.exp(-0.5 * ((i - c + d) / sig) ** 2).sum() for i in range(N)]) / (sig * np.sqrt(2 * np.pi))
    want = 2.5 * g1(5)[:, None] * g1(9)[None, :]
    assert np.abs(b - want).max() < 1e-12
    assert abs(b.sum() - 2.5) < 1e-12                               # mass conserved
    assert np.abs(blur(a, 0.0) - a).max() < 1e-13                   # sigma = 0: identity
    # independent library route: numpy's FFT with the same transfer function
    k = np.fft.fftfreq(N, 1.0 / N)
    H = np.exp(-2 * np.pi ** 2 * sig ** 2 * (k[:, None] ** 2 + k[None, :] ** 2) / N ** 2)
    r = np.random.default_rng(2).uniform(size=(N, N))
    assert np.abs(blur(r, sig) - np.fft.ifft2(np.fft.fft2(r) * H).real).max() < 1e-12
    # a size that is not a power of two (reading A20): the same closed form and library route
    N = 24
    a = np.zeros((N, N))
    a[20, 3] = 1.5
    d = N * np.arange(-4, 5)
    g1 = lambda c: np.array([np.exp(-0.5 * ((i - c + d) / sig) ** 2).sum() for i in range(N)]) / (sig * np.sqrt(2 * np.pi))
    assert np.abs(blur(a, sig) - 1.5 * g1(20)[:, None] * g1(3)[None, :]).max() < 1e-12
    k = np.fft.fftfreq(N, 1.0 / N)
    H = np.exp(-2 * np.pi ** 2 * sig ** 2 * (k[:, None] ** 2 + k[None, :] ** 2) / N ** 2)
    r = np.random.default_rng(3).uniform(size=(N, N))
    assert np.abs(blur(r, sig) - np.fft.ifft2(np.fft.fft2(r) * H).real).max() < 1e-12


def _sw_plan(g, S):
    Np, N = g.shape[0], g.shape[-1]
    o = Oracle(N, Np)
    o.set_data(np.ones((Np, N, N)))
    o.set_support(S)
    o.set_estimate(g)
    return o


def test_shrinkwrap_threshold_support_and_idempotence():
    N, Np = 32, 3
    rng = np.random.default_rng(9)
    g = np.zeros((Np, N, N), complex)
    g[:, 10:20, 8:22] = rng.uniform(0.5, 1.0, size=(Np, 10, 14)) * np.exp(1j * rng.uniform(0, 6, size=(Np, 10, 14)))
    g[:, 2, 2] = 5.0                                                # a bright pixel OUTSIDE the current support
    S = np.zeros((Np, N, N), np.uint8)
    S[:, 6:26, 4:28] = 1
    # sigma = 0: no blur, the new support is |S g| >= thr max|S g| exactly (the outside pixel is ignored)
    o = _sw_plan(g, S)
    o.shrinkwrap(0.0, 0.2)
    a = np.abs(g) * S
    want = (a >= 0.2 * a.max(axis=(1, 2), keepdims=True)).astype(np.uint8)
    assert np.array_equal(o.get_support(), want) and want[:, 2, 2].max() == 0
    # idempotent on a binary image with sigma = 0
    ob = _sw_plan(want.astype(complex), want)
    ob.shrinkwrap(0.0, 0.5)
    assert np.array_equal(ob.get_support(), want)
    # with a blur: against numpy's FFT, away from the threshold
    o = _sw_plan(g, S)
    b = o.shrinkwrap(1.5, 0.2, want_blurred=True)
    k = np.fft.fftfreq(N, 1.0 / N)
    H = np.exp(-2 * np.pi ** 2 * 1.5 ** 2 * (k[:, None] ** 2 + k[None, :] ** 2) / N ** 2)
    ref = np.fft.ifft2(np.fft.fft2(a) * H).real
    assert np.abs(b - ref).max() < 1e-12
    clear = np.abs(ref - 0.2 * ref.max(axis=(1, 2), keepdims=True)) > 1e-9
    assert np.array_equal(o.get_support()[clear], (ref >= 0.2 * ref.max(axis=(1, 2), keepdims=True))[clear].astype(np.uint8))
    assert o.get_support().sum() > want.sum()                       # the blur widens the thresholded region
    # an empty estimate gives an empty support
    oz = _sw_plan(np.zeros((Np, N, N), complex), S)
    oz.shrinkwrap(1.0, 0.2)
    assert oz.get_support().sum() == 0


# ---------------------------------------------------------------- f1: Step A
def test_prereconstruct_is_the_uncoupled_loop_on_one_projection():
    p = cpra_inputs.make_problem(2, Np=4, N=32)
    g0 = p.estimate.astype(np.complex128)
    a = Oracle(p.N, p.Np).load(p)
    a.prereconstruct(2, 5, 0.9)
    out = a.get_projections(0)
    for n in (0, 1, 3):
        assert np.array_equal(out[n], g0[n])                        # the other projections are untouched
    assert a.iteration == 0
    # the same five iterations through the loop with the coupling switched off (K = 0)
    b = Oracle(p.N, p.Np).load(p, alpha=(1.0,))
    b.iterate(5, 0.9)
    assert np.abs(out[2] - b.get_projections(0)[2]).max() <= 1e-13 * np.abs(g0).max()
    assert np.abs(out[2] - g0[2]).max() > 1e-3 * np.abs(g0).max()


# ---------------------------------------------------------------- f1: Step C
def test_center_of_mass_closed_forms():
    N = 16
    a = np.zeros((N, N), complex)
    a[N // 2 + 3, N // 2 - 5] = 2.0j                                # a delta: its position, whatever its phase
    assert center_of_mass(a) == (3.0, -5.0)
    a[N // 2 + 3, N // 2 - 1] = -6.0                                # two masses 2 and 6 on one row
    cy, cx = center_of_mass(a)
    assert abs(cy - 3.0) < 1e-15 and abs(cx - (-5 * 2 - 1 * 6) / 8) < 1e-15
    assert center_of_mass(np.zeros((N, N), complex)) == (0.0, 0.0)


def _episode(Np, N, seed):
    """A compact asymmetric complex blob per projection, centre of mass near the centre pixel."""
    rng = np.random.default_rng(seed)
    e = np.zeros((Np, N, N), complex)
    e[:, N // 2 - 3:N // 2 + 4, N // 2 - 2:N // 2 + 5] = rng.uniform(0.2, 1.0, size=(Np, 7, 7)) * np.exp(1j * rng.uniform(0, 6, size=(Np, 7, 7)))
    e[:, N // 2 - 3, N // 2 - 2] = 3.0                              # a heavy corner: clearly not centro-symmetric
    return e


def _twin(e):
    N = e.shape[-1]
    i = (N - np.arange(N)) % N
    return np.conj(e[..., i, :][..., :, i])


def _merge(episodes, errors, N, Np, NL, n_ref=0):
    o = Oracle(N, Np)
    o.merge_begin(NL)
    for e, E in zip(episodes, errors):
        o.merge_offer(e, E)
    return o, o.merge_finish(n_ref)


def test_merge_keeps_the_lowest_errors():
    N, Np = 16, 3
    eps = [_episode(Np, N, s) for s in range(6)]
    errs = [0.5, 0.2, 0.9, 0.1, 0.3, 0.05]
    o = Oracle(N, Np)
    o.merge_begin(3)
    for e, E in zip(eps, errs):
        o.merge_offer(e, E)
    assert sorted(o.merge_errors()) == [0.05, 0.1, 0.2]             # N_l lowest of N_r


def test_merge_of_copies_is_the_identity_and_undoes_shift_twin_and_phase():
    """Step C on N_l versions of ONE episode that differ exactly by the ambiguities the paper lists
    (PAPER.md:64 displacement, :70 central inversion) and by the free global phase of an unconstrained
    iterate: the result is the centred episode itself (averaging equal things is the identity)."""
    N, Np = 16, 4
    base = _episode(Np, N, 1)
    # centre it first (whole pixels), so that "the centred episode" is known in closed form
    ref = np.empty_like(base)
    for n in range(Np):
        cy, cx = center_of_mass(base[n])
        ref[n] = np.roll(base[n], (-int(np.floor(cy + 0.5)), -int(np.floor(cx + 0.5))), axis=(0, 1))
        cy, cx = center_of_mass(ref[n])
        assert abs(cy) <= 0.5 and abs(cx) <= 0.5
    v1 = np.stack([np.roll(ref[n], (2 - n, n - 1), axis=(0, 1)) for n in range(Np)])        # displaced, per PO
    v2 = _twin(ref) * np.exp(0.8j)                                                            # twin + phase
    v3 = np.roll(_twin(ref), (1, -2), axis=(1, 2)) * np.exp(-2.1j)                            # all three
    o, (out, sh, tw) = _merge([ref, v1, v2, v3], [0.1, 0.2, 0.3, 0.4], N, Np, 4)
    assert np.abs(out - ref).max() < 1e-13
    assert list(tw) == [0, 0, 1, 1]
    assert [tuple(sh[1, n]) for n in range(Np)] == [(-(2 - n), -(n - 1)) for n in range(Np)]
    assert np.all(sh[0] == 0)
    # the twin of a centred PO is centred on the same pixel or one off (|com| <= 1/2 flips sign): whole-pixel
    # shifts of v2 are 0 here because ref's centre of mass is not on a half-pixel
    # the decision uses ONE PO (n_ref); summed over all POs (n_ref = -1) it is the same here
    o, (out_all, _, tw_all) = _merge([ref, v1, v2, v3], [0.1, 0.2, 0.3, 0.4], N, Np, 4, n_ref=-1)
    assert list(tw_all) == [0, 0, 1, 1] and np.abs(out_all - ref).max() < 1e-13


def test_merge_distance_zero_to_one_version_positive_to_the_other():
    """the distance to the best episode is taken for the PO and for its central inversion; for
    an episode that IS the twin of the best one, the inverted version is at distance 0 and the plain one is
    not -- and the average of the best episode with its own twin, once corrected, is the best episode."""
    N, Np = 16, 2
    ref = _episode(Np, N, 3)
    for n in range(Np):
        cy, cx = center_of_mass(ref[n])
        ref[n] = np.roll(ref[n], (-int(np.floor(cy + 0.5)), -int(np.floor(cx + 0.5))), axis=(0, 1))
    t = _twin(ref)
    d_plain = np.linalg.norm(t[0] - ref[0])
    d_inv = np.linalg.norm(_twin(t)[0] - ref[0])
    assert d_inv == 0.0 and d_plain > 0.5 * np.linalg.norm(ref[0])
    _, (out, sh, tw) = _merge([ref, t], [0.1, 0.2], N, Np, 2)
    assert list(tw) == [0, 1] and np.abs(out - ref).max() < 1e-13
    # offered the other way round the twin is the best episode and the result is the twin (the ambiguity
    # is resolved relative to the best episode, not absolutely)
    _, (out2, _, tw2) = _merge([ref, t], [0.2, 0.1], N, Np, 2)
    assert list(tw2) == [1, 0] and np.abs(out2 - t).max() < 1e-13


def test_merge_averages_different_episodes():
    N, Np = 16, 2
    a, b = _episode(Np, N, 5), _episode(Np, N, 6)
    o, (out, sh, tw) = _merge([a, b], [0.1, 0.2], N, Np, 2)
    # by hand with numpy: shifts, then twin / phase of b against a on PO 0, then the mean
    def centred(e):
        r = np.empty_like(e)
        for n in range(Np):
            cy, cx = center_of_mass(e[n])
            f = lambda c: -int(np.floor(c + 0.5)) if c >= 0 else int(np.floor(-c + 0.5))
            r[n] = np.roll(e[n], (f(cy), f(cx)), axis=(0, 1))
        return r
    ca, cb = centred(a), centred(b)
    c, ct = np.vdot(ca[0], cb[0]), np.vdot(ca[0], _twin(cb)[0])
    if abs(ct) > abs(c):
        cb, c = _twin(cb), ct
    cb = cb * np.conj(c) / abs(c)
    assert np.abs(out - 0.5 * (ca + cb)).max() < 1e-13
    assert abs(np.vdot(ca[0], cb[0]).imag) < 1e-12 and np.vdot(ca[0], cb[0]).real > 0     # phases aligned


def test_merge_offer_from_the_plan_takes_the_supported_estimate_and_its_error():
    p = cpra_inputs.make_problem(2, Np=4, N=32)
    o = Oracle(p.N, p.Np).load(p)
    o.iterate(3, 0.9)
    o.merge_begin(2)
    o.merge_offer()
    assert o.merge_errors()[0] == o.get_error()[1]
    out, sh, tw = o.merge_finish(0)
    s = o.get_projections(1)
    want = np.stack([np.roll(s[n], tuple(sh[0, n]), axis=(0, 1)) for n in range(p.Np)])
    assert np.abs(out - want).max() == 0.0


# ---------------------------------------------------------------- f3: 3D transform
def test_fft3_against_numpy_and_round_trip():
    for N in (4, 8, 16, 12, 20):       # 12, 20: not powers of two (reading A20: the definition, line by line)
        rng = np.random.default_rng(N)
        v = rng.normal(size=(N, N, N)) + 1j * rng.normal(size=(N, N, N))
        F = fft3(v, -1)
        assert np.abs(F - np.fft.fftn(v)).max() < 1e-12 * np.abs(F).max()
        assert np.abs(fft3(F, +1) - v).max() < 1e-13
    # a delta at (z0, y0, x0): plane wave with the e^{-2 pi i ...} sign on every axis, axes not swapped
    N = 8
    d = np.zeros((N, N, N), complex)
    d[1, 2, 3] = 1.0
    kz, ky, kx = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    assert np.abs(fft3(d, -1) - np.exp(-2j * np.pi * (1 * kz + 2 * ky + 3 * kx) / N)).max() < 1e-13


def test_fft3_of_the_assembled_spectrum_returns_the_object(tiny_problem):
    """Step D end to end on the oracle: slices of the true projections -> E(q) -> inverse 3D FT ~ the
    object (up to the interpolation between slices): correlation with the true object close to 1."""
    p = tiny_problem
    N = p.N
    o = Oracle(N, p.Np)
    o.set_data(np.ones((p.Np, N, N)), None, p.angles)
    o.set_support(np.ones((p.Np, N, N), np.uint8))
    o.set_estimate(p.projections)
    vol, w = o.assemble_3d()
    rec = fft3(vol, +1)
    pad = np.zeros((N, N, N))
    off = (N - p.obj.shape[0]) // 2
    pad[off:off + p.obj.shape[0], off:off + p.obj.shape[0], off:off + p.obj.shape[0]] = p.obj
    corr = abs(np.vdot(pad, rec)) / (np.linalg.norm(pad) * np.linalg.norm(rec))
    assert corr > 0.97, corr


# ---------------------------------------------------------------- f3: Step D's iterations
def _cube_case(N=16, seed=3):
    rng = np.random.default_rng(seed)
    obj = np.zeros((N, N, N), complex)
    obj[5:11, 4:12, 6:10] = rng.uniform(0.3, 1.0, size=(6, 8, 4)) * np.exp(1j * rng.uniform(0, 1, size=(6, 8, 4)))
    S3 = np.zeros((N, N, N), np.uint8)
    S3[4:12, 3:13, 5:11] = 1
    E = np.fft.fftn(obj)
    return obj, S3, E, rng


def test_refine_3d_closed_forms():
    obj, S3, E, rng = _cube_case()
    N = obj.shape[0]
    ones = np.ones((N, N, N))
    # everything known: one iteration is S3 . F^-1[E] = the object (its support lies inside S3), error 0
    o, err = refine_3d(E, ones, S3, 2)
    assert np.abs(o - obj).max() < 1e-13 and err.max() < 1e-13
    # nothing constrained in real space (S3 = 1): the object is F^-1 of the zero-filled spectrum, error 0
    W = (rng.uniform(size=(N, N, N)) < 0.5).astype(float)
    o, err = refine_3d(E, W, np.ones((N, N, N), np.uint8), 3)
    assert np.abs(o - np.fft.ifftn(E * (W > 0))).max() < 1e-13 and err.max() < 1e-13
    # one iteration by hand with numpy's FFT (independent library): object and error
    o1, e1 = refine_3d(E, W, S3, 1)
    want = np.fft.ifftn(E * (W > 0)) * S3
    assert np.abs(o1 - want).max() < 1e-13
    Fp = np.fft.fftn(want)
    assert abs(e1[0] - np.sqrt((np.abs(Fp - E)[W > 0] ** 2).sum() / (np.abs(E)[W > 0] ** 2).sum())) < 1e-13
    # second iteration: the unknown voxels carry F' of the first, the known ones E again
    o2, _ = refine_3d(E, W, S3, 2)
    assert np.abs(o2 - np.fft.ifftn(np.where(W > 0, E, Fp)) * S3).max() < 1e-13


def test_refine_3d_at_a_size_that_is_not_a_power_of_two():
    """Reading A20 carried to Step D: N = 12, two iterations by hand with numpy's FFT."""
    obj, S3, E, rng = _cube_case(N=12, seed=5)
    W = (rng.uniform(size=(12, 12, 12)) < 0.6).astype(float)
    o2, e2 = refine_3d(E, W, S3, 2)
    o1 = np.fft.ifftn(E * (W > 0)) * S3
    F1 = np.fft.fftn(o1)
    want = np.fft.ifftn(np.where(W > 0, E, F1)) * S3
    assert np.abs(o2 - want).max() < 1e-13
    den = (np.abs(E)[W > 0] ** 2).sum()
    assert abs(e2[0] - np.sqrt((np.abs(F1 - E)[W > 0] ** 2).sum() / den)) < 1e-13
    assert abs(e2[1] - np.sqrt((np.abs(np.fft.fftn(want) - E)[W > 0] ** 2).sum() / den)) < 1e-13


def test_refine_3d_sw_closed_forms():
    """Reading A30: the 3D support update inside Step D's iterations, by hand with numpy's FFT."""
    obj, S3, E, rng = _cube_case()
    N = obj.shape[0]
    W = (rng.uniform(size=(N, N, N)) < 0.6).astype(float)
    # never updating = refine_3d, support untouched
    o0, e0 = refine_3d(E, W, S3, 4)
    o1, e1, s1 = refine_3d_sw(E, W, S3, 4, 0, 1.0, 0.1)
    assert np.array_equal(o0, o1) and np.array_equal(e0, e1) and np.array_equal(s1, S3)
    o1, e1, s1 = refine_3d_sw(E, W, S3, 4, 4, 1.0, 0.1)          # the only multiple of 4 is the last iteration: no update
    assert np.array_equal(o0, o1) and np.array_equal(s1, S3)
    # one update after iteration 2 of 3, sigma = 0: the new support is the threshold of |O_2| itself
    o2, _ = refine_3d(E, W, S3, 2)
    thr = 0.2
    want_s = (np.abs(o2) >= thr * np.abs(o2).max()).astype(np.uint8)
    o3, e3, s3, b3 = refine_3d_sw(E, W, S3, 3, 2, 0.0, thr, want_blurred=True)
    clear = np.abs(np.abs(o2) - thr * np.abs(o2).max()) > 1e-12
    assert np.abs(b3 - np.abs(o2)).max() < 1e-13
    assert np.array_equal(s3[clear], want_s[clear]) and 0 < s3.sum() < S3.sum()
    # ... and iteration 3 ran against it: by hand
    F2 = np.fft.fftn(o2)
    F = np.where(W > 0, E, F2)
    want_o = np.fft.ifftn(F) * s3
    assert np.abs(o3 - want_o).max() < 1e-13
    assert abs(e3[2] - np.sqrt((np.abs(np.fft.fftn(want_o) - E)[W > 0] ** 2).sum() / (np.abs(E)[W > 0] ** 2).sum())) < 1e-13
    # sigma > 0: the blur is the 3D Gaussian transfer function (numpy route), real part
    sig = 1.5
    _, _, s4, b4 = refine_3d_sw(E, W, S3, 3, 2, sig, thr, want_blurred=True)
    k = np.fft.fftfreq(N, 1.0 / N)
    H = np.exp(-2 * np.pi ** 2 * sig ** 2 * (k[:, None, None] ** 2 + k[None, :, None] ** 2 + k[None, None, :] ** 2) / N ** 2)
    wb = np.fft.ifftn(np.fft.fftn(np.abs(o2)) * H).real
    assert np.abs(b4 - wb).max() < 1e-13
    clear = np.abs(wb - thr * wb.max()) > 1e-12
    assert np.array_equal(s4[clear], (wb >= thr * wb.max()).astype(np.uint8)[clear])
    assert abs(wb.sum() - np.abs(o2).sum()) < 1e-10               # the blur conserves the mass
    # nothing left: an all-zero estimate empties the support
    _, _, s5 = refine_3d_sw(np.zeros_like(E), W, S3, 3, 1, 1.0, 0.1)
    assert s5.sum() == 0


def test_backproject_support_closed_forms(tiny_problem):
    """Reading A29: the visual hull of the 2D supports."""
    N = 32
    c = N // 2
    def plan(S, angles):
        o = Oracle(N, len(angles))
        o.set_data(np.ones((len(angles), N, N)), None, np.asarray(angles, float))
        o.set_support(S)
        return o
    yy, xx = np.meshgrid(np.arange(N) - c, np.arange(N) - c, indexing="ij")
    rad = np.hypot(yy, xx)
    # full supports: everything whose footprint stays on the detector at every angle (the inscribed cylinder) stays
    full = plan(np.ones((3, N, N), np.uint8), [0.0, 0.7, 2.0]).backproject_support()
    assert full[:, rad <= c - 1].all() and np.array_equal(full[0], full[N - 1])
    assert plan(np.ones((1, N, N), np.uint8), [0.0]).backproject_support()[:, :, :N - 1].all()
    # one projection at 0 degrees: S3[z][y][x] = S[z][x] or S[z][x + 1] for every y (u = x exactly: the footprint rule
    # looks at columns u and u + 1); at 90 degrees u = y
    rng = np.random.default_rng(4)
    S = (rng.uniform(size=(1, N, N)) < 0.3).astype(np.uint8)
    dil = S[0] | np.concatenate([S[0][:, 1:], np.zeros((N, 1), np.uint8)], axis=1)
    s3 = plan(S, [0.0]).backproject_support()
    assert np.array_equal(s3, np.broadcast_to(dil[:, None, :], (N, N, N)))
    s3 = plan(S, [np.pi / 2]).backproject_support()
    # cos(pi/2) = 6e-17: u = y up to rounding, so columns y and y + 1 (or y - 1 and y) are looked at: the hull contains S[z][y]
    assert np.all(s3[:, :, :][np.broadcast_to(S[0][:, :, None].astype(bool), (N, N, N))])
    # a strip |u - c| <= r at many angles: the hull is the cylinder of radius r (up to the one-pixel footprint)
    r = 6
    strip = np.zeros((N, N), np.uint8)
    strip[:, c - r:c + r + 1] = 1
    angles = np.linspace(0, np.pi, 36, endpoint=False)
    s3 = plan(np.broadcast_to(strip, (36, N, N)).copy(), angles).backproject_support()
    assert s3[:, rad <= r - 0.5].all() and not s3[:, rad >= r + 1.5].any()
    # an empty row z in one projection empties the slab z
    S2 = np.ones((4, N, N), np.uint8)
    S2[2, 5, :] = 0
    s3 = plan(S2, [0.0, 0.5, 1.0, 1.5]).backproject_support()
    assert not s3[5].any() and s3[4][rad <= c - 1].all() and s3[6][rad <= c - 1].all()
    # physics: the supports of an object's true projections contain the object
    p = tiny_problem
    o = Oracle(p.N, p.Np)
    o.set_data(np.ones((p.Np, p.N, p.N)), None, p.angles)
    o.set_support((np.abs(p.projections) > 0).astype(np.uint8))
    hull = o.backproject_support()
    pad = np.zeros((p.N,) * 3)
    off = (p.N - p.obj.shape[0]) // 2
    pad[off:off + p.obj.shape[0], off:off + p.obj.shape[0], off:off + p.obj.shape[0]] = np.abs(p.obj)
    assert hull[pad > 0].all() and hull.sum() < 0.5 * p.N ** 3          # (every voxel adds a positive amount to its footprint)


def test_refine_3d_error_never_increases_and_recovers_the_object():
    """Alternating projections between two convex sets (known Fourier samples / support): the distance to
    the data cannot grow, and with half of the spectrum known and a tight support the object comes back."""
    obj, S3, E, rng = _cube_case()
    N = obj.shape[0]
    W = (rng.uniform(size=(N, N, N)) < 0.5).astype(float)
    o, err = refine_3d(E, W, S3, 60)
    assert np.all(np.diff(err) <= 1e-12) and err[-1] < 0.05 * err[0]
    assert np.linalg.norm(o - obj) < 0.05 * np.linalg.norm(obj)
    assert np.abs(o[S3 == 0]).max() == 0.0


# ---------------------------------------------------------------- f4: FSC and PRTF
def test_fsc_closed_forms():
    N = 16
    rng = np.random.default_rng(8)
    F = rng.normal(size=(N, N, N)) + 1j * rng.normal(size=(N, N, N))
    ns = N // 2 + 1
    assert np.abs(fsc(F, F) - 1.0).max() < 1e-14
    assert np.abs(fsc(F, -F) + 1.0).max() < 1e-14
    assert np.abs(fsc(F, 1j * F)).max() < 1e-14                       # quadrature: Re<F, iF> = 0
    assert np.abs(fsc(F, 3.0 * F) - 1.0).max() < 1e-14                # scale invariant
    # shells: a spectrum living on one voxel k correlates only in shell round(|k|); outside N/2 it is left out
    for k, sh in (((0, 0, 0), 0), ((3, -4, 0), 5), ((-2, 2, 1), 3), ((5, 5, 5), None)):
        D = np.zeros((N, N, N), complex)
        D[k[0] % N, k[1] % N, k[2] % N] = 1.0
        f = fsc(D + 1e-30 * 0, D)
        want = np.zeros(ns)
        if sh is not None:
            want[sh] = 1.0
        assert np.array_equal(f, want), (k, f)
    # against a numpy restatement on random pairs
    G = rng.normal(size=(N, N, N)) + 1j * rng.normal(size=(N, N, N)) + 0.5 * F
    k = np.fft.fftfreq(N, 1.0 / N)
    r = np.floor(np.sqrt(k[:, None, None] ** 2 + k[None, :, None] ** 2 + k[None, None, :] ** 2) + 0.5).astype(int)
    want = np.array([(F[r == s] * np.conj(G[r == s])).sum().real / np.sqrt((np.abs(F[r == s]) ** 2).sum() * (np.abs(G[r == s]) ** 2).sum())
                     for s in range(ns)])
    assert np.abs(fsc(F, G) - want).max() < 1e-13 and 0.2 < want[4] < 0.7


def test_prtf_closed_forms():
    p = cpra_inputs.make_problem(1, Np=4, noise=False)
    P = p.projections
    I_c = np.fft.fftshift(np.abs(np.fft.fft2(P)) ** 2, axes=(-2, -1))
    mask = np.ones((p.Np, p.N, p.N), np.uint8)
    mask[:, p.N // 2 - 1:p.N // 2 + 2, p.N // 2 - 1:p.N // 2 + 2] = 0      # a 3 x 3 beamstop: rings 0 and 1 unmeasured
    o = Oracle(p.N, p.Np)
    o.set_data(I_c, mask)
    t = o.prtf(P)
    assert t[0] == 0.0 and t[1] == 0.0                                # empty rings
    assert np.abs(t[2:] - 1.0).max() < 1e-9                           # the true projections reproduce the amplitudes
    assert np.abs(o.prtf(0.25 * np.exp(0.3j) * P)[2:] - 0.25).max() < 1e-9
    # averaging two reconstructions with opposite phases of one pixel ring kills that ring: PRTF measures phase consistency
    G = np.fft.fft2(P)
    k = np.fft.fftfreq(p.N, 1.0 / p.N)
    ring = np.floor(np.sqrt(k[:, None] ** 2 + k[None, :] ** 2) + 0.5).astype(int) == 6
    G2 = G.copy()
    G2[:, ring] *= -1.0
    t2 = o.prtf(0.5 * (P + np.fft.ifft2(G2)))
    assert abs(t2[6]) < 1e-9 and np.abs(np.delete(t2[2:], 4) - 1.0).max() < 1e-9


# ---------------------------------------------------------------- f2: positivity
def test_positivity_closed_form():
    """Nothing measured (M = 0: g' = g), K = 0: with positivity a pixel inside the support keeps g where Re g >= 0 and
    gets the feedback value elsewhere -- HIO (1 - beta) g, RAAR (1 - beta) g, ER 0 -- exactly like a pixel outside the
    support; without the flag the inside pixels are untouched."""
    N, Np, beta = 8, 2, 0.9
    g = _stack(Np, N, 41)
    S = np.zeros((Np, N, N), np.uint8)
    S[:, 2:6, 1:7] = 1
    inside = S.astype(bool)
    neg = g.real < 0
    for rule, outside in (("hio", 1 - beta), ("raar", 1 - beta), ("er", 0.0)):
        for pos in (0, 1):
            o = Oracle(N, Np)
            o.set_data(np.ones((Np, N, N)), np.zeros((Np, N, N), np.uint8))
            o.set_support(S)
            o.set_carousel([1.0], 1)
            o.set_update(rule)
            o.set_positivity(pos)
            o.set_estimate(g)
            o.iterate(1, beta)
            out = o.get_projections(0)
            keep = inside & ~(neg & bool(pos))
            assert np.abs(out[keep] - g[keep]).max() < 1e-14, (rule, pos)
            assert np.abs(out[~keep] - outside * g[~keep]).max() < 1e-14, (rule, pos)
    assert (inside & neg).sum() > 5 and (inside & ~neg).sum() > 5


# ---------------------------------------------------------------- consistency of one episode before Step D (A28)
def test_align_episode_restores_phases_and_twins_of_true_projections():
    """The projections of one object all have the same total (line integrals), and neighbours are
    similar.  A stack of true projections whose members were multiplied by arbitrary unit phases, and
    some replaced by their twins conj(P(-r)), comes back exactly."""
    p = cpra_inputs.make_problem(1, Np=12, noise=False)
    P = p.projections
    tot = P.sum(axis=(1, 2))
    assert np.abs(tot - tot[0]).max() < 2e-3 * abs(tot[0]) and tot[0].real > 0      # the identity itself (bilinear rotation: to 1e-3)
    rng = np.random.default_rng(3)
    N = p.N
    i = (N - np.arange(N)) % N
    tw = lambda a: np.conj(a[..., i, :][..., :, i])
    for n_ref, twinned in ((0, [3, 4, 5, 9]), (6, [0, 1, 11]), (2, [])):
        ep = P * np.exp(1j * rng.uniform(0, 2 * np.pi, size=p.Np))[:, None, None]
        for n in twinned:
            ep[n] = tw(ep[n])
        out, fl = align_episode(ep, n_ref)
        assert np.abs(out - P).max() < 1e-10 * np.abs(P).max(), (n_ref, twinned)
        assert sorted(np.flatnonzero(fl)) == sorted(twinned)
    # if the reference projection itself is a twin the whole stack comes out as the twin object: consistent again
    ep = P.copy()
    ep[0] = tw(ep[0])
    out, fl = align_episode(ep, 0)
    assert np.abs(out - tw(P)).max() < 1e-10 * np.abs(P).max() and fl.sum() == p.Np - 1
    # invariants on arbitrary data: totals real and positive, Fourier moduli untouched
    g = _stack(5, 8, 77)
    out, _ = align_episode(g, 2)
    s = out.sum(axis=(1, 2))
    assert np.abs(s.imag).max() < 1e-12 and s.real.min() > 0
    assert np.abs(np.abs(np.fft.fft2(out)) - np.abs(np.fft.fft2(g))).max() < 1e-11
