"""Parity of the steps around the loop (seam of a 180 degree scan, shrink-wrap, Step A,
Step C, the 3D transform of Step D) with the FP64 oracle, through the C ABI.  Integer outputs (support
bits, shifts, twin decisions) are compared exactly; where floating point decides a bit, the pixels whose
value lies within rounding of the threshold are set aside and counted.

Run on the B200 box:  python -m pytest tests -m gpu -x -q"""
import numpy as np
import pytest

import cpra_inputs
from conftest import rel_l2

pytestmark = pytest.mark.gpu
TOL_1 = 1e-5
TOL_E = 1e-4


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "the gpu-marked tests need a CUDA device"
    return torch


def _gpu(problem, alpha=(0.6, 0.2), n_ei=1, flags=0):
    import paper_2402_05283_b200 as cpra
    return cpra.Plan(problem.N, problem.Np, flags=flags).load(problem, alpha, n_ei)


def _oracle(problem, alpha=(0.6, 0.2), n_ei=1):
    from oracle import Oracle
    return Oracle(problem.N, problem.Np).load(problem, alpha, n_ei)


def _get(plan, which=0):
    return plan.get_projections(which).cpu().numpy()


# ------------------------------------------------------------------------------------------------
# f2: mirrored wrap at the seam of a [0, 180) scan, every kernel family that evaluates the mix
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,Np,alpha,n_ei,flags", [
    (64, 7, (0.6, 0.2), 1, 0),            # whole-image kernel, K = 1
    (128, 6, (0.5, 0.2, 0.05), 1, 0),     # whole-image kernel, K = 2
    (256, 6, (0.6, 0.2), 1, 0),           # tile kernels
    (256, 7, (0.4, 0.15, 0.1, 0.05), 2, 0),
    (512, 7, (0.6, 0.2), 1, 0),           # fused inverse-row / forward-row kernel: mirrored halo tiles
    (512, 3, (0.6, 0.2), 1, 0),           # every projection is a seam neighbour
    (512, 7, (0.6, 0.2), 2, 0),
    (512, 6, (0.6, 0.2), 1, 4),           # CPRA_FLAG_NO_WALK: the tile kernels at N = 512
    (512, 5, (0.5, 0.2, 0.05), 1, 0),
    (1024, 3, (0.6, 0.2), 1, 0),
])
def test_seam_flip(torch_cuda, N, Np, alpha, n_ei, flags):
    p = cpra_inputs.random_stack(N, Np, seed=900 + N + Np, beamstop=3)
    o = _oracle(p, alpha, n_ei).set_seam(1)
    g = _gpu(p, alpha, n_ei, flags).set_seam(True)
    lit = _oracle(p, alpha, n_ei)
    for plan in (o, g, lit):
        plan.iterate(4, 0.9)
    ref = o.get_projections(0)
    assert rel_l2(_get(g), ref) <= 4 * TOL_1
    assert rel_l2(lit.get_projections(0), ref) > 1e-2                 # the flag matters on this input
    E, Eg = g.get_error()
    assert abs(float(Eg.cpu()[0]) - o.get_error()[1]) <= TOL_E * o.get_error()[1]
    # split calls: K1 / K3 and the fused kernel alternate, bit-identical
    h = _gpu(p, alpha, n_ei, flags).set_seam(True)
    for k in (1, 2, 1):
        h.iterate(k, 0.9)
    assert np.array_equal(_get(h).view(np.uint32), _get(g).view(np.uint32))


def test_seam_flip_on_config_2_and_3(torch_cuda):
    for cfg, Np in ((2, 12), (3, 6)):
        p = cpra_inputs.make_problem(cfg, Np=Np)
        o, g = _oracle(p).set_seam(1), _gpu(p).set_seam(True)
        o.iterate(3, p.beta)
        g.iterate(3, p.beta)
        assert rel_l2(_get(g), o.get_projections(0)) <= 3 * TOL_1, cfg


# ------------------------------------------------------------------------------------------------
# f2: shrink-wrap
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,Np,N", [(1, 8, None), (2, 12, None), (3, 6, None), (4, 4, None), (5, 3, None), (1, 5, 160), (1, 4, 48)])
def test_shrinkwrap(torch_cuda, cfg, Np, N):
    p = cpra_inputs.make_problem(cfg, Np=Np, N=N)
    o, g = _oracle(p), _gpu(p)
    o.iterate(5, p.beta)
    g.iterate(5, p.beta)
    sigma, thr = 2.0, 0.15
    bo = o.shrinkwrap(sigma, thr, want_blurred=True)
    bg = g.shrinkwrap(sigma, thr, want_blurred=True).cpu().numpy().astype(np.float64)
    mx = bo.max(axis=(1, 2), keepdims=True)
    assert np.abs(bg - bo).max() <= 2e-5 * mx.max()
    So, Sg = o.get_support(), g.get_support().cpu().numpy()
    clear = np.abs(bo - thr * mx) > 5e-5 * mx                         # away from the threshold the bit is unique
    assert np.array_equal(So[clear], Sg[clear])
    assert (~clear).mean() < 2e-3
    assert 0 < Sg.sum() < p.support.sum() * 1.5
    # the loop goes on with the new support: same support on both sides, then two more iterations
    o.set_support(Sg)
    o.iterate(2, p.beta)
    g.iterate(2, p.beta)
    assert rel_l2(_get(g), o.get_projections(0)) <= 1e-4             # 7 iterations of drift
    assert rel_l2(_get(g, 1), o.get_projections(1)) <= 1e-4


def test_shrinkwrap_sigma_zero_and_empty(torch_cuda):
    import paper_2402_05283_b200 as cpra
    p = cpra_inputs.random_stack(64, 4, seed=71)
    g = _gpu(p)
    g.shrinkwrap(0.0, 0.5)
    a = np.abs(p.estimate) * p.support
    b = np.abs(a - 0.5 * a.max(axis=(1, 2), keepdims=True)) > 1e-5 * a.max()
    want = a >= 0.5 * a.max(axis=(1, 2), keepdims=True)
    assert np.array_equal(g.get_support().cpu().numpy()[b].astype(bool), want[b])
    z = cpra_inputs.random_stack(64, 4, seed=72)
    z.estimate[:] = 0
    g = _gpu(z)
    g.shrinkwrap(1.0, 0.2)
    assert int(g.get_support().sum()) == 0
    with pytest.raises(cpra.CpraError) as e:
        g.shrinkwrap(-1.0, 0.2)
    assert e.value.code == cpra.ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------------
# f1: Step A
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,Np,n,k", [(64, 5, 0, 3), (64, 5, 4, 4), (256, 4, 2, 3), (512, 3, 1, 2), (1024, 2, 1, 1)])
def test_prereconstruct(torch_cuda, N, Np, n, k):
    import paper_2402_05283_b200 as cpra
    p = cpra_inputs.random_stack(N, Np, seed=500 + N + k, beamstop=3)
    alpha = (0.6, 0.2) if Np >= 3 else (1.0,)
    o, g = _oracle(p, alpha), _gpu(p, alpha)
    o.prereconstruct(n, k, 0.9)
    g.prereconstruct(n, k, 0.9)
    out, ref = _get(g), o.get_projections(0)
    assert rel_l2(out[n], ref[n]) <= k * TOL_1
    for m in range(Np):
        if m != n:
            assert np.array_equal(out[m], p.estimate[m])              # untouched, bit for bit
    assert g.iteration == 0
    with pytest.raises(cpra.CpraError) as e:
        g.get_error()
    assert e.value.code == cpra.ERR_NOT_READY
    # Step B follows on the pre-reconstructed stack
    o.iterate(2, 0.9)
    g.iterate(2, 0.9)
    assert rel_l2(_get(g), o.get_projections(0)) <= (k + 2) * TOL_1


def test_prereconstruct_many_iterations(torch_cuda):
    """N_i^pre = 200 iterations on PO 0: the same as 200 iterations of the uncoupled loop for that
    projection (up to the drift of 200 chaotic iterations through different kernels), the others untouched."""
    p = cpra_inputs.make_problem(1, Np=4)
    loop = _gpu(p, (1.0,))
    loop.iterate(201, p.beta)
    e_loop = loop.get_error()[0].cpu().numpy()
    one = _gpu(p, (1.0,))
    one.iterate(1, p.beta)
    e_one = one.get_error()[0].cpu().numpy()
    g = _gpu(p, (1.0,))
    g.prereconstruct(0, 200, p.beta)
    g.iterate(1, p.beta)
    e = g.get_error()[0].cpu().numpy()
    assert abs(e[0] - e_loop[0]) <= 0.05 * e_loop[0] and e[0] > 100 * e_one[0]
    assert np.array_equal(e[1:], e_one[1:])


# ------------------------------------------------------------------------------------------------
# f1: Step C
# ------------------------------------------------------------------------------------------------
def _blob_episode(Np, N, seed):
    rng = np.random.default_rng(seed)
    e = np.zeros((Np, N, N), np.complex64)
    h = N // 2
    e[:, h - 5:h + 6, h - 4:h + 7] = (rng.uniform(0.2, 1.0, size=(Np, 11, 11)) * np.exp(1j * rng.uniform(0, 6, size=(Np, 11, 11)))).astype(np.complex64)
    e[:, h - 5, h - 4] = 3.0
    return e


def _twin(e):
    N = e.shape[-1]
    i = (N - np.arange(N)) % N
    return np.conj(e[..., i, :][..., :, i])


@pytest.mark.parametrize("N,Np,n_ref", [(32, 3, 0), (64, 5, 2), (64, 4, -1), (256, 2, 1)])
def test_merge_against_oracle(torch_cuda, N, Np, n_ref):
    import paper_2402_05283_b200 as cpra
    from oracle import Oracle
    base = _blob_episode(Np, N, 1)
    eps = [base,
           np.stack([np.roll(base[n], (3 - n, n - 2), axis=(0, 1)) for n in range(Np)]),
           (_twin(base) * np.exp(0.8j)).astype(np.complex64),
           _blob_episode(Np, N, 2),
           (np.roll(_twin(_blob_episode(Np, N, 3)), (2, -3), axis=(1, 2)) * np.exp(-2j)).astype(np.complex64),
           _blob_episode(Np, N, 4)]
    errs = [0.30, 0.20, 0.25, 0.10, 0.40, 0.15]
    o = Oracle(N, Np)
    o.merge_begin(4)
    g = cpra.Plan(N, Np)
    g.merge_begin(4)
    for e, E in zip(eps, errs):
        o.merge_offer(e, E)
        g.merge_offer(torch_cuda.from_numpy(np.ascontiguousarray(e)).cuda(), E)
    Eg, cnt = g.merge_errors()
    assert int(cnt.cpu()[0]) == 4 and np.array_equal(Eg.cpu().numpy(), o.merge_errors())     # same slots, same errors
    out_o, sh_o, tw_o = o.merge_finish(n_ref)
    out_g, sh_g, tw_g = g.merge_finish(n_ref)
    assert np.array_equal(sh_g.cpu().numpy(), sh_o) and np.array_equal(tw_g.cpu().numpy(), tw_o)
    assert tw_o.sum() >= 1 and np.abs(sh_o).sum() > 0
    assert rel_l2(out_g.cpu().numpy(), out_o) <= 1e-6
    assert np.array_equal(g.merge_get(1).cpu().numpy(), eps[1])


def test_merge_of_restarts_from_the_plan(torch_cuda):
    """Steps A + B + C on config 1: N_r = 6 random restarts, N_l = 3 kept, each restart pre-reconstructs PO 0
    and runs the coupled loop; the bank is fed from the plan on the device.  Decisions equal the oracle's;
    the merged episode agrees to the drift of the iterates it is made of."""
    import paper_2402_05283_b200 as cpra
    from oracle import Oracle
    p = cpra_inputs.make_problem(1, Np=8)
    g = cpra.Plan(p.N, p.Np).load(p)
    o = Oracle(p.N, p.Np).load(p)
    g.merge_begin(3)
    o.merge_begin(3)
    for r in range(6):
        g0 = cpra_inputs.random_phase_estimate(p.intensity, p.mask, r)
        g.set_estimate(torch_cuda.from_numpy(g0).cuda())
        o.set_estimate(g0)
        for plan in (g, o):
            plan.prereconstruct(0, 6, p.beta)
            plan.iterate(6, p.beta)
            plan.merge_offer()
    Eg, cnt = g.merge_errors()
    Eo = o.merge_errors()
    assert int(cnt.cpu()[0]) == 3 and np.abs(Eg.cpu().numpy() - Eo).max() <= TOL_E * Eo.max()
    out_o, sh_o, tw_o = o.merge_finish(0)
    out_g, sh_g, tw_g = g.merge_finish(0)
    assert np.array_equal(tw_g.cpu().numpy(), tw_o)
    assert (sh_g.cpu().numpy() != sh_o).mean() <= 0.05                  # a centre of mass within 1e-5 of a half pixel may round either way
    if np.array_equal(sh_g.cpu().numpy(), sh_o):
        assert rel_l2(out_g.cpu().numpy(), out_o) <= 2e-4


# ------------------------------------------------------------------------------------------------
# f3: the 3D transform of Step D
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [16, 32, 64, 128, 256, 20, 48, 160])
def test_fft3(torch_cuda, N):
    import paper_2402_05283_b200 as cpra
    rng = np.random.default_rng(N)
    v = (rng.normal(size=(N, N, N)) + 1j * rng.normal(size=(N, N, N))).astype(np.complex64)
    plan = cpra.Plan(N, N)
    d = torch_cuda.from_numpy(v).cuda()
    F = plan.fft3(d, -1)
    ref = np.fft.fftn(v.astype(np.complex128))
    assert rel_l2(F.cpu().numpy(), ref) <= 3e-6
    B = plan.fft3(F, +1).cpu().numpy()
    assert rel_l2(B, v) <= 4e-6
    if N <= 64:
        from oracle import fft3
        assert rel_l2(F.cpu().numpy(), fft3(v, -1)) <= 3e-6
    dl = np.zeros((N, N, N), np.complex64)
    dl[1, 2, 3] = 1.0
    Fd = plan.fft3(torch_cuda.from_numpy(dl).cuda(), -1).cpu().numpy()
    kz, ky, kx = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    assert np.abs(Fd - np.exp(-2j * np.pi * (kz + 2 * ky + 3 * kx) / N)).max() < 2e-5
    with pytest.raises(cpra.CpraError) as e:
        cpra.Plan(N, N + 1).fft3(d, -1)
    assert e.value.code in (cpra.ERR_INVALID_ARG,)


def test_step_d_assemble_then_inverse_3d(torch_cuda):
    """Steps D's two transforms chained on the device: slices of the true projections -> E(q) -> O(r),
    against the same chain on the oracle, and against the object itself (correlation)."""
    import paper_2402_05283_b200 as cpra
    from oracle import Oracle, fft3
    p = cpra_inputs.make_problem(1, keep_object=True, noise=False)
    N = p.N
    g = cpra.Plan(N, p.Np)
    g.set_data(torch_cuda.from_numpy(p.intensity).cuda(), None, p.angles)
    g.set_support(torch_cuda.ones((p.Np, N, N), dtype=torch_cuda.uint8, device="cuda"))
    g.set_estimate(torch_cuda.from_numpy(p.projections.astype(np.complex64)).cuda())
    vol, w = g.assemble_3d()
    rec = cpra.Plan(N, N).fft3(vol, +1).cpu().numpy()
    o = Oracle(N, p.Np)
    o.set_data(np.ones((p.Np, N, N)), None, p.angles)
    o.set_support(np.ones((p.Np, N, N), np.uint8))
    o.set_estimate(p.projections.astype(np.complex64))
    ref = fft3(o.assemble_3d()[0], +1)
    assert rel_l2(rec, ref) <= 3 * TOL_1
    pad = np.zeros((N, N, N))
    off = (N - p.obj.shape[0]) // 2
    pad[off:off + p.obj.shape[0], off:off + p.obj.shape[0], off:off + p.obj.shape[0]] = p.obj
    assert abs(np.vdot(pad, rec)) / (np.linalg.norm(pad) * np.linalg.norm(rec)) > 0.97


@pytest.mark.parametrize("N", [16, 64, 128, 48])
def test_refine_3d(torch_cuda, N):
    """Step D's iterations on the device against the oracle: half of the spectrum known, a box support."""
    import paper_2402_05283_b200 as cpra
    from oracle import refine_3d
    rng = np.random.default_rng(N)
    h = N // 2
    obj = np.zeros((N, N, N), np.complex64)
    a = max(2, N // 6)
    obj[h - a:h + a, h - a + 1:h + a, h - a:h + a - 1] = (rng.uniform(0.3, 1.0, size=(2 * a, 2 * a - 1, 2 * a - 1)) *
                                                          np.exp(1j * rng.uniform(0, 1, size=(2 * a, 2 * a - 1, 2 * a - 1)))).astype(np.complex64)
    S3 = np.zeros((N, N, N), np.uint8)
    S3[h - a - 1:h + a + 1, h - a:h + a + 1, h - a - 1:h + a] = 1
    E = np.fft.fftn(obj.astype(np.complex128)).astype(np.complex64)
    W = (rng.uniform(size=(N, N, N)) < 0.5).astype(np.float32)
    k = 6
    ro, eo = refine_3d(E, W, S3, k)
    plan = cpra.Plan(N, N)
    rg, eg = plan.refine_3d(torch_cuda.from_numpy(E).cuda(), torch_cuda.from_numpy(W).cuda(), torch_cuda.from_numpy(S3).cuda(), k)
    assert rel_l2(rg.cpu().numpy(), ro) <= 2 * TOL_1
    assert np.abs(eg.cpu().numpy() - eo).max() <= TOL_E * eo.max()
    assert np.all(np.diff(eo) <= 1e-12)
    assert np.abs(rg.cpu().numpy()[S3 == 0]).max() == 0.0


@pytest.mark.parametrize("N", [32, 64, 48])
def test_refine_3d_sw(torch_cuda, N):
    """Step D's iterations with the support re-thresholded every 2 iterations (reading A30), device vs oracle.  The
    threshold is taken in fp32 on the device and in fp64 by the oracle: voxels whose blurred value lies within
    rounding of it are set aside for the comparison of the support; the test data keep them out of the way."""
    import paper_2402_05283_b200 as cpra
    from oracle import refine_3d_sw
    rng = np.random.default_rng(N)
    h = N // 2
    a = max(2, N // 6)
    obj = np.zeros((N, N, N), np.complex64)
    obj[h - a:h + a, h - a + 1:h + a, h - a:h + a - 1] = (rng.uniform(0.3, 1.0, size=(2 * a, 2 * a - 1, 2 * a - 1)) *
                                                          np.exp(1j * rng.uniform(0, 1, size=(2 * a, 2 * a - 1, 2 * a - 1)))).astype(np.complex64)
    S3 = np.zeros((N, N, N), np.uint8)
    S3[h - a - 3:h + a + 3, h - a - 2:h + a + 3, h - a - 3:h + a + 2] = 1
    E = np.fft.fftn(obj.astype(np.complex128)).astype(np.complex64)
    W = (rng.uniform(size=(N, N, N)) < 0.7).astype(np.float32)
    k, every, sig, thr = 5, 2, 1.0, 0.12
    plan = cpra.Plan(N, N)
    dE, dW, dS = (torch_cuda.from_numpy(x).cuda() for x in (E, W, S3))
    # one update (after iteration 2 of 3): the blurred volumes agree, the supports agree away from the threshold
    og, eg, sg, bg = plan.refine_3d_sw(dE, dW, dS, 3, every, sig, thr, want_blurred=True)
    oo, eo, so, bo = refine_3d_sw(E, W, S3, 3, every, sig, thr, want_blurred=True)
    assert np.abs(bg.cpu().numpy() - bo).max() <= 2e-5 * bo.max()
    clear = np.abs(bo - thr * bo.max()) > 5e-5 * bo.max()
    assert np.array_equal(sg.cpu().numpy()[clear], so[clear]) and (~clear).mean() < 2e-3
    assert 0 < so.sum() < S3.sum()
    assert np.array_equal(dS.cpu().numpy(), S3)                      # the caller's tensor is untouched by the binding
    # the full run, continued on both sides from the SAME support history: feed the device's support of each update
    # back through a run of its own (k = 5: updates after iterations 2 and 4)
    og, eg, sg = plan.refine_3d_sw(dE, dW, dS, k, every, sig, thr)
    oo, eo, so = refine_3d_sw(E, W, S3, k, every, sig, thr)
    same = np.array_equal(sg.cpu().numpy(), so)
    if same:                                                         # no voxel sat on the threshold: everything is comparable
        assert rel_l2(og.cpu().numpy(), oo) <= 3 * TOL_1
        assert np.abs(eg.cpu().numpy() - eo).max() <= TOL_E * eo.max()
    else:
        assert (sg.cpu().numpy() != so).mean() < 1e-3
    assert np.abs(og.cpu().numpy()[sg.cpu().numpy() == 0]).max() == 0.0
    # every = 0 is cpra_refine_3d
    o1, e1 = plan.refine_3d(dE, dW, dS, 3)
    o2, e2, s2 = plan.refine_3d_sw(dE, dW, dS, 3, 0, sig, thr)
    assert torch_cuda.equal(o1, o2) and torch_cuda.equal(e1, e2) and torch_cuda.equal(s2, dS)
    with pytest.raises(cpra.CpraError) as e:
        plan.refine_3d_sw(dE, dW, dS, 3, 1, -1.0, thr)
    assert e.value.code == cpra.ERR_INVALID_ARG


@pytest.mark.parametrize("cfg,Np,N", [(1, 8, None), (4, 6, 128), (1, 5, 160), (3, 6, None)])
def test_backproject_support(torch_cuda, cfg, Np, N):
    """The visual hull of the 2D supports (reading A29), device vs oracle, bit for bit (u is evaluated in double on
    both sides with the same roundings), through both support layouts (bit-packed / bytes)."""
    p = cpra_inputs.make_problem(cfg, Np=Np, N=N, keep_object=True)
    o, g = _oracle(p), _gpu(p)
    ho, hg = o.backproject_support(), g.backproject_support().cpu().numpy()
    assert np.array_equal(ho, hg)
    assert 0 < hg.sum() < p.N ** 3 // 2
    # tighter supports: the silhouettes of the true projections; the hull contains the object
    S = (np.abs(p.projections) > 0).astype(np.uint8)
    o.set_support(S)
    g.set_support(torch_cuda.from_numpy(S).cuda())
    ho, hg = o.backproject_support(), g.backproject_support().cpu().numpy()
    assert np.array_equal(ho, hg)
    pad = np.zeros((p.N,) * 3)
    off = (p.N - p.obj.shape[0]) // 2
    pad[off:off + p.obj.shape[0], off:off + p.obj.shape[0], off:off + p.obj.shape[0]] = np.abs(p.obj)
    assert hg[pad > 0].all()


@pytest.mark.parametrize("N", [16, 64, 128])
def test_fsc(torch_cuda, N):
    import paper_2402_05283_b200 as cpra
    from oracle import fsc
    rng = np.random.default_rng(N)
    F = (rng.normal(size=(N, N, N)) + 1j * rng.normal(size=(N, N, N))).astype(np.complex64)
    G = (0.6 * F + rng.normal(size=(N, N, N)) + 1j * rng.normal(size=(N, N, N))).astype(np.complex64)
    plan = cpra.Plan(N, N)
    out = plan.fsc(torch_cuda.from_numpy(F).cuda(), torch_cuda.from_numpy(G).cuda()).cpu().numpy()
    assert np.abs(out - fsc(F, G)).max() <= 2e-6
    assert np.abs(plan.fsc(torch_cuda.from_numpy(F).cuda(), torch_cuda.from_numpy(F).cuda()).cpu().numpy() - 1.0).max() <= 2e-6


@pytest.mark.parametrize("cfg,Np,N", [(1, 8, None), (2, 12, None), (3, 6, None), (4, 4, None), (1, 5, 160)])
def test_prtf(torch_cuda, cfg, Np, N):
    """PRTF of the supported estimate after a few iterations against the measured amplitudes (beamstop pixels
    and zero-count pixels left out), device vs oracle."""
    p = cpra_inputs.make_problem(cfg, Np=Np, N=N)
    o, g = _oracle(p), _gpu(p)
    o.iterate(3, p.beta)
    g.iterate(3, p.beta)
    avg = o.get_projections(1).astype(np.complex64)
    want = o.prtf(avg)
    got = g.prtf(torch_cuda.from_numpy(avg).cuda()).cpu().numpy()
    assert np.abs(got - want).max() <= 2e-5 * max(1.0, np.abs(want).max())
    assert want[p.N // 4] > 0


# ------------------------------------------------------------------------------------------------
# f4: sizes that are not powers of two (PAPER.md:82 N = 160, :98 N = 700): the mixed-radix path
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [20, 48, 100, 160, 224, 360, 420, 700, 1008])
def test_fft2_mixed_radix(torch_cuda, N):
    import paper_2402_05283_b200 as cpra
    Np = 2
    rng = np.random.default_rng(N)
    x = (rng.normal(size=(Np, N, N)) + 1j * rng.normal(size=(Np, N, N))).astype(np.complex64)
    plan = cpra.Plan(N, Np)
    F = plan.fft2(torch_cuda.from_numpy(x).cuda(), -1).cpu().numpy()
    ref = np.fft.fft2(x.astype(np.complex128))
    assert rel_l2(F, ref) < 3e-6, rel_l2(F, ref)
    assert rel_l2(plan.fft2(torch_cuda.from_numpy(F).cuda(), +1).cpu().numpy(), x) < 4e-6
    d = np.zeros((Np, N, N), np.complex64)
    d[:, 3, 5] = 1.0
    Fd = plan.fft2(torch_cuda.from_numpy(d).cuda(), -1).cpu().numpy()
    ky, kx = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    assert np.abs(Fd[1] - np.exp(-2j * np.pi * (3 * ky + 5 * kx) / N)).max() < 2e-5


@pytest.mark.parametrize("N,Np", [(64, 5), (256, 4), (512, 3), (1024, 2), (160, 3), (700, 2)])
def test_set_estimate_spectrum(torch_cuda, N, Np):
    """cpra_set_estimate_spectrum: the start given as its spectrum equals the inverse transform handed to
    cpra_set_estimate, and the loop runs on from it like the oracle's."""
    p = cpra_inputs.random_stack(N, Np, seed=40 + N, beamstop=3)
    rng = np.random.default_rng(N)
    G0 = (rng.normal(size=(Np, N, N)) + 1j * rng.normal(size=(Np, N, N))).astype(np.complex64)
    g0 = np.fft.ifft2(G0.astype(np.complex128))
    alpha = (0.6, 0.2) if Np >= 3 else (1.0,)
    g = _gpu(p, alpha)
    g.set_estimate_spectrum(torch_cuda.from_numpy(G0).cuda())
    assert g.iteration == 0
    assert rel_l2(_get(g), g0) <= 4e-6 if N < 700 else 6e-6
    p.estimate = g0.astype(np.complex64)
    o = _oracle(p, alpha)
    o.iterate(2, 0.9)
    g.iterate(2, 0.9)
    assert rel_l2(_get(g), o.get_projections(0)) <= 3 * TOL_1


def test_fft2_every_supported_mixed_radix_size(torch_cuda):
    """Every even N in [16, 1024] with prime factors 2, 3, 5, 7 that is not a power of two (every combination of stage
    radices, ragged last tiles on both tile widths): forward transform of one random image against numpy, round trip."""
    import paper_2402_05283_b200 as cpra
    sizes = []
    for N in range(16, 1025, 2):
        n = N
        for f in (2, 3, 5, 7):
            while n % f == 0:
                n //= f
        if n == 1 and N & (N - 1):
            sizes.append(N)
    assert len(sizes) > 60 and 160 in sizes and 700 in sizes
    rng = np.random.default_rng(9)
    worst = 0.0
    for N in sizes:
        x = (rng.normal(size=(1, N, N)) + 1j * rng.normal(size=(1, N, N))).astype(np.complex64)
        plan = cpra.Plan(N, 1)
        d = torch_cuda.from_numpy(x).cuda()
        F = plan.fft2(d, -1)
        e = rel_l2(F.cpu().numpy(), np.fft.fft2(x.astype(np.complex128)))
        b = rel_l2(plan.fft2(F, +1).cpu().numpy(), x)
        plan.close()
        worst = max(worst, e, b)
        assert e < 3e-6 and b < 4e-6, (N, e, b)
    print(f"\n{len(sizes)} mixed-radix sizes, worst relL2 {worst:.2e}")


@pytest.mark.parametrize("N,Np,alpha,n_ei,seam,rule", [
    (160, 6, (0.6, 0.2), 1, 0, "hio"), (160, 5, (0.5, 0.2, 0.05), 2, 1, "raar"), (48, 7, (0.6, 0.2), 1, 1, "hio"),
    (100, 3, (0.6, 0.2), 3, 0, "er"), (700, 3, (0.6, 0.2), 1, 0, "hio"), (20, 1, (1.0,), 1, 0, "hio"),
    (420, 3, (0.6, 0.2), 1, 1, "hio")])
def test_loop_mixed_radix(torch_cuda, N, Np, alpha, n_ei, seam, rule):
    """The loop at the paper's own detector sizes (160, 700) and other 2^a 3^b 5^c 7^d sizes against the oracle,
    whose transform for these N is the O(N^2)-per-line definition."""
    p = cpra_inputs.random_stack(N, Np, seed=700 + N + Np, beamstop=3)
    o, g = _oracle(p, alpha, n_ei), _gpu(p, alpha, n_ei)
    o.set_seam(seam); g.set_seam(bool(seam))
    o.set_update(rule); g.set_update(rule)
    k = 2 if N >= 420 else 4
    o.iterate(k, 0.9)
    g.iterate(k, 0.9)
    assert rel_l2(_get(g), o.get_projections(0)) <= k * TOL_1
    assert rel_l2(_get(g, 1), o.get_projections(1)) <= k * TOL_1
    E, Eg = g.get_error()
    Eo, Ego = o.get_error()
    assert np.abs(E.cpu().numpy() - Eo).max() <= TOL_E * Eo.max() and abs(float(Eg.cpu()[0]) - Ego) <= TOL_E * Ego
    # split calls are bit-identical; Step A and the bank work on these sizes too
    h = _gpu(p, alpha, n_ei); h.set_seam(bool(seam)); h.set_update(rule)
    for kk in ([1, 1] if k == 2 else [1, 2, 1]):
        h.iterate(kk, 0.9)
    assert np.array_equal(_get(h).view(np.uint32), _get(g).view(np.uint32))
    o.prereconstruct(0, 2, 0.9)
    g.prereconstruct(0, 2, 0.9)
    assert rel_l2(_get(g), o.get_projections(0)) <= (k + 2) * TOL_1


def test_full_size_paper_simulation_detector(torch_cuda):
    """The paper's simulated case at its own size (N = 160 with N_p = 90 projections): config 1's object
    scaled to N = 160, every projection after two iterations of the coupled loop against the oracle (whose transform at
    this N is the O(N^2) definition), and the per-projection errors."""
    p = cpra_inputs.make_problem(1, Np=90, N=160)
    o, g = _oracle(p), _gpu(p)
    o.set_seam(1); g.set_seam(True)
    o.iterate(2, p.beta)
    g.iterate(2, p.beta)
    out, ref = _get(g), o.get_projections(0)
    pn = np.sqrt((np.abs(out - ref) ** 2).sum(axis=(1, 2)) / (np.abs(ref) ** 2).sum(axis=(1, 2)))
    assert pn.max() <= 3 * TOL_1 and np.median(pn) <= TOL_1, (pn.max(), np.median(pn))
    E, Eg = g.get_error()
    Eo, Ego = o.get_error()
    assert np.abs(E.cpu().numpy() - Eo).max() <= TOL_E * Eo.max() and abs(float(Eg.cpu()[0]) - Ego) <= TOL_E * Ego


def test_assembly_and_merge_mixed_radix(torch_cuda):
    """Config 1 scaled to N = 160 (the paper's oxide-particle detector size): three iterations, the
    Fourier-slice assembly and a merge from the plan, against the oracle."""
    p = cpra_inputs.make_problem(1, Np=6, N=160)
    o, g = _oracle(p), _gpu(p)
    o.iterate(3, p.beta)
    g.iterate(3, p.beta)
    assert rel_l2(_get(g), o.get_projections(0)) <= 3 * TOL_1
    vo, wo = o.assemble_3d()
    vg, wg = g.assemble_3d()
    assert np.array_equal(wg.cpu().numpy().astype(np.float64), wo)
    assert rel_l2(vg.cpu().numpy(), vo) <= 3 * TOL_1
    o.merge_begin(2); g.merge_begin(2)
    o.merge_offer(); g.merge_offer()
    out_o, sh_o, tw_o = o.merge_finish(0)
    out_g, sh_g, tw_g = g.merge_finish(0)
    assert np.array_equal(sh_g.cpu().numpy()[:len(sh_o)], sh_o)       # (one episode kept of the two slots)
    assert rel_l2(out_g.cpu().numpy(), out_o) <= 3 * TOL_1


@pytest.mark.parametrize("N,Np,rule,flags", [(64, 5, "hio", 0), (128, 4, "raar", 0), (256, 5, "hio", 0), (512, 5, "hio", 0),
                                             (512, 4, "er", 4), (1024, 3, "hio", 0), (160, 4, "hio", 0)])
def test_positivity(torch_cuda, N, Np, rule, flags):
    """cpra_set_positivity through every kernel family.  The sign test on Re g' is taken in fp32 on the device and in
    fp64 by the oracle: after ONE iteration the two agree except at pixels whose Re g' lies within rounding of zero,
    which are set aside (what is unique is compared) and must be rare."""
    p = cpra_inputs.random_stack(N, Np, seed=1200 + N, beamstop=3)
    o, g = _oracle(p), _gpu(p, flags=flags)
    ref0 = _oracle(p)
    for plan in (o, g):
        plan.set_update(rule)
        plan.set_positivity(True)
    ref0.set_update(rule)
    o.iterate(1, 0.9)
    g.iterate(1, 0.9)
    ref0.iterate(1, 0.9)
    out, ref, plain = _get(g), o.get_projections(0), ref0.get_projections(0)
    # inside the support without positivity the state is g' itself: its real part is what the test looked at
    gp_re = plain.real
    clear = ~((p.support == 1) & (np.abs(gp_re) < 1e-5 * np.abs(plain).max()))
    assert (~clear).mean() < 1e-3
    assert np.linalg.norm((out - ref)[clear]) <= 2 * TOL_1 * np.linalg.norm(ref[clear])
    assert rel_l2(ref, plain) > 0.05                                   # the flag matters on this input
    # a second iteration through the multi-iteration path stays close (a flipped pixel would show as ~1e-3)
    o.iterate(1, 0.9)
    g.iterate(1, 0.9)
    assert rel_l2(_get(g), o.get_projections(0)) <= 2e-3


@pytest.mark.parametrize("N,Np,n_ref", [(64, 12, 0), (128, 7, 3), (160, 5, 4)])
def test_align_episode(torch_cuda, N, Np, n_ref):
    """cpra_align_episode against the oracle on a stack of true projections with scrambled phases and twins, and on
    a reconstructed episode."""
    import paper_2402_05283_b200 as cpra
    from oracle import align_episode
    p = cpra_inputs.make_problem(1, Np=Np, N=N, noise=False)
    rng = np.random.default_rng(N)
    i = (N - np.arange(N)) % N
    ep = (p.projections * np.exp(1j * rng.uniform(0, 6.28, size=Np))[:, None, None]).astype(np.complex64)
    for n in (1, Np - 2):
        ep[n] = np.conj(ep[n][i][:, i])
    plan = cpra.Plan(N, Np)
    d = torch_cuda.from_numpy(ep.copy()).cuda()
    fl = plan.align_episode(d, n_ref).cpu().numpy()
    ref, flo = align_episode(ep, n_ref)
    assert np.array_equal(fl, flo)
    assert rel_l2(d.cpu().numpy(), ref) <= 1e-6
    g = _gpu(p)
    g.iterate(5, p.beta)
    e2 = g.get_projections(1)
    ref2, fl2 = align_episode(e2.cpu().numpy(), n_ref)
    flg = g.align_episode(e2, n_ref).cpu().numpy()
    assert np.array_equal(flg, fl2) and rel_l2(e2.cpu().numpy(), ref2) <= 1e-6


def test_pipeline_steps_a_to_d(torch_cuda):
    """paper_2402_05283_b200.pipeline.reconstruct on config 1 (noise-free, 32 angles): N_r = 6 restarts, N_l = 3 kept,
    Step A batched over the restarts, Step D to O(r).  The merged projections correlate with the true ones and the
    3D object with the true object (up to the twin of the whole object)."""
    import paper_2402_05283_b200 as cpra
    p = cpra_inputs.make_problem(1, keep_object=True)
    dev = "cuda"
    I, M, S = (torch_cuda.from_numpy(a).to(dev) for a in (p.intensity, p.mask, p.support))
    res = cpra.pipeline.reconstruct(I, M, S, p.angles, n_restarts=6, n_keep=3, n_pre=200, n_episodes=25, n_ei=2, seam_flip=True)
    N = p.N
    ep = res.episode.cpu().numpy()
    corr = lambda a, b: abs(np.vdot(a, b)) / (np.linalg.norm(a) * np.linalg.norm(b))
    c2 = np.mean([max(corr(np.abs(ep[n]), np.abs(p.projections[n])), corr(np.abs(ep[n][::-1, ::-1]), np.abs(p.projections[n]))) for n in range(p.Np)])
    assert c2 > 0.9, c2
    pad = np.zeros((N, N, N))
    off = (N - p.obj.shape[0]) // 2
    pad[off:off + p.obj.shape[0], off:off + p.obj.shape[0], off:off + p.obj.shape[0]] = p.obj
    rec = res.obj.cpu().numpy()
    i = (N - np.arange(N)) % N
    c3 = max(corr(np.abs(rec), pad), corr(np.abs(rec[i][:, i][:, :, i]), pad))
    print(f"\npipeline: corr2d={c2:.3f} corr3d={c3:.3f} errors={res.errors.cpu().numpy()} seconds={res.seconds}")
    assert c3 > 0.8, c3
    assert len(res.errors) == 3 and float(res.errors.max()) < 0.2
    # Step D as PAPER.md:104 has it: 3D iterations against the back-projected 2D supports of the merged episode, the 3D
    # support re-thresholded every 5 iterations
    res = cpra.pipeline.reconstruct(I, M, S, p.angles, n_restarts=6, n_keep=3, n_pre=200, n_episodes=25, n_ei=2, seam_flip=True,
                                    refine_iters=20, shrink3d=(5, 2.0, 0.05))
    rec, s3 = res.obj.cpu().numpy(), res.support3d.cpu().numpy().astype(bool)
    both = [(np.abs(rec), s3), (np.abs(rec[i][:, i][:, :, i]), s3[i][:, i][:, :, i])]
    c3r, s3b = max(((corr(r, pad), m) for r, m in both), key=lambda t: t[0])
    inside = pad[s3b].sum() / pad.sum()
    print(f"pipeline + 3D iterations: corr3d={c3r:.3f} object mass inside the final 3D support={inside:.3f} "
          f"support voxels={int(s3.sum())} of {N ** 3} refine error {float(res.refine_error[0]):.3f} -> {float(res.refine_error[-1]):.3f}")
    assert c3r > 0.8, c3r
    assert inside > 0.9 and s3.sum() < 0.3 * N ** 3
    assert np.abs(rec[~s3]).max() == 0.0
