"""The seeded input generator: determinism, shapes, conventions (SURVEY.md 8(d) recipe)."""
import numpy as np

import cpra_inputs


def test_projector_c_equals_numpy_and_axis_sum():
    rng = np.random.default_rng(0)
    obj = rng.uniform(size=(8, 8, 8)) + 1j * rng.uniform(size=(8, 8, 8))
    ang = np.array([0.0, 0.3, np.pi / 2, 2.0, np.pi, 4.0])
    a = cpra_inputs.project(obj, 16, ang)
    b = cpra_inputs.project_numpy(obj, 16, ang)
    assert np.abs(a - b).max() < 1e-12
    pad = np.zeros((16, 16, 16), complex)
    pad[4:12, 4:12, 4:12] = obj
    assert np.abs(a[0] - pad.sum(axis=1)).max() < 1e-13          # theta = 0: plain sum along y


def test_problem_is_deterministic_and_well_formed():
    p1 = cpra_inputs.make_problem(2, Np=6, N=32)
    p2 = cpra_inputs.make_problem(2, Np=6, N=32)
    for f in ("intensity", "mask", "support", "estimate", "angles"):
        assert np.array_equal(getattr(p1, f), getattr(p2, f)), f
    assert p1.intensity.dtype == np.float32 and p1.estimate.dtype == np.complex64
    assert p1.mask.dtype == np.uint8 and p1.support.dtype == np.uint8
    N = p1.N
    # detector-centred: the brightest pixel region is at the centre; beamstop zeros sit there
    assert p1.mask[0, N // 2, N // 2] == 0 and p1.mask[0, 0, 0] == 1
    assert (p1.mask[0] == 0).sum() == 25
    # Poisson counts: integers, total close to the photon budget
    assert np.all(p1.intensity == np.round(p1.intensity))
    assert abs(p1.intensity[0].sum() / 1e7 - 1) < 0.01
    # support contains the bulk of the true projection and stays inside the half-size box
    P = np.abs(p1.projections)
    assert (P * p1.support).sum() > 0.95 * P.sum()
    # oversampling: projected object occupies < N/2 * sqrt(2) in u
    cols = np.where(p1.support.any(axis=(0, 1)))[0]
    assert cols.max() - cols.min() < 0.75 * N


def test_configs_match_baseline_json():
    import json, os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cfgs = json.load(open(os.path.join(root, "BASELINE.json")))["configs"]
    want = {1: (64, 32), 2: (128, 90), 3: (256, 180), 4: (512, 360), 5: (1024, 180)}
    for i, (N, Np) in want.items():
        assert cpra_inputs.CONFIGS[i]["N"] == N and cpra_inputs.CONFIGS[i]["Np"] == Np
        assert f"N={N}" in cfgs[i - 1] or f"{N}³" in cfgs[i - 1] or f"{N}×{N}" in cfgs[i - 1]
