"""cpra_fsc_static (include/cpra.h): the entry point that allocates no device memory -- its scratch is a fixed
__device__ array inside libcpra.so -- against the existing path cpra_fsc (plan + workspace), on two calls in a row.

Collected last on purpose (the file name): the suite runs with pytest -x."""
import numpy as np
import pytest

TOL_FSC = 2e-6      # the bar of tests/test_gpu_next.py::test_fsc


def _pair(N, seed):
    rng = np.random.default_rng(seed)
    F = (rng.normal(size=(N, N, N)) + 1j * rng.normal(size=(N, N, N))).astype(np.complex64)
    G = (0.6 * F + rng.normal(size=(N, N, N)) + 1j * rng.normal(size=(N, N, N))).astype(np.complex64)
    return F, G


@pytest.mark.gpu
def test_fsc_static_matches_the_plan_path_on_two_calls_in_a_row():
    import torch
    import paper_2402_05283_b200 as cpra
    # two different problems and sizes, the larger one first: what the first call leaves in the shared array
    # (shells 33 .. 64 too) must not reach the second result
    cases = [(128, 11), (64, 12)]
    outs, wants = [], []
    for N, seed in cases:
        F, G = (torch.from_numpy(a).cuda() for a in _pair(N, seed))
        out = torch.full((N // 2 + 1,), float("nan"), dtype=torch.float32, device="cuda")   # caller-owned output
        res = cpra.fsc_static(F, G, out)
        assert res.data_ptr() == out.data_ptr()
        outs.append(out)
        plan = cpra.Plan(N, N)
        wants.append(plan.fsc(F, G))
        plan.close()
    torch.cuda.synchronize()
    for (N, _), out, want in zip(cases, outs, wants):
        o, w = out.cpu().numpy(), want.cpu().numpy()
        assert np.all(np.isfinite(o)) and o.shape == (N // 2 + 1,)
        assert np.abs(o - w).max() <= TOL_FSC
    # the same inputs again: the array is cleared by every call, so the result does not accumulate
    N, seed = cases[1]
    F, G = (torch.from_numpy(a).cuda() for a in _pair(N, seed))
    again = cpra.fsc_static(F, G, torch.empty(N // 2 + 1, dtype=torch.float32, device="cuda")).cpu().numpy()
    assert np.abs(again - wants[1].cpu().numpy()).max() <= TOL_FSC
    assert np.abs(cpra.fsc_static(F, F).cpu().numpy() - 1.0).max() <= TOL_FSC


@pytest.mark.gpu
def test_fsc_static_refuses_sizes_beyond_its_array():
    import torch
    import paper_2402_05283_b200 as cpra
    L = cpra.lib()
    buf = torch.zeros(16, dtype=torch.float32, device="cuda")     # never touched: the size check comes first
    p = buf.data_ptr()
    assert L.cpra_fsc_static(cpra.binding.FSC_STATIC_MAX_N + 2, p, p, p, None) == cpra.ERR_UNSUPPORTED_SIZE
    assert L.cpra_fsc_static(63, p, p, p, None) == cpra.ERR_INVALID_ARG
    assert L.cpra_fsc_static(64, None, p, p, None) == cpra.ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert float(buf.abs().max()) == 0.0
