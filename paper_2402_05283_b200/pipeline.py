"""CPRA as the paper composes it (Fig. 2), on top of the C-ABI calls: orchestration only.

    Step A  pre-reconstruct projection 0 from a random start -- for ALL N_r restarts at once: the
            N_r random starts of that one projection are a stack of their own (a plan with N_r images of the same
            data, coupling off), so the N_i^pre conventional iterations run batched instead of one image at a time
    Step B  per restart: N_e episodes of N_ei iterations of the coupled loop (cpra_iterate with n_ei = N_ei)
    Step C  the bank keeps the N_l lowest-error episodes (cpra_merge_offer, decided on the device); centre of mass,
            twin selection, average (cpra_merge_finish)
            then cpra_align_episode: the projections of the merged episode are given one common phase gauge and one
            twin choice (reading A28) -- without it the slices of an unconstrained complex iterate do not fit together
    Step D  Fourier-slice assembly of the merged episode (cpra_assemble_3d), then optionally the inverse 3D
            transform / the iterations against a 3D support (cpra_fft3 / cpra_refine_3d / cpra_refine_3d_sw); the 3D
            support is the caller's or the back-projection of the merged episode's 2D supports (cpra_shrinkwrap on the
            merged episode, then cpra_backproject_support: PAPER.md:104)

Every arithmetic step runs in the library's kernels; this module only allocates torch tensors, draws the random
starting phases (torch's generator on the device: input generation, not part of the method) and calls the binding."""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import Optional


from . import binding


@dataclass
class CpraResult:
    episode: "object"            # merged episode, complex64 [Np, N, N] (device)
    errors: "object"             # float64 [N_l] errors of the kept restarts (device)
    shifts: "object"             # int32 [N_l, Np, 2]
    twins: "object"              # int32 [N_l]
    spectrum: "object" = None    # complex64 [N, N, N], the assembled E(q) (device) if assemble=True
    weight: "object" = None      # float32 [N, N, N]
    obj: "object" = None         # complex64 [N, N, N], O(r) if a 3D step was asked for
    refine_error: "object" = None
    support3d: "object" = None   # u8 [N, N, N]: the 3D support Step D ended with
    seconds: dict = None


def native_amplitudes(intensity, mask):
    """M sqrt(max(I, 0)) in native order (zero frequency at index 0) from detector-centred intensities: the modulus of
    every random-phase start (the same for all restarts: computed once)."""
    import torch
    N = intensity.shape[-1]
    A = torch.sqrt(torch.clamp(intensity.to(torch.float32), min=0.0))
    if mask is not None:
        A = A * mask.to(torch.float32)
    return torch.roll(A, shifts=(-(N // 2), -(N // 2)), dims=(-2, -1)).contiguous()


def random_phase_spectra(intensity, mask, seed: int, amplitudes=None):
    """G0 = M sqrt(I) e^{i phi}, phi ~ U[0, 2 pi) per pixel (reading A15; "random initial guess"), native
    order, complex64 [n, N, N]: the spectrum of a random start (input generation: torch's generator on the device).
    amplitudes = native_amplitudes(intensity, mask), computed once for many restarts."""
    import torch
    A = native_amplitudes(intensity, mask) if amplitudes is None else amplitudes
    gen = torch.Generator(device=A.device)
    gen.manual_seed(int(seed))
    phi = torch.empty(A.shape, device=A.device, dtype=torch.float32).uniform_(0.0, 2.0 * math.pi, generator=gen)
    return torch.polar(A, phi)


def random_phase_starts(plan, intensity, mask, seed: int, amplitudes=None):
    """Random-phase starts g0 = F^-1[G0] of random_phase_spectra, through the library's own cpra_fft2; complex64 [n, N, N]."""
    return plan.fft2(random_phase_spectra(intensity, mask, seed, amplitudes), +1)


def reconstruct(intensity, mask, support, angles, n_restarts: int, n_keep: int, n_pre: int, n_episodes: int, n_ei: int,
                beta: float = 0.9, alpha=(0.6, 0.2), update: str = "hio", seam_flip: bool = False, seed: int = 0,
                shrinkwrap: Optional[tuple] = None, assemble: bool = True, support3d=None, refine_iters: int = 0,
                n_ref: int = 0, align: bool = True, step3d: bool = True, shrink3d: Optional[tuple] = None,
                support2d_for_3d: tuple = (3.0, 0.03)) -> CpraResult:
    """Steps A-D.  intensity fp32 [Np, N, N], mask u8 [Np, N, N] or None, support u8 [Np, N, N]: CUDA tensors;
    angles: Np radians (host).  shrinkwrap = (sigma, threshold): one support update at the end of every episode
    (PAPER.md:104).  refine_iters > 0: Step D's iterations against support3d (u8 [N, N, N]) or, if that is None, against
    the back-projection of the 2D supports that a shrink-wrap with support2d_for_3d = (sigma, threshold) finds on the
    merged episode; shrink3d = (every, sigma, threshold): the 3D support is re-thresholded every `every` iterations
    (PAPER.md:104).  refine_iters == 0 with assemble: E(q) and O(r) = F3^-1[E] (step3d=False: E(q) only)."""
    import torch
    Np, N = int(intensity.shape[0]), int(intensity.shape[-1])
    dev = intensity.device
    sec = {}

    def timed(name, t0):
        t1 = torch.cuda.Event(enable_timing=True)
        t1.record()
        torch.cuda.synchronize(dev)
        sec[name] = t0.elapsed_time(t1) * 1e-3

    def start():
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    # ---- Step A, batched over the restarts: N_r starts of projection 0, no coupling -------------------------------
    t0 = start()
    pre = None
    if n_pre > 0:
        pa = binding.Plan(N, n_restarts)
        pa.set_data(intensity[:1].expand(n_restarts, N, N).contiguous(),
                    None if mask is None else mask[:1].expand(n_restarts, N, N).contiguous(), None)
        pa.set_support(support[:1].expand(n_restarts, N, N).contiguous())
        pa.set_carousel((1.0,), 1)
        pa.set_update(update)
        I0 = intensity[:1].expand(n_restarts, N, N).contiguous()
        M0 = None if mask is None else mask[:1].expand(n_restarts, N, N).contiguous()
        pa.set_estimate_spectrum(random_phase_spectra(I0, M0, seed))
        pa.iterate(n_pre, beta)
        # the restarts take their projection 0 from here: as spectra, which is how the starts are handed over
        pre = pa.fft2(pa.get_projections(binding.ITERATE), -1)
        pa.close()
    timed("step_a", t0)

    # ---- Steps B and C ----------------------------------------------------------------------------------------------
    t0 = start()
    plan = binding.Plan(N, Np)
    plan.set_data(intensity, mask, angles)
    plan.set_carousel(alpha, n_ei)
    plan.set_update(update)
    plan.set_seam(seam_flip)
    plan.merge_begin(n_keep)
    amplitudes = native_amplitudes(intensity, mask)
    for r in range(n_restarts):
        plan.set_support(support)
        G0 = random_phase_spectra(intensity, mask, seed + 7919 * (r + 1), amplitudes)
        if pre is not None:
            G0[0] = pre[r]
        plan.set_estimate_spectrum(G0)
        for _ in range(n_episodes):
            plan.iterate(n_ei, beta)
            if shrinkwrap is not None:
                plan.shrinkwrap(float(shrinkwrap[0]), float(shrinkwrap[1]))
        plan.merge_offer()
    episode, shifts, twins = plan.merge_finish(n_ref)
    if align:
        plan.align_episode(episode, n_ref)          # one phase gauge and one twin choice for the whole stack (reading A28)
    errors, count = plan.merge_errors()
    timed("steps_b_c", t0)
    res = CpraResult(episode=episode, errors=errors[:int(count.cpu()[0])], shifts=shifts, twins=twins, seconds=sec)

    # ---- Step D -----------------------------------------------------------------------------------------------------
    if assemble:
        t0 = start()
        # the merged episode is already restricted to (shifted) supports: assemble it as it is
        plan.set_support(torch.ones((Np, N, N), dtype=torch.uint8, device=dev))
        plan.set_estimate(episode)
        res.spectrum, res.weight = plan.assemble_3d()
        timed("assemble", t0)
        if step3d:
            t0 = start()
            if refine_iters > 0 and support3d is None:
                # the 2D supports of the merged projections, projected back
                plan.shrinkwrap(float(support2d_for_3d[0]), float(support2d_for_3d[1]))
                support3d = plan.backproject_support()
            plan.close()
            p3 = binding.Plan(N, N)
            if refine_iters > 0:
                if shrink3d is not None:
                    res.obj, res.refine_error, res.support3d = p3.refine_3d_sw(res.spectrum, res.weight, support3d, refine_iters,
                                                                               int(shrink3d[0]), float(shrink3d[1]), float(shrink3d[2]))
                else:
                    res.obj, res.refine_error = p3.refine_3d(res.spectrum, res.weight, support3d, refine_iters)
                    res.support3d = support3d
            else:
                res.obj = p3.fft3(res.spectrum, +1)
            p3.close()
            timed("step_d_3d", t0)
    plan.close()
    return res
