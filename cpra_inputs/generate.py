"""Seeded synthetic inputs for the CPRA iteration loop (shared by the oracle tests and the GPU tests).

This module is *input generation only*.  It holds none of the method's arithmetic: no mix, no
modulus projection, no HIO, no error metric, no assembly.  It builds a voxel object, projects it
(the forward model of PAPER.md:31-44, Eq. (1)-(3)), forms intensities with numpy's library FFT,
adds Poisson noise, and derives masks, supports and random-phase initial estimates.  Neither
``oracle/`` nor ``paper_2402_05283_b200/`` is imported here, and neither imports the other.

The recipes follow BASELINE.json's five configs / SURVEY.md 8(d); they are synthetic stand-ins for
the paper's workloads (Li-rich layered-oxide particle PAPER.md:80, S. aureus cell PAPER.md:98,
performance sweep PAPER.md:106), which are not available.  DESIGN.md section "Input recipe" states
every choice made here.

Conventions:
  * arrays O[z][y][x]; projections P[n][z][u], rotation about z, angles in radians;
  * forward FT  e^{-2 pi i ...} unnormalised (numpy.fft.fft2);
  * intensities and masks are *detector-centred* (DC at index N/2, i.e. numpy.fft.fftshift of the
    native order); projected objects, supports and estimates are centred at pixel (N/2, N/2).
"""
from __future__ import annotations

import ctypes
import dataclasses
import math
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SEED_BASE = 240205283 * 10

# id -> recipe.  n_in = inner (unpadded) object grid = N/2 (oversampling).
CONFIGS = {
    1: dict(name="tiny", N=64, Np=32, range_deg=180.0, photons=None, beamstop=0, iters=50,
            complex_obj=False, support_r=2),
    2: dict(name="ellipsoids128", N=128, Np=90, range_deg=180.0, photons=1e7, beamstop=5, iters=200,
            complex_obj=False, support_r=3),
    3: dict(name="oxide256", N=256, Np=180, range_deg=180.0, photons=1e8, beamstop=9, iters=500,
            complex_obj=False, support_r=3),
    4: dict(name="cell512", N=512, Np=360, range_deg=360.0, photons=1e9, beamstop=15, iters=300,
            complex_obj=True, support_r=3),
    5: dict(name="large1024", N=1024, Np=180, range_deg=180.0, photons=None, beamstop=0, iters=100,
            complex_obj=False, support_r=3),
}


@dataclasses.dataclass
class Problem:
    """One CPRA input set.  All arrays are C-contiguous."""
    config: int
    N: int
    Np: int
    angles: np.ndarray        # [Np] float64, radians
    intensity: np.ndarray     # [Np,N,N] float32, detector-centred
    mask: np.ndarray          # [Np,N,N] uint8, detector-centred, 1 = measured
    support: np.ndarray       # [Np,N,N] uint8, 1 = inside
    estimate: np.ndarray      # [Np,N,N] complex64, initial guess g^0
    projections: np.ndarray   # [Np,N,N] complex128, the true projected objects (not an input)
    obj: Optional[np.ndarray]  # [n_in]^3 inner object (None if dropped to save memory)
    beta: float = 0.9
    iters: int = 0


# ----------------------------------------------------------------------------------------------
# projector (C helper with a numpy fallback)
# ----------------------------------------------------------------------------------------------
_lib = None


def build_projector(force: bool = False) -> str:
    """Compile cpra_inputs/projector.c -> libcpra_projector.so (gcc, OpenMP).  Returns the path."""
    src = os.path.join(_HERE, "projector.c")
    out = os.path.join(_HERE, "libcpra_projector.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", out, src, "-lm"])
    return out


def _projector():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build_projector())
        _lib.cpra_project.restype = None
        _lib.cpra_project.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
                                      ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    return _lib


def project(obj: np.ndarray, N: int, angles: np.ndarray) -> np.ndarray:
    """Line-integral projections of obj[z][y][x] (inner grid, centred in an N grid) rotated about z.

    Returns P[n][z][u] complex128 (imaginary part zero for a real object)."""
    nin = obj.shape[0]
    assert obj.shape == (nin, nin, nin) and (N - nin) % 2 == 0
    angles = np.ascontiguousarray(angles, dtype=np.float64)
    Np = len(angles)
    re = np.ascontiguousarray(obj.real, dtype=np.float64)
    out_re = np.zeros((Np, N, N), dtype=np.float64)
    if np.iscomplexobj(obj):
        im = np.ascontiguousarray(obj.imag, dtype=np.float64)
        out_im = np.zeros((Np, N, N), dtype=np.float64)
        _projector().cpra_project(re.ctypes.data, im.ctypes.data, nin, N, Np, angles.ctypes.data,
                                  out_re.ctypes.data, out_im.ctypes.data)
        return out_re + 1j * out_im
    _projector().cpra_project(re.ctypes.data, None, nin, N, Np, angles.ctypes.data,
                              out_re.ctypes.data, None)
    return out_re.astype(np.complex128)


def project_numpy(obj: np.ndarray, N: int, angles: np.ndarray) -> np.ndarray:
    """Pure-numpy restatement of `project` (slow; used to cross-check the C helper on small cases)."""
    nin = obj.shape[0]
    off = (N - nin) // 2
    c = N // 2
    pad = np.zeros((nin, nin + 2, nin + 2), dtype=np.complex128)   # one zero voxel all round
    pad[:, 1:-1, 1:-1] = obj
    out = np.zeros((len(angles), N, N), dtype=np.complex128)
    u = (np.arange(N) - c)[:, None]
    s = (np.arange(N) - c)[None, :]
    for n, th in enumerate(angles):
        ct, st = math.cos(th), math.sin(th)
        x = u * ct - s * st + c - off + 1.0      # +1: index into the padded slice
        y = u * st + s * ct + c - off + 1.0
        ok = (x >= 0) & (y >= 0) & (x < nin + 1) & (y < nin + 1)
        x = np.where(ok, x, 0.0)
        y = np.where(ok, y, 0.0)
        x0 = np.floor(x).astype(np.int64)
        y0 = np.floor(y).astype(np.int64)
        wx = x - x0
        wy = y - y0
        v = (pad[:, y0, x0] * ((1 - wy) * (1 - wx)) + pad[:, y0, x0 + 1] * ((1 - wy) * wx)
             + pad[:, y0 + 1, x0] * (wy * (1 - wx)) + pad[:, y0 + 1, x0 + 1] * (wy * wx))
        v = np.where(ok[None], v, 0.0)
        out[n, off:off + nin, :] = v.sum(axis=2)
    return out


# ----------------------------------------------------------------------------------------------
# objects
# ----------------------------------------------------------------------------------------------
def _add_ellipsoid(vol, centre, axes, value, mode="add"):
    """vol[z][y][x] += value inside the ellipsoid; centre/axes given as (x, y, z)."""
    n = vol.shape[0]
    lo = [max(0, int(math.floor(centre[i] - axes[i]))) for i in range(3)]
    hi = [min(n, int(math.ceil(centre[i] + axes[i])) + 1) for i in range(3)]
    if any(h <= l for l, h in zip(lo, hi)):
        return
    x = (np.arange(lo[0], hi[0]) - centre[0]) / axes[0]
    y = (np.arange(lo[1], hi[1]) - centre[1]) / axes[1]
    z = (np.arange(lo[2], hi[2]) - centre[2]) / axes[2]
    inside = (z[:, None, None] ** 2 + y[None, :, None] ** 2 + x[None, None, :] ** 2) <= 1.0
    sub = vol[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]]
    if mode == "add":
        sub[inside] += value
    else:
        sub[inside] = value


def _add_gaussian(vol, centre, sigma, amp):
    n = vol.shape[0]
    r = 4.0 * sigma
    lo = [max(0, int(math.floor(centre[i] - r))) for i in range(3)]
    hi = [min(n, int(math.ceil(centre[i] + r)) + 1) for i in range(3)]
    if any(h <= l for l, h in zip(lo, hi)):
        return
    gx = np.exp(-0.5 * ((np.arange(lo[0], hi[0]) - centre[0]) / sigma) ** 2)
    gy = np.exp(-0.5 * ((np.arange(lo[1], hi[1]) - centre[1]) / sigma) ** 2)
    gz = np.exp(-0.5 * ((np.arange(lo[2], hi[2]) - centre[2]) / sigma) ** 2)
    vol[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] += amp * gz[:, None, None] * gy[None, :, None] * gx[None, None, :]


def make_object(config: int, nin: int, rng: np.random.Generator) -> np.ndarray:
    """The inner-grid object of BASELINE.json config `config`, voxelised on nin^3 (scaled if nin
    differs from the config's own inner grid).  Real float64, or complex128 for config 4."""
    ref = CONFIGS[config]["N"] // 2
    sc = nin / ref                       # geometric scale when a config is run at another N
    c = nin / 2.0
    vol = np.zeros((nin, nin, nin), dtype=np.float64)
    if config == 1:
        # solid ellipsoid (semi-axes 10, 8, 6 along x, y, z), density 1, + 5 Gaussian blobs inside
        ax = np.array([10.0, 8.0, 6.0]) * sc
        _add_ellipsoid(vol, (c, c, c), ax, 1.0)
        for _ in range(5):
            d = rng.normal(size=3)
            d /= np.linalg.norm(d)
            pos = c + d * ax * rng.uniform(0.0, 0.6)
            _add_gaussian(vol, pos, 2.0 * sc, rng.uniform(0.2, 0.8))
        return vol
    if config == 2:
        for _ in range(12):
            ax = rng.uniform(4.0, 14.0, size=3) * sc
            pos = c + rng.uniform(-14.0, 14.0, size=3) * sc
            _add_ellipsoid(vol, pos, ax, rng.uniform(0.3, 1.0))
        return vol
    if config == 3:
        # faceted particle: sphere r=50 cut by 8 random half-spaces; 6 alternating layers; 10 voids
        r0 = 50.0 * sc
        g = np.arange(nin) - c
        Z, Y, X = g[:, None, None], g[None, :, None], g[None, None, :]
        inside = (X * X + Y * Y + Z * Z) <= r0 * r0
        for _ in range(8):
            nrm = rng.normal(size=3)
            nrm /= np.linalg.norm(nrm)
            d = rng.uniform(0.55, 0.9) * r0
            inside &= (X * nrm[0] + Y * nrm[1] + Z * nrm[2]) <= d
        layer = np.floor((g + r0) / (2.0 * r0 / 6.0)).astype(np.int64) % 2      # along z
        dens = np.where(layer == 0, 0.6, 1.0)[:, None, None]
        vol = np.where(inside, dens, 0.0) * np.ones((nin, nin, nin))
        for _ in range(10):
            pos = c + rng.uniform(-0.5, 0.5, size=3) * r0
            rad = rng.uniform(2.0, 6.0) * sc
            _add_ellipsoid(vol, pos, (rad, rad, rad), 0.0, mode="set")
        return np.ascontiguousarray(vol)
    if config == 4:
        # spherical shell (outer r 110, wall 6, density 1), interior 0.15, 40 Gaussian inclusions;
        # complex object O = rho * exp(i * 0.1 * rho)   ("phase term 0.1 x density")
        ro, wall = 110.0 * sc, 6.0 * sc
        g = np.arange(nin) - c
        r2 = g[:, None, None] ** 2 + g[None, :, None] ** 2 + g[None, None, :] ** 2
        vol = np.where(r2 <= ro * ro, np.where(r2 >= (ro - wall) ** 2, 1.0, 0.15), 0.0)
        del r2
        for _ in range(40):
            d = rng.normal(size=3)
            d /= np.linalg.norm(d)
            pos = c + d * rng.uniform(0.0, 0.85) * (ro - wall)
            _add_gaussian(vol, pos, rng.uniform(2.0, 8.0) * sc, rng.uniform(0.05, 0.3))
        return vol * np.exp(1j * 0.1 * vol)
    if config == 5:
        for _ in range(60):
            ax = rng.uniform(10.0, 60.0, size=3) * sc
            pos = c + rng.uniform(-0.25, 0.25, size=3) * nin
            _add_ellipsoid(vol, pos, ax, rng.uniform(0.2, 1.0))
        return vol
    raise ValueError(f"unknown config {config}")


# ----------------------------------------------------------------------------------------------
# problem assembly
# ----------------------------------------------------------------------------------------------
def _dilate(b: np.ndarray, r: int) -> np.ndarray:
    """Binary dilation of the last two axes by a (2r+1)x(2r+1) square, zero boundary."""
    out = b.copy()
    for axis in (-2, -1):
        acc = out.copy()
        for d in range(1, r + 1):
            for sgn in (1, -1):
                sh = np.roll(out, sgn * d, axis=axis)
                idx = [slice(None)] * out.ndim
                idx[axis] = slice(0, d) if sgn == 1 else slice(-d, None)
                sh[tuple(idx)] = False
                acc |= sh
        out = acc
    return out


def angles_for(config: int, Np: int) -> np.ndarray:
    return np.deg2rad(CONFIGS[config]["range_deg"]) * np.arange(Np, dtype=np.float64) / Np


def random_phase_estimate(intensity_c: np.ndarray, mask: np.ndarray, rng) -> np.ndarray:
    """Random-phase start ("random initial guess"):
    g0_n = F^-1[M_n sqrt(I_n) e^{i phi}], phi ~ U[0, 2 pi) iid per pixel.  `rng`: a numpy Generator
    or an integer seed (one restart of PAPER.md:64's N_r random restarts per seed)."""
    if not isinstance(rng, np.random.Generator):
        rng = np.random.default_rng(np.random.SeedSequence([SEED_BASE, 9, int(rng)]))
    Np, N = intensity_c.shape[0], intensity_c.shape[-1]
    est = np.empty((Np, N, N), dtype=np.complex64)
    for n in range(Np):
        A_native = np.fft.ifftshift(np.sqrt(np.maximum(intensity_c[n].astype(np.float64), 0.0)) * mask[n])
        phi = rng.uniform(0.0, 2.0 * math.pi, size=(N, N))
        est[n] = np.fft.ifft2(A_native * np.exp(1j * phi)).astype(np.complex64)
    return est


def make_problem(config: int, Np: Optional[int] = None, N: Optional[int] = None,
                 seed_offset: int = 0, keep_object: bool = False,
                 noise: bool = True) -> Problem:
    """Build the inputs of BASELINE.json config `config` (optionally with fewer angles Np, or at
    another grid size N: the object is scaled with N).  Deterministic in (config, Np, N, seed_offset)."""
    cfg = CONFIGS[config]
    N = int(N or cfg["N"])
    Np = int(Np or cfg["Np"])
    nin = N // 2
    ss = np.random.SeedSequence(SEED_BASE + config + 1000 * seed_offset)
    rng_obj, rng_noise, rng_phase = (np.random.default_rng(s) for s in ss.spawn(3))

    obj = make_object(config, nin, rng_obj)
    angles = angles_for(config, Np)
    P = project(obj, N, angles)                                   # [Np,N,N] complex128

    # intensities, native order -> detector-centred
    I = np.abs(np.fft.fft2(P)) ** 2
    if cfg["photons"] is not None and noise:
        for n in range(Np):
            scale = cfg["photons"] / I[n].sum()
            I[n] = rng_noise.poisson(I[n] * scale).astype(np.float64)   # photon counts, not rescaled
            P[n] *= math.sqrt(scale)                                    # truth on the same scale
    I_c = np.fft.fftshift(I, axes=(-2, -1)).astype(np.float32)

    mask = np.ones((Np, N, N), dtype=np.uint8)
    b = cfg["beamstop"]
    if b:
        lo = N // 2 - b // 2
        mask[:, lo:lo + b, lo:lo + b] = 0

    if config == 1:
        # support = projected ellipsoid indicator dilated by 2 px
        ell = np.zeros((nin, nin, nin))
        _add_ellipsoid(ell, (nin / 2.0,) * 3, np.array([10.0, 8.0, 6.0]) * (nin / 32.0), 1.0)
        sup = np.abs(project(ell, N, angles)) > 1e-9
    else:
        a = np.abs(P)
        sup = a > 0.2 * a.max(axis=(-2, -1), keepdims=True)
    support = _dilate(sup, cfg["support_r"]).astype(np.uint8)

    est = random_phase_estimate(I_c, mask, rng_phase)

    return Problem(config=config, N=N, Np=Np, angles=angles,
                   intensity=np.ascontiguousarray(I_c), mask=np.ascontiguousarray(mask),
                   support=np.ascontiguousarray(support), estimate=np.ascontiguousarray(est),
                   projections=P, obj=obj if keep_object else None,
                   beta=0.9, iters=cfg["iters"])


def random_stack(N: int, Np: int, seed: int, support_frac: float = 0.4, beamstop: int = 0):
    """A structureless seeded problem (random complex estimate, random positive intensities, a
    centred square support, optional beamstop) for edge-case and API tests at arbitrary (N, Np)."""
    rng = np.random.default_rng(SEED_BASE + 77 + seed)
    est = (rng.normal(size=(Np, N, N)) + 1j * rng.normal(size=(Np, N, N))).astype(np.complex64)
    I = (rng.gamma(2.0, 50.0, size=(Np, N, N))).astype(np.float32)
    mask = np.ones((Np, N, N), dtype=np.uint8)
    if beamstop:
        lo = N // 2 - beamstop // 2
        mask[:, lo:lo + beamstop, lo:lo + beamstop] = 0
    support = np.zeros((Np, N, N), dtype=np.uint8)
    h = max(1, int(N * support_frac / 2))
    support[:, N // 2 - h:N // 2 + h, N // 2 - h:N // 2 + h] = 1
    # make the support differ between projections so that index mix-ups show
    for n in range(Np):
        support[n, (N // 2 + h + n) % N, N // 2] = 1
    angles = np.pi * np.arange(Np) / Np
    return Problem(config=0, N=N, Np=Np, angles=angles, intensity=I, mask=mask, support=support,
                   estimate=est, projections=est.astype(np.complex128), obj=None, beta=0.9, iters=0)
