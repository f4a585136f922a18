"""ctypes binding of oracle/cpra_oracle.c -- TEST INFRASTRUCTURE (see the C file's header).

`Oracle(N, Np)` mirrors the product's C ABI (cpra_plan / set_data / set_support / set_carousel /
set_estimate / iterate / get_error / get_projections / assemble_3d) with host numpy arrays, FP64
internally.  `Oracle(..., precision="f32")` loads the float build of the same source, used only to
report the drift of an fp32 state next to the GPU's; it is never the reference.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBS = {}


def build_oracle(force: bool = False) -> dict:
    """gcc-compile cpra_oracle.c into liboracle.so (double) and liboracle_f32.so (float)."""
    src = os.path.join(_HERE, "cpra_oracle.c")
    outs = {}
    for prec, define in (("f64", "double"), ("f32", "float")):
        out = os.path.join(_HERE, "liboracle.so" if prec == "f64" else "liboracle_f32.so")
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c99",
                                   f"-DORACLE_REAL={define}", "-o", out, src, "-lm"])
        outs[prec] = out
    return outs


def _lib(precision: str = "f64"):
    if precision not in _LIBS:
        lib = ctypes.CDLL(build_oracle()[precision])
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        lib.oracle_plan.argtypes = [ctypes.POINTER(vp), ci, ci]
        lib.oracle_destroy.argtypes = [vp]
        lib.oracle_set_data.argtypes = [vp, vp, vp, vp]
        lib.oracle_set_support.argtypes = [vp, vp]
        lib.oracle_set_carousel.argtypes = [vp, ci, vp, ci]
        lib.oracle_set_update.argtypes = [vp, ci]
        lib.oracle_set_estimate.argtypes = [vp, vp]
        lib.oracle_set_iteration.argtypes = [vp, ctypes.c_long]
        lib.oracle_get_iteration.argtypes = [vp]
        lib.oracle_get_iteration.restype = ctypes.c_long
        lib.oracle_iterate.argtypes = [vp, ci, cd]
        lib.oracle_get_error.argtypes = [vp, vp, vp]
        lib.oracle_get_projections.argtypes = [vp, ci, vp]
        lib.oracle_assemble_3d.argtypes = [vp, vp, vp]
        lib.oracle_fft2.argtypes = [vp, vp, ci, ci, ci]
        lib.oracle_dft2_naive.argtypes = [vp, vp, ci, ci]
        lib.oracle_mix.argtypes = [vp, vp, ci, ci, ci, vp]
        lib.oracle_modulus.argtypes = [vp, vp, vp, ci, vp]
        lib.oracle_hio.argtypes = [vp, vp, vp, ci, cd]
        lib.oracle_real_name.restype = ctypes.c_char_p
        lib.oracle_set_seam.argtypes = [vp, ci]
        lib.oracle_set_positivity.argtypes = [vp, ci]
        lib.oracle_mix_seam.argtypes = [vp, vp, ci, ci, ci, vp, ci]
        lib.oracle_blur.argtypes = [vp, vp, ci, cd]
        lib.oracle_shrinkwrap.argtypes = [vp, cd, cd, vp]
        lib.oracle_get_support.argtypes = [vp, vp]
        lib.oracle_prereconstruct.argtypes = [vp, ci, ci, cd]
        lib.oracle_center_of_mass.argtypes = [vp, ci, vp, vp]
        lib.oracle_merge_begin.argtypes = [vp, ci]
        lib.oracle_merge_offer.argtypes = [vp, vp, cd]
        lib.oracle_merge_errors.argtypes = [vp, vp, vp]
        lib.oracle_merge_finish.argtypes = [vp, ci, vp, vp, vp]
        lib.oracle_fft3.argtypes = [vp, vp, ci, ci]
        lib.oracle_align_episode.argtypes = [vp, ci, ci, ci, vp]
        lib.oracle_refine_3d.argtypes = [vp, vp, vp, ci, ci, vp, vp]
        lib.oracle_refine_3d_sw.argtypes = [vp, vp, vp, ci, ci, ci, cd, cd, vp, vp, vp]
        lib.oracle_backproject_support.argtypes = [vp, vp]
        lib.oracle_fsc.argtypes = [vp, vp, ci, vp]
        lib.oracle_prtf.argtypes = [vp, vp, vp]
        _LIBS[precision] = lib
    return _LIBS[precision]


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"{what} returned {code}")
        self.code = code


def _chk(code, what):
    if code != 0:
        raise OracleError(code, what)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def fft2(stack, sign=-1, precision="f64"):
    """Radix-2 2D FFT of an image or a stack [count,N,N] (sign=-1 forward, +1 inverse/N^2)."""
    a = _c128(stack)
    N = a.shape[-1]
    out = np.empty_like(a)
    _chk(_lib(precision).oracle_fft2(a.ctypes.data, out.ctypes.data, N, a.size // (N * N), sign), "oracle_fft2")
    return out


def dft2_naive(img, sign=-1):
    a = _c128(img)
    out = np.empty_like(a)
    _chk(_lib().oracle_dft2_naive(a.ctypes.data, out.ctypes.data, a.shape[-1], sign), "oracle_dft2_naive")
    return out


def mix(stack, alpha, precision="f64"):
    a = _c128(stack)
    Np, N = a.shape[0], a.shape[-1]
    al = np.ascontiguousarray(alpha, dtype=np.float64)
    out = np.empty_like(a)
    _chk(_lib(precision).oracle_mix(a.ctypes.data, out.ctypes.data, N, Np, len(al) - 1, al.ctypes.data), "oracle_mix")
    return out


def modulus(G, A, M, precision="f64"):
    """Fourier-modulus constraint on one native-order image.  Returns (G', num)."""
    g = _c128(G).copy()
    a = np.ascontiguousarray(A, dtype=np.float64)
    m = np.ascontiguousarray(M, dtype=np.uint8)
    num = ctypes.c_double(0.0)
    _chk(_lib(precision).oracle_modulus(g.ctypes.data, a.ctypes.data, m.ctypes.data, g.shape[-1],
                                        ctypes.addressof(num)), "oracle_modulus")
    return g, num.value


def hio(ghat, gp, S, beta, precision="f64"):
    a = _c128(ghat).copy()
    b = _c128(gp)
    s = np.ascontiguousarray(S, dtype=np.uint8)
    _chk(_lib(precision).oracle_hio(a.ctypes.data, b.ctypes.data, s.ctypes.data, a.shape[-1], float(beta)), "oracle_hio")
    return a


def mix_seam(stack, alpha, flip, precision="f64"):
    """Eq. (4) with the seam flag of reading A5b (flip=1: neighbours across the ends of the stack mirrored in u)."""
    a = _c128(stack)
    Np, N = a.shape[0], a.shape[-1]
    al = np.ascontiguousarray(alpha, dtype=np.float64)
    out = np.empty_like(a)
    _chk(_lib(precision).oracle_mix_seam(a.ctypes.data, out.ctypes.data, N, Np, len(al) - 1, al.ctypes.data, int(flip)), "oracle_mix_seam")
    return out


def blur(img, sigma, precision="f64"):
    """Periodic Gaussian blur of one real N x N image (the blur of the shrink-wrap update)."""
    a = np.ascontiguousarray(img, dtype=np.float64)
    out = np.empty_like(a)
    _chk(_lib(precision).oracle_blur(a.ctypes.data, out.ctypes.data, a.shape[-1], float(sigma)), "oracle_blur")
    return out


def center_of_mass(img):
    """(cy, cx) of |img| about the centre pixel (N/2, N/2)."""
    a = _c128(img)
    cy, cx = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _chk(_lib().oracle_center_of_mass(a.ctypes.data, a.shape[-1], ctypes.addressof(cy), ctypes.addressof(cx)), "oracle_center_of_mass")
    return cy.value, cx.value


def fft3(vol, sign=-1, precision="f64"):
    """3D FFT of a cube [N,N,N] (z, y, x) as x, y and z lines of the radix-2 routine (sign=+1: inverse, /N^3)."""
    a = _c128(vol)
    out = np.empty_like(a)
    _chk(_lib(precision).oracle_fft3(a.ctypes.data, out.ctypes.data, a.shape[-1], sign), "oracle_fft3")
    return out


def refine_3d(E, W, S3, k):
    """Step D's iterations (reading A26): returns (object [N,N,N] complex128, err[k])."""
    e = _c128(E)
    w = np.ascontiguousarray(W, dtype=np.float64)
    s3 = np.ascontiguousarray(S3, dtype=np.uint8)
    obj = np.empty_like(e)
    err = np.empty(int(k), dtype=np.float64)
    _chk(_lib().oracle_refine_3d(e.ctypes.data, w.ctypes.data, s3.ctypes.data, e.shape[-1], int(k), obj.ctypes.data, err.ctypes.data),
         "oracle_refine_3d")
    return obj, err


def refine_3d_sw(E, W, S3, k, every, sigma, threshold, want_blurred=False):
    """Step D's iterations with the 3D support re-thresholded every `every` iterations (readings A26, A30): returns
    (object [N,N,N] complex128, err[k], final support u8 [N,N,N][, the blurred |O| of the last update])."""
    e = _c128(E)
    w = np.ascontiguousarray(W, dtype=np.float64)
    s3 = np.ascontiguousarray(S3, dtype=np.uint8).copy()
    obj = np.empty_like(e)
    err = np.empty(int(k), dtype=np.float64)
    bl = np.zeros(s3.shape, dtype=np.float64) if want_blurred else None
    _chk(_lib().oracle_refine_3d_sw(e.ctypes.data, w.ctypes.data, s3.ctypes.data, e.shape[-1], int(k), int(every), float(sigma),
                                    float(threshold), obj.ctypes.data, err.ctypes.data, None if bl is None else bl.ctypes.data),
         "oracle_refine_3d_sw")
    return (obj, err, s3, bl) if want_blurred else (obj, err, s3)


def align_episode(episode, n_ref=0):
    """Phase gauge and twin chain of one episode (reading A28): returns (aligned copy, flips int32[Np])."""
    e = _c128(episode).copy()
    Np, N = e.shape[0], e.shape[-1]
    fl = np.zeros(Np, dtype=np.int32)
    _chk(_lib().oracle_align_episode(e.ctypes.data, N, Np, int(n_ref), fl.ctypes.data), "oracle_align_episode")
    return e, fl


def fsc(F1, F2):
    """Fourier shell correlation of two 3D spectra: N/2 + 1 values."""
    a, b = _c128(F1), _c128(F2)
    out = np.empty(a.shape[-1] // 2 + 1, dtype=np.float64)
    _chk(_lib().oracle_fsc(a.ctypes.data, b.ctypes.data, a.shape[-1], out.ctypes.data), "oracle_fsc")
    return out


class Oracle:
    """The CPRA loop on the host in FP64 (or fp32 with precision='f32'; drift display only)."""

    def __init__(self, N: int, Np: int, precision: str = "f64"):
        self._l = _lib(precision)
        self.N, self.Np = int(N), int(Np)
        h = ctypes.c_void_p()
        _chk(self._l.oracle_plan(ctypes.byref(h), self.N, self.Np), "oracle_plan")
        self._h = h

    def __del__(self):
        if getattr(self, "_h", None):
            self._l.oracle_destroy(self._h)
            self._h = None

    def set_data(self, intensity, mask=None, angles=None):
        I = np.ascontiguousarray(intensity, dtype=np.float64)
        assert I.shape == (self.Np, self.N, self.N)
        m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
        a = None if angles is None else np.ascontiguousarray(angles, dtype=np.float64)
        _chk(self._l.oracle_set_data(self._h, I.ctypes.data, None if m is None else m.ctypes.data,
                                     None if a is None else a.ctypes.data), "oracle_set_data")

    def set_support(self, support):
        s = np.ascontiguousarray(support, dtype=np.uint8)
        assert s.shape == (self.Np, self.N, self.N)
        _chk(self._l.oracle_set_support(self._h, s.ctypes.data), "oracle_set_support")

    def set_carousel(self, alpha, n_ei=1):
        al = np.ascontiguousarray(alpha, dtype=np.float64)
        _chk(self._l.oracle_set_carousel(self._h, len(al) - 1, al.ctypes.data, int(n_ei)), "oracle_set_carousel")

    def set_estimate(self, g0):
        g = _c128(g0)
        assert g.shape == (self.Np, self.N, self.N)
        _chk(self._l.oracle_set_estimate(self._h, g.ctypes.data), "oracle_set_estimate")

    def set_iteration(self, t):
        _chk(self._l.oracle_set_iteration(self._h, int(t)), "oracle_set_iteration")

    @property
    def iteration(self):
        return int(self._l.oracle_get_iteration(self._h))

    def set_update(self, rule):
        """Real-space update of step 6: "hio" (default), "raar" or "er" (reading A22)."""
        _chk(self._l.oracle_set_update(self._h, {"hio": 0, "raar": 1, "er": 2}[rule]), "oracle_set_update")
        return self

    def iterate(self, k, beta=0.9):
        _chk(self._l.oracle_iterate(self._h, int(k), float(beta)), "oracle_iterate")

    def get_error(self):
        E = np.empty(self.Np, dtype=np.float64)
        Eg = ctypes.c_double(0.0)
        _chk(self._l.oracle_get_error(self._h, E.ctypes.data, ctypes.addressof(Eg)), "oracle_get_error")
        return E, Eg.value

    def get_projections(self, which=0):
        out = np.empty((self.Np, self.N, self.N), dtype=np.complex128)
        _chk(self._l.oracle_get_projections(self._h, int(which), out.ctypes.data), "oracle_get_projections")
        return out

    def assemble_3d(self, want_weight=True):
        vol = np.empty((self.N,) * 3, dtype=np.complex128)
        w = np.empty((self.N,) * 3, dtype=np.float64) if want_weight else None
        _chk(self._l.oracle_assemble_3d(self._h, vol.ctypes.data, None if w is None else w.ctypes.data),
             "oracle_assemble_3d")
        return (vol, w) if want_weight else vol

    # -- seam, shrink-wrap, Step A, Step C ------------------------------------------
    def set_positivity(self, on):
        _chk(self._l.oracle_set_positivity(self._h, int(bool(on))), "oracle_set_positivity")
        return self

    def set_seam(self, flip):
        _chk(self._l.oracle_set_seam(self._h, int(bool(flip))), "oracle_set_seam")
        return self

    def shrinkwrap(self, sigma, threshold, want_blurred=False):
        b = np.empty((self.Np, self.N, self.N), dtype=np.float64) if want_blurred else None
        _chk(self._l.oracle_shrinkwrap(self._h, float(sigma), float(threshold), None if b is None else b.ctypes.data),
             "oracle_shrinkwrap")
        return b

    def get_support(self):
        S = np.empty((self.Np, self.N, self.N), dtype=np.uint8)
        _chk(self._l.oracle_get_support(self._h, S.ctypes.data), "oracle_get_support")
        return S

    def backproject_support(self):
        """The 3D support from the 2D supports and the angles (reading A29): u8 [N, N, N] (z, y, x)."""
        S3 = np.empty((self.N, self.N, self.N), dtype=np.uint8)
        _chk(self._l.oracle_backproject_support(self._h, S3.ctypes.data), "oracle_backproject_support")
        return S3

    def prereconstruct(self, n, k, beta=0.9):
        _chk(self._l.oracle_prereconstruct(self._h, int(n), int(k), float(beta)), "oracle_prereconstruct")

    def merge_begin(self, NL):
        _chk(self._l.oracle_merge_begin(self._h, int(NL)), "oracle_merge_begin")

    def merge_offer(self, episode=None, E=0.0):
        e = None if episode is None else _c128(episode)
        _chk(self._l.oracle_merge_offer(self._h, None if e is None else e.ctypes.data, float(E)), "oracle_merge_offer")

    def merge_errors(self):
        n = ctypes.c_int(0)
        _chk(self._l.oracle_merge_errors(self._h, None, ctypes.addressof(n)), "oracle_merge_errors")
        E = np.empty(n.value, dtype=np.float64)
        _chk(self._l.oracle_merge_errors(self._h, E.ctypes.data, ctypes.addressof(n)), "oracle_merge_errors")
        return E

    def merge_finish(self, n_ref=0):
        """Returns (final episode [Np,N,N] complex128, shifts [kept,Np,2] int32, twins [kept] int32)."""
        kept = len(self.merge_errors())
        out = np.empty((self.Np, self.N, self.N), dtype=np.complex128)
        sh = np.zeros((kept, self.Np, 2), dtype=np.int32)
        tw = np.zeros(kept, dtype=np.int32)
        _chk(self._l.oracle_merge_finish(self._h, int(n_ref), out.ctypes.data, sh.ctypes.data, tw.ctypes.data), "oracle_merge_finish")
        return out, sh, tw

    def prtf(self, avg):
        a = _c128(avg)
        out = np.empty(self.N // 2 + 1, dtype=np.float64)
        _chk(self._l.oracle_prtf(self._h, a.ctypes.data, out.ctypes.data), "oracle_prtf")
        return out

    def load(self, problem, alpha=(0.6, 0.2), n_ei=1):
        """Convenience: feed a cpra_inputs.Problem."""
        self.set_data(problem.intensity, problem.mask, problem.angles)
        self.set_support(problem.support)
        self.set_carousel(alpha, n_ei)
        self.set_estimate(problem.estimate)
        return self
