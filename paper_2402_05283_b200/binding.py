"""Thin ctypes binding of libcpra.so (include/cpra.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device
memory and streams only.  Nothing here falls back to the CPU: if the library cannot be loaded, or
a call fails, a `CpraError` is raised."""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

CPRA_OK = 0
ERR_INVALID_ARG, ERR_UNSUPPORTED_SIZE, ERR_NOT_READY, ERR_WORKSPACE, ERR_CUDA, ERR_INVALID_VALUE = -1, -2, -3, -4, -5, -6
ITERATE, SUPPORTED = 0, 1
FLAG_DEFAULT, FLAG_FORCE_MULTIPASS, FLAG_NO_CHUNKING, FLAG_NO_WALK = 0, 1, 2, 4
MAX_K = 8
FSC_STATIC_MAX_N = 1024
PROFILE_CLASSES = 5
PROFILE_NAMES = ("row_fwd", "col", "row_inv", "image", "walk")

_vp, _ci, _cf, _cl, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_long, ctypes.c_size_t

# name -> (restype, argtypes): every symbol include/cpra.h declares
SIGNATURES = {
    "cpra_plan": (_ci, [ctypes.POINTER(_vp), _ci, _ci, ctypes.c_uint, _vp]),
    "cpra_workspace_bytes": (_ci, [_vp, ctypes.POINTER(_sz)]),
    "cpra_bind_workspace": (_ci, [_vp, _vp, _sz]),
    "cpra_set_data": (_ci, [_vp, _vp, _vp, _vp]),
    "cpra_set_support": (_ci, [_vp, _vp]),
    "cpra_set_carousel": (_ci, [_vp, _ci, _vp, _ci]),
    "cpra_set_estimate": (_ci, [_vp, _vp]),
    "cpra_set_estimate_spectrum": (_ci, [_vp, _vp]),
    "cpra_get_iteration": (_ci, [_vp, ctypes.POINTER(_cl)]),
    "cpra_set_iteration": (_ci, [_vp, _cl]),
    "cpra_iterate": (_ci, [_vp, _ci, _cf]),
    "cpra_get_error": (_ci, [_vp, _vp, _vp]),
    "cpra_get_projections": (_ci, [_vp, _ci, _vp]),
    "cpra_assemble_3d": (_ci, [_vp, _vp, _vp]),
    "cpra_fft2": (_ci, [_vp, _vp, _vp, _ci]),
    "cpra_host_staging_bytes": (_ci, [_vp, ctypes.POINTER(_sz)]),
    "cpra_reconstruct_host": (_ci, [_vp, _vp, _sz, _vp, _vp, _vp, _vp, _vp, _ci, _cf, _vp, _vp, _vp]),
    "cpra_set_chunk": (_ci, [_vp, _ci]),
    "cpra_set_update": (_ci, [_vp, _ci]),
    "cpra_profile": (_ci, [_vp, _ci]),
    "cpra_profile_read": (_ci, [_vp, _vp, _vp]),
    "cpra_launch_count": (_ci, [_vp, ctypes.POINTER(_cl)]),
    "cpra_set_seam": (_ci, [_vp, _ci]),
    "cpra_set_positivity": (_ci, [_vp, _ci]),
    "cpra_set_cluster": (_ci, [_vp, _ci]),
    "cpra_set_walk_ctas": (_ci, [_vp, _ci]),
    "cpra_shrinkwrap": (_ci, [_vp, _cf, _cf, _vp]),
    "cpra_get_support": (_ci, [_vp, _vp]),
    "cpra_prereconstruct": (_ci, [_vp, _ci, _ci, _cf]),
    "cpra_merge_bytes": (_ci, [_vp, _ci, ctypes.POINTER(_sz)]),
    "cpra_merge_bind": (_ci, [_vp, _vp, _sz, _ci]),
    "cpra_merge_offer": (_ci, [_vp, _vp, ctypes.c_double]),
    "cpra_merge_errors": (_ci, [_vp, _vp, _vp]),
    "cpra_merge_get": (_ci, [_vp, _ci, _vp]),
    "cpra_merge_finish": (_ci, [_vp, _ci, _vp, _vp, _vp]),
    "cpra_align_episode": (_ci, [_vp, _vp, _ci, _vp]),
    "cpra_fft3": (_ci, [_vp, _vp, _vp, _ci]),
    "cpra_refine_3d": (_ci, [_vp, _vp, _vp, _vp, _ci, _vp, _vp]),
    "cpra_refine_3d_sw": (_ci, [_vp, _vp, _vp, _vp, _ci, _ci, _cf, _cf, _vp, _vp, _vp]),
    "cpra_backproject_support": (_ci, [_vp, _vp]),
    "cpra_fsc": (_ci, [_vp, _vp, _vp, _vp]),
    "cpra_prtf": (_ci, [_vp, _vp, _vp]),
    "cpra_fsc_static": (_ci, [_ci, _vp, _vp, _vp, _vp]),
    "cpra_destroy": (_ci, [_vp]),
    "cpra_status_string": (ctypes.c_char_p, [_ci]),
}

_LIB = None


class CpraError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = int(code)
        name = lib().cpra_status_string(self.code).decode() if _LIB is not None else str(code)
        super().__init__(f"{what} failed: {name} ({self.code})")


def lib_path() -> str:
    return _build.LIB


def lib() -> ctypes.CDLL:
    """Load libcpra.so (building it first if the sources are newer).  Raises if unavailable."""
    global _LIB
    if _LIB is None:
        path = _build.build()
        if not os.path.exists(path):
            raise OSError(f"{path} is missing and could not be built; there is no fallback path")
        L = ctypes.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)      # AttributeError if the symbol is not exported
            fn.restype, fn.argtypes = res, args
        _LIB = L
    return _LIB


def _chk(code: int, what: str) -> None:
    if code != CPRA_OK:
        raise CpraError(code, what)


def _dptr(t, dtype, nelem=None):
    """Device pointer of a contiguous CUDA torch tensor (checked)."""
    import torch
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda or not t.is_contiguous():
        raise TypeError("expected a contiguous CUDA torch tensor")
    if t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    if nelem is not None and t.numel() != nelem:
        raise ValueError(f"expected {nelem} elements, got {t.numel()}")
    return t.data_ptr()


def fsc_static(F1, F2, out=None):
    """cpra_fsc_static: the Fourier shell correlation of two complex64 [N, N, N] CUDA tensors with no plan, no
    workspace and no device allocation inside the call (its scratch is a fixed __device__ array in libcpra.so;
    N even, N <= FSC_STATIC_MAX_N; calls that overlap on the GPU race on that array).  `out`: float32 [N/2 + 1]
    CUDA tensor to write into -- pass one where nothing may be allocated; otherwise torch allocates it here."""
    import torch
    N = int(F1.shape[-1])
    if out is None:
        out = torch.empty(N // 2 + 1, dtype=torch.float32, device=F1.device)
    with torch.cuda.device(F1.device):      # the array's address is looked up for the CURRENT device
        rc = lib().cpra_fsc_static(N, _dptr(F1, torch.complex64, N ** 3), _dptr(F2, torch.complex64, N ** 3),
                                   _dptr(out, torch.float32, N // 2 + 1), torch.cuda.current_stream(F1.device).cuda_stream)
    if rc == ERR_UNSUPPORTED_SIZE:
        raise CpraError(rc, f"cpra_fsc_static (N = {N} exceeds the static scratch, N <= {FSC_STATIC_MAX_N})")
    _chk(rc, "cpra_fsc_static")
    return out


class Plan:
    """One CPRA problem: N x N pixels, Np projections, on the current CUDA device and stream.

    Mirrors the C ABI one to one: set_data / set_support / set_carousel / set_estimate / iterate /
    get_error / get_projections / assemble_3d (+ fft2, reconstruct_host).  Tensors are torch CUDA
    tensors owned by the caller; complex arrays are torch.complex64."""

    def __init__(self, N: int, Np: int, flags: int = FLAG_DEFAULT, stream=None, device=None):
        import torch
        self._l = lib()
        self.N, self.Np = int(N), int(Np)
        self._h = _vp()
        self._ws = None
        if not torch.cuda.is_available():
            # validate the sizes first so that argument errors are reported as such
            _chk(self._l.cpra_plan(ctypes.byref(self._h), self.N, self.Np, flags, None), "cpra_plan")
            self.close()
            raise CpraError(ERR_CUDA, "cpra_plan (no CUDA device; there is no CPU fallback)")
        self.device = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        _chk(self._l.cpra_plan(ctypes.byref(self._h), self.N, self.Np, flags, _vp(self.stream.cuda_stream)), "cpra_plan")
        nbytes = _sz()
        _chk(self._l.cpra_workspace_bytes(self._h, ctypes.byref(nbytes)), "cpra_workspace_bytes")
        self.workspace_bytes = int(nbytes.value)
        self._ws = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=self.device)
        _chk(self._l.cpra_bind_workspace(self._h, _vp(self._ws.data_ptr()), self.workspace_bytes), "cpra_bind_workspace")
        self._stage = None
        self._px = self.Np * self.N * self.N

    # -- lifetime ---------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._l.cpra_destroy(self._h)
            self._h = _vp()
        self._ws = None
        self._stage = None
        self._bank = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C ABI, one method per call ------------------------------------------------------------
    def set_data(self, intensity, mask=None, angles=None):
        import torch
        a = None
        if angles is not None:
            a = np.ascontiguousarray(np.asarray(angles, dtype=np.float64))
            if a.shape != (self.Np,):
                raise ValueError("angles must have Np entries")
        _chk(self._l.cpra_set_data(self._h, _dptr(intensity, torch.float32, self._px),
                                   _dptr(mask, torch.uint8, self._px),
                                   None if a is None else a.ctypes.data), "cpra_set_data")

    def set_support(self, support):
        import torch
        _chk(self._l.cpra_set_support(self._h, _dptr(support, torch.uint8, self._px)), "cpra_set_support")

    def set_carousel(self, alpha, n_ei=1):
        al = np.ascontiguousarray(np.asarray(alpha, dtype=np.float64))
        _chk(self._l.cpra_set_carousel(self._h, len(al) - 1, al.ctypes.data, int(n_ei)), "cpra_set_carousel")

    def set_estimate(self, g0):
        import torch
        _chk(self._l.cpra_set_estimate(self._h, _dptr(g0, torch.complex64, self._px)), "cpra_set_estimate")

    def set_estimate_spectrum(self, G0):
        """cpra_set_estimate_spectrum: the starting estimate as F^-1 of a natural-order spectrum complex64 [Np, N, N]."""
        import torch
        _chk(self._l.cpra_set_estimate_spectrum(self._h, _dptr(G0, torch.complex64, self._px)), "cpra_set_estimate_spectrum")

    @property
    def iteration(self) -> int:
        t = _cl()
        _chk(self._l.cpra_get_iteration(self._h, ctypes.byref(t)), "cpra_get_iteration")
        return int(t.value)

    @iteration.setter
    def iteration(self, t: int):
        _chk(self._l.cpra_set_iteration(self._h, int(t)), "cpra_set_iteration")

    def set_chunk(self, images: int):
        _chk(self._l.cpra_set_chunk(self._h, int(images)), "cpra_set_chunk")

    def set_walk_ctas(self, per_sm: int):
        _chk(self._l.cpra_set_walk_ctas(self._h, int(per_sm)), "cpra_set_walk_ctas")
        return self

    def set_cluster(self, ctas_per_image: int):
        _chk(self._l.cpra_set_cluster(self._h, int(ctas_per_image)), "cpra_set_cluster")
        return self

    def iterate(self, k: int, beta: float = 0.9):
        _chk(self._l.cpra_iterate(self._h, int(k), float(beta)), "cpra_iterate")

    def get_error(self):
        """(E[Np], E_global[1]) as CUDA float32 tensors (no host sync)."""
        import torch
        E = torch.empty(self.Np, dtype=torch.float32, device=self.device)
        Eg = torch.empty(1, dtype=torch.float32, device=self.device)
        _chk(self._l.cpra_get_error(self._h, E.data_ptr(), Eg.data_ptr()), "cpra_get_error")
        return E, Eg

    def get_projections(self, which: int = ITERATE, out=None):
        import torch
        if out is None:
            out = torch.empty((self.Np, self.N, self.N), dtype=torch.complex64, device=self.device)
        _chk(self._l.cpra_get_projections(self._h, int(which), _dptr(out, torch.complex64, self._px)), "cpra_get_projections")
        return out

    def assemble_3d(self, want_weight: bool = True):
        import torch
        vol = torch.empty((self.N,) * 3, dtype=torch.complex64, device=self.device)
        w = torch.empty((self.N,) * 3, dtype=torch.float32, device=self.device) if want_weight else None
        _chk(self._l.cpra_assemble_3d(self._h, vol.data_ptr(), None if w is None else w.data_ptr()), "cpra_assemble_3d")
        return (vol, w) if want_weight else vol

    def fft2(self, stack, sign: int = -1):
        import torch
        out = torch.empty_like(stack)
        _chk(self._l.cpra_fft2(self._h, _dptr(stack, torch.complex64, self._px), out.data_ptr(), int(sign)), "cpra_fft2")
        return out

    def set_update(self, rule: str):
        """Real-space update rule: "hio" (default), "raar" or "er"."""
        _chk(self._l.cpra_set_update(self._h, {"hio": 0, "raar": 1, "er": 2}[rule]), "cpra_set_update")
        return self

    # -- around the loop -------------------------------------------------------------
    def set_positivity(self, on: bool):
        _chk(self._l.cpra_set_positivity(self._h, int(bool(on))), "cpra_set_positivity")
        return self

    def set_seam(self, flip: bool):
        _chk(self._l.cpra_set_seam(self._h, int(bool(flip))), "cpra_set_seam")
        return self

    def shrinkwrap(self, sigma: float, threshold: float, want_blurred: bool = False):
        import torch
        b = torch.empty((self.Np, self.N, self.N), dtype=torch.float32, device=self.device) if want_blurred else None
        _chk(self._l.cpra_shrinkwrap(self._h, float(sigma), float(threshold), None if b is None else b.data_ptr()), "cpra_shrinkwrap")
        return b

    def get_support(self):
        import torch
        S = torch.empty((self.Np, self.N, self.N), dtype=torch.uint8, device=self.device)
        _chk(self._l.cpra_get_support(self._h, S.data_ptr()), "cpra_get_support")
        return S

    def prereconstruct(self, n: int, k: int, beta: float = 0.9):
        _chk(self._l.cpra_prereconstruct(self._h, int(n), int(k), float(beta)), "cpra_prereconstruct")

    def merge_begin(self, n_keep: int):
        """Allocate (torch) and bind the bank of the n_keep lowest-error episodes."""
        import torch
        nb = _sz()
        _chk(self._l.cpra_merge_bytes(self._h, int(n_keep), ctypes.byref(nb)), "cpra_merge_bytes")
        self._bank = torch.empty(int(nb.value), dtype=torch.uint8, device=self.device)
        self._n_keep = int(n_keep)
        _chk(self._l.cpra_merge_bind(self._h, _vp(self._bank.data_ptr()), int(nb.value), int(n_keep)), "cpra_merge_bind")

    def merge_offer(self, episode=None, E: float = 0.0):
        import torch
        _chk(self._l.cpra_merge_offer(self._h, _dptr(episode, torch.complex64, self._px), float(E)), "cpra_merge_offer")

    def merge_errors(self):
        """(errors double[n_keep] CUDA tensor in slot order, count int32[1] CUDA tensor)."""
        import torch
        E = torch.empty(self._n_keep, dtype=torch.float64, device=self.device)
        c = torch.empty(1, dtype=torch.int32, device=self.device)
        _chk(self._l.cpra_merge_errors(self._h, E.data_ptr(), c.data_ptr()), "cpra_merge_errors")
        return E, c

    def merge_get(self, slot: int):
        import torch
        out = torch.empty((self.Np, self.N, self.N), dtype=torch.complex64, device=self.device)
        _chk(self._l.cpra_merge_get(self._h, int(slot), out.data_ptr()), "cpra_merge_get")
        return out

    def merge_finish(self, n_ref: int = 0):
        """(final episode complex64 [Np,N,N], shifts int32 [n_keep,Np,2], twins int32 [n_keep]) on the device."""
        import torch
        out = torch.empty((self.Np, self.N, self.N), dtype=torch.complex64, device=self.device)
        sh = torch.zeros((self._n_keep, self.Np, 2), dtype=torch.int32, device=self.device)
        tw = torch.zeros(self._n_keep, dtype=torch.int32, device=self.device)
        _chk(self._l.cpra_merge_finish(self._h, int(n_ref), out.data_ptr(), sh.data_ptr(), tw.data_ptr()), "cpra_merge_finish")
        return out, sh, tw

    def align_episode(self, episode, n_ref: int = 0):
        """Phase gauge and twin chain of one episode, in place; returns the flips (int32 [Np], device)."""
        import torch
        fl = torch.zeros(self.Np, dtype=torch.int32, device=self.device)
        _chk(self._l.cpra_align_episode(self._h, _dptr(episode, torch.complex64, self._px), int(n_ref), fl.data_ptr()), "cpra_align_episode")
        return fl

    def fft3(self, vol, sign: int = -1):
        import torch
        out = torch.empty_like(vol)
        _chk(self._l.cpra_fft3(self._h, _dptr(vol, torch.complex64, self.N ** 3), out.data_ptr(), int(sign)), "cpra_fft3")
        return out

    def refine_3d(self, E, W, S3, k: int):
        """Step D's iterations: (object complex64 [N,N,N], err float32 [k]) on the device."""
        import torch
        n3 = self.N ** 3
        obj = torch.empty((self.N,) * 3, dtype=torch.complex64, device=self.device)
        err = torch.empty(int(k), dtype=torch.float32, device=self.device)
        _chk(self._l.cpra_refine_3d(self._h, _dptr(E, torch.complex64, n3), _dptr(W, torch.float32, n3), _dptr(S3, torch.uint8, n3),
                                    int(k), obj.data_ptr(), err.data_ptr()), "cpra_refine_3d")
        return obj, err

    def refine_3d_sw(self, E, W, S3, k: int, every: int, sigma: float, threshold: float, want_blurred: bool = False):
        """cpra_refine_3d_sw: returns (object complex64 [N, N, N], err float32 [k], support u8 [N, N, N] after the last
        update[, blurred float32 [N, N, N]]).  S3 is copied: the caller's tensor is not modified."""
        import torch
        n3 = self.N ** 3
        obj = torch.empty((self.N, self.N, self.N), dtype=torch.complex64, device=self.device)
        err = torch.empty(int(k), dtype=torch.float32, device=self.device)
        s3 = S3.clone().contiguous()
        bl = torch.zeros((self.N, self.N, self.N), dtype=torch.float32, device=self.device) if want_blurred else None
        _chk(self._l.cpra_refine_3d_sw(self._h, _dptr(E, torch.complex64, n3), _dptr(W, torch.float32, n3), _dptr(s3, torch.uint8, n3),
                                       int(k), int(every), float(sigma), float(threshold), obj.data_ptr(), err.data_ptr(),
                                       None if bl is None else bl.data_ptr()), "cpra_refine_3d_sw")
        return (obj, err, s3, bl) if want_blurred else (obj, err, s3)

    def backproject_support(self):
        """cpra_backproject_support: the visual hull of the current 2D supports, u8 [N, N, N] (z, y, x)."""
        import torch
        S3 = torch.empty((self.N, self.N, self.N), dtype=torch.uint8, device=self.device)
        _chk(self._l.cpra_backproject_support(self._h, S3.data_ptr()), "cpra_backproject_support")
        return S3

    def fsc(self, F1, F2):
        import torch
        out = torch.empty(self.N // 2 + 1, dtype=torch.float32, device=self.device)
        _chk(self._l.cpra_fsc(self._h, _dptr(F1, torch.complex64, self.N ** 3), _dptr(F2, torch.complex64, self.N ** 3), out.data_ptr()), "cpra_fsc")
        return out

    def prtf(self, avg):
        import torch
        out = torch.empty(self.N // 2 + 1, dtype=torch.float32, device=self.device)
        _chk(self._l.cpra_prtf(self._h, _dptr(avg, torch.complex64, self._px), out.data_ptr()), "cpra_prtf")
        return out

    def profile(self, enable: bool):
        _chk(self._l.cpra_profile(self._h, int(bool(enable))), "cpra_profile")

    def profile_read(self):
        """{class name: (milliseconds, launches)} accumulated since the last read (synchronises)."""
        ms = (ctypes.c_double * PROFILE_CLASSES)()
        cnt = (_cl * PROFILE_CLASSES)()
        _chk(self._l.cpra_profile_read(self._h, ms, cnt), "cpra_profile_read")
        return {n: (float(ms[i]), int(cnt[i])) for i, n in enumerate(PROFILE_NAMES)}

    @property
    def launch_count(self) -> int:
        c = _cl()
        _chk(self._l.cpra_launch_count(self._h, ctypes.byref(c)), "cpra_launch_count")
        return int(c.value)

    # -- host-buffer end-to-end call ---------------------------------------------------------------
    def host_staging_bytes(self) -> int:
        b = _sz()
        _chk(self._l.cpra_host_staging_bytes(self._h, ctypes.byref(b)), "cpra_host_staging_bytes")
        return int(b.value)

    def reconstruct_host(self, intensity, mask, angles, support, g0, k, beta=0.9, out=None, want_error=True):
        """Host (CPU, ideally pinned) torch tensors or numpy arrays in, host arrays out.
        Returns (projections complex64 [Np,N,N] host, E[Np] host, E_global float)."""
        import torch

        def hptr(x, dtype, n):
            if x is None:
                return None, None
            t = torch.as_tensor(x)
            if t.is_cuda or not t.is_contiguous() or t.dtype != dtype or t.numel() != n:
                raise TypeError("expected a contiguous host tensor of the right dtype and size")
            return t, t.data_ptr()

        if self._stage is None:
            self._stage = torch.empty(self.host_staging_bytes(), dtype=torch.uint8, device=self.device)
        keep = []
        tI, pI = hptr(intensity, torch.float32, self._px); keep.append(tI)
        tM, pM = hptr(mask, torch.uint8, self._px); keep.append(tM)
        tS, pS = hptr(support, torch.uint8, self._px); keep.append(tS)
        tG, pG = hptr(g0, torch.complex64, self._px); keep.append(tG)
        a = None if angles is None else np.ascontiguousarray(np.asarray(angles, dtype=np.float64))
        if out is None:
            out = torch.empty((self.Np, self.N, self.N), dtype=torch.complex64).pin_memory()
        E = torch.empty(self.Np + 1, dtype=torch.float32).pin_memory() if want_error else None
        _chk(self._l.cpra_reconstruct_host(
            self._h, self._stage.data_ptr(), self._stage.numel(), pI, pM,
            None if a is None else a.ctypes.data, pS, pG, int(k), float(beta), out.data_ptr(),
            None if E is None else E.data_ptr(),
            None if E is None else E.data_ptr() + 4 * self.Np), "cpra_reconstruct_host")
        if E is None:
            return out, None, None
        return out, E[:self.Np], float(E[self.Np])

    # -- convenience --------------------------------------------------------------------------------
    def load(self, problem, alpha=(0.6, 0.2), n_ei=1):
        """Upload a cpra_inputs.Problem (numpy) and set everything."""
        import torch
        dev = self.device
        self.set_data(torch.from_numpy(problem.intensity).to(dev), torch.from_numpy(problem.mask).to(dev), problem.angles)
        self.set_support(torch.from_numpy(problem.support).to(dev))
        self.set_carousel(alpha, n_ei)
        self.set_estimate(torch.from_numpy(problem.estimate).to(dev))
        return self
