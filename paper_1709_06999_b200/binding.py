"""ctypes binding of include/galario_b200.h (same names, argument marshalling only)."""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Optional

import numpy as np
import torch

import os

_HERE = Path(__file__).resolve().parent
# GALARIO_B200_LIB points at another build of the same library (e.g. one compiled with different -D tuning flags).
_LIB_PATH = Path(os.environ.get("GALARIO_B200_LIB", _HERE / "libgalario_b200.so"))
_lib: Optional[ctypes.CDLL] = None

_vp, _i, _d, _i64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_int64


class GalarioError(RuntimeError):
    pass


def library_path() -> Path:
    return _LIB_PATH


def load_library() -> ctypes.CDLL:
    """Load the C-ABI library.  Fails loudly when it has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise GalarioError(f"{_LIB_PATH} is missing: run `python -m paper_1709_06999_b200.build` "
                               "(or __graft_entry__.build()).  There is no CPU fallback.")
        lib = ctypes.CDLL(str(_LIB_PATH))
        lib.gal_strerror.restype = ctypes.c_char_p
        lib.gal_plan_workspace_bytes.restype = ctypes.c_size_t
        lib.gal_last_oob_count.restype = _i64
        lib.gal_plan_launch_count.restype = _i64
        lib.gal_plan_create.argtypes = [ctypes.POINTER(_vp), _i, _i, _i, _i]
        for name in ("gal_plan_destroy", "gal_plan_workspace_bytes", "gal_last_oob_count", "gal_last_cuda_error",
                     "gal_plan_launch_count"):
            getattr(lib, name).argtypes = [_vp]
        lib.gal_plan_timing_enable.argtypes = [_vp, _i]
        lib.gal_plan_timing_read.argtypes = [_vp, _vp, _vp]
        lib.gal_get_image_size.argtypes = [_vp, _vp, _i64, _d, _d, _d, _vp, _vp]
        lib.gal_plan_set_pruning.argtypes = [_vp, _i]
        lib.gal_plan_set_option.argtypes = [_vp, _i, _d]
        lib.gal_plan_unbind_uv.argtypes = [_vp]
        lib.gal_last_extent_violations.argtypes = [_vp]
        lib.gal_last_extent_violations.restype = _i64
        for s in ("f64", "f32"):
            getattr(lib, f"gal_plan_bind_uv_{s}").argtypes = [_vp, _vp, _vp, _i64, _i, _vp]
        lib.gal_plan_unbind_obs.argtypes = [_vp]
        for s in ("f64", "f32"):
            getattr(lib, f"gal_plan_bind_obs_{s}").argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _i64, _i, _vp]
        lib.gal_last_uv_extent.argtypes = [_vp, _vp]
        for s in ("f64", "f32"):
            getattr(lib, f"gal_sweep_{s}").argtypes = [_vp, _vp, _i, _d, _d, _d, _d, _vp, _vp]
            getattr(lib, f"gal_fft2_shifted_{s}").argtypes = [_vp, _vp, _vp, _vp]
            getattr(lib, f"gal_sample_image_{s}").argtypes = [_vp, _vp, _d, _vp, _vp, _i64, _d, _d, _d, _vp, _vp]
            getattr(lib, f"gal_chi2_image_{s}").argtypes = [_vp, _vp, _d, _vp, _vp, _vp, _vp, _vp, _i64, _d, _d, _d,
                                                            _vp, _vp]
            getattr(lib, f"gal_chi2_image_host_{s}").argtypes = [_vp, _vp, _d, _vp, _vp, _vp, _vp, _vp, _i64, _d, _d,
                                                                 _d, _vp, _vp]
            getattr(lib, f"gal_sample_profile_{s}").argtypes = [_vp, _vp, _i, _d, _d, _d, _vp, _vp, _i64, _d, _d, _d,
                                                                _d, _vp, _vp]
            getattr(lib, f"gal_chi2_profile_{s}").argtypes = [_vp, _vp, _i, _d, _d, _d, _vp, _vp, _vp, _vp, _vp, _i64,
                                                              _d, _d, _d, _d, _vp, _vp]
            getattr(lib, f"gal_chi2_image_batch_{s}").argtypes = [_vp, _vp, _i, _d, _vp, _vp, _vp, _vp, _vp, _i64, _d,
                                                                  _d, _d, _vp, _vp, _vp]
        for s in ("f64", "f32"):
            getattr(lib, f"gal_chi2_image_sets_{s}").argtypes = [_vp, _vp, _i, _d, _vp, _vp, _vp, _vp, _vp, _i64, _d, _d,
                                                                 _d, _vp, _vp, _vp]
        for s in ("f64", "f32"):
            getattr(lib, f"gal_sample_profile_hankel_{s}").argtypes = [_vp, _vp, _i, _d, _d, _vp, _vp, _i64, _d, _d, _d, _d,
                                                                       _vp, _vp]
            getattr(lib, f"gal_chi2_profile_hankel_{s}").argtypes = [_vp, _vp, _i, _d, _d, _vp, _vp, _vp, _vp, _vp, _i64,
                                                                     _d, _d, _d, _d, _vp, _vp]
        for s in ("f64", "f32"):
            getattr(lib, f"gal_sample_image_multi_{s}").argtypes = [_vp, _vp, _d, _vp, _vp, _i64, _i, _vp, _vp, _vp, _vp,
                                                                    _vp, _vp]
            getattr(lib, f"gal_chi2_image_multi_{s}").argtypes = [_vp, _vp, _d, _vp, _vp, _vp, _vp, _vp, _i64, _i, _vp,
                                                                  _vp, _vp, _vp, _vp, _vp]
        for s in ("f64", "f32"):
            getattr(lib, f"gal_sample_image_host_{s}").argtypes = [_vp, _vp, _d, _vp, _vp, _i64, _d, _d, _d, _vp, _vp]
            getattr(lib, f"gal_chi2_profile_host_{s}").argtypes = [_vp, _vp, _i, _d, _d, _d, _vp, _vp, _vp, _vp, _vp, _i64,
                                                                   _d, _d, _d, _d, _vp, _vp]
            getattr(lib, f"gal_sample_profile_host_{s}").argtypes = [_vp, _vp, _i, _d, _d, _d, _vp, _vp, _i64, _d, _d, _d,
                                                                     _d, _vp, _vp]
        lib.gal_chi2_profile_hankel_noalloc_f64.argtypes = [_i, _vp, _i, _d, _d, _vp, _vp, _vp, _vp, _vp, _i64, _d, _d,
                                                            _d, _d, _vp, _vp]
        lib.gal_noalloc_scratch_bytes.restype = ctypes.c_size_t
        lib.gal_measure_fp64_fma_peak.argtypes = [_i, _vp, _vp]
        _lib = lib
    return _lib


def _check(rc: int, what: str, plan: "Plan" = None) -> None:
    if rc != 0:
        msg = load_library().gal_strerror(rc).decode()
        extra = f" (cudaError {load_library().gal_last_cuda_error(plan._h)})" if plan is not None and rc == -3 else ""
        raise GalarioError(f"{what}: {msg}{extra}")


def get_image_size(u, v, PB: float = 0.0, f_min: float = 5.0, f_max: float = 2.5):
    """(N_lm, dxy) for the uv coverage (host arrays, wavelengths): Eq. 19-24."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    v = np.ascontiguousarray(v, dtype=np.float64)
    if u.shape != v.shape:
        raise GalarioError("u and v must have the same shape")
    n, d = ctypes.c_int(0), ctypes.c_double(0.0)
    _check(load_library().gal_get_image_size(u.ctypes.data, v.ctypes.data, u.size, float(PB), float(f_min),
                                             float(f_max), ctypes.addressof(n), ctypes.addressof(d)),
           "gal_get_image_size")
    return n.value, d.value


def measure_fp64_peak(device: int = 0):
    """(TFLOP/s, ms of the best launch): the FP64 FMA rate measured on `device` (gal_measure_fp64_fma_peak)."""
    tf, ms = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(load_library().gal_measure_fp64_fma_peak(int(device), ctypes.addressof(tf), ctypes.addressof(ms)),
           "gal_measure_fp64_fma_peak")
    return tf.value, ms.value


NOALLOC_MAX_POINTS = 1 << 20          # GAL_NOALLOC_MAX_POINTS of the header


def chi2ProfileHankelNoAlloc(I, Rmin, dR, u, v, re_obs, im_obs, w, out, dRA=0.0, dDec=0.0, PA=0.0, inc=0.0):
    """chi2Profile by the direct Hankel transform (Eq. 25) for callers that may not allocate device memory.

    Every other call of this package goes through a ``Plan``, and creating a plan calls ``cudaMalloc``.  A program
    that lives inside a fixed device-memory budget (its host application split the GPU up at start-up, it runs as a
    memory-capped MPS client, the GPU is already full) or that cannot tolerate the device-wide synchronisation of
    ``cudaMalloc`` in its inner loop uses this function instead: no plan, no allocation of any kind — neither in the
    library nor here, which is why ``out`` (a 1-element float64 CUDA tensor for the result) is a required argument
    and is returned as it is.  The reduction scratch is a 65 792-byte static array inside the library that every GPU
    holds until the process exits; its size limits the call to ``NOALLOC_MAX_POINTS`` = 1 048 576 points (more
    raises ``GalarioError``; split the set and add the results).

    All tensors are contiguous float64 CUDA tensors on one device.  The call is asynchronous on torch's current
    stream.  The first call on each GPU also looks up the scratch array's device address and loads the library's
    device code there: make one small call at start-up, before capturing any stream and before the time-critical
    part.  All calls on a GPU share the one array — calls that may overlap (several streams or threads) race and
    return wrong sums; keep them on one stream."""
    lib = load_library()
    if not torch.cuda.is_available():
        raise GalarioError("no CUDA device: the galario-b200 path has no CPU fallback")
    dev = None
    M = u.numel() if isinstance(u, torch.Tensor) else -1
    for t, what, n in ((I, "I", None), (u, "u", M), (v, "v", M), (re_obs, "re_obs", M), (im_obs, "im_obs", M), (w, "w", M),
                       (out, "out", 1)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise GalarioError(f"{what} must be a contiguous float64 CUDA tensor")
        if n is not None and t.numel() != n:
            raise GalarioError(f"{what} has {t.numel()} elements, expected {n}")
        dev = t.get_device() if dev is None else dev
        if t.get_device() != dev:
            raise GalarioError(f"{what} lives on cuda:{t.get_device()}, I on cuda:{dev}")
    if dev != torch.cuda.current_device():
        raise GalarioError(f"the tensors live on cuda:{dev} but torch's current device (whose stream is used) is "
                           f"cuda:{torch.cuda.current_device()}")
    rc = lib.gal_chi2_profile_hankel_noalloc_f64(dev, I.data_ptr(), I.numel(), Rmin, dR, u.data_ptr(), v.data_ptr(),
                                                 re_obs.data_ptr(), im_obs.data_ptr(), w.data_ptr(), M, dRA, dDec, PA,
                                                 inc, out.data_ptr(), _stream())
    if rc != 0:
        extra = f" (cudaError {lib.gal_noalloc_last_cuda_error()})" if rc == -3 else ""
        raise GalarioError(f"gal_chi2_profile_hankel_noalloc_f64: {lib.gal_strerror(rc).decode()}{extra}")
    return out


def _stream() -> int:
    # (the raw handle of torch's current stream; small calls are bound by the host's issue rate, so the cheap accessor)
    return torch._C._cuda_getCurrentRawStream(torch.cuda.current_device())


class Plan:
    """gal_plan: owns the twiddle table, the half-plane spectrum workspace and the reduction scratch."""

    def __init__(self, nxy: int, batch: int = 1, dtype: torch.dtype = torch.float64, device: int = 0):
        if dtype not in (torch.float64, torch.float32):
            raise GalarioError("dtype must be torch.float64 or torch.float32")
        if not torch.cuda.is_available():
            raise GalarioError("no CUDA device: the galario-b200 path has no CPU fallback")
        self.nxy, self.batch, self.dtype, self.device = int(nxy), int(batch), dtype, int(device)
        self._sfx = "f64" if dtype == torch.float64 else "f32"
        self._cdtype = torch.complex128 if dtype == torch.float64 else torch.complex64
        self._lib = load_library()
        self._fns = {}
        h = _vp()
        _check(self._lib.gal_plan_create(ctypes.byref(h), self.nxy, self.batch, 64 if dtype == torch.float64 else 32,
                                         self.device), "gal_plan_create")
        self._h = h
        self._bound_uv = None       # tensors of the current gal_plan_bind_uv / gal_plan_bind_obs (kept alive, see bind_uv)
        self._bound_obs = None

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            self._lib.gal_plan_destroy(h)
            self._h = None

    # -- helpers ---------------------------------------------------------------------------
    def _fn(self, name):
        f = self._fns.get(name)
        if f is None:
            f = self._fns[name] = getattr(self._lib, f"gal_{name}_{self._sfx}")
        return f

    def _dev(self, t: torch.Tensor, what: str, numel: Optional[int] = None) -> int:
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == self.dtype and t.is_contiguous()):
            raise GalarioError(f"{what} must be a contiguous CUDA tensor of dtype {self.dtype}")
        if t.get_device() != self.device:
            raise GalarioError(f"{what} lives on cuda:{t.get_device()}, the plan on cuda:{self.device}")
        if numel is not None and t.numel() != numel:
            raise GalarioError(f"{what} has {t.numel()} elements, expected {numel}")
        return t.data_ptr()

    def _out(self, out, numel: int, dtype, like: torch.Tensor) -> torch.Tensor:
        if out is None:
            return torch.empty(numel, dtype=dtype, device=like.device)
        if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == dtype and out.is_contiguous()
                and out.numel() == numel and out.device.index == self.device):
            raise GalarioError(f"out must be a contiguous cuda:{self.device} tensor of {numel} x {dtype}")
        return out

    def workspace_bytes(self) -> int:
        return int(self._lib.gal_plan_workspace_bytes(self._h))

    def last_oob_count(self) -> int:
        return int(self._lib.gal_last_oob_count(self._h))

    def launch_count(self) -> int:
        return int(self._lib.gal_plan_launch_count(self._h))

    def timing_enable(self, max_calls: int) -> None:
        _check(self._lib.gal_plan_timing_enable(self._h, int(max_calls)), "gal_plan_timing_enable", self)

    def timing_read(self):
        """Average ms of (uv-extent kernel, row pass, column pass, sampling kernel) over the recorded calls, and
        their number."""
        ms = (ctypes.c_double * 4)()
        n = ctypes.c_int64(0)
        _check(self._lib.gal_plan_timing_read(self._h, ctypes.addressof(ms), ctypes.addressof(n)),
               "gal_plan_timing_read", self)
        return [ms[0], ms[1], ms[2], ms[3]], n.value

    def set_pruning(self, mode: int) -> None:
        """0 = never, 1 = automatic (default), 2 = always: see gal_plan_set_pruning."""
        _check(self._lib.gal_plan_set_pruning(self._h, int(mode)), "gal_plan_set_pruning", self)

    OPTIONS = {"row_mode": 1, "batch_chunk": 2, "speculate": 3, "spec_min_bytes": 4, "batch_conc": 5, "row_prefetch": 6,
               "row_x2_one_cta": 7}                          # GAL_OPT_* of the header

    def set_option(self, name: str, value) -> None:
        """Tuning options (gal_plan_set_option): kernel forms / launch geometries, never results."""
        if name not in self.OPTIONS:
            raise GalarioError(f"unknown option {name!r}; one of {sorted(self.OPTIONS)}")
        _check(self._lib.gal_plan_set_option(self._h, self.OPTIONS[name], float(value)), "gal_plan_set_option", self)

    @staticmethod
    def _placements(placements):
        """[(dRA, dDec, PA[, scale]), ...] -> four host double arrays."""
        a = np.array([tuple(pl) + (1.0,) * (4 - len(pl)) for pl in placements], dtype=np.float64).reshape(-1, 4)
        return [np.ascontiguousarray(a[:, i]) for i in range(4)]

    def sampleImageMulti(self, image, dxy, u, v, placements, out=None):
        """sum_s scale_s * sampleImage(image; dRA_s, dDec_s, PA_s): one transform, S placements."""
        M = u.numel()
        out = self._out(out, M, self._cdtype, u)
        dRA, dDec, PA, sc = self._placements(placements)
        _check(self._fn("sample_image_multi")(self._h, self._dev(image, "image", self.nxy ** 2), dxy, self._dev(u, "u"),
                                              self._dev(v, "v", M), M, len(dRA), dRA.ctypes.data, dDec.ctypes.data,
                                              PA.ctypes.data, sc.ctypes.data, out.data_ptr(), _stream()),
               "gal_sample_image_multi", self)
        return out

    def chi2ImageMulti(self, image, dxy, u, v, re_obs, im_obs, w, placements, out=None):
        M = u.numel()
        out = self._out(out, 1, torch.float64, u)
        dRA, dDec, PA, sc = self._placements(placements)
        _check(self._fn("chi2_image_multi")(self._h, self._dev(image, "image", self.nxy ** 2), dxy, self._dev(u, "u"),
                                            self._dev(v, "v", M), self._dev(re_obs, "re_obs", M), self._dev(im_obs, "im_obs", M),
                                            self._dev(w, "w", M), M, len(dRA), dRA.ctypes.data, dDec.ctypes.data,
                                            PA.ctypes.data, sc.ctypes.data, out.data_ptr(), _stream()),
               "gal_chi2_image_multi", self)
        return out

    def bind_uv(self, u, v) -> None:
        """Promise that u and v ([M] or [C][M] CUDA tensors) keep their contents: later calls that pass these
        very tensors skip the per-call uv-extent kernel (gal_plan_bind_uv)."""
        C = 1 if u.dim() == 1 else u.shape[0]
        M = u.shape[-1]
        _check(self._fn("plan_bind_uv")(self._h, self._dev(u, "u"), self._dev(v, "v", u.numel()), M, C, _stream()),
               "gal_plan_bind_uv", self)
        # The binding is identified by device addresses.  Keep the tensors alive until unbind / rebind: torch's caching
        # allocator would otherwise hand a freed tensor's address to NEW data, which would then match the old binding.
        self._bound_uv = (u, v)
        self._bound_obs = None

    def bind_obs(self, u, v, re_obs, im_obs, w) -> None:
        """Promise that the five observation arrays ([M] or [C][M]) keep their contents: later chi2 calls that pass
        these very tensors sample the plan's private, uv-sorted copy (gal_plan_bind_obs)."""
        C = 1 if u.dim() == 1 else u.shape[0]
        M = u.shape[-1]
        n = u.numel()
        _check(self._fn("plan_bind_obs")(self._h, self._dev(u, "u"), self._dev(v, "v", n), self._dev(re_obs, "re_obs", n),
                                         self._dev(im_obs, "im_obs", n), self._dev(w, "w", n), M, C, _stream()),
               "gal_plan_bind_obs", self)
        # as bind_uv: the five addresses ARE the binding, so the tensors must not be freed (and their addresses
        # recycled for other data, which would silently sample the plan's old private copy) while it stands
        self._bound_uv = (u, v)
        self._bound_obs = (u, v, re_obs, im_obs, w)

    def unbind_obs(self) -> None:
        _check(self._lib.gal_plan_unbind_obs(self._h), "gal_plan_unbind_obs", self)
        self._bound_obs = None

    def unbind_uv(self) -> None:
        _check(self._lib.gal_plan_unbind_uv(self._h), "gal_plan_unbind_uv", self)
        self._bound_uv = None
        self._bound_obs = None

    def last_extent_violations(self) -> int:
        return int(self._lib.gal_last_extent_violations(self._h))

    def last_uv_extent(self):
        """(kumax, kvs_min, kvs_max) the most recent call's transform was pruned to."""
        ext = (ctypes.c_int * 3)()
        _check(self._lib.gal_last_uv_extent(self._h, ctypes.addressof(ext)), "gal_last_uv_extent", self)
        return int(ext[0]), int(ext[1]), int(ext[2])

    # -- the paper's calls ---------------------------------------------------------------------
    def sweep(self, I, Rmin, dR, dxy, inc=0.0, out=None):
        out = torch.empty((self.nxy, self.nxy), dtype=self.dtype, device=I.device) if out is None else out
        _check(self._fn("sweep")(self._h, self._dev(I, "I"), I.numel(), Rmin, dR, dxy, inc, self._dev(out, "out", self.nxy ** 2),
                                 _stream()), "gal_sweep", self)
        return out

    def fft2_shifted(self, image, out=None):
        if out is None:
            out = torch.empty((self.nxy, self.nxy // 2 + 1), dtype=self._cdtype, device=image.device)
        out = self._out(out, self.nxy * (self.nxy // 2 + 1), self._cdtype, image)
        _check(self._fn("fft2_shifted")(self._h, self._dev(image, "image", self.nxy ** 2), out.data_ptr(), _stream()),
               "gal_fft2_shifted", self)
        return out

    def sampleImage(self, image, dxy, u, v, PA=0.0, dRA=0.0, dDec=0.0, out=None):
        M = u.numel()
        out = self._out(out, M, self._cdtype, u)
        _check(self._fn("sample_image")(self._h, self._dev(image, "image", self.nxy ** 2), dxy, self._dev(u, "u"), self._dev(v, "v", M),
                                        M, dRA, dDec, PA, out.data_ptr(), _stream()), "gal_sample_image", self)
        return out

    def chi2Image(self, image, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, out=None):
        out = self._out(out, 1, torch.float64, u)
        M = u.numel()
        _check(self._fn("chi2_image")(self._h, self._dev(image, "image", self.nxy ** 2), dxy, self._dev(u, "u"), self._dev(v, "v", M),
                                      self._dev(re_obs, "re_obs", M), self._dev(im_obs, "im_obs", M), self._dev(w, "w", M),
                                      M, dRA, dDec, PA, out.data_ptr(), _stream()), "gal_chi2_image", self)
        return out

    def sampleProfile(self, I, Rmin, dR, dxy, u, v, inc=0.0, PA=0.0, dRA=0.0, dDec=0.0, out=None):
        M = u.numel()
        out = self._out(out, M, self._cdtype, u)
        _check(self._fn("sample_profile")(self._h, self._dev(I, "I"), I.numel(), Rmin, dR, dxy, self._dev(u, "u"),
                                          self._dev(v, "v", M), M, dRA, dDec, PA, inc, out.data_ptr(), _stream()),
               "gal_sample_profile", self)
        return out

    def chi2Profile(self, I, Rmin, dR, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, inc=0.0, out=None):
        out = self._out(out, 1, torch.float64, u)
        M = u.numel()
        _check(self._fn("chi2_profile")(self._h, self._dev(I, "I"), I.numel(), Rmin, dR, dxy, self._dev(u, "u"),
                                        self._dev(v, "v", M), self._dev(re_obs, "re_obs", M), self._dev(im_obs, "im_obs", M),
                                        self._dev(w, "w", M), M, dRA, dDec, PA, inc, out.data_ptr(), _stream()),
               "gal_chi2_profile", self)
        return out

    def sampleProfileHankel(self, I, Rmin, dR, u, v, inc=0.0, PA=0.0, dRA=0.0, dDec=0.0, out=None):
        """sampleProfile by the direct Hankel transform of Eq. 25 (no image, no FFT)."""
        M = u.numel()
        out = self._out(out, M, self._cdtype, u)
        _check(self._fn("sample_profile_hankel")(self._h, self._dev(I, "I"), I.numel(), Rmin, dR, self._dev(u, "u"),
                                                 self._dev(v, "v", M), M, dRA, dDec, PA, inc, out.data_ptr(), _stream()),
               "gal_sample_profile_hankel", self)
        return out

    def chi2ProfileHankel(self, I, Rmin, dR, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, inc=0.0, out=None):
        M = u.numel()
        out = self._out(out, 1, torch.float64, u)
        _check(self._fn("chi2_profile_hankel")(self._h, self._dev(I, "I"), I.numel(), Rmin, dR, self._dev(u, "u"),
                                               self._dev(v, "v", M), self._dev(re_obs, "re_obs", M),
                                               self._dev(im_obs, "im_obs", M), self._dev(w, "w", M), M, dRA, dDec,
                                               PA, inc, out.data_ptr(), _stream()), "gal_chi2_profile_hankel", self)
        return out

    def chi2ImageBatch(self, images, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, out=None):
        """images [C][n][n]; u, v, re_obs, im_obs, w [C][M].  Returns (chi2[C], total[1]) on the device."""
        C, M = images.shape[0], u.shape[1]
        out = self._out(out, C + 1, torch.float64, u)
        n = C * M
        _check(self._fn("chi2_image_batch")(self._h, self._dev(images, "images", C * self.nxy ** 2), C, dxy, self._dev(u, "u", n),
                                            self._dev(v, "v", n), self._dev(re_obs, "re_obs", n), self._dev(im_obs, "im_obs", n),
                                            self._dev(w, "w", n), M, dRA, dDec, PA, out.data_ptr(),
                                            out.data_ptr() + 8 * C, _stream()), "gal_chi2_image_batch", self)
        return out[:C], out[C:]

    def chi2ImageSets(self, image, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, out=None):
        """K observation sets ([K][M] tensors, K <= the plan's batch) against ONE image: one transform, one sampling
        launch over the sets (gal_chi2_image_sets).  Returns (chi2_per_set[K], chi2_total[1])."""
        if u.dim() != 2:
            raise GalarioError("u, v, re_obs, im_obs, w must be [K][M]")
        K, M = u.shape
        n = K * M
        out = self._out(out, K + 1, torch.float64, u)
        _check(self._fn("chi2_image_sets")(self._h, self._dev(image, "image", self.nxy ** 2), K, dxy, self._dev(u, "u"),
                                           self._dev(v, "v", n), self._dev(re_obs, "re_obs", n),
                                           self._dev(im_obs, "im_obs", n), self._dev(w, "w", n), M, dRA, dDec, PA,
                                           out.data_ptr(), out.data_ptr() + 8 * K, _stream()), "gal_chi2_image_sets", self)
        return out[:K], out[K:]

    # -- host-pointer calls (numpy / CPU tensors in, Python float or numpy out) ------------------
    def _host(self, a, what):
        a = a.numpy() if isinstance(a, torch.Tensor) else a
        want = np.float64 if self.dtype == torch.float64 else np.float32
        if not (isinstance(a, np.ndarray) and a.dtype == want and a.flags.c_contiguous):
            raise GalarioError(f"{what} must be a C-contiguous host array of dtype {want.__name__}")
        return a.ctypes.data

    def chi2Image_host(self, image, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0) -> float:
        out = ctypes.c_double(0.0)
        _check(self._fn("chi2_image_host")(self._h, self._host(image, "image"), dxy, self._host(u, "u"),
                                           self._host(v, "v"), self._host(re_obs, "re_obs"),
                                           self._host(im_obs, "im_obs"), self._host(w, "w"), u.size if isinstance(u, np.ndarray) else u.numel(),
                                           dRA, dDec, PA, ctypes.addressof(out), _stream()), "gal_chi2_image_host", self)
        return out.value

    def _host_n(self, a, what, n=None):
        """Host array -> address, with its length checked (a short array would be an out-of-bounds host read)."""
        p = self._host(a, what)
        size = a.size if isinstance(a, np.ndarray) else a.numel()
        if n is not None and size != n:
            raise GalarioError(f"{what} has {size} elements, expected {n}")
        return p

    def sampleImage_host(self, image, dxy, u, v, PA=0.0, dRA=0.0, dDec=0.0) -> np.ndarray:
        M = u.size if isinstance(u, np.ndarray) else u.numel()
        out = np.empty(M, dtype=np.complex128 if self.dtype == torch.float64 else np.complex64)
        _check(self._fn("sample_image_host")(self._h, self._host_n(image, "image", self.nxy ** 2), dxy, self._host(u, "u"),
                                             self._host_n(v, "v", M), M, dRA, dDec, PA, out.ctypes.data, _stream()),
               "gal_sample_image_host", self)
        return out

    def chi2Profile_host(self, I, Rmin, dR, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, inc=0.0) -> float:
        out = ctypes.c_double(0.0)
        n = I.size if isinstance(I, np.ndarray) else I.numel()
        M = u.size if isinstance(u, np.ndarray) else u.numel()
        _check(self._fn("chi2_profile_host")(self._h, self._host(I, "I"), n, Rmin, dR, dxy, self._host(u, "u"),
                                             self._host_n(v, "v", M), self._host_n(re_obs, "re_obs", M),
                                             self._host_n(im_obs, "im_obs", M), self._host_n(w, "w", M), M, dRA, dDec, PA,
                                             inc, ctypes.addressof(out), _stream()), "gal_chi2_profile_host", self)
        return out.value

    def sampleProfile_host(self, I, Rmin, dR, dxy, u, v, inc=0.0, PA=0.0, dRA=0.0, dDec=0.0) -> np.ndarray:
        n = I.size if isinstance(I, np.ndarray) else I.numel()
        M = u.size if isinstance(u, np.ndarray) else u.numel()
        out = np.empty(M, dtype=np.complex128 if self.dtype == torch.float64 else np.complex64)
        _check(self._fn("sample_profile_host")(self._h, self._host(I, "I"), n, Rmin, dR, dxy, self._host(u, "u"),
                                               self._host_n(v, "v", M), M, dRA, dDec, PA, inc, out.ctypes.data, _stream()),
               "gal_sample_profile_host", self)
        return out


# -- module-level calls in the paper's style, with a plan cache -------------------------------------
_plans: dict = {}


def get_plan(nxy: int, batch: int = 1, dtype: torch.dtype = torch.float64, device: Optional[int] = None) -> Plan:
    device = torch.cuda.current_device() if device is None else device
    key = (int(nxy), int(batch), dtype, int(device))
    if key not in _plans:
        _plans[key] = Plan(nxy, batch, dtype, device)
    return _plans[key]


def _plan_for(t: torch.Tensor, nxy: int, batch: int = 1) -> Plan:
    if not (isinstance(t, torch.Tensor) and t.is_cuda):
        raise GalarioError("inputs must be CUDA tensors (there is no CPU path)")
    return get_plan(nxy, batch, t.dtype, t.device.index)


def sampleImage(image, dxy, u, v, PA=0.0, dRA=0.0, dDec=0.0):
    return _plan_for(image, image.shape[-1]).sampleImage(image, dxy, u, v, PA, dRA, dDec)


def chi2Image(image, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0):
    return _plan_for(image, image.shape[-1]).chi2Image(image, dxy, u, v, re_obs, im_obs, w, dRA, dDec, PA)


def sampleProfile(I, Rmin, dR, nxy, dxy, u, v, inc=0.0, PA=0.0, dRA=0.0, dDec=0.0):
    return _plan_for(I, nxy).sampleProfile(I, Rmin, dR, dxy, u, v, inc, PA, dRA, dDec)


def chi2Profile(I, Rmin, dR, nxy, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, inc=0.0):
    return _plan_for(I, nxy).chi2Profile(I, Rmin, dR, dxy, u, v, re_obs, im_obs, w, dRA, dDec, PA, inc)


def sweep(I, Rmin, dR, nxy, dxy, inc=0.0):
    return _plan_for(I, nxy).sweep(I, Rmin, dR, dxy, inc)


def chi2ImageBatch(images, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0):
    return _plan_for(images, images.shape[-1], images.shape[0]).chi2ImageBatch(images, dxy, u, v, re_obs, im_obs, w,
                                                                              dRA, dDec, PA)


def fft2_shifted(image):
    return _plan_for(image, image.shape[-1]).fft2_shifted(image)
