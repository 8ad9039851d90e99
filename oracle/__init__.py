"""ctypes front end of the CPU oracle (``galario_oracle.cpp``).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.  Nothing
under ``paper_1709_06999_b200/`` imports it, and it imports nothing from there.

The functions mirror the paper's names: ``sampleImage``,
``chi2Image``, ``sampleProfile``, ``chi2Profile``, ``sweep``, plus the intermediate
``spectrum`` (``fftshift(rfft2(fftshift(image)), axes=0)``) and the batched cube
of DESIGN.md reading A17.  All arithmetic happens in the C++ file; this module only marshals
numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "galario_oracle.cpp"
_LIB = _HERE / "liboracle.so"

_c_double_p = ctypes.POINTER(ctypes.c_double)
_c_int64_p = ctypes.POINTER(ctypes.c_int64)


def build(force: bool = False) -> Path:
    """Compile the oracle with g++ (-O2, C++17).  Building the checker is not using it."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-pthread", str(_SRC), "-o", str(tmp)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(str(build()))
        _lib.orc_chi2.restype = ctypes.c_double
    return _lib


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a: np.ndarray):
    return a.ctypes.data_as(_c_double_p)


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise ValueError(f"oracle {what} failed with code {rc}")


def host_threads() -> int:
    return os.cpu_count() or 1


def sweep(I, Rmin, dR, nxy, dxy, inc=0.0) -> np.ndarray:
    I = _f64(I)
    img = np.empty((nxy, nxy), dtype=np.float64)
    _check(lib().orc_sweep(_p(I), ctypes.c_int(I.size), ctypes.c_double(Rmin), ctypes.c_double(dR),
                           ctypes.c_int(nxy), ctypes.c_double(dxy), ctypes.c_double(inc), _p(img)), "sweep")
    return img


def spectrum(image, nthreads: int = 1, long_double: bool = False) -> np.ndarray:
    """Shifted half-plane spectrum G[nxy][nxy/2+1] (complex128)."""
    image = _f64(image)
    n = image.shape[0]
    assert image.shape == (n, n)
    G = np.empty((n, n // 2 + 1), dtype=np.complex128)
    fn = lib().orc_spectrum_ld if long_double else lib().orc_spectrum
    _check(fn(_p(image), ctypes.c_int(n), G.ctypes.data_as(_c_double_p), ctypes.c_int(nthreads)), "spectrum")
    return G


def sample_spectrum(G, dxy, u, v, dRA=0.0, dDec=0.0, PA=0.0, nthreads: int = 1, return_oob: bool = False):
    G = np.ascontiguousarray(G, dtype=np.complex128)
    n = G.shape[0]
    assert G.shape == (n, n // 2 + 1)
    u, v = _f64(u), _f64(v)
    M = u.size
    vis = np.empty(M, dtype=np.complex128)
    oob = ctypes.c_int64(0)
    _check(lib().orc_sample_spectrum(G.ctypes.data_as(_c_double_p), ctypes.c_int(n), ctypes.c_double(dxy), _p(u),
                                     _p(v), ctypes.c_int64(M), ctypes.c_double(dRA), ctypes.c_double(dDec),
                                     ctypes.c_double(PA), vis.ctypes.data_as(_c_double_p), ctypes.byref(oob),
                                     ctypes.c_int(nthreads)), "sample_spectrum")
    return (vis, oob.value) if return_oob else vis


def sampleImage(image, dxy, u, v, PA=0.0, dRA=0.0, dDec=0.0, nthreads: int = 1, long_double: bool = False,
                return_oob: bool = False):
    image = _f64(image)
    n = image.shape[0]
    assert image.shape == (n, n)
    u, v = _f64(u), _f64(v)
    M = u.size
    vis = np.empty(M, dtype=np.complex128)
    oob = ctypes.c_int64(0)
    fn = lib().orc_sample_image_ld if long_double else lib().orc_sample_image
    _check(fn(_p(image), ctypes.c_int(n), ctypes.c_double(dxy), _p(u), _p(v), ctypes.c_int64(M),
              ctypes.c_double(dRA), ctypes.c_double(dDec), ctypes.c_double(PA), vis.ctypes.data_as(_c_double_p),
              ctypes.byref(oob), ctypes.c_int(nthreads)), "sampleImage")
    return (vis, oob.value) if return_oob else vis


def chi2(vis, re_obs, im_obs, w, nthreads: int = 1) -> float:
    vis = np.ascontiguousarray(vis, dtype=np.complex128)
    re_obs, im_obs, w = _f64(re_obs), _f64(im_obs), _f64(w)
    return float(lib().orc_chi2(vis.ctypes.data_as(_c_double_p), _p(re_obs), _p(im_obs), _p(w),
                                ctypes.c_int64(vis.size), ctypes.c_int(nthreads)))


def chi2Image(image, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, nthreads: int = 1) -> float:
    image = _f64(image)
    n = image.shape[0]
    u, v, re_obs, im_obs, w = _f64(u), _f64(v), _f64(re_obs), _f64(im_obs), _f64(w)
    out = ctypes.c_double(0.0)
    _check(lib().orc_chi2_image(_p(image), ctypes.c_int(n), ctypes.c_double(dxy), _p(u), _p(v), _p(re_obs),
                                _p(im_obs), _p(w), ctypes.c_int64(u.size), ctypes.c_double(dRA),
                                ctypes.c_double(dDec), ctypes.c_double(PA), ctypes.byref(out), None,
                                ctypes.c_int(nthreads)), "chi2Image")
    return out.value


def sampleProfile(I, Rmin, dR, nxy, dxy, u, v, inc=0.0, PA=0.0, dRA=0.0, dDec=0.0, nthreads: int = 1):
    I, u, v = _f64(I), _f64(u), _f64(v)
    M = u.size
    vis = np.empty(M, dtype=np.complex128)
    _check(lib().orc_sample_profile(_p(I), ctypes.c_int(I.size), ctypes.c_double(Rmin), ctypes.c_double(dR),
                                    ctypes.c_int(nxy), ctypes.c_double(dxy), _p(u), _p(v), ctypes.c_int64(M),
                                    ctypes.c_double(dRA), ctypes.c_double(dDec), ctypes.c_double(PA),
                                    ctypes.c_double(inc), vis.ctypes.data_as(_c_double_p), None,
                                    ctypes.c_int(nthreads)), "sampleProfile")
    return vis


def chi2Profile(I, Rmin, dR, nxy, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, inc=0.0,
                nthreads: int = 1) -> float:
    I, u, v, re_obs, im_obs, w = _f64(I), _f64(u), _f64(v), _f64(re_obs), _f64(im_obs), _f64(w)
    out = ctypes.c_double(0.0)
    _check(lib().orc_chi2_profile(_p(I), ctypes.c_int(I.size), ctypes.c_double(Rmin), ctypes.c_double(dR),
                                  ctypes.c_int(nxy), ctypes.c_double(dxy), _p(u), _p(v), _p(re_obs), _p(im_obs),
                                  _p(w), ctypes.c_int64(u.size), ctypes.c_double(dRA), ctypes.c_double(dDec),
                                  ctypes.c_double(PA), ctypes.c_double(inc), ctypes.byref(out), None,
                                  ctypes.c_int(nthreads)), "chi2Profile")
    return out.value


def chi2ImageBatch(images, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, nthreads: int = 1,
                   return_oob: bool = False):
    """images [C][n][n]; u, v, re_obs, im_obs, w [C][M].  Returns (chi2[C], total[, out-of-grid points])."""
    images = _f64(images)
    C, n, _ = images.shape
    u, v, re_obs, im_obs, w = _f64(u), _f64(v), _f64(re_obs), _f64(im_obs), _f64(w)
    M = u.shape[1]
    per = np.empty(C, dtype=np.float64)
    tot = ctypes.c_double(0.0)
    oob = ctypes.c_int64(0)
    _check(lib().orc_chi2_image_batch(_p(images), ctypes.c_int(C), ctypes.c_int(n), ctypes.c_double(dxy), _p(u),
                                      _p(v), _p(re_obs), _p(im_obs), _p(w), ctypes.c_int64(M),
                                      ctypes.c_double(dRA), ctypes.c_double(dDec), ctypes.c_double(PA), _p(per),
                                      ctypes.byref(tot), ctypes.byref(oob), ctypes.c_int(nthreads)), "chi2ImageBatch")
    return (per, tot.value, oob.value) if return_oob else (per, tot.value)


def chi2ImageSets(image, dxy, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, nthreads: int = 1,
                  return_oob: bool = False):
    """K observation sets against ONE model image ("fit simultaneously several observations"; SURVEY.md
    8(f) row 3): u, v, re_obs, im_obs, w are [K][M]; the result is chi2Image of the image with every set in turn, and
    their sum in set order.  Written out as exactly that loop.  Returns (chi2[K], total[, out-of-grid points])."""
    u, v, re_obs, im_obs, w = _f64(u), _f64(v), _f64(re_obs), _f64(im_obs), _f64(w)
    K = u.shape[0]
    per = np.empty(K, dtype=np.float64)
    oob = 0
    for k in range(K):
        if return_oob:
            _, n = sampleImage(image, dxy, u[k], v[k], PA, dRA, dDec, return_oob=True, nthreads=nthreads)
            oob += n
        per[k] = chi2Image(image, dxy, u[k], v[k], re_obs[k], im_obs[k], w[k], dRA, dDec, PA, nthreads=nthreads)
    tot = 0.0
    for k in range(K):
        tot += per[k]
    return (per, tot, oob) if return_oob else (per, tot)


def sampleProfileHankel(I, Rmin, dR, u, v, inc=0.0, PA=0.0, dRA=0.0, dDec=0.0, nthreads: int = 1):
    """Direct Hankel-transform evaluation of Eq. 25 on the profile grid; no image, no FFT."""
    I, u, v = _f64(I), _f64(u), _f64(v)
    M = u.size
    vis = np.empty(M, dtype=np.complex128)
    _check(lib().orc_sample_profile_hankel(_p(I), ctypes.c_int(I.size), ctypes.c_double(Rmin), ctypes.c_double(dR),
                                           _p(u), _p(v), ctypes.c_int64(M), ctypes.c_double(dRA),
                                           ctypes.c_double(dDec), ctypes.c_double(PA), ctypes.c_double(inc),
                                           vis.ctypes.data_as(_c_double_p), ctypes.c_int(nthreads)),
           "sampleProfileHankel")
    return vis


def chi2ProfileHankel(I, Rmin, dR, u, v, re_obs, im_obs, w, dRA=0.0, dDec=0.0, PA=0.0, inc=0.0,
                      nthreads: int = 1) -> float:
    I, u, v, re_obs, im_obs, w = _f64(I), _f64(u), _f64(v), _f64(re_obs), _f64(im_obs), _f64(w)
    out = ctypes.c_double(0.0)
    _check(lib().orc_chi2_profile_hankel(_p(I), ctypes.c_int(I.size), ctypes.c_double(Rmin), ctypes.c_double(dR),
                                         _p(u), _p(v), _p(re_obs), _p(im_obs), _p(w), ctypes.c_int64(u.size),
                                         ctypes.c_double(dRA), ctypes.c_double(dDec), ctypes.c_double(PA),
                                         ctypes.c_double(inc), ctypes.byref(out), ctypes.c_int(nthreads)),
           "chi2ProfileHankel")
    return out.value
