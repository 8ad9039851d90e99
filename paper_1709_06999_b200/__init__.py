"""galario-b200: the GALARIO hot path (arXiv:1709.06999) as hand-written sm_100a CUDA kernels.

Thin binding over the C ABI of ``include/galario_b200.h``: argument marshalling only, every step
of the path runs in the kernels of ``csrc/``.  PyTorch is used for device memory and streams.
There is no CPU fallback: if ``libgalario_b200.so`` is missing or no CUDA device is present the
calls raise.

Paper-style calls::

    from paper_1709_06999_b200 import sampleImage, chi2Image, sampleProfile, chi2Profile, sweep
    vis  = sampleImage(image, dxy, u, v, PA=PA, dRA=dRA, dDec=dDec)        # CUDA tensors in and out
    chi2 = chi2Image(image, dxy, u, v, re_obs, im_obs, w, dRA, dDec, PA)   # 1-element CUDA tensor
"""
from .binding import (Plan, GalarioError, library_path, load_library, sampleImage, chi2Image, sampleProfile,
                      chi2Profile, sweep, chi2ImageBatch, fft2_shifted, get_plan, get_image_size,
                      chi2ProfileHankelNoAlloc, NOALLOC_MAX_POINTS, measure_fp64_peak)

__all__ = ["Plan", "GalarioError", "library_path", "load_library", "sampleImage", "chi2Image", "sampleProfile",
           "chi2Profile", "sweep", "chi2ImageBatch", "fft2_shifted", "get_plan", "get_image_size",
           "chi2ProfileHankelNoAlloc", "NOALLOC_MAX_POINTS", "measure_fp64_peak"]
