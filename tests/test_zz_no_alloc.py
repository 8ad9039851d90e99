"""The allocation-free entry point, gal_chi2_profile_hankel_noalloc_f64 (binding: chi2ProfileHankelNoAlloc).

Some users of this library are not allowed to call cudaMalloc: a fitting code confined to a fixed slice of the GPU
by its host application (or by an MPS memory cap, or because the rest of the run already fills the card), and code in
a latency-critical loop that cannot take cudaMalloc's device-wide synchronisation.  They cannot create a ``Plan``
(gal_plan_create allocates the workspace), so the library gives them one plan-less call whose reduction scratch is a
static 65 792-byte device array inside the library image; the price is a hard limit of 1 048 576 points per call.

What is checked here: the new call against the existing plan-based chi2ProfileHankel on the same inputs, at the chi2
tolerance of the other GPU tests (relative 1e-10; the two differ only in summation order), on TWO CALLS IN A ROW issued
without a host synchronisation between them — the second with fewer points than the first, so that the shared array
still holds partial sums of the first call beyond the part the second one writes, and a stale ticket or a stale slot
would show.  Then the limit, M = 0, and a raw ctypes call with bad arguments.

This file is collected last on purpose (``pytest --collect-only``: the name sorts after every other test file): the
suite runs with ``pytest -x``, which stops at the first failure, and a failure here must not hide the parity tests.  It
builds its own inputs and shares no state with them, so it passes both alone in a fresh process — where its first
call is the one that looks up the scratch array's address — and at the end of the whole suite.
"""
import ctypes

import numpy as np
import pytest
import torch

import workloads as W

pytestmark = pytest.mark.gpu

ARCSEC = np.pi / 648000.0
TOL_CHI2_F64 = 1e-10          # as tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def g():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1709_06999_b200 as pkg
    pkg.load_library()          # fails loudly if the extension is missing
    return pkg


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), device="cuda")


def test_two_calls_in_a_row_match_the_plan_based_call(g):
    # first call: 40 001 points = 313 tiles of 128 with a ragged tail, inclined, rotated, offset;
    # second call: 5 003 points = 40 tiles, other profile length, no offset (phase factor switched off)
    wa = W.config(1, nxy=256, M=40_001, nr=700)
    wb = W.config(1, nxy=256, M=5_003, nr=333)
    A = [dev(a) for a in (wa.profile, wa.u, wa.v, wa.re_obs, wa.im_obs, wa.w)]
    B = [dev(a) for a in (wb.profile, wb.u, wb.v, wb.re_obs, wb.im_obs, wb.w)]
    argsA = dict(dRA=0.11 * ARCSEC, dDec=-0.07 * ARCSEC, PA=wa.PA, inc=np.deg2rad(45.0))
    argsB = dict(dRA=0.0, dDec=0.0, PA=0.4, inc=0.0)
    outA, outB, outA2 = (torch.full((1,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3))

    # the two calls under test, back to back on one stream, then the first one again (run-to-run bit equality)
    r = g.chi2ProfileHankelNoAlloc(A[0], wa.Rmin, wa.dR, *A[1:], outA, **argsA)
    assert r is outA                                         # the caller's tensor, not a new one
    g.chi2ProfileHankelNoAlloc(B[0], wb.Rmin, wb.dR, *B[1:], outB, **argsB)
    g.chi2ProfileHankelNoAlloc(A[0], wa.Rmin, wa.dR, *A[1:], outA2, **argsA)
    torch.cuda.synchronize()
    a, b, a2 = float(outA[0]), float(outB[0]), float(outA2[0])

    plan = g.Plan(64)                                        # the existing path (its nxy plays no role here)
    ra = float(plan.chi2ProfileHankel(A[0], wa.Rmin, wa.dR, *A[1:], **argsA).cpu()[0])
    rb = float(plan.chi2ProfileHankel(B[0], wb.Rmin, wb.dR, *B[1:], **argsB).cpu()[0])
    assert np.isfinite(ra) and ra > 0 and np.isfinite(rb) and rb > 0
    assert abs(a - ra) <= TOL_CHI2_F64 * abs(ra), (a, ra)
    assert abs(b - rb) <= TOL_CHI2_F64 * abs(rb), (b, rb)
    assert a2 == a                                           # fixed tiles, fixed order: the same bits
    assert ra != rb                                          # (the two calls really were different problems)


def test_limit_empty_set_and_bad_arguments(g):
    lib = g.load_library()
    assert g.NOALLOC_MAX_POINTS == 1 << 20 and lib.gal_noalloc_scratch_bytes() == 256 + 8 * (1 << 20) // 128
    w = W.config(1, nxy=256, M=300, nr=100)
    prof, u, v, re, im, wt = (dev(a) for a in (w.profile, w.u, w.v, w.re_obs, w.im_obs, w.w))
    out = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")

    # one point beyond the limit: refused with its own error code before anything is launched, `out` untouched
    big = torch.zeros(g.NOALLOC_MAX_POINTS + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(g.GalarioError, match="GAL_NOALLOC_MAX_POINTS"):
        g.chi2ProfileHankelNoAlloc(prof, w.Rmin, w.dR, big, big, big, big, big, out)
    torch.cuda.synchronize()
    assert float(out[0]) == 7.0
    del big

    # M = 0: chi2 of no points is 0
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    g.chi2ProfileHankelNoAlloc(prof, w.Rmin, w.dR, e, e, e, e, e, out)
    assert float(out[0]) == 0.0

    # and the call still works after the refusals
    g.chi2ProfileHankelNoAlloc(prof, w.Rmin, w.dR, u, v, re, im, wt, out, PA=w.PA, inc=w.inc)
    ref = float(g.Plan(64).chi2ProfileHankel(prof, w.Rmin, w.dR, u, v, re, im, wt, 0.0, 0.0, w.PA, w.inc).cpu()[0])
    assert abs(float(out[0]) - ref) <= TOL_CHI2_F64 * abs(ref)

    # binding checks: a short array, a wrong dtype, a missing output
    with pytest.raises(g.GalarioError):
        g.chi2ProfileHankelNoAlloc(prof, w.Rmin, w.dR, u, v[:-1], re, im, wt, out)
    with pytest.raises(g.GalarioError):
        g.chi2ProfileHankelNoAlloc(prof, w.Rmin, w.dR, u, v, re, im, wt, out.float())
    with pytest.raises(g.GalarioError):
        g.chi2ProfileHankelNoAlloc(prof, w.Rmin, w.dR, u, v, re, im, wt, None)

    # raw C ABI: invalid arguments come back as -1 (GAL_ERR_INVALID_ARGUMENT), an over-long set as -6
    f = lib.gal_chi2_profile_hankel_noalloc_f64
    p = lambda t: t.data_ptr()
    good = [0, p(prof), 100, w.Rmin, w.dR, p(u), p(v), p(re), p(im), p(wt), 300, 0.0, 0.0, 0.0, 0.0, p(out), None]
    def call(**kw):
        a = list(good)
        for k, val in kw.items():
            a[int(k[1:])] = val
        return f(*a)
    assert call() == 0
    assert call(a0=-1) == -1 and call(a0=64) == -1           # device
    assert call(a1=None) == -1 and call(a2=1) == -1          # profile, nr < 2
    assert call(a4=0.0) == -1                                # dR
    assert call(a5=None) == -1 and call(a9=None) == -1       # u, w
    assert call(a10=-1) == -1                                # M < 0
    assert call(a14=np.pi / 2) == -1 and call(a13=float("nan")) == -1
    assert call(a15=None) == -1                              # chi2_out
    assert call(a10=(1 << 20) + 1) == -6
    assert lib.gal_strerror(-6).startswith(b"M exceeds GAL_NOALLOC_MAX_POINTS")
    torch.cuda.synchronize()
