"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Run on the B200 box with ``-m gpu``.

Tolerances (BASELINE.json north_star; reading A13 for "relative"):
  fp64: per visibility  |dV| / max(|V_oracle|, 1e-6 peak) <= 1e-9;   chi2 relative <= 1e-10
  fp32: per visibility  |dV| <= 1e-4 peak;                           chi2 relative <= 1e-4
  FFT stage alone (fp64): <= 1e-12 of the spectrum's peak.
Integer decisions (the cell a point falls in, the out-of-grid count, the sweep's hard edge) are
taken by both sides in double with the listing's operation order, so they are compared exactly.
"""
import numpy as np
import pytest
import torch

import workloads as W

pytestmark = pytest.mark.gpu

ARCSEC = np.pi / 648000.0
TOL_VIS_F64, TOL_CHI2_F64 = 1e-9, 1e-10
TOL_VIS_F32, TOL_CHI2_F32 = 1e-4, 1e-4


@pytest.fixture(scope="module")
def g():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1709_06999_b200 as pkg
    pkg.load_library()          # fails loudly if the extension is missing
    return pkg


def dev(a, dtype=None):
    t = torch.as_tensor(np.ascontiguousarray(a), device="cuda")
    return t if dtype is None else t.to(dtype)


def rel_err(vis, ref):
    peak = np.abs(ref).max()
    return (np.abs(vis - ref) / np.maximum(np.abs(ref), 1e-6 * peak)).max()


def threads(orc):
    return orc.host_threads()


# ---------------------------------------------------------------------------------------------
# S2+S3+S4: the transform alone, every supported size (several tiles, both FFT code paths)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [8, 16, 32, 64, 128, 256, 512, 1024, 2048, 4096, 8192, 16384])
def test_fft2_shifted_matches_oracle_f64(g, orc, n):
    rng = np.random.default_rng(n)
    img = rng.standard_normal((n, n))
    img[n // 2, n // 2] += 5.0
    ref = orc.spectrum(img, nthreads=threads(orc))
    out = g.Plan(n).fft2_shifted(dev(img)).cpu().numpy()
    assert out.shape == ref.shape
    assert np.abs(out - ref).max() <= 1e-12 * np.abs(ref).max()


@pytest.mark.parametrize("n", [8, 64, 512, 4096, 8192, 16384])
def test_fft2_shifted_matches_oracle_f32(g, orc, n):
    rng = np.random.default_rng(n + 1)
    img = rng.random((n, n)).astype(np.float32)
    ref = orc.spectrum(img.astype(np.float64), nthreads=threads(orc))
    out = g.Plan(n, dtype=torch.float32).fft2_shifted(dev(img)).cpu().numpy()
    assert np.abs(out - ref).max() <= 2e-6 * np.abs(ref).max()


def test_fft_delta_and_sign_fold(g):
    """Delta a px East / b px North of the centre -> exp(+2 pi i (ku a + kv b)/n): pins the (-1)^(ku+kv)
    fold of the centre shift and the row fold of the v shift directly on the GPU."""
    n, a, b = 256, 3, -5
    img = np.zeros((n, n))
    img[n // 2 - b, n // 2 - a] = 1.0
    out = g.Plan(n).fft2_shifted(dev(img)).cpu().numpy()
    ku = np.arange(n // 2 + 1)[None, :]
    kv = (np.arange(n) - n // 2)[:, None]
    assert np.abs(out - np.exp(2j * np.pi * (ku * a + kv * b) / n)).max() <= 1e-13


# ---------------------------------------------------------------------------------------------
# S1: sweep
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,inc", [(64, 0.0), (256, 0.6), (1024, np.deg2rad(45.0))])
def test_sweep_matches_oracle(g, orc, n, inc):
    w = W.config(1, nxy=n, M=10, nr=700)
    ref = orc.sweep(w.profile, w.Rmin, w.dR, n, w.dxy, inc)
    out = g.Plan(n).sweep(dev(w.profile), w.Rmin, w.dR, w.dxy, inc).cpu().numpy()
    assert np.array_equal(out == 0, ref == 0)                 # hard edge and zero centre decided identically
    assert np.array_equal(out, ref)                           # same operations, same rounding
    out32 = g.Plan(n, dtype=torch.float32).sweep(dev(w.profile.astype(np.float32)), w.Rmin, w.dR, w.dxy, inc)
    ref32 = orc.sweep(w.profile.astype(np.float32).astype(np.float64), w.Rmin, w.dR, n, w.dxy, inc)
    assert np.array_equal(out32.cpu().numpy(), ref32.astype(np.float32))


# ---------------------------------------------------------------------------------------------
# the five configs, reduced (oracle in seconds, several tiles, ragged tails) ...
# ---------------------------------------------------------------------------------------------
REDUCED = [
    (0, dict(nxy=256, M=10_000)),                     # config 0 is already small: run it as written
    (1, dict(nxy=512, M=50_001, nr=1000)),
    (2, dict(nxy=1024, M=200_003)),
    (3, dict(nxy=2048, M=300_007, n_src=120)),
]


def run_gpu(g, w, dtype=torch.float64):
    plan = g.Plan(w.nxy, 1, dtype)
    t = lambda a: dev(a)
    if w.entry == "chi2Profile":
        vis = plan.sampleProfile(t(w.profile), w.Rmin, w.dR, w.dxy, t(w.u), t(w.v), w.inc, w.PA, w.dRA, w.dDec)
        oob = plan.last_oob_count()
        chi2 = plan.chi2Profile(t(w.profile), w.Rmin, w.dR, w.dxy, t(w.u), t(w.v), t(w.re_obs), t(w.im_obs), t(w.w),
                                w.dRA, w.dDec, w.PA, w.inc)
    else:
        vis = plan.sampleImage(t(w.image), w.dxy, t(w.u), t(w.v), w.PA, w.dRA, w.dDec)
        oob = plan.last_oob_count()
        chi2 = plan.chi2Image(t(w.image), w.dxy, t(w.u), t(w.v), t(w.re_obs), t(w.im_obs), t(w.w), w.dRA, w.dDec, w.PA)
    return vis.cpu().numpy(), float(chi2.cpu()[0]), oob


def run_oracle(orc, w):
    f = lambda a: np.asarray(a, dtype=np.float64)
    nt = threads(orc)
    if w.entry == "chi2Profile":
        image = orc.sweep(f(w.profile), w.Rmin, w.dR, w.nxy, w.dxy, w.inc)
    else:
        image = f(w.image)
    vis, oob = orc.sampleImage(image, w.dxy, f(w.u), f(w.v), w.PA, w.dRA, w.dDec, nthreads=nt, return_oob=True)
    chi2 = orc.chi2(vis, f(w.re_obs), f(w.im_obs), f(w.w))
    return vis, chi2, oob


@pytest.mark.parametrize("idx,kw", REDUCED)
def test_configs_reduced_f64(g, orc, idx, kw):
    w = W.config(idx, **kw)
    vis, chi2, oob = run_gpu(g, w)
    ref, ref_chi2, ref_oob = run_oracle(orc, w)
    assert oob == ref_oob
    assert rel_err(vis, ref) <= TOL_VIS_F64
    assert abs(chi2 - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2)


@pytest.mark.parametrize("idx,kw", REDUCED)
def test_configs_reduced_f32(g, orc, idx, kw):
    w = W.config(idx, **kw).as_f32()
    vis, chi2, oob = run_gpu(g, w, torch.float32)
    ref, ref_chi2, ref_oob = run_oracle(orc, w)              # fp64 oracle on the fp32-rounded inputs (A14)
    assert oob == ref_oob
    assert np.abs(vis - ref).max() <= TOL_VIS_F32 * np.abs(ref).max()
    assert abs(chi2 - ref_chi2) <= TOL_CHI2_F32 * abs(ref_chi2)


def test_config4_reduced_batch(g, orc):
    w = W.config(4, nxy=256, M=20_011, C=5)
    plan = g.Plan(w.nxy, 5)
    per, tot = plan.chi2ImageBatch(dev(w.image), w.dxy, dev(w.u), dev(w.v), dev(w.re_obs), dev(w.im_obs), dev(w.w),
                                   w.dRA, w.dDec, w.PA)
    rper, rtot = orc.chi2ImageBatch(w.image, w.dxy, w.u, w.v, w.re_obs, w.im_obs, w.w, w.dRA, w.dDec, w.PA,
                                    nthreads=threads(orc))
    per, tot = per.cpu().numpy(), float(tot.cpu()[0])
    assert np.abs(per - rper).max() <= TOL_CHI2_F64 * np.abs(rper).max()
    assert abs(tot - rtot) <= TOL_CHI2_F64 * abs(rtot)
    # a batch of C is exactly C single calls (same kernels, same reduction geometry per channel is not
    # promised, so compare at the chi2 tolerance) and a smaller C on a larger plan works
    p1 = g.Plan(w.nxy, 1)
    for c in (0, 4):
        one = p1.chi2Image(dev(w.image[c]), w.dxy, dev(w.u[c]), dev(w.v[c]), dev(w.re_obs[c]), dev(w.im_obs[c]),
                           dev(w.w[c]), w.dRA, w.dDec, w.PA)
        assert abs(float(one.cpu()[0]) - rper[c]) <= TOL_CHI2_F64 * abs(rper[c])
    per3, tot3 = plan.chi2ImageBatch(dev(w.image[:3]), w.dxy, dev(w.u[:3]), dev(w.v[:3]), dev(w.re_obs[:3]),
                                     dev(w.im_obs[:3]), dev(w.w[:3]), w.dRA, w.dDec, w.PA)
    assert np.abs(per3.cpu().numpy() - rper[:3]).max() <= TOL_CHI2_F64 * np.abs(rper).max()
    assert abs(float(tot3.cpu()[0]) - rper[:3].sum()) <= TOL_CHI2_F64 * rper[:3].sum()


# ---------------------------------------------------------------------------------------------
# ... and at BASELINE.json's full sizes, in the launch configuration bench.py times
# ---------------------------------------------------------------------------------------------
def test_config1_full(g, orc):
    w = W.config(1)
    vis, chi2, oob = run_gpu(g, w)
    ref, ref_chi2, ref_oob = run_oracle(orc, w)
    assert oob == ref_oob
    assert rel_err(vis, ref) <= TOL_VIS_F64
    assert abs(chi2 - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2)


def test_config2_full(g, orc):
    w = W.config(2)
    vis, chi2, oob = run_gpu(g, w)
    ref, ref_chi2, ref_oob = run_oracle(orc, w)
    assert oob == ref_oob
    assert rel_err(vis, ref) <= TOL_VIS_F64
    assert abs(chi2 - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2)


@pytest.fixture(scope="module")
def cfg3_full():
    return W.config(3)


def test_config3_full_f64(g, orc, cfg3_full):
    w = cfg3_full
    vis, chi2, oob = run_gpu(g, w)
    ref, ref_chi2, ref_oob = run_oracle(orc, w)
    assert oob == ref_oob
    assert rel_err(vis, ref) <= TOL_VIS_F64
    assert abs(chi2 - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2)
    # determinism: fixed reduction tree, no floating-point atomics
    _, chi2b, _ = run_gpu(g, w)
    assert chi2b == chi2


def test_config3_full_f32(g, orc, cfg3_full):
    w = cfg3_full.as_f32()
    vis, chi2, oob = run_gpu(g, w, torch.float32)
    ref, ref_chi2, ref_oob = run_oracle(orc, w)
    assert oob == ref_oob
    assert np.abs(vis - ref).max() <= TOL_VIS_F32 * np.abs(ref).max()
    assert abs(chi2 - ref_chi2) <= TOL_CHI2_F32 * abs(ref_chi2)


def test_config4_full(g, orc):
    """All 128 channels at the launch geometry bench.py times (grid.y = 128), each against the oracle, the total
    against the oracle's, and the out-of-grid count against the oracle's summed count."""
    w = W.config(4)
    C = w.image.shape[0]
    plan = g.Plan(w.nxy, C)
    per, tot = plan.chi2ImageBatch(dev(w.image), w.dxy, dev(w.u), dev(w.v), dev(w.re_obs), dev(w.im_obs), dev(w.w),
                                   w.dRA, w.dDec, w.PA)
    oob = plan.last_oob_count()
    per, tot = per.cpu().numpy(), float(tot.cpu()[0])
    rper, rtot, roob = orc.chi2ImageBatch(w.image, w.dxy, w.u, w.v, w.re_obs, w.im_obs, w.w, w.dRA, w.dDec, w.PA,
                                          nthreads=threads(orc), return_oob=True)
    assert per.shape == rper.shape == (C,)
    assert (np.abs(per - rper) <= TOL_CHI2_F64 * np.abs(rper)).all(), np.argmax(np.abs(per - rper) / np.abs(rper))
    assert abs(tot - rtot) <= TOL_CHI2_F64 * abs(rtot)
    assert oob == roob and oob > 0      # 16 km at 230 GHz reaches index 609 > 512: some points wrap (reading A6)


def test_config4_reduced_batch_f32(g, orc):
    """gal_chi2_image_batch_f32 against the fp64 oracle on the fp32-rounded inputs (reading A14), per channel and
    total, at the fp32 chi2 tolerance; the out-of-grid count is an integer decision taken in double on both sides."""
    w = W.config(4, nxy=256, M=20_011, C=5).as_f32()
    plan = g.Plan(w.nxy, 5, torch.float32)
    per, tot = plan.chi2ImageBatch(dev(w.image), w.dxy, dev(w.u), dev(w.v), dev(w.re_obs), dev(w.im_obs), dev(w.w),
                                   w.dRA, w.dDec, w.PA)
    oob = plan.last_oob_count()
    f = lambda a: np.asarray(a, dtype=np.float64)
    rper, rtot, roob = orc.chi2ImageBatch(f(w.image), w.dxy, f(w.u), f(w.v), f(w.re_obs), f(w.im_obs), f(w.w),
                                          w.dRA, w.dDec, w.PA, nthreads=threads(orc), return_oob=True)
    per, tot = per.cpu().numpy(), float(tot.cpu()[0])
    assert (np.abs(per - rper) <= TOL_CHI2_F32 * np.abs(rper)).all()
    assert abs(tot - rtot) <= TOL_CHI2_F32 * abs(rtot)
    assert oob == roob


# ---------------------------------------------------------------------------------------------
# direct Hankel evaluation of Eq. 25 against the oracle's
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("M,nr,inc", [(20_003, 2000, np.deg2rad(45.0)), (777, 333, 0.0), (1, 2, 0.3)])
def test_hankel_profile_matches_oracle(g, orc, M, nr, inc):
    w = W.config(1, nxy=256, M=M, nr=nr)
    plan = g.Plan(64)                                                   # no image: nxy plays no role
    prof, u, v, re, im, wt = (dev(a) for a in (w.profile, w.u, w.v, w.re_obs, w.im_obs, w.w))
    dRA, dDec, PA = 0.11 * ARCSEC, -0.07 * ARCSEC, w.PA
    vis = plan.sampleProfileHankel(prof, w.Rmin, w.dR, u, v, inc, PA, dRA, dDec).cpu().numpy()
    ref = orc.sampleProfileHankel(w.profile, w.Rmin, w.dR, w.u, w.v, inc, PA, dRA, dDec, nthreads=threads(orc))
    assert np.abs(vis - ref).max() <= 1e-9 * np.abs(ref).max()
    chi2 = float(plan.chi2ProfileHankel(prof, w.Rmin, w.dR, u, v, re, im, wt, dRA, dDec, PA, inc).cpu()[0])
    ref_chi2 = orc.chi2ProfileHankel(w.profile, w.Rmin, w.dR, w.u, w.v, w.re_obs, w.im_obs, w.w, dRA, dDec, PA, inc,
                                     nthreads=threads(orc))
    assert abs(chi2 - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2)
    # no offset: the phase factor is exactly 1 and the visibilities are real
    v0 = plan.sampleProfileHankel(prof, w.Rmin, w.dR, u, v, inc, PA).cpu().numpy()
    assert np.all(v0.imag == 0.0)
    # rho = 0: the total flux of the swept disc (trapezoid of 2 pi I r cos inc)
    z = torch.zeros(1, dtype=torch.float64, device="cuda")
    f0 = plan.sampleProfileHankel(prof, w.Rmin, w.dR, z, z, inc).cpu().numpy()[0].real
    R = w.Rmin + w.dR * np.arange(nr)
    flux = 2 * np.pi * np.cos(inc) * np.trapezoid(w.profile * R, dx=w.dR)
    assert abs(f0 - flux) <= 1e-12 * abs(flux)


def test_hankel_profile_f32_and_agreement_with_the_fft_route(g, orc):
    w = W.config(1, nxy=512, M=5_001, nr=1000)
    wf = w.as_f32()
    f = lambda a: np.asarray(a, dtype=np.float64)
    p32 = g.Plan(64, 1, torch.float32)
    prof, u, v, re, im, wt = (dev(a) for a in (wf.profile, wf.u, wf.v, wf.re_obs, wf.im_obs, wf.w))
    vis = p32.sampleProfileHankel(prof, w.Rmin, w.dR, u, v, w.inc, w.PA, 1e-7, 2e-7).cpu().numpy()
    ref = orc.sampleProfileHankel(f(wf.profile), w.Rmin, w.dR, f(wf.u), f(wf.v), w.inc, w.PA, 1e-7, 2e-7,
                                  nthreads=threads(orc))
    assert np.abs(vis - ref).max() <= TOL_VIS_F32 * np.abs(ref).max()
    chi2 = float(p32.chi2ProfileHankel(prof, w.Rmin, w.dR, u, v, re, im, wt, 1e-7, 2e-7, w.PA, w.inc).cpu()[0])
    rc = orc.chi2(ref, f(wf.re_obs), f(wf.im_obs), f(wf.w))
    assert abs(chi2 - rc) <= TOL_CHI2_F32 * abs(rc)
    # the two GPU routes (FFT + interpolation, direct Hankel) see the same sky: they differ by the bilinear
    # interpolation error of the FFT route and by the pixelisation of this workload's cusped profile (R^-0.7, empty
    # centre pixel, reading A5): about ten per cent of the peak at this 5" field of view.  The tight
    # statement of their agreement (1e-5 at the uv-grid nodes) is an oracle pin.
    plan = g.Plan(w.nxy)
    d = lambda a: dev(a)
    a = plan.sampleProfile(d(w.profile), w.Rmin, w.dR, w.dxy, d(w.u), d(w.v), w.inc, w.PA).cpu().numpy()
    b = plan.sampleProfileHankel(d(w.profile), w.Rmin, w.dR, d(w.u), d(w.v), w.inc, w.PA).cpu().numpy()
    assert np.abs(a - b).max() <= 0.15 * np.abs(b).max()


# ---------------------------------------------------------------------------------------------
# identities that hold at any size, on the GPU itself
# ---------------------------------------------------------------------------------------------
def test_sampleProfile_is_sampleImage_of_sweep_bit_for_bit(g):
    """PAPER.md:402.  The fused row loader and the standalone sweep kernel share one device function."""
    w = W.config(1, nxy=512, M=30_000, nr=1000)
    plan = g.Plan(w.nxy)
    a = plan.sampleProfile(dev(w.profile), w.Rmin, w.dR, w.dxy, dev(w.u), dev(w.v), w.inc, w.PA, 1e-7, -2e-7)
    img = plan.sweep(dev(w.profile), w.Rmin, w.dR, w.dxy, w.inc)
    b = plan.sampleImage(img, w.dxy, dev(w.u), dev(w.v), w.PA, 1e-7, -2e-7)
    assert torch.equal(a, b)


def test_point_source_closed_form_on_gpu(g):
    n, dxy = 1024, 0.01 * ARCSEC
    img = np.zeros((n, n))
    img[n // 2, n // 2] = 1.0
    rng = np.random.default_rng(3)
    du = 1.0 / (n * dxy)
    q, az = rng.uniform(0, 0.45 * n, 100_000) * du, rng.uniform(0, 2 * np.pi, 100_000)
    u, v = q * np.cos(az), q * np.sin(az)
    dRA, dDec = 0.4 * ARCSEC, -0.25 * ARCSEC
    vis = g.Plan(n).sampleImage(dev(img), dxy, dev(u), dev(v), 0.9, dRA, dDec).cpu().numpy()
    assert np.abs(vis - np.exp(2j * np.pi * (u * dRA + v * dDec))).max() <= 1e-12


def test_chi2_properties_on_gpu(g):
    w = W.config(0)
    plan = g.Plan(w.nxy)
    t = dev
    vis = plan.sampleImage(t(w.image), w.dxy, t(w.u), t(w.v), w.PA, w.dRA, w.dDec)
    vr, vi = vis.real.contiguous(), vis.imag.contiguous()
    zero = plan.chi2Image(t(w.image), w.dxy, t(w.u), t(w.v), vr, vi, t(w.w), w.dRA, w.dDec, w.PA)
    assert float(zero.cpu()[0]) == 0.0                       # V_obs = V exactly -> 0 exactly
    z = torch.zeros_like(vr)
    c0 = float(plan.chi2Image(t(w.image), w.dxy, t(w.u), t(w.v), z, z, t(w.w), w.dRA, w.dDec, w.PA).cpu()[0])
    expect = float((t(w.w) * (vr * vr + vi * vi)).sum().cpu())
    assert abs(c0 - expect) <= 1e-12 * expect
    c3 = float(plan.chi2Image(t(w.image), w.dxy, t(w.u), t(w.v), z, z, 3.0 * t(w.w), w.dRA, w.dDec, w.PA).cpu()[0])
    assert abs(c3 - 3.0 * c0) <= 1e-13 * c3


# ---------------------------------------------------------------------------------------------
# pruned transform and the two streaming paths of the sampler
# ---------------------------------------------------------------------------------------------
def numpy_extent(w, n):
    """The listing's index arithmetic, operation by operation in numpy doubles."""
    c, s = np.cos(w.PA), np.sin(w.PA)
    du = 1.0 / (n * w.dxy)
    urot, vrot = w.u * c - w.v * s, w.u * s + w.v * c
    uidx = np.abs(urot) / du
    vidx = np.where(urot < 0, n / 2 - vrot / du, n / 2 + vrot / du)
    inside = (uidx <= n / 2 - 1.0) & (vidx >= 0.0) & (vidx < n - 1)
    if not inside.all():
        return (n // 2, 0, n - 1)
    ix, iy = np.floor(uidx).astype(int), np.floor(vidx).astype(int)
    # the cell of the dead slots (column 0..1, rows n/2..n/2+1) is always part of the extent
    return (max(ix.max() + 1, 1), min(iy.min(), n // 2), max(iy.max() + 1, n // 2 + 1))


@pytest.mark.parametrize("idx,kw", [(1, dict(nxy=512, M=50_001, nr=1000)), (2, dict(nxy=1024, M=200_003)),
                                    (3, dict(nxy=2048, M=300_007, n_src=120)), (0, dict(nxy=256, M=10_000))])
def test_pruned_transform_changes_nothing(g, idx, kw):
    """The same call with the transform pruned to the uv extent and with the full transform: bit-identical
    visibilities and chi2, and the extent is exactly what the index arithmetic of the listing gives."""
    w = W.config(idx, **kw)
    plan = g.Plan(w.nxy)
    # poison the workspace with the spectrum of another image first
    other = np.random.default_rng(5).standard_normal((w.nxy, w.nxy)) * 1e6
    plan.set_pruning(0)
    plan.sampleImage(dev(other), w.dxy, dev(w.u), dev(w.v), w.PA, w.dRA, w.dDec)
    assert plan.last_uv_extent() == (w.nxy // 2, 0, w.nxy - 1)
    res = {}
    for mode in (2, 0, 1):
        plan.set_pruning(mode)
        res[mode] = run_gpu_on(plan, w)
        if mode == 2:
            assert plan.last_uv_extent() == numpy_extent(w, w.nxy)
    for mode in (0, 1):
        assert np.array_equal(res[2][0], res[mode][0])
        assert res[2][1] == res[mode][1]
        assert res[2][2] == res[mode][2]


def run_gpu_on(plan, w):
    t = dev
    if w.entry == "chi2Profile":
        vis = plan.sampleProfile(t(w.profile), w.Rmin, w.dR, w.dxy, t(w.u), t(w.v), w.inc, w.PA, w.dRA, w.dDec)
        oob = plan.last_oob_count()
        chi2 = plan.chi2Profile(t(w.profile), w.Rmin, w.dR, w.dxy, t(w.u), t(w.v), t(w.re_obs), t(w.im_obs), t(w.w),
                                w.dRA, w.dDec, w.PA, w.inc)
    else:
        vis = plan.sampleImage(t(w.image), w.dxy, t(w.u), t(w.v), w.PA, w.dRA, w.dDec)
        oob = plan.last_oob_count()
        chi2 = plan.chi2Image(t(w.image), w.dxy, t(w.u), t(w.v), t(w.re_obs), t(w.im_obs), t(w.w), w.dRA, w.dDec, w.PA)
    return vis.cpu().numpy(), float(chi2.cpu()[0]), oob


def test_pruned_batch_and_f32(g):
    w = W.config(4, nxy=256, M=20_000, C=4)
    plan = g.Plan(w.nxy, 4)
    out = {}
    for mode in (0, 2):
        plan.set_pruning(mode)
        per, tot = plan.chi2ImageBatch(dev(w.image), w.dxy, dev(w.u), dev(w.v), dev(w.re_obs), dev(w.im_obs),
                                       dev(w.w), w.dRA, w.dDec, w.PA)
        out[mode] = (per.cpu().numpy(), float(tot.cpu()[0]))
    assert np.array_equal(out[0][0], out[2][0]) and out[0][1] == out[2][1]
    w3 = W.config(3, nxy=1024, M=100_003, n_src=50).as_f32()
    p32 = g.Plan(w3.nxy, 1, torch.float32)
    r = {}
    for mode in (0, 2):
        p32.set_pruning(mode)
        r[mode] = run_gpu_on(p32, w3)
    assert np.array_equal(r[0][0], r[2][0]) and r[0][1] == r[2][1]
    ext = p32.last_uv_extent()
    assert ext[0] < w3.nxy // 2 and ext[1] > 0 and ext[2] < w3.nxy - 1


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_unaligned_arrays_take_the_plain_load_path(g, dtype):
    """Tiles are streamed by TMA bulk copies when every per-point array is 16-byte aligned, by plain loads
    otherwise; both give the same bits."""
    w = W.config(3, nxy=512, M=70_001, n_src=30)
    if dtype == torch.float32:
        w = w.as_f32()
    plan = g.Plan(w.nxy, 1, dtype)
    arrs = [w.u, w.v, w.re_obs, w.im_obs, w.w]
    al = [dev(a) for a in arrs]
    un = [dev(np.concatenate([a[:1], a]))[1:] for a in arrs]              # data_ptr offset by one element
    assert all(x.data_ptr() % 16 == 0 for x in al) and all(x.data_ptr() % 16 != 0 for x in un)
    img = dev(w.image)
    va = plan.sampleImage(img, w.dxy, al[0], al[1], w.PA, w.dRA, w.dDec)
    vu = plan.sampleImage(img, w.dxy, un[0], un[1], w.PA, w.dRA, w.dDec)
    assert torch.equal(va, vu)
    ca = plan.chi2Image(img, w.dxy, *al, w.dRA, w.dDec, w.PA)
    cu = plan.chi2Image(img, w.dxy, *un, w.dRA, w.dDec, w.PA)
    assert float(ca.cpu()[0]) == float(cu.cpu()[0])


def test_bound_uv_set(g):
    """gal_plan_bind_uv: calls on a bound uv set skip the uv-extent kernel (3 launches instead of 4), use an extent
    that contains the exact one for any PA, give bit-identical results, and a broken promise is detected."""
    w = W.config(3, nxy=2048, M=300_007, n_src=120)
    img, u, v, re, im, wt = (dev(a) for a in (w.image, w.u, w.v, w.re_obs, w.im_obs, w.w))
    free, bound = g.Plan(w.nxy), g.Plan(w.nxy)
    bound.bind_uv(u, v)
    for PA in (w.PA, 0.3, 2.5, -1.2):
        a = free.sampleImage(img, w.dxy, u, v, PA, w.dRA, w.dDec)
        exact = free.last_uv_extent()
        n0 = bound.launch_count()
        b = bound.sampleImage(img, w.dxy, u, v, PA, w.dRA, w.dDec)
        assert bound.launch_count() - n0 == 3
        ext = bound.last_uv_extent()
        assert ext[0] >= exact[0] and ext[1] <= exact[1] and ext[2] >= exact[2] and ext[0] < w.nxy // 2
        assert torch.equal(a, b) and bound.last_extent_violations() == 0
        ca = free.chi2Image(img, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, PA)
        cb = bound.chi2Image(img, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, PA)
        assert float(ca.cpu()[0]) == float(cb.cpu()[0]) and bound.last_extent_violations() == 0
    # other arrays of the same size are not the bound set: the call computes its own extent
    u2 = u.clone()
    n0 = bound.launch_count()
    bound.sampleImage(img, w.dxy, u2, v, w.PA, w.dRA, w.dDec)
    assert bound.launch_count() - n0 == 4 and bound.last_extent_violations() == 0
    # a broken promise (contents changed in place) is reported: by the counter, and loudly by the next call
    u.mul_(1.7)
    bound.sampleImage(img, w.dxy, u, v, w.PA, w.dRA, w.dDec)
    assert bound.last_extent_violations() > 0
    with pytest.raises(g.GalarioError, match="bound"):
        bound.sampleImage(img, w.dxy, u, v, w.PA, w.dRA, w.dDec)
    # ... which also dropped the binding: the plan works again, unbound
    c = bound.sampleImage(img, w.dxy, u, v, w.PA, w.dRA, w.dDec)
    assert bound.last_extent_violations() == 0 and torch.equal(c, free.sampleImage(img, w.dxy, u, v, w.PA, w.dRA, w.dDec))
    # an explicit unbind after polling the counter clears the pending error as well
    bound.bind_uv(u, v)
    u.mul_(1.3)
    bound.sampleImage(img, w.dxy, u, v, w.PA, w.dRA, w.dDec)
    assert bound.last_extent_violations() > 0
    bound.unbind_uv()
    c = bound.sampleImage(img, w.dxy, u, v, w.PA, w.dRA, w.dDec)
    assert torch.equal(c, free.sampleImage(img, w.dxy, u, v, w.PA, w.dRA, w.dDec))
    # the multi-source call verifies a bound set too: same results while the promise holds, reported when it breaks
    pl = [(w.dRA, w.dDec, w.PA), (-2 * w.dRA, w.dDec, 0.4, 0.3)]
    u.copy_(dev(w.u))                                        # (back to the original baselines)
    bound.bind_uv(u, v)
    m = bound.sampleImageMulti(img, w.dxy, u, v, pl)
    assert bound.last_extent_violations() == 0 and bound.last_uv_extent()[0] < w.nxy // 2
    assert torch.equal(m, free.sampleImageMulti(img, w.dxy, u, v, pl))
    u.mul_(1.4)
    bound.sampleImageMulti(img, w.dxy, u, v, pl)
    assert bound.last_extent_violations() > 0
    with pytest.raises(g.GalarioError, match="bound"):
        bound.sampleImageMulti(img, w.dxy, u, v, pl)
    assert torch.equal(bound.sampleImageMulti(img, w.dxy, u, v, pl), free.sampleImageMulti(img, w.dxy, u, v, pl))


@pytest.mark.parametrize("idx,kw,dtype", [(2, dict(nxy=1024, M=200_003), torch.float64),
                                          (3, dict(nxy=2048, M=300_007, n_src=120), torch.float64),
                                          (3, dict(nxy=2048, M=300_007, n_src=120), torch.float32),
                                          (0, dict(), torch.float64)])
def test_bound_observation_set(g, orc, idx, kw, dtype):
    """gal_plan_bind_obs: chi2 calls on a bound observation set sample the plan's private, uv-sorted copy.  The sum
    runs over the same points in another order: against the oracle at the chi2 tolerance, bit-identical from call to
    call and from binding to binding (the permutation is unique), three launches per call, no uv-extent kernel."""
    w = W.config(idx, **kw)
    f32 = dtype == torch.float32
    if f32:
        w = w.as_f32()
    tol = TOL_CHI2_F32 if f32 else TOL_CHI2_F64
    f = lambda a: np.asarray(a, dtype=np.float64)
    ref, roob = orc.sampleImage(f(w.image), w.dxy, f(w.u), f(w.v), w.PA, w.dRA, w.dDec, nthreads=threads(orc), return_oob=True)
    ref_chi2 = orc.chi2(ref, f(w.re_obs), f(w.im_obs), f(w.w))
    plan = g.Plan(w.nxy, 1, dtype)
    img, u, v, re, im, wt = (dev(a) for a in (w.image, w.u, w.v, w.re_obs, w.im_obs, w.w))
    plan.bind_obs(u, v, re, im, wt)
    n0 = plan.launch_count()
    a = float(plan.chi2Image(img, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA).cpu()[0])
    assert plan.launch_count() - n0 == 3
    assert plan.last_oob_count() == roob
    assert abs(a - ref_chi2) <= tol * abs(ref_chi2)
    b = float(plan.chi2Image(img, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA).cpu()[0])
    plan.bind_obs(u, v, re, im, wt)
    c = float(plan.chi2Image(img, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA).cpu()[0])
    assert a == b == c
    # another PA and offset on the same binding (the sort is rotation-agnostic)
    ref2 = orc.sampleImage(f(w.image), w.dxy, f(w.u), f(w.v), w.PA + 1.0, -w.dRA, 2 * w.dDec, nthreads=threads(orc))
    d = float(plan.chi2Image(img, w.dxy, u, v, re, im, wt, -w.dRA, 2 * w.dDec, w.PA + 1.0).cpu()[0])
    r2 = orc.chi2(ref2, f(w.re_obs), f(w.im_obs), f(w.w))
    assert abs(d - r2) <= tol * abs(r2)
    # sampleImage on the bound (u, v) keeps the caller's order
    vis = plan.sampleImage(img, w.dxy, u, v, w.PA, w.dRA, w.dDec).cpu().numpy()
    if f32:
        assert np.abs(vis - ref).max() <= TOL_VIS_F32 * np.abs(ref).max()
    else:
        assert rel_err(vis, ref) <= TOL_VIS_F64
    # other observation pointers: the (u, v) binding still applies, the private copy does not
    re2 = re.clone()
    e = float(plan.chi2Image(img, w.dxy, u, v, re2, im, wt, w.dRA, w.dDec, w.PA).cpu()[0])
    assert abs(e - ref_chi2) <= tol * abs(ref_chi2)
    # the copy is private: changing the caller's arrays has no effect until the set is bound again
    re.add_(1.0)
    assert float(plan.chi2Image(img, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA).cpu()[0]) == a
    plan.unbind_obs()
    changed = float(plan.chi2Image(img, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA).cpu()[0])
    rc = orc.chi2(ref, f(w.re_obs) + 1.0, f(w.im_obs), f(w.w))
    assert abs(changed - rc) <= tol * abs(rc)


def test_bound_observation_set_batch_and_profile(g, orc):
    w = W.config(4, nxy=256, M=20_000, C=5)
    plan = g.Plan(w.nxy, 5)
    img, u, v, re, im, wt = (dev(a) for a in (w.image, w.u, w.v, w.re_obs, w.im_obs, w.w))
    plan.bind_obs(u, v, re, im, wt)
    per, tot = plan.chi2ImageBatch(img, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA)
    rper, rtot, roob = orc.chi2ImageBatch(w.image, w.dxy, w.u, w.v, w.re_obs, w.im_obs, w.w, w.dRA, w.dDec, w.PA,
                                          nthreads=threads(orc), return_oob=True)
    assert (np.abs(per.cpu().numpy() - rper) <= TOL_CHI2_F64 * np.abs(rper)).all()
    assert abs(float(tot.cpu()[0]) - rtot) <= TOL_CHI2_F64 * abs(rtot)
    assert plan.last_oob_count() == roob
    w1 = W.config(1, nxy=512, M=50_001, nr=1000)
    p1 = g.Plan(w1.nxy)
    prof, u, v, re, im, wt = (dev(a) for a in (w1.profile, w1.u, w1.v, w1.re_obs, w1.im_obs, w1.w))
    p1.bind_obs(u, v, re, im, wt)
    c = float(p1.chi2Profile(prof, w1.Rmin, w1.dR, w1.dxy, u, v, re, im, wt, w1.dRA, w1.dDec, w1.PA, w1.inc).cpu()[0])
    r = orc.chi2Profile(w1.profile, w1.Rmin, w1.dR, w1.nxy, w1.dxy, w1.u, w1.v, w1.re_obs, w1.im_obs, w1.w, w1.dRA,
                        w1.dDec, w1.PA, w1.inc, nthreads=threads(orc))
    assert abs(c - r) <= TOL_CHI2_F64 * abs(r)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_multi_source_composition(g, orc, dtype):
    """one model image placed S times, V = sum_s scale_s V_s with one transform; against the oracle's
    single-source visibilities summed in numpy, and chi2 against the oracle's chi2 of that sum."""
    w = W.config(3, nxy=1024, M=120_011, n_src=40)
    if dtype == torch.float32:
        w = w.as_f32()
    f = lambda a: np.asarray(a, dtype=np.float64)
    places = [(w.dRA, w.dDec, w.PA), (-2e-7, 3e-7, 0.4, 0.5), (5e-7, 1e-7, 2.0, 2.0), (0.0, 0.0, -1.0, 0.25)]
    ref = sum(sc * orc.sampleImage(f(w.image), w.dxy, f(w.u), f(w.v), PA, dRA, dDec, nthreads=threads(orc))
              for dRA, dDec, PA, sc in [p + (1.0,) * (4 - len(p)) for p in places])
    ref_chi2 = orc.chi2(ref, f(w.re_obs), f(w.im_obs), f(w.w))
    plan = g.Plan(w.nxy, 1, dtype)
    img, u, v, re, im, wt = (dev(a) for a in (w.image, w.u, w.v, w.re_obs, w.im_obs, w.w))
    res = {}
    for mode in (1, 0):
        plan.set_pruning(mode)
        vis = plan.sampleImageMulti(img, w.dxy, u, v, places)
        chi2 = float(plan.chi2ImageMulti(img, w.dxy, u, v, re, im, wt, places).cpu()[0])
        res[mode] = (vis.cpu().numpy(), chi2)
    vis, chi2 = res[1]
    assert np.array_equal(vis, res[0][0]) and chi2 == res[0][1]          # pruning (union of the extents) changes nothing
    if dtype == torch.float64:
        assert rel_err(vis, ref) <= TOL_VIS_F64 and abs(chi2 - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2)
        one = plan.sampleImageMulti(img, w.dxy, u, v, places[:1])
        assert torch.equal(one, plan.sampleImage(img, w.dxy, u, v, w.PA, w.dRA, w.dDec))   # S = 1 is the plain call
    else:
        assert np.abs(vis - ref).max() <= TOL_VIS_F32 * np.abs(ref).max()
        assert abs(chi2 - ref_chi2) <= TOL_CHI2_F32 * abs(ref_chi2)


def test_multi_source_with_out_of_grid_points(g, orc):
    """Multi-source on config 0 (7.5 % of the points leave the half-plane grid after the rotation, reading A6): the
    union of the extents is the whole plane; S = 2 exercises one accumulate step, S = 3 two; the out-of-grid count
    is summed over the sources."""
    w = W.config(0)
    plan = g.Plan(w.nxy)
    img, u, v, re, im, wt = (dev(a) for a in (w.image, w.u, w.v, w.re_obs, w.im_obs, w.w))
    for places in ([(w.dRA, w.dDec, w.PA), (1e-7, -2e-7, 1.1, 0.5)],
                   [(w.dRA, w.dDec, w.PA, 0.7), (0.0, 0.0, 0.0, 1.0), (-3e-7, 2e-7, 2.5, 0.3)]):
        ref, roob = 0.0, 0
        for dRA, dDec, PA, sc in [p + (1.0,) * (4 - len(p)) for p in places]:
            vs, o = orc.sampleImage(w.image, w.dxy, w.u, w.v, PA, dRA, dDec, nthreads=threads(orc), return_oob=True)
            ref, roob = ref + sc * vs, roob + o
        vis = plan.sampleImageMulti(img, w.dxy, u, v, places).cpu().numpy()
        assert plan.last_oob_count() == roob and roob > 0
        assert plan.last_uv_extent() == (w.nxy // 2, 0, w.nxy - 1)
        assert rel_err(vis, ref) <= TOL_VIS_F64
        chi2 = float(plan.chi2ImageMulti(img, w.dxy, u, v, re, im, wt, places).cpu()[0])
        ref_chi2 = orc.chi2(ref, w.re_obs, w.im_obs, w.w)
        assert abs(chi2 - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2)


def test_multi_source_single_launch_long_lists_and_bound_set(g, orc):
    """The S placements are looped inside ONE sampling launch: launch accounting, a list longer
    than one chunk of placements (sum carried through vis / a plan-owned sum for chi2), and chi2 on a bound
    observation set."""
    w = W.config(2, nxy=512, M=60_007)
    plan = g.Plan(w.nxy)
    plan.set_pruning(2)                 # (automatic mode does not prune a spectrum this small)
    img, u, v, re, im, wt = (dev(a) for a in (w.image, w.u, w.v, w.re_obs, w.im_obs, w.w))
    rng = np.random.default_rng(3)
    mk = lambda S: [(float(a), float(b), float(c), float(d)) for a, b, c, d in
                    zip(rng.uniform(-3e-7, 3e-7, S), rng.uniform(-3e-7, 3e-7, S), rng.uniform(0, 3.1, S), rng.uniform(0.1, 1.0, S))]
    for S in (4, 16, 17, 37):
        places = mk(S)
        ref, roob = 0.0, 0
        for dRA, dDec, PA, sc in places:
            vs, o = orc.sampleImage(w.image, w.dxy, w.u, w.v, PA, dRA, dDec, nthreads=threads(orc), return_oob=True)
            ref, roob = ref + sc * vs, roob + o
        ref_chi2 = orc.chi2(ref, w.re_obs, w.im_obs, w.w)
        n0 = plan.launch_count()
        vis = plan.sampleImageMulti(img, w.dxy, u, v, places).cpu().numpy()
        nchunks = (S + 15) // 16
        assert plan.launch_count() - n0 == 4 + nchunks          # radius, extent, row, column + one launch per chunk
        assert plan.last_oob_count() == roob
        assert rel_err(vis, ref) <= TOL_VIS_F64
        chi2 = float(plan.chi2ImageMulti(img, w.dxy, u, v, re, im, wt, places).cpu()[0])
        assert abs(chi2 - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2)
    # bound observation set: no extent kernels at all, the private sorted copy is sampled
    plan.bind_obs(u, v, re, im, wt)
    n0 = plan.launch_count()
    b = float(plan.chi2ImageMulti(img, w.dxy, u, v, re, im, wt, places).cpu()[0])
    assert plan.launch_count() - n0 == 2 + nchunks
    assert abs(b - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2)
    vis_b = plan.sampleImageMulti(img, w.dxy, u, v, places).cpu().numpy()     # caller's order
    assert rel_err(vis_b, ref) <= TOL_VIS_F64
    plan.unbind_obs()
    # a following plain call finds its per-call state re-armed
    c = float(plan.chi2Image(img, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA).cpu()[0])
    rv, ro = orc.sampleImage(w.image, w.dxy, w.u, w.v, w.PA, w.dRA, w.dDec, nthreads=threads(orc), return_oob=True)
    r = orc.chi2(rv, w.re_obs, w.im_obs, w.w)
    assert abs(c - r) <= TOL_CHI2_F64 * abs(r) and plan.last_oob_count() == ro


def test_per_call_state_across_calls(g, orc):
    """The out-of-grid counter and the uv extent belong to ONE call: the two device copies of that state are used
    alternately and re-armed by the sampler of the call before (or by an explicit copy after an M = 0 call)."""
    w = W.config(0)
    plan = g.Plan(w.nxy)
    plan.set_pruning(2)                 # always compute the extent (automatic mode skips it for a spectrum this small)
    t = dev
    _, ref_oob = orc.sampleImage(w.image, w.dxy, w.u, w.v, w.PA, w.dRA, w.dDec, return_oob=True)
    assert ref_oob > 0
    inside = (np.hypot(w.u, w.v) < 0.3 / w.dxy)
    ui, vi = w.u[inside], w.v[inside]
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    for rep in range(3):
        plan.sampleImage(t(w.image), w.dxy, t(w.u), t(w.v), w.PA, w.dRA, w.dDec)
        assert plan.last_oob_count() == ref_oob and plan.last_uv_extent() == (w.nxy // 2, 0, w.nxy - 1)
        plan.chi2Image(t(w.image), w.dxy, t(ui), t(vi), t(w.re_obs[inside]), t(w.im_obs[inside]), t(w.w[inside]),
                       w.dRA, w.dDec, w.PA)
        ext = plan.last_uv_extent()
        assert plan.last_oob_count() == 0 and ext[0] < w.nxy // 2 and ext[1] > 0 and ext[2] < w.nxy - 1
        if rep == 1:
            plan.chi2Image(t(w.image), w.dxy, e, e, e, e, e)
            assert plan.last_oob_count() == 0


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_speculative_extent_and_its_second_pass(g, orc, dtype):
    """Automatic pruning, unbound uv, nxy = 2048 / 4096: from the second call on the transform is pruned to the extent
    the call before derived from its points' largest baseline (no uv-extent kernel), every point is verified against
    it, and a call whose points reach further repeats itself on the device (one conditional kernel).  Whatever the
    history, every result equals the one of a plan that never prunes — bit for bit, except for a repeated call, whose
    row pass is the plain kernel's (last bits of the transform) — and the out-of-grid count is the oracle's."""
    w = W.config(2, nxy=2048, M=300_007)
    f32 = dtype == torch.float32
    if f32:
        w = w.as_f32()
    fresh = g.Plan(w.nxy, 1, dtype)
    fresh.set_pruning(0)
    plan = g.Plan(w.nxy, 1, dtype)                      # prune mode 1 (default)
    plan.set_option("spec_min_bytes", 0)                # speculate at this test's size too
    image = dev(w.image)
    N = w.nxy

    def both(scale, PA, dRA, what, repeated=False):
        u, v = dev(w.u * scale), dev(w.v * scale)
        n0 = plan.launch_count()
        if what == "chi2":
            args = (image, w.dxy, u, v, dev(w.re_obs), dev(w.im_obs), dev(w.w), dRA, w.dDec, PA)
            a, b = plan.chi2Image(*args).cpu().numpy(), fresh.chi2Image(*args).cpu().numpy()
        else:
            a = plan.sampleImage(image, w.dxy, u, v, PA, dRA, w.dDec).cpu().numpy()
            b = fresh.sampleImage(image, w.dxy, u, v, PA, dRA, w.dDec).cpu().numpy()
        if repeated:
            tol = 1e-5 if f32 else 1e-11
            assert np.abs(a - b).max() <= tol * np.abs(b).max(), (scale, PA, what)
        else:
            assert np.array_equal(a, b), (scale, PA, what)
        assert plan.last_oob_count() == fresh.last_oob_count()
        return plan.last_uv_extent(), plan.launch_count() - n0

    e1, n1 = both(1.0, w.PA, w.dRA, "chi2")             # uv-extent kernel: the exact extent
    e2, n2 = both(1.0, w.PA, w.dRA, "chi2")             # speculates on the radius extent of call 1: symmetric, a superset
    assert n1 == 4 and n2 == 4                          # (extent, row, column, sampling) / (row, column, sampling, conditional)
    assert e2[0] >= e1[0] and e2[1] <= e1[1] and e2[2] >= e1[2] and e2[0] < N // 2
    assert e2[1] + e2[2] == N
    e3, _ = both(1.0, w.PA + 0.7, 2 * w.dRA, "sample")  # any rotation stays inside the radius extent
    assert e3 == e2
    e4, _ = both(1.6, w.PA, w.dRA, "chi2", repeated=True)     # longer baselines: verification fails, second pass on the new extent
    assert e4[0] > e2[0] and e4[1] < e2[1]
    e5, _ = both(1.0, w.PA - 0.3, w.dRA, "sample")      # shorter again: speculates on call 4's (larger) extent, no second pass
    assert e5 == e4
    e6, _ = both(1.0, w.PA, w.dRA, "chi2")              # and back to the extent of the data
    assert e6 == e2
    # points beyond the grid: the derived extent is the whole plane, results and counts still equal
    e7, _ = both(8.0, w.PA, w.dRA, "chi2", repeated=True)
    assert e7 == (N // 2, 0, N - 1) and plan.last_oob_count() > 0
    e8, _ = both(8.0, w.PA, w.dRA, "sample")
    assert e8 == (N // 2, 0, N - 1)
    e9, _ = both(1.0, w.PA, w.dRA, "chi2")              # whole-plane speculation can not fail
    assert e9 == (N // 2, 0, N - 1)
    assert both(1.0, w.PA, w.dRA, "chi2")[0] == e2
    both(1.7, w.PA, w.dRA, "sample", repeated=True)     # a repeated sampleImage
    # against the oracle once, on the state this history has left behind (a repeated call)
    f = lambda a: np.asarray(a, dtype=np.float64)
    us, vs = (w.u * 1.9).astype(w.u.dtype), (w.v * 1.9).astype(w.v.dtype)
    ref = orc.chi2Image(f(w.image), w.dxy, f(us), f(vs), f(w.re_obs), f(w.im_obs), f(w.w), w.dRA, w.dDec, w.PA)
    got = float(plan.chi2Image(image, w.dxy, dev(us), dev(vs), dev(w.re_obs), dev(w.im_obs), dev(w.w),
                               w.dRA, w.dDec, w.PA).cpu()[0])
    assert abs(got - ref) <= (TOL_CHI2_F32 if f32 else TOL_CHI2_F64) * abs(ref)


@pytest.mark.parametrize("nxy,dtype", [(2048, torch.float64), (4096, torch.float64), (2048, torch.float32), (4096, torch.float32)])
def test_second_pass_of_a_speculative_call_against_the_oracle(g, orc, nxy, dtype):
    """The conditional second pass (redo.cuh) at BOTH sizes it is built for, incl. the headline's nxy = 4096: after a
    speculating call on short baselines the uv set grows, the sampler's verification fails and the persistent kernel
    repeats row pass, column pass and sampling on the device.  Its visibilities and chi2 are compared with the ORACLE
    at the tolerances of every other parity test (reading A13), with the out-of-grid count and the extent."""
    f32 = dtype == torch.float32
    w = W.config(3, nxy=nxy, M=150_001, n_src=40)
    if f32:
        w = w.as_f32()
    f = lambda a: np.asarray(a, dtype=np.float64)
    plan = g.Plan(nxy, 1, dtype)                             # prune mode 1 (default)
    plan.set_option("spec_min_bytes", 0)                     # speculate at this test's M too
    image, obs = dev(w.image), (dev(w.re_obs), dev(w.im_obs), dev(w.w))
    small = (dev(w.u * 0.5), dev(w.v * 0.5))
    N = nxy

    def prime():                                             # two calls on the short baselines: the 2nd speculates
        plan.chi2Image(image, w.dxy, *small, *obs, w.dRA, w.dDec, w.PA)
        n0 = plan.launch_count()
        plan.chi2Image(image, w.dxy, *small, *obs, w.dRA, w.dDec, w.PA)
        assert plan.launch_count() - n0 == 4                 # row, column, sampling, conditional kernel: no extent pass
        return plan.last_uv_extent()

    for scale, wraps in ((1.0, False), (5.0, True)):         # grown set inside the grid / beyond it (whole plane, A6)
        us, vs = (w.u * scale).astype(w.u.dtype), (w.v * scale).astype(w.v.dtype)
        u, v = dev(us), dev(vs)
        ref, ref_oob = orc.sampleImage(f(w.image), w.dxy, f(us), f(vs), w.PA, w.dRA, w.dDec, return_oob=True,
                                       nthreads=threads(orc))
        ref_chi2 = orc.chi2(ref, f(w.re_obs), f(w.im_obs), f(w.w))
        peak = np.abs(ref).max()
        # sampleImage through the second pass
        e_small = prime()
        vis = plan.sampleImage(image, w.dxy, u, v, w.PA, w.dRA, w.dDec).cpu().numpy()
        e_big = plan.last_uv_extent()
        assert e_big[0] > e_small[0] and e_big[1] < e_small[1] and e_big[2] > e_small[2]      # the call did repeat itself
        assert (e_big == (N // 2, 0, N - 1)) == wraps
        assert plan.last_oob_count() == ref_oob and (ref_oob > 0) == wraps
        if f32:
            assert np.abs(vis - ref).max() <= TOL_VIS_F32 * peak
        else:
            assert rel_err(vis, ref) <= TOL_VIS_F64
        # chi2Image through the second pass
        prime()
        chi2 = float(plan.chi2Image(image, w.dxy, u, v, *obs, w.dRA, w.dDec, w.PA).cpu()[0])
        assert plan.last_uv_extent() == e_big and plan.last_oob_count() == ref_oob
        assert abs(chi2 - ref_chi2) <= (TOL_CHI2_F32 if f32 else TOL_CHI2_F64) * abs(ref_chi2)
        # and the call after it speculates on the grown extent: no second pass, same numbers
        chi2b = float(plan.chi2Image(image, w.dxy, u, v, *obs, w.dRA, w.dDec, w.PA).cpu()[0])
        assert abs(chi2b - ref_chi2) <= (TOL_CHI2_F32 if f32 else TOL_CHI2_F64) * abs(ref_chi2)


def test_second_passes_of_two_plans_under_contention(g):
    """The second pass is one persistent kernel with grid barriers, so all of its CTAs must be resident together.  It is
    launched cooperatively: two plans on two streams that BOTH repeat a call at the same moment — each grid wants every
    SM — and a third stream that keeps the SMs busy with long direct-Hankel launches must all finish (a plain launch
    could place part of each grid and spin for ever), with the results of a never-pruning plan."""
    w = W.config(3, nxy=2048, M=150_001, n_src=40)
    image, obs = dev(w.image), (dev(w.re_obs), dev(w.im_obs), dev(w.w))
    small, big = (dev(w.u * 0.5), dev(w.v * 0.5)), (dev(w.u), dev(w.v))
    fresh = g.Plan(w.nxy)
    fresh.set_pruning(0)
    ref_small = float(fresh.chi2Image(image, w.dxy, *small, *obs, w.dRA, w.dDec, w.PA).cpu()[0])
    ref_big = float(fresh.chi2Image(image, w.dxy, *big, *obs, w.dRA, w.dDec, w.PA).cpu()[0])
    plans = [g.Plan(w.nxy), g.Plan(w.nxy)]
    for p in plans:
        p.set_option("spec_min_bytes", 0)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    filler_stream, filler_plan = torch.cuda.Stream(), g.Plan(64)
    w1 = W.config(1, nxy=256, M=60_000, nr=2000)
    fill = [dev(a) for a in (w1.profile, w1.u, w1.v, w1.re_obs, w1.im_obs, w1.w)]
    torch.cuda.synchronize()
    outs = ([], [])
    for it in range(8):
        with torch.cuda.stream(filler_stream):               # some milliseconds of CTAs on every SM
            filler_plan.chi2ProfileHankel(fill[0], w1.Rmin, w1.dR, *fill[1:], 0.0, 0.0, w1.PA, w1.inc)
        for p, st, o in zip(plans, streams, outs):
            with torch.cuda.stream(st):                      # small, small (speculates), big (verification fails: second pass)
                a = p.chi2Image(image, w.dxy, *small, *obs, w.dRA, w.dDec, w.PA)
                b = p.chi2Image(image, w.dxy, *small, *obs, w.dRA, w.dDec, w.PA)
                c = p.chi2Image(image, w.dxy, *big, *obs, w.dRA, w.dDec, w.PA)
                o.append((a, b, c))
    torch.cuda.synchronize()
    for o in outs:
        for a, b, c in o:
            for got, ref in ((a, ref_small), (b, ref_small), (c, ref_big)):
                assert abs(float(got[0]) - ref) <= TOL_CHI2_F64 * abs(ref)
    for p in plans:
        assert p.last_uv_extent()[0] < w.nxy // 2 and p.last_oob_count() == 0


def test_batched_calls_back_to_back_read_the_extent_after_the_wait(g):
    """Small grids, always-prune mode, C > 1, points beyond the grid (so the exact extent is the WHOLE plane and the
    spectrum takes the single-value layout, while the armed default says 'pair'), many calls issued back to back with
    no host synchronisation: the kernels of consecutive calls are co-resident through programmatic dependent launch,
    so a sampler that read the extent before its griddepcontrol.wait would pick the wrong layout / plane offset.
    Every call must equal the never-pruning plan's result, bit for bit."""
    w = W.config(4, nxy=128, M=60_000, C=6)
    u, v = dev(w.u), dev(w.v)                                # at this nxy: far beyond the grid in every channel
    args = (dev(w.image), w.dxy, u, v, dev(w.re_obs), dev(w.im_obs), dev(w.w), w.dRA, w.dDec, w.PA)
    ref_plan = g.Plan(w.nxy, 6)
    ref_plan.set_pruning(0)
    rper, rtot = ref_plan.chi2ImageBatch(*args)
    assert ref_plan.last_oob_count() > 0
    plan = g.Plan(w.nxy, 6)
    plan.set_pruning(2)
    outs = [plan.chi2ImageBatch(*args) for _ in range(40)]   # no synchronisation in between
    torch.cuda.synchronize()
    assert plan.last_uv_extent() == (w.nxy // 2, 0, w.nxy - 1)
    for per, tot in outs:
        assert torch.equal(per, rper) and torch.equal(tot, rtot)
    # the same with in-grid points in between (pair layout <-> single layout from one call to the next)
    ui, vi = dev(w.u * 0.08), dev(w.v * 0.08)                # (longest baseline at 49 of 64 cells)
    argi = (args[0], w.dxy, ui, vi) + args[4:]
    iper, itot = ref_plan.chi2ImageBatch(*argi)
    assert ref_plan.last_oob_count() == 0
    mixed = [plan.chi2ImageBatch(*(args if k % 2 else argi)) for k in range(40)]
    torch.cuda.synchronize()
    for k, (per, tot) in enumerate(mixed):
        assert torch.equal(per, rper if k % 2 else iper) and torch.equal(tot, rtot if k % 2 else itot), k


@pytest.mark.parametrize("nxy", [2048, 4096])
def test_row_pass_variant_follows_the_expected_extent(g, nxy):
    """At nxy = 2048 / 4096 (fp64) the plan picks the row-pass form from the extent it EXPECTS — a hint the sampler of
    the call before leaves in mapped host memory, read without synchronising: several rows per CTA (whole sectors)
    for a whole-plane transform, one row per CTA when the row-transformed image stays in the L2.  Both forms do the
    same arithmetic: whatever the history of a plan, its results equal, bit for bit, those of a plan that never
    prunes (which always takes the first form)."""
    w = W.config(2, nxy=nxy, M=100_003)
    image = dev(w.image)
    ref_plan = g.Plan(nxy)
    ref_plan.set_pruning(0)
    plan = g.Plan(nxy)
    plan.set_option("speculate", 0)                          # this test is about the row-pass forms (the speculative
                                                             # extent has its own, above)
    obs = (dev(w.re_obs), dev(w.im_obs), dev(w.w))
    for scale in (1.0, 1.0, 1.0, 9.0, 9.0, 1.0, 1.0):        # in-grid (pruned), then wrapping (whole plane), then back
        u, v = dev(w.u * scale), dev(w.v * scale)
        a = plan.chi2Image(image, w.dxy, u, v, *obs, w.dRA, w.dDec, w.PA)
        b = ref_plan.chi2Image(image, w.dxy, u, v, *obs, w.dRA, w.dDec, w.PA)
        torch.cuda.synchronize()                             # (the hint of this call is in host memory now)
        assert torch.equal(a, b), scale
        va = plan.sampleImage(image, w.dxy, u, v, w.PA, w.dRA, w.dDec)
        vb = ref_plan.sampleImage(image, w.dxy, u, v, w.PA, w.dRA, w.dDec)
        torch.cuda.synchronize()
        assert torch.equal(va, vb), scale
        whole = plan.last_uv_extent() == (nxy // 2, 0, nxy - 1)
        assert whole == (scale > 1.0)


# ---------------------------------------------------------------------------------------------
# edge cases
# ---------------------------------------------------------------------------------------------
def test_edge_points_and_wrap(g, orc):
    """Exact nodes, u' = 0 and -0.0, the top row, the Nyquist column, and points beyond the grid."""
    n, dxy = 64, 0.05 * ARCSEC
    du = 1.0 / (n * dxy)
    img = np.random.default_rng(0).random((n, n))
    u = np.array([0.0, -0.0, 2.0, -3.0, 0.0, n / 2.0, -n / 2.0, n / 2 + 0.5, -(n / 2 + 2.0), 3.0, 3.0, 2.0, 1e-300,
                  n / 2 - 1e-9, 75.3, -140.7]) * du
    v = np.array([0.0, 1.5, 1.0, 4.0, n / 2 - 1.0, 2.5, -1.0, 0.0, 1.0, n / 2 - 0.5, -n / 2 - 0.25, n / 2 - 1.0, -0.0,
                  -n / 2, 99.1, -64.0]) * du
    plan = g.Plan(n)
    for PA, dRA, dDec in ((0.0, 0.0, 0.0), (0.0, 1e-7, 2e-7), (1.1, -3e-7, 1e-7)):
        vis = plan.sampleImage(dev(img), dxy, dev(u), dev(v), PA, dRA, dDec).cpu().numpy()
        oob = plan.last_oob_count()
        ref, ref_oob = orc.sampleImage(img, dxy, u, v, PA, dRA, dDec, return_oob=True)
        assert oob == ref_oob
        assert rel_err(vis, ref) <= TOL_VIS_F64


def test_empty_single_and_ragged_M(g, orc):
    w = W.config(0)
    plan = g.Plan(w.nxy)
    t = dev
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    assert plan.sampleImage(t(w.image), w.dxy, e, e).numel() == 0
    assert float(plan.chi2Image(t(w.image), w.dxy, e, e, e, e, e).cpu()[0]) == 0.0
    for M in (1, 31, 257, 9_999):
        s = slice(0, M)
        vis = plan.sampleImage(t(w.image), w.dxy, t(w.u[s]), t(w.v[s]), w.PA, w.dRA, w.dDec).cpu().numpy()
        ref = orc.sampleImage(w.image, w.dxy, w.u[s], w.v[s], w.PA, w.dRA, w.dDec)
        assert rel_err(vis, ref) <= TOL_VIS_F64
        c = float(plan.chi2Image(t(w.image), w.dxy, t(w.u[s]), t(w.v[s]), t(w.re_obs[s]), t(w.im_obs[s]), t(w.w[s]),
                                 w.dRA, w.dDec, w.PA).cpu()[0])
        r = orc.chi2(ref, w.re_obs[s], w.im_obs[s], w.w[s])
        assert abs(c - r) <= TOL_CHI2_F64 * abs(r)


def test_smallest_and_largest_nxy_end_to_end(g, orc):
    for n, M in ((8, 100), (4096, 1000), (8192, 50_001), (16384, 50_001)):
        rng = np.random.default_rng(n)
        dxy = 0.01 * ARCSEC
        du = 1.0 / (n * dxy)
        img = rng.random((n, n))
        u, v = rng.uniform(-0.45 * n, 0.45 * n, M) * du, rng.uniform(-0.45 * n, 0.45 * n, M) * du
        plan = g.Plan(n)
        vis = plan.sampleImage(dev(img), dxy, dev(u), dev(v), 0.3, 1e-7, 1e-7).cpu().numpy()
        ref = orc.sampleImage(img, dxy, u, v, 0.3, 1e-7, 1e-7, nthreads=threads(orc))
        assert rel_err(vis, ref) <= TOL_VIS_F64
        # chi2 at the same size: observations = the oracle's visibilities + noise, seeded weights
        re_o = ref.real + 1e-3 * rng.standard_normal(M)
        im_o = ref.imag + 1e-3 * rng.standard_normal(M)
        wt = rng.lognormal(np.log(1e6), 0.5, M)
        chi2 = float(plan.chi2Image(dev(img), dxy, dev(u), dev(v), dev(re_o), dev(im_o), dev(wt), 1e-7, 1e-7, 0.3).cpu()[0])
        ref_chi2 = orc.chi2(ref, re_o, im_o, wt)
        assert abs(chi2 - ref_chi2) <= TOL_CHI2_F64 * abs(ref_chi2), n


def test_error_codes(g):
    lib = g.load_library()
    import ctypes
    h = ctypes.c_void_p()
    assert lib.gal_plan_create(ctypes.byref(h), 100, 1, 64, 0) == -1        # not a power of two
    assert lib.gal_plan_create(ctypes.byref(h), 256, 0, 64, 0) == -1        # batch < 1
    assert lib.gal_plan_create(ctypes.byref(h), 256, 1, 16, 0) == -1        # precision
    assert lib.gal_plan_create(ctypes.byref(h), 32768, 1, 64, 0) == -4      # unsupported size
    assert lib.gal_plan_create(None, 256, 1, 64, 0) == -1
    plan = g.Plan(64)
    img = torch.zeros(64, 64, dtype=torch.float64, device="cuda")
    x = torch.zeros(10, dtype=torch.float64, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    f = lib.gal_chi2_image_f64
    ok = (plan._h, img.data_ptr(), 1e-7, x.data_ptr(), x.data_ptr(), x.data_ptr(), x.data_ptr(), x.data_ptr(), 10,
          0.0, 0.0, 0.0, out.data_ptr(), None)
    assert f(*ok) == 0
    bad = lambda i, val: f(*[val if j == i else a for j, a in enumerate(ok)])
    assert bad(1, None) == -1 and bad(3, None) == -1 and bad(7, None) == -1 and bad(12, None) == -1
    assert bad(2, 0.0) == -1 and bad(2, -1.0) == -1 and bad(8, -5) == -1 and bad(9, float("nan")) == -1
    assert lib.gal_chi2_image_f32(*ok) == -1                                 # plan precision mismatch
    # an image or a visibility buffer at an odd element offset is refused, not faulted on
    big = torch.zeros(64 * 64 + 1, dtype=torch.float64, device="cuda")
    assert bad(1, big.data_ptr() + 8) == -1
    vis = torch.zeros(2 * 10 + 1, dtype=torch.float64, device="cuda")
    sa = lib.gal_sample_image_f64
    assert sa(plan._h, img.data_ptr(), 1e-7, x.data_ptr(), x.data_ptr(), 10, 0.0, 0.0, 0.0, vis.data_ptr(), None) == 0
    assert sa(plan._h, img.data_ptr(), 1e-7, x.data_ptr(), x.data_ptr(), 10, 0.0, 0.0, 0.0, vis.data_ptr() + 8, None) == -1
    spec = torch.zeros(2 * 64 * 33 + 1, dtype=torch.float64, device="cuda")
    assert lib.gal_fft2_shifted_f64(plan._h, img.data_ptr(), spec.data_ptr() + 8, None) == -1
    assert lib.gal_fft2_shifted_f64(plan._h, big.data_ptr() + 8, spec.data_ptr(), None) == -1
    prof = torch.ones(10, dtype=torch.float64, device="cuda")
    sw = lib.gal_sweep_f64
    assert sw(plan._h, prof.data_ptr(), 10, 0.0, 1e-7, 1e-7, 0.0, img.data_ptr(), None) == 0
    assert sw(plan._h, prof.data_ptr(), 1, 0.0, 1e-7, 1e-7, 0.0, img.data_ptr(), None) == -1     # nr < 2
    assert sw(plan._h, prof.data_ptr(), 10, 0.0, 0.0, 1e-7, 0.0, img.data_ptr(), None) == -1     # dR <= 0
    assert sw(plan._h, prof.data_ptr(), 10, 0.0, 1e-7, 1e-7, 1.6, img.data_ptr(), None) == -1    # |inc| >= pi/2
    with pytest.raises(g.GalarioError):
        g.Plan(64, 2).chi2ImageBatch(torch.zeros(3, 64, 64, dtype=torch.float64, device="cuda"), 1e-7,
                                     torch.zeros(3, 4, dtype=torch.float64, device="cuda"),
                                     torch.zeros(3, 4, dtype=torch.float64, device="cuda"),
                                     torch.zeros(3, 4, dtype=torch.float64, device="cuda"),
                                     torch.zeros(3, 4, dtype=torch.float64, device="cuda"),
                                     torch.zeros(3, 4, dtype=torch.float64, device="cuda"))       # C > plan batch
    torch.cuda.synchronize()


def test_host_pointer_calls_match_device_calls(g, orc):
    w = W.config(0)
    plan = g.Plan(w.nxy)
    c_host = plan.chi2Image_host(w.image, w.dxy, w.u, w.v, w.re_obs, w.im_obs, w.w, w.dRA, w.dDec, w.PA)
    c_dev = float(plan.chi2Image(dev(w.image), w.dxy, dev(w.u), dev(w.v), dev(w.re_obs), dev(w.im_obs), dev(w.w),
                                 w.dRA, w.dDec, w.PA).cpu()[0])
    assert c_host == c_dev
    v_host = plan.sampleImage_host(w.image, w.dxy, w.u, w.v, w.PA, w.dRA, w.dDec)
    v_dev = plan.sampleImage(dev(w.image), w.dxy, dev(w.u), dev(w.v), w.PA, w.dRA, w.dDec).cpu().numpy()
    assert np.array_equal(v_host, v_dev)
    w1 = W.config(1, nxy=256, M=5000, nr=500)
    p1 = g.Plan(w1.nxy)
    ch = p1.chi2Profile_host(w1.profile, w1.Rmin, w1.dR, w1.dxy, w1.u, w1.v, w1.re_obs, w1.im_obs, w1.w, 0.0, 0.0,
                             w1.PA, w1.inc)
    r = orc.chi2Profile(w1.profile, w1.Rmin, w1.dR, w1.nxy, w1.dxy, w1.u, w1.v, w1.re_obs, w1.im_obs, w1.w, 0.0, 0.0,
                        w1.PA, w1.inc)
    assert abs(ch - r) <= TOL_CHI2_F64 * abs(r)
    vp_host = p1.sampleProfile_host(w1.profile, w1.Rmin, w1.dR, w1.dxy, w1.u, w1.v, w1.inc, w1.PA, 1e-7, -2e-7)
    vp_dev = p1.sampleProfile(dev(w1.profile), w1.Rmin, w1.dR, w1.dxy, dev(w1.u), dev(w1.v), w1.inc, w1.PA, 1e-7, -2e-7)
    assert np.array_equal(vp_host, vp_dev.cpu().numpy())
    with pytest.raises(g.GalarioError):
        p1.sampleProfile_host(w1.profile, w1.Rmin, w1.dR, w1.dxy, w1.u, w1.v[:-1])
    # the single-precision library offers the same calls
    wf, w1f = w.as_f32(), w1.as_f32()
    q, q1 = g.Plan(w.nxy, 1, torch.float32), g.Plan(w1.nxy, 1, torch.float32)
    vh = q.sampleImage_host(wf.image, w.dxy, wf.u, wf.v, w.PA, w.dRA, w.dDec)
    vd = q.sampleImage(dev(wf.image), w.dxy, dev(wf.u), dev(wf.v), w.PA, w.dRA, w.dDec).cpu().numpy()
    assert vh.dtype == np.complex64 and np.array_equal(vh, vd)
    ch32 = q1.chi2Profile_host(w1f.profile, w1.Rmin, w1.dR, w1.dxy, w1f.u, w1f.v, w1f.re_obs, w1f.im_obs, w1f.w, 0.0, 0.0,
                               w1.PA, w1.inc)
    cd32 = float(q1.chi2Profile(dev(w1f.profile), w1.Rmin, w1.dR, w1.dxy, dev(w1f.u), dev(w1f.v), dev(w1f.re_obs),
                                dev(w1f.im_obs), dev(w1f.w), 0.0, 0.0, w1.PA, w1.inc).cpu()[0])
    assert ch32 == cd32 and abs(ch32 - r) <= TOL_CHI2_F32 * abs(r)
    vph = q1.sampleProfile_host(w1f.profile, w1.Rmin, w1.dR, w1.dxy, w1f.u, w1f.v, w1.inc, w1.PA)
    vpd = q1.sampleProfile(dev(w1f.profile), w1.Rmin, w1.dR, w1.dxy, dev(w1f.u), dev(w1f.v), w1.inc, w1.PA).cpu().numpy()
    assert np.array_equal(vph, vpd)


def test_paper_style_module_calls(g, orc):
    w = W.config(0)
    vis = g.sampleImage(dev(w.image), w.dxy, dev(w.u), dev(w.v), PA=w.PA, dRA=w.dRA, dDec=w.dDec).cpu().numpy()
    ref = orc.sampleImage(w.image, w.dxy, w.u, w.v, PA=w.PA, dRA=w.dRA, dDec=w.dDec)
    assert rel_err(vis, ref) <= TOL_VIS_F64
    c = g.chi2Image(dev(w.image), w.dxy, dev(w.u), dev(w.v), dev(w.re_obs), dev(w.im_obs), dev(w.w), w.dRA, w.dDec, w.PA)
    r = orc.chi2(ref, w.re_obs, w.im_obs, w.w)
    assert abs(float(c.cpu()[0]) - r) <= TOL_CHI2_F64 * abs(r)


def test_binding_rejects_short_arrays_and_wrong_outputs(g):
    """The multi-source and direct-Hankel methods of the binding check what they hand to the C ABI (a short array or a
    wrong-typed output would be an out-of-bounds device access), and a NaN coordinate cannot be bound."""
    w = W.config(1, nxy=64, M=500, nr=100)
    plan = g.Plan(64)
    img = torch.zeros(64, 64, dtype=torch.float64, device="cuda")
    prof, u, v, re, im, wt = (dev(a) for a in (w.profile, w.u, w.v, w.re_obs, w.im_obs, w.w))
    pl = [(0.0, 0.0, 0.0), (1e-7, 0.0, 0.3, 0.5)]
    bad_out = torch.empty(500, dtype=torch.complex64, device="cuda")
    for call in (lambda: plan.sampleImageMulti(img, w.dxy, u, v[:-1], pl),
                 lambda: plan.sampleImageMulti(img, w.dxy, u, v, pl, out=bad_out),
                 lambda: plan.sampleImageMulti(img[:32], w.dxy, u, v, pl),
                 lambda: plan.chi2ImageMulti(img, w.dxy, u, v, re, im[:-3], wt, pl),
                 lambda: plan.chi2ImageMulti(img, w.dxy, u, v, re, im, wt, pl, out=torch.empty(1, device="cuda")),
                 lambda: plan.sampleProfileHankel(prof, w.Rmin, w.dR, u, v[:10]),
                 lambda: plan.sampleProfileHankel(prof, w.Rmin, w.dR, u, v, out=bad_out),
                 lambda: plan.chi2ProfileHankel(prof, w.Rmin, w.dR, u, v, re, im, wt[:-1]),
                 lambda: plan.chi2ProfileHankel(prof, w.Rmin, w.dR, u, v, re, im, wt, out=torch.empty(2, dtype=torch.float64, device="cuda")),
                 lambda: plan.bind_uv(u, v[:-1])):
        with pytest.raises(g.GalarioError):
            call()
    assert plan.sampleImageMulti(img, w.dxy, u, v, pl).shape == (500,)       # and the good calls still go through
    un = u.clone()
    un[17] = float("nan")
    with pytest.raises(g.GalarioError):
        plan.bind_uv(un, v)                                  # the radius reduction must not drop a NaN
    with pytest.raises(g.GalarioError):
        plan.bind_obs(u, un, re, im, wt)
    plan.bind_uv(u, v)
    plan.unbind_uv()
    plan.set_option("batch_conc", 4)
    with pytest.raises(g.GalarioError):
        plan.set_option("no_such_option", 1)
    with pytest.raises(g.GalarioError):
        plan.set_option("row_mode", 9)


# ---------------------------------------------------------------------------------------------
# K observation sets against one model image in one call (second alternative)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype,M", [(torch.float64, 40_004), (torch.float64, 40_003), (torch.float32, 40_004)])
def test_observation_sets_against_one_image(g, orc, dtype, M):
    """gal_chi2_image_sets: ONE transform, grid.y over the sets.  Every set's chi2, the total, the out-of-grid count
    against the oracle's loop over chi2Image; sets of different reach (one of them beyond the grid), data and weights;
    16-byte aligned rows (TMA path, M = 40 004) and ragged ones (plain loads); pruned to the union of the extents."""
    f32 = dtype == torch.float32
    w = W.config(3, nxy=1024, M=M, n_src=40)
    if f32:
        w = w.as_f32()
    tol = TOL_CHI2_F32 if f32 else TOL_CHI2_F64
    f = lambda a: np.asarray(a, dtype=np.float64)
    K = 4
    for scales, mode in (((0.9, 0.7, 0.5, 0.3), 2), ((1.0, 0.5, 3.0, 0.7), 1), ((0.9, 0.7, 0.5, 0.3), 0)):
        st = lambda a, sc=False: np.ascontiguousarray(np.stack(
            [np.roll(a, 997 * k) * (a.dtype.type(scales[k]) if sc else a.dtype.type(1)) for k in range(K)]))
        u, v, ro, io, wt = st(w.u, True), st(w.v, True), st(w.re_obs), st(w.im_obs), st(w.w)
        wt = np.ascontiguousarray(wt * np.arange(1, K + 1, dtype=wt.dtype)[:, None])
        plan = g.Plan(w.nxy, K, dtype)
        plan.set_pruning(mode)
        n0 = plan.launch_count()
        per, tot = plan.chi2ImageSets(dev(w.image), w.dxy, dev(u), dev(v), dev(ro), dev(io), dev(wt), w.dRA, w.dDec, w.PA)
        per, tot = per.cpu().numpy(), float(tot.cpu()[0])
        assert plan.launch_count() - n0 <= 4                  # [extent,] one transform (1-2 kernels), ONE sampling launch
        rper, rtot, roob = orc.chi2ImageSets(f(w.image), w.dxy, f(u), f(v), f(ro), f(io), f(wt), w.dRA, w.dDec, w.PA,
                                             nthreads=threads(orc), return_oob=True)
        assert (np.abs(per - rper) <= tol * np.abs(rper)).all(), (scales, mode)
        assert abs(tot - rtot) <= tol * abs(rtot)
        assert plan.last_oob_count() == roob and (roob > 0) == (max(scales) > 0.95)   # (longest baseline: 548 of 512 cells)
        ext = plan.last_uv_extent()
        if mode == 2:
            assert ext[0] < w.nxy // 2                        # pruned to the union of the sets' extents
        # each set alone through the single-set call: the same numbers to rounding (other partial-sum grouping)
        one = g.Plan(w.nxy, 1, dtype)
        for k in (0, K - 1):
            c = float(one.chi2Image(dev(w.image), w.dxy, dev(u[k]), dev(v[k]), dev(ro[k]), dev(io[k]), dev(wt[k]),
                                    w.dRA, w.dDec, w.PA).cpu()[0])
            assert abs(c - per[k]) <= (1e-5 if f32 else 1e-12) * abs(c)
    with pytest.raises(g.GalarioError):
        g.Plan(w.nxy, 2, dtype).chi2ImageSets(dev(w.image), w.dxy, dev(u), dev(v), dev(ro), dev(io), dev(wt))   # K > plan batch


def test_two_hundred_mixed_calls_on_one_plan_against_the_oracle(g, orc):
    """Stand-in for the sanitizer pass this pool does not allow: 200 calls on ONE plan in a
    seeded random order — chi2Image and sampleImage, six uv sets of two lengths (ragged and 16-byte aligned) and four
    reaches (so the speculative extent shrinks, grows, fails and repeats itself on the device, and wraps to the whole
    plane), bound observation sets coming and going — issued in bursts of 20 without host synchronisation, every
    result compared with the oracle's for that uv set.  State leaking from one call into the next (tickets, the
    alternating call state, extents, the second pass's counters) would show as a wrong number."""
    w = W.config(3, nxy=2048, M=120_000, n_src=40)
    f = lambda a: np.asarray(a, dtype=np.float64)
    image = dev(w.image)
    variants = []
    for M, scale in ((120_000, 1.0), (50_001, 0.5), (120_000, 1.8), (50_001, 2.5), (120_000, 0.3), (50_001, 1.0)):
        u, v = w.u[:M] * scale, w.v[:M] * scale
        ro, io, wt = w.re_obs[:M], w.im_obs[:M], w.w[:M]
        vis, oob = orc.sampleImage(f(w.image), w.dxy, u, v, w.PA, w.dRA, w.dDec, return_oob=True, nthreads=threads(orc))
        variants.append(dict(d=[dev(a) for a in (u, v, ro, io, wt)], vis=vis, chi2=orc.chi2(vis, ro, io, wt), oob=oob))
    assert any(x["oob"] > 0 for x in variants) and any(x["oob"] == 0 for x in variants)
    plan = g.Plan(w.nxy)
    plan.set_option("spec_min_bytes", 0)
    rng = np.random.default_rng(2024)
    n_calls, n_bound = 0, 0
    for burst in range(10):
        issued = []
        bind_k = int(rng.integers(len(variants))) if burst % 3 == 2 else None
        if bind_k is not None:
            plan.bind_obs(*variants[bind_k]["d"])
        for _ in range(20):
            k = int(rng.integers(len(variants)))
            x = variants[k]
            if rng.random() < 0.3:
                issued.append((k, "vis", plan.sampleImage(image, w.dxy, x["d"][0], x["d"][1], w.PA, w.dRA, w.dDec)))
            else:
                issued.append((k, "chi2", plan.chi2Image(image, w.dxy, *x["d"], w.dRA, w.dDec, w.PA)))
                n_bound += bind_k == k
            n_calls += 1
        torch.cuda.synchronize()
        assert plan.last_oob_count() == variants[issued[-1][0]]["oob"]
        for k, what, out in issued:
            x = variants[k]
            if what == "vis":
                assert rel_err(out.cpu().numpy(), x["vis"]) <= TOL_VIS_F64, (burst, k)
            else:
                assert abs(float(out.cpu()[0]) - x["chi2"]) <= TOL_CHI2_F64 * abs(x["chi2"]), (burst, k)
        if bind_k is not None:
            plan.unbind_obs()
    assert n_calls == 200 and n_bound > 0
