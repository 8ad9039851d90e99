"""Pins of the CPU oracle against things other than itself (run with -m "not gpu").

The paper prints no numeric visibility or chi-square anywhere, so the pins are:
brute-force evaluation of the sky-coordinate Fourier sum (no FFT, no abs/conj fold), the
paper's own Appendix-D listing re-run on numpy.fft + scipy, closed forms
(point source, Gaussian), symmetries (Hermitian, Parseval, PA = 90/180 deg, image roll ==
phase ramp) and scipy.interp1d for the sweep.  Each is chosen so that a dropped term, a wrong
sign or index, or a transposed operand in oracle/galario_oracle.cpp fails at least one.
"""
import numpy as np
import pytest
from scipy.interpolate import RectBivariateSpline, interp1d

ARCSEC = np.pi / 648000.0


# ---------------------------------------------------------------------------------------
# independent restatements used as pins
# ---------------------------------------------------------------------------------------
def brute_node(image, dxy, ku, kv):
    """sum_ij A[i][j] exp(+2 pi i (ku du l_j + kv du m_i)) for ANY integers ku, kv (reading A1).
    No FFT, no shift, no Hermitian fold: periodicity and symmetry come out of the sum itself."""
    n = image.shape[0]
    lj = (n // 2 - np.arange(n))          # in pixels; du * dxy = 1/n
    mi = (n // 2 - np.arange(n))
    ph_l = np.exp(2j * np.pi * ku * lj / n)
    ph_m = np.exp(2j * np.pi * kv * mi / n)
    return ph_m @ image @ ph_l


def brute_sample(image, dxy, u, v, dRA, dDec, PA):
    """Bilinear interpolation of the FULL periodic plane of brute_node at the rotated point,
    times exp(+2 pi i (u dRA + v dDec)).  No abs(u), no conjugation branch."""
    n = image.shape[0]
    du = 1.0 / (n * dxy)
    out = np.empty(u.size, dtype=complex)
    c, s = np.cos(PA), np.sin(PA)
    cache = {}

    def node(ku, kv):
        if (ku, kv) not in cache:
            cache[(ku, kv)] = brute_node(image, dxy, ku, kv)
        return cache[(ku, kv)]

    for k in range(u.size):
        ur, vr = u[k] * c - v[k] * s, u[k] * s + v[k] * c
        x, y = ur / du, vr / du
        ix, iy = int(np.floor(x)), int(np.floor(y))
        tx, ty = x - ix, y - iy
        val = ((1 - ty) * ((1 - tx) * node(ix, iy) + tx * node(ix + 1, iy)) +
               ty * ((1 - tx) * node(ix, iy + 1) + tx * node(ix + 1, iy + 1)))
        out[k] = val * np.exp(2j * np.pi * (u[k] * dRA + v[k] * dDec))
    return out


def listing_chi2Image(image, dxy, u, v, vis_obs_re, vis_obs_im, weights, dRA=0., dDec=0., PA=0.):
    """The paper's py_chi2Image with the OCR damage repaired as in DESIGN.md
    reading A4; library routines do the work (numpy.fft, scipy RectBivariateSpline)."""
    nxy = image.shape[0]
    dRA = dRA * 2. * np.pi
    dDec = dDec * 2. * np.pi
    du = 1. / (nxy * dxy)
    fft_r2c_shifted = np.fft.fftshift(np.fft.rfft2(np.fft.fftshift(image)), axes=0)
    cos_PA, sin_PA = np.cos(PA), np.sin(PA)
    urot = u * cos_PA - v * sin_PA
    vrot = u * sin_PA + v * cos_PA
    dRArot = dRA * cos_PA - dDec * sin_PA
    dDecrot = dRA * sin_PA + dDec * cos_PA
    urot_idx = np.abs(urot) / du
    vrot_idx = nxy / 2. + vrot / du
    uneg = urot < 0.
    vrot_idx[uneg] = nxy / 2 - vrot[uneg] / du
    u_axis = np.linspace(0., nxy // 2, nxy // 2 + 1)
    v_axis = np.linspace(0., nxy - 1, nxy)
    f_re = RectBivariateSpline(v_axis, u_axis, fft_r2c_shifted.real, kx=1, ky=1, s=0)
    ReInt = f_re.ev(vrot_idx, urot_idx)
    f_im = RectBivariateSpline(v_axis, u_axis, fft_r2c_shifted.imag, kx=1, ky=1, s=0)
    ImInt = f_im.ev(vrot_idx, urot_idx)
    ImInt[uneg] *= -1.
    theta = urot * dRArot + vrot * dDecrot
    vis = (ReInt + 1j * ImInt) * (np.cos(theta) + 1j * np.sin(theta))
    chi2 = np.sum(((vis.real - vis_obs_re) ** 2. + (vis.imag - vis_obs_im) ** 2.) * weights)
    return chi2, vis


def listing_sweep(intensity, Rmin, dR, nxy, dxy, inc=0.):
    """Image stage of the paper's py_chi2Profile, on scipy.interp1d."""
    inc_cos = np.cos(inc)
    nrad = len(intensity)
    gridrad = np.linspace(Rmin, Rmin + dR * (nrad - 1), nrad)
    ncol, nrow = nxy, nxy
    x = (np.linspace(0.5, -0.5 + 1. / float(ncol), ncol)) * dxy * ncol
    y = (np.linspace(0.5, -0.5 + 1. / float(nrow), nrow)) * dxy * nrow
    x_axis, y_axis = np.meshgrid(x / inc_cos, y)
    x_meshgrid = np.sqrt(x_axis ** 2. + y_axis ** 2.)
    intensity = intensity * dxy ** 2.
    f = interp1d(gridrad, intensity, kind='linear', fill_value=0., bounds_error=False, assume_sorted=True)
    return f(x_meshgrid)


def in_range_uv(rng, M, n, dxy, frac=0.45):
    """Points whose rotated index stays inside the half-plane grid for any PA."""
    du = 1.0 / (n * dxy)
    q = rng.uniform(0.0, frac * n, M) * du
    az = rng.uniform(0, 2 * np.pi, M)
    return q * np.cos(az), q * np.sin(az)


# ---------------------------------------------------------------------------------------
# O2+O3+O4: spectrum
# ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [8, 16, 30, 64, 128, 256])
def test_spectrum_nodes_vs_brute_force(orc, n):
    rng = np.random.default_rng(n)
    img = rng.standard_normal((n, n))
    G = orc.spectrum(img)
    assert G.shape == (n, n // 2 + 1)
    peak = np.abs(G).max()
    nodes = [(ku, kvs) for ku in range(n // 2 + 1) for kvs in range(n)]
    if len(nodes) > 400:
        pick = rng.choice(len(nodes), 400, replace=False)
        nodes = [nodes[p] for p in pick] + [(0, 0), (n // 2, 0), (0, n - 1), (n // 2, n // 2), (1, n // 2 + 1)]
    for ku, kvs in nodes:
        ref = brute_node(img, 1.0, ku, kvs - n // 2)
        assert abs(G[kvs, ku] - ref) <= 1e-12 * peak, (ku, kvs)


@pytest.mark.parametrize("n", [16, 64, 128, 512])
def test_spectrum_vs_numpy_listing_line(orc, n):
    """PAPER.md:659 verbatim on numpy (library routine) — covers direct-DFT and radix-2 paths."""
    img = np.random.default_rng(7 + n).random((n, n))
    ref = np.fft.fftshift(np.fft.rfft2(np.fft.fftshift(img)), axes=0)
    G = orc.spectrum(img)
    assert np.abs(G - ref).max() <= 1e-12 * np.abs(ref).max()
    Gl = orc.spectrum(img, long_double=True)
    assert np.abs(G - Gl).max() <= 1e-12 * np.abs(ref).max()
    Gt = orc.spectrum(img, nthreads=3)
    assert np.array_equal(G, Gt)


@pytest.mark.parametrize("n", [32, 256])
def test_parseval_half_plane(orc, n):
    img = np.random.default_rng(3).standard_normal((n, n))
    G = orc.spectrum(img)
    wgt = np.full(n // 2 + 1, 2.0)
    wgt[0] = wgt[-1] = 1.0
    lhs = (np.abs(G) ** 2 * wgt[None, :]).sum() / n ** 2
    assert lhs == pytest.approx((img ** 2).sum(), rel=1e-12)


@pytest.mark.parametrize("n", [32, 128])
def test_delta_offset_gives_plane_wave_nodes(orc, n):
    """Delta at [n/2 - b][n/2 - a] (a px East, b px North) -> G = exp(+2 pi i (ku a + kv b)/n)."""
    a, b = 3, -5
    img = np.zeros((n, n))
    img[n // 2 - b, n // 2 - a] = 1.0
    G = orc.spectrum(img)
    ku = np.arange(n // 2 + 1)[None, :]
    kv = (np.arange(n) - n // 2)[:, None]
    ref = np.exp(2j * np.pi * (ku * a + kv * b) / n)
    assert np.abs(G - ref).max() <= 1e-12


def test_centred_gaussian_nodes_closed_form(orc):
    """Elliptical Gaussian (flux F) centred on [n/2][n/2]: node values F exp(-2 pi^2 (sl^2 u^2 + sm^2 v^2)),
    purely real.  Catches a swapped axis (sl != sm) and any stray sign/shift (imaginary part)."""
    n, dxy, F = 256, 0.02 * ARCSEC, 1.7
    sl, sm = 3.0 * dxy, 5.5 * dxy
    c = (n // 2 - np.arange(n)) * dxy
    img = np.exp(-0.5 * ((c[None, :] / sl) ** 2 + (c[:, None] / sm) ** 2)) * (F * dxy ** 2 / (2 * np.pi * sl * sm))
    G = orc.spectrum(img)
    du = 1.0 / (n * dxy)
    uu = np.arange(n // 2 + 1)[None, :] * du
    vv = (np.arange(n) - n // 2)[:, None] * du
    ref = F * np.exp(-2 * np.pi ** 2 * (sl ** 2 * uu ** 2 + sm ** 2 * vv ** 2))
    assert np.abs(G - ref).max() <= 1e-12 * F


# ---------------------------------------------------------------------------------------
# O5+O6+O7: sampling
# ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,PA,dRA,dDec", [(16, 0.0, 0.0, 0.0), (16, 0.7, 0.3, -0.2), (32, 2.1, -1.3, 0.9),
                                           (30, -0.4, 0.25, 0.5)])
def test_sample_vs_brute_force_full_plane(orc, n, PA, dRA, dDec):
    """End-to-end pin at nxy <= 64, including points beyond the half-plane grid (reading A6),
    exact-node points, u' = 0 and the top row."""
    rng = np.random.default_rng(100 + n)
    dxy = 0.05 * ARCSEC
    du = 1.0 / (n * dxy)
    img = rng.random((n, n))
    u = rng.uniform(-0.9 * n, 0.9 * n, 60) * du
    v = rng.uniform(-0.9 * n, 0.9 * n, 60) * du
    u[:6] = np.array([0.0, 2.0, -3.0, 0.0, n / 2.0, -n / 2.0]) * du
    v[:6] = np.array([0.0, 1.0, 4.0, (n / 2 - 1.0), 2.5, -1.0]) * du
    dRA, dDec = dRA * dxy * 3, dDec * dxy * 3
    vis = orc.sampleImage(img, dxy, u, v, PA=PA, dRA=dRA, dDec=dDec)
    ref = brute_sample(img, dxy, u, v, dRA, dDec, PA)
    peak = np.abs(ref).max()
    assert np.abs(vis - ref).max() <= 1e-12 * peak
    visl = orc.sampleImage(img, dxy, u, v, PA=PA, dRA=dRA, dDec=dDec, long_double=True)
    assert np.abs(visl - ref).max() <= 1e-12 * peak


@pytest.mark.parametrize("n", [64, 128, 256])
def test_chi2Image_vs_appendix_D_listing(orc, n):
    rng = np.random.default_rng(n)
    dxy = 0.01 * ARCSEC
    img = rng.random((n, n)) ** 3
    M = 3000
    u, v = in_range_uv(rng, M, n, dxy)
    u[0], v[0] = 0.0, 0.0
    ro, io, w = rng.standard_normal(M), rng.standard_normal(M), rng.uniform(0.5, 2.0, M)
    dRA, dDec, PA = 0.31 * ARCSEC, -0.17 * ARCSEC, 0.83
    chi2_ref, vis_ref = listing_chi2Image(img, dxy, u, v, ro, io, w, dRA, dDec, PA)
    vis, oob = orc.sampleImage(img, dxy, u, v, PA=PA, dRA=dRA, dDec=dDec, return_oob=True)
    assert oob == 0
    assert np.abs(vis - vis_ref).max() <= 1e-12 * np.abs(vis_ref).max()
    assert orc.chi2Image(img, dxy, u, v, ro, io, w, dRA, dDec, PA) == pytest.approx(chi2_ref, rel=1e-12)
    assert orc.chi2Image(img, dxy, u, v, ro, io, w, dRA, dDec, PA, nthreads=4) == pytest.approx(chi2_ref, rel=1e-12)
    assert np.array_equal(orc.sampleImage(img, dxy, u, v, PA=PA, dRA=dRA, dDec=dDec, nthreads=4), vis)


def test_point_source_unit_amplitude_linear_phase(orc):
    """Delta at the centre pixel: V = exp(+2 pi i (u dRA + v dDec)) for any PA."""
    n, dxy = 128, 0.01 * ARCSEC
    img = np.zeros((n, n))
    img[n // 2, n // 2] = 1.0
    rng = np.random.default_rng(5)
    u, v = in_range_uv(rng, 2000, n, dxy)
    dRA, dDec = 0.4 * ARCSEC, -0.25 * ARCSEC
    for PA in (0.0, 0.5, 2.0):
        vis = orc.sampleImage(img, dxy, u, v, PA=PA, dRA=dRA, dDec=dDec)
        ref = np.exp(2j * np.pi * (u * dRA + v * dDec))
        assert np.abs(vis - ref).max() <= 1e-13


def test_image_roll_equals_phase_ramp_at_nodes(orc):
    """Moving the image a px East and b px North == dRA = a dxy, dDec = b dxy, exactly at nodes."""
    n, dxy = 64, 0.02 * ARCSEC
    rng = np.random.default_rng(11)
    img = np.zeros((n, n))
    img[20:44, 20:44] = rng.random((24, 24))
    a, b = 4, -6
    rolled = np.roll(np.roll(img, -a, axis=1), -b, axis=0)     # col j -> j - a (East), row i -> i - b (North)
    du = 1.0 / (n * dxy)
    ku, kv = np.meshgrid(np.arange(-n // 4, n // 4), np.arange(-n // 4, n // 4))
    u, v = (ku.ravel() * du).astype(float), (kv.ravel() * du).astype(float)
    v1 = orc.sampleImage(rolled, dxy, u, v)
    v2 = orc.sampleImage(img, dxy, u, v, dRA=a * dxy, dDec=b * dxy)
    assert np.abs(v1 - v2).max() <= 1e-12 * np.abs(v1).max()


def test_hermitian_symmetry(orc):
    n, dxy = 128, 0.01 * ARCSEC
    rng = np.random.default_rng(2)
    img = rng.random((n, n))
    u, v = in_range_uv(rng, 1000, n, dxy)
    kw = dict(PA=0.6, dRA=0.2 * ARCSEC, dDec=0.1 * ARCSEC)
    a = orc.sampleImage(img, dxy, u, v, **kw)
    b = orc.sampleImage(img, dxy, -u, -v, **kw)
    assert np.abs(a - np.conj(b)).max() <= 1e-13 * np.abs(a).max()


def test_PA_90_and_180_identities(orc):
    """PA = 90 deg == sampling A_rot[i][j] = A[j][(n - i) % n] with PA = 0 (reading A3);
    PA = 180 deg with no offsets == complex conjugate of PA = 0."""
    n, dxy = 64, 0.02 * ARCSEC
    rng = np.random.default_rng(9)
    img = rng.random((n, n))
    u, v = in_range_uv(rng, 500, n, dxy, frac=0.3)
    i, j = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    rot = img[j, (n - i) % n]
    a = orc.sampleImage(img, dxy, u, v, PA=np.pi / 2)
    b = orc.sampleImage(rot, dxy, u, v, PA=0.0)
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    c = orc.sampleImage(img, dxy, u, v, PA=np.pi)
    d = orc.sampleImage(img, dxy, u, v, PA=0.0)
    assert np.abs(c - np.conj(d)).max() <= 1e-12 * np.abs(d).max()


def test_offnode_gaussian_within_bilinear_bound(orc):
    """Off-node values of a centred Gaussian stay within du^2/8 (|V_uu| + |V_vv|)_max of the closed form."""
    n, dxy = 256, 0.02 * ARCSEC
    sl, sm = 4.0 * dxy, 6.0 * dxy
    c = (n // 2 - np.arange(n)) * dxy
    img = np.exp(-0.5 * ((c[None, :] / sl) ** 2 + (c[:, None] / sm) ** 2)) * (dxy ** 2 / (2 * np.pi * sl * sm))
    rng = np.random.default_rng(1)
    u, v = in_range_uv(rng, 4000, n, dxy, frac=0.3)
    vis = orc.sampleImage(img, dxy, u, v)
    ref = np.exp(-2 * np.pi ** 2 * (sl ** 2 * u ** 2 + sm ** 2 * v ** 2))
    du = 1.0 / (n * dxy)
    bound = du ** 2 / 8 * 4 * np.pi ** 2 * (sl ** 2 + sm ** 2)
    err = np.abs(vis - ref).max()
    assert 1e-6 < err <= bound * 1.01        # it IS an approximation, and it obeys the bound
    assert np.abs(vis.imag).max() <= 1e-14


def test_oob_count_and_wrap(orc):
    n, dxy = 32, 0.05 * ARCSEC
    du = 1.0 / (n * dxy)
    img = np.random.default_rng(0).random((n, n))
    u = np.array([1.5, n / 2 + 0.5, -(n / 2 + 2.0), 3.0, 3.0, 2.0]) * du
    v = np.array([2.0, 0.0, 1.0, n / 2 - 0.5, -n / 2 - 0.25, n / 2 - 1.0]) * du
    vis, oob = orc.sampleImage(img, dxy, u, v, return_oob=True)
    assert oob == 4
    assert np.abs(vis - brute_sample(img, dxy, u, v, 0, 0, 0)).max() <= 1e-12 * np.abs(vis).max()


# ---------------------------------------------------------------------------------------
# O1: sweep
# ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("inc", [0.0, 0.6, np.deg2rad(45.0)])
def test_sweep_vs_listing_interp1d(orc, inc):
    n, dxy = 96, 0.03 * ARCSEC
    nr, Rmin, dR = 300, 1e-3 * ARCSEC, 4e-3 * ARCSEC      # Rmax = 1.197" < half field 1.44": hard edge inside
    R = Rmin + dR * np.arange(nr)
    I = (R / ARCSEC + 0.05) ** -0.7 * np.exp(-R / ARCSEC) * 1e10
    img = orc.sweep(I, Rmin, dR, n, dxy, inc)
    ref = listing_sweep(I, Rmin, dR, n, dxy, inc)
    assert img[n // 2, n // 2] == 0.0 and ref[n // 2, n // 2] == 0.0          # r = 0 < Rmin (reading A5)
    assert (ref == 0).sum() > n and np.array_equal(img == 0, ref == 0)          # same support (hard edge)
    assert np.abs(img - ref).max() <= 1e-13 * ref.max()


def test_sweep_edges_and_inclination_stretch(orc):
    n, dxy = 64, 0.01 * ARCSEC
    nr = 17
    dR = dxy            # Rmax = 16 px exactly on a pixel centre along the North-South axis
    I = np.linspace(2.0, 1.0, nr)
    img = orc.sweep(I, 0.0, dR, n, dxy, 0.0)
    assert img[n // 2, n // 2] == pytest.approx(2.0 * dxy ** 2, rel=1e-15)   # Rmin = 0: centre = I[0] dxy^2
    assert img[n // 2 - 16, n // 2] == pytest.approx(1.0 * dxy ** 2, rel=1e-12)   # r == Rmax inclusive
    assert img[n // 2 - 17, n // 2] == 0.0
    assert img[n // 2 - 3, n // 2] == pytest.approx(I[3] * dxy ** 2, rel=1e-12)   # North
    assert img[n // 2, n // 2 - 3] == pytest.approx(I[3] * dxy ** 2, rel=1e-12)   # East, face-on: symmetric
    inc = np.deg2rad(60.0)         # cos = 0.5: East-West compressed by 2, no flux factor (reading A9)
    img2 = orc.sweep(I, 0.0, dR, n, dxy, inc)
    assert img2[n // 2, n // 2 - 3] == pytest.approx(I[6] * dxy ** 2, rel=1e-9)
    assert img2[n // 2 - 3, n // 2] == pytest.approx(I[3] * dxy ** 2, rel=1e-12)


def test_sampleProfile_is_sampleImage_of_sweep(orc):
    """identical 'at machine precision' — here bit for bit."""
    rng = np.random.default_rng(4)
    n, dxy = 128, 0.02 * ARCSEC
    nr, Rmin, dR = 200, 1e-4 * ARCSEC, 5e-3 * ARCSEC
    I = rng.random(nr) * 1e10
    u, v = in_range_uv(rng, 500, n, dxy)
    kw = dict(PA=0.3, dRA=0.1 * ARCSEC, dDec=-0.2 * ARCSEC)
    a = orc.sampleProfile(I, Rmin, dR, n, dxy, u, v, inc=0.5, **kw)
    b = orc.sampleImage(orc.sweep(I, Rmin, dR, n, dxy, 0.5), dxy, u, v, **kw)
    assert np.array_equal(a, b)
    ro, io, w = rng.standard_normal(500), rng.standard_normal(500), rng.random(500)
    c1 = orc.chi2Profile(I, Rmin, dR, n, dxy, u, v, ro, io, w, inc=0.5, **kw)
    assert c1 == orc.chi2(a, ro, io, w)


def test_gaussian_profile_vs_hankel_closed_form(orc):
    """E1: face-on Gaussian profile exp(-r^2/2s^2) -> V = 2 pi s^2 exp(-2 pi^2 s^2 rho^2).
    A sanity bound (the profile is linearly interpolated), at the paper's quoted 1e-5 level."""
    n, dxy = 512, 0.01 * ARCSEC
    s = 0.25 * ARCSEC
    dR = dxy / 10
    nr = int(2.5 * ARCSEC / dR)
    R = dR * np.arange(nr)
    I = np.exp(-0.5 * (R / s) ** 2)
    du = 1.0 / (n * dxy)
    ku, kv = np.meshgrid(np.arange(0, 40, 3), np.arange(-40, 40, 7))
    u, v = ku.ravel() * du, kv.ravel() * du
    vis = orc.sampleProfile(I, 0.0, dR, n, dxy, u, v)
    ref = 2 * np.pi * s ** 2 * np.exp(-2 * np.pi ** 2 * s ** 2 * (u ** 2 + v ** 2))
    assert np.abs(vis - ref).max() <= 1e-5 * ref.max()
    assert np.abs(vis.imag).max() <= 1e-12 * ref.max()


# ---------------------------------------------------------------------------------------
# O8: chi2
# ---------------------------------------------------------------------------------------
def test_chi2_invariants(orc):
    rng = np.random.default_rng(8)
    M = 10001
    vis = rng.standard_normal(M) + 1j * rng.standard_normal(M)
    w = rng.uniform(0.1, 3.0, M)
    assert orc.chi2(vis, vis.real, vis.imag, w) == 0.0
    assert orc.chi2(vis, np.zeros(M), np.zeros(M), w) == pytest.approx(float(np.sum(w * np.abs(vis) ** 2)), rel=1e-13)
    assert orc.chi2(vis, np.zeros(M), np.zeros(M), np.zeros(M)) == 0.0
    ro, io = rng.standard_normal(M), rng.standard_normal(M)
    c = orc.chi2(vis, ro, io, w)
    assert orc.chi2(vis, ro, io, 3.0 * w) == pytest.approx(3.0 * c, rel=1e-13)
    import math
    exact = math.fsum(((vis.real - ro) ** 2 + (vis.imag - io) ** 2) * w)
    assert c == pytest.approx(exact, rel=1e-14)
    assert orc.chi2(vis, ro, io, w, nthreads=5) == pytest.approx(exact, rel=1e-14)
    # only the real residual / only the imaginary residual: catches a dropped term
    assert orc.chi2(vis, vis.real, io, w) == pytest.approx(float(np.sum(w * (vis.imag - io) ** 2)), rel=1e-13)
    assert orc.chi2(vis, ro, vis.imag, w) == pytest.approx(float(np.sum(w * (vis.real - ro) ** 2)), rel=1e-13)


def test_batch_is_a_loop_over_channels(orc):
    rng = np.random.default_rng(12)
    C, n, M, dxy = 3, 32, 200, 0.05 * ARCSEC
    imgs = rng.random((C, n, n))
    du = 1.0 / (n * dxy)
    u, v = rng.uniform(-0.4 * n, 0.4 * n, (C, M)) * du, rng.uniform(-0.4 * n, 0.4 * n, (C, M)) * du
    ro, io, w = rng.standard_normal((C, M)), rng.standard_normal((C, M)), rng.random((C, M))
    per, tot = orc.chi2ImageBatch(imgs, dxy, u, v, ro, io, w, dRA=1e-7, dDec=-2e-7, PA=0.4)
    for c in range(C):
        assert per[c] == orc.chi2Image(imgs[c], dxy, u[c], v[c], ro[c], io[c], w[c], 1e-7, -2e-7, 0.4)
    assert tot == pytest.approx(per.sum(), rel=1e-15)


def test_observation_sets_against_one_image_closed_form(orc):
    """chi2ImageSets pinned by a closed form, not by itself: a point source of flux F at the phase centre has a
    constant spectrum, which bilinear interpolation reproduces exactly, so V = F exp(2 pi i (u dRA + v dDec)) at
    every point and chi2 of set k is a plain numpy sum over THAT set's arrays.  The sets differ in
    length scale, observations and weights, so a mixed-up set index (u of one set with the weights of another, a
    total that skips a set) fails."""
    rng = np.random.default_rng(5)
    K, n, M, dxy, F = 4, 32, 300, 0.05 * ARCSEC, 2.5
    img = np.zeros((n, n))
    img[n // 2, n // 2] = F
    du = 1.0 / (n * dxy)
    scale = np.array([0.1, 0.2, 0.3, 0.4])[:, None]
    u, v = rng.uniform(-n, n, (K, M)) * du * scale, rng.uniform(-n, n, (K, M)) * du * scale
    ro, io, w = rng.standard_normal((K, M)), rng.standard_normal((K, M)), rng.random((K, M)) * np.arange(1, K + 1)[:, None]
    dRA, dDec = 0.31 * ARCSEC, -0.17 * ARCSEC
    per, tot = orc.chi2ImageSets(img, dxy, u, v, ro, io, w, dRA, dDec, 0.0)
    V = F * np.exp(2j * np.pi * (u * dRA + v * dDec))
    ref = (w * ((V.real - ro) ** 2 + (V.imag - io) ** 2)).sum(axis=1)
    assert per.shape == (K,) and np.allclose(per, ref, rtol=1e-11, atol=0)
    assert tot == pytest.approx(ref.sum(), rel=1e-11)
    assert len(set(np.round(per, 6))) == K                   # the sets really are different problems
    # with the out-of-grid count: the sum over the sets
    per2, tot2, oob = orc.chi2ImageSets(img, dxy, u * 8, v * 8, ro, io, w, dRA, dDec, 0.0, return_oob=True)
    assert oob == sum(orc.sampleImage(img, dxy, u[k] * 8, v[k] * 8, 0.0, dRA, dDec, return_oob=True)[1] for k in range(K)) > 0


# ---------------------------------------------------------------------------------------
# H1: direct Hankel evaluation of Eq. 25 — oracle.sampleProfileHankel / chi2ProfileHankel
# ---------------------------------------------------------------------------------------
def _rot(u, v, PA):
    return u * np.cos(PA) - v * np.sin(PA), u * np.sin(PA) + v * np.cos(PA)


def test_hankel_gaussian_closed_form_with_trapezoid_error_term(orc):
    """I(r) = exp(-r^2 / 2 s^2) on [0, Rmax]:  V(rho) = 2 pi s^2 exp(-2 pi^2 s^2 rho^2)  (closed form of Eq. 25).
    The composite trapezoid rule differs from the integral by the Euler-Maclaurin term h^2/12 [f'(Rmax) - f'(0)]
    with f = I J0 r, f'(0) = I(0) = 1, f'(Rmax) ~ 0: a constant -2 pi h^2 / 12 for every rho.  With that term the
    oracle must hit the closed form to O(h^4): a dropped 2 pi, r weight, end-point half weight or a J1 in place
    of J0 fails by orders of magnitude."""
    s, h, nr = 0.2 * ARCSEC, 1e-3 * ARCSEC, 4001
    R = h * np.arange(nr)
    I = np.exp(-R ** 2 / (2 * s * s))
    rho = np.array([0.0, 1e4, 1e5, 3e5, 6e5, 1e6, 3e6])
    V = orc.sampleProfileHankel(I, 0.0, h, rho, np.zeros_like(rho))
    closed = 2 * np.pi * s * s * np.exp(-2 * np.pi ** 2 * s * s * rho ** 2)
    peak = closed[0]
    assert np.abs(V.imag).max() == 0.0                                   # real for a centred axisymmetric source
    assert np.abs(V.real - (closed - 2 * np.pi * h * h / 12)).max() <= 2e-9 * peak
    assert np.abs(V.real - closed).max() >= 1e-6 * peak                  # ... and the term is really there
    # the same points on any azimuth (rho only) and chi2 on top of it
    az = np.linspace(0.1, 6.0, rho.size)
    V2 = orc.sampleProfileHankel(I, 0.0, h, rho * np.cos(az), rho * np.sin(az))
    assert np.abs(V2 - V).max() <= 1e-13 * peak
    import math
    re_o, im_o, w = closed * 0.9, np.full(rho.size, 1e-13), np.linspace(1.0, 2.0, rho.size) * 1e22
    chi2 = orc.chi2ProfileHankel(I, 0.0, h, rho, np.zeros_like(rho), re_o, im_o, w)
    ref = math.fsum(w * ((V.real - re_o) ** 2 + (V.imag - im_o) ** 2))
    assert abs(chi2 - ref) <= 1e-13 * ref


def test_hankel_annulus_closed_form(orc):
    """Sharp ring I = 1 on [a0, a1] (the paper's template (c), Eq. 28), Rmin = a0 > 0:
    int r J0(k r) dr = r J1(k r) / k, so V = (a1 J1(2 pi rho a1) - a0 J1(2 pi rho a0)) / rho; trapezoid error term
    h^2/12 [f'(a1) - f'(a0)], f' = J0(k r) - k r J1(k r).  Pins J0 (through J1 = -J0'), the r weight, Rmin and the
    grid R_k = Rmin + k dR."""
    from scipy.special import j0, j1
    a0, a1, nr = 0.2 * ARCSEC, 0.5 * ARCSEC, 3001
    h = (a1 - a0) / (nr - 1)
    I = np.ones(nr)
    rho = np.array([2e4, 1.1e5, 4.3e5, 9.7e5])
    V = orc.sampleProfileHankel(I, a0, h, np.zeros_like(rho), rho)      # along v: rho = abs(v)
    k = 2 * np.pi * rho
    exact = (a1 * j1(k * a1) - a0 * j1(k * a0)) / rho
    fp = lambda r: j0(k * r) - k * r * j1(k * r)
    corr = 2 * np.pi * h * h / 12 * (fp(a1) - fp(a0))
    peak = np.pi * (a1 * a1 - a0 * a0)
    assert np.abs(V.real - (exact + corr)).max() <= 1e-9 * peak
    assert np.abs(V.imag).max() == 0.0


def test_hankel_inclination_PA_and_phase(orc):
    """The swept image is I(sqrt((l / cos inc)^2 + m^2)): for a Gaussian profile an elliptical
    Gaussian with sigma_l = s cos inc, sigma_m = s, whose transform is 2 pi s^2 cos inc exp(-2 pi^2 s^2
    ((u' cos inc)^2 + v'^2)) at the rotated point (Eq. 11-12), times exp(+2 pi i (u dRA + v dDec)) (reading A1/A3).
    Pins the cos inc factor, which axis is compressed, the rotation sense and the phase sign."""
    s, h, nr = 0.15 * ARCSEC, 5e-4 * ARCSEC, 5001
    R = h * np.arange(nr)
    I = np.exp(-R ** 2 / (2 * s * s))
    rng = np.random.default_rng(5)
    u, v = rng.uniform(-8e5, 8e5, 40), rng.uniform(-8e5, 8e5, 40)
    inc, PA, dRA, dDec = 0.9, 0.7, 0.31 * ARCSEC, -0.17 * ARCSEC
    V = orc.sampleProfileHankel(I, 0.0, h, u, v, inc, PA, dRA, dDec)
    ur, vr = _rot(u, v, PA)
    ci = np.cos(inc)
    amp = 2 * np.pi * s * s * ci * np.exp(-2 * np.pi ** 2 * s * s * ((ur * ci) ** 2 + vr ** 2)) - 2 * np.pi * ci * h * h / 12
    ref = amp * np.exp(2j * np.pi * (u * dRA + v * dDec))
    assert np.abs(V - ref).max() <= 5e-9 * 2 * np.pi * s * s
    # the wrong axis or the wrong rotation sense is far outside that tolerance
    wrong = 2 * np.pi * s * s * ci * np.exp(-2 * np.pi ** 2 * s * s * (ur ** 2 + (vr * ci) ** 2))
    assert np.abs(np.abs(V) - wrong).max() >= 1e-3 * 2 * np.pi * s * s


def test_hankel_agrees_with_sampleProfile_at_the_papers_level(orc):
    """sampleProfile (sweep + FFT + bilinear interpolation) and the analytic Eq. 25 agree to a
    fractional difference generally below 1e-5.  Template (a) of the paper (Eq. 26): Gaussian disc
    with a Gaussian ring, inclined.  The bilinear interpolation error of the FFT route is (du 2 pi sigma)^2 / 8 of
    the peak off the nodes of the uv grid (per cent level at this field of view), so the two
    evaluations are compared AT the nodes (u, v) = (ku, kv) du with PA = 0, where interpolation is exact and only
    the pixelisation of the swept image separates them.  Two different evaluations of the same sky: agreement at
    the paper's level pins the normalisation (dxy^2, 2 pi, cos inc) and the geometry of one against the other."""
    nxy, dxy = 1024, 0.004 * ARCSEC
    du = 1.0 / (nxy * dxy)
    h, nr = 2e-4 * ARCSEC, 9000                                         # Rmax = 1.8"
    R = h * np.arange(nr)                 # Rmin = 0: with Rmin > 0 the sweep leaves the centre pixel empty (reading A5),
    Ra = R / ARCSEC                       # a constant I(0) dxy^2 = 5.6e-5 of the peak in every visibility
    I = (np.exp(-(Ra / 0.2) ** 2) + 0.3 * np.exp(-((Ra - 0.4) / 0.15) ** 2)) * 1e10
    rng = np.random.default_rng(11)
    ku, kv = rng.integers(-40, 41, 300), rng.integers(-40, 41, 300)     # up to 1000 klambda-ish: V spans 6 decades
    u, v = ku * du, kv * du
    inc = 0.5
    Vh = orc.sampleProfileHankel(I, R[0], h, u, v, inc, 0.0, 2e-7, -1e-7)
    Vf = orc.sampleProfile(I, R[0], h, nxy, dxy, u, v, inc, 0.0, 2e-7, -1e-7)
    peak = np.abs(Vh).max()
    assert np.abs(Vh - Vf).max() <= 1e-5 * peak
    # off the nodes and rotated, the difference is the interpolation error: inside its analytic bound, far above 1e-5
    uo, vo = (ku + 0.5) * du, (kv + 0.5) * du
    Vho = orc.sampleProfileHankel(I, R[0], h, uo, vo, inc, 1.1)
    Vfo = orc.sampleProfile(I, R[0], h, nxy, dxy, uo, vo, inc, 1.1)
    assert 1e-4 * peak <= np.abs(Vho - Vfo).max() <= 0.05 * peak
