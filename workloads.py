"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md "Inputs").

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no FFT, no bilinear interpolation of a spectrum, no sweep of a profile, no
chi-square.  It imports neither ``oracle`` nor the CUDA binding.  What it does hold is the
*synthetic sky*: images drawn from closed-form brightness distributions, (u, v) tracks from
textbook earth-rotation synthesis, and "observed" visibilities that are the *continuous* Fourier
transform of that sky (closed form for Gaussians and point sources, the Hankel integral of
PAPER.md:368 Eq. 25 for axisymmetric discs) plus Gaussian noise.  The paper measures on its
authors' own uv tables and images, which are not public and not in this container
(PAPER.md:396, 408); these inputs take their shapes (PAPER.md:316-338 Table 1, :430) and stand
in for them.

Conventions (readings A1, A2, A10): images are [row][col], row 0 = North, col 0 =
East, origin at pixel [n/2][n/2]; sky offsets l (East) = (n/2 - col) dxy, m (North) =
(n/2 - row) dxy; the observed sky is the model rotated by PA (East of North) about the phase
centre and then moved by (dRA, dDec); the Fourier sign is the one of the paper's Appendix D
listing, V(u, v) = sum A exp(+2 pi i (u l + v m)).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

ARCSEC = np.pi / 648000.0
C_LIGHT = 299792458.0  # m/s
_SEED0 = 1000


@dataclass
class Workload:
    """One problem instance.  Arrays are numpy float64 unless ``precision == 'f32'``."""
    name: str
    entry: str                      # 'chi2Image' | 'chi2Profile' | 'chi2ImageBatch'
    nxy: int
    dxy: float
    u: np.ndarray                   # [M] or [C][M]
    v: np.ndarray
    re_obs: np.ndarray
    im_obs: np.ndarray
    w: np.ndarray
    dRA: float
    dDec: float
    PA: float
    image: Optional[np.ndarray] = None      # [n][n] or [C][n][n]
    profile: Optional[np.ndarray] = None    # [nr]
    Rmin: float = 0.0
    dR: float = 0.0
    inc: float = 0.0
    precision: str = "f64"
    meta: dict = field(default_factory=dict)

    @property
    def M(self) -> int:
        return int(self.u.shape[-1])

    def as_f32(self) -> "Workload":
        """fp32 variant (reading A14): every array rounded to float32; scalars unchanged."""
        def r(a):
            return None if a is None else np.ascontiguousarray(a, dtype=np.float32)
        return Workload(self.name + "-f32", self.entry, self.nxy, self.dxy, r(self.u), r(self.v), r(self.re_obs),
                        r(self.im_obs), r(self.w), self.dRA, self.dDec, self.PA, r(self.image), r(self.profile),
                        self.Rmin, self.dR, self.inc, "f32", dict(self.meta))


# -----------------------------------------------------------------------------------------
# (u, v) generators
# -----------------------------------------------------------------------------------------
def uv_uniform(rng, M, dxy, frac=0.45):
    """cfg 0: u, v ~ U(-frac/dxy, +frac/dxy) independently (wavelengths)."""
    lim = frac / dxy
    return rng.uniform(-lim, lim, M), rng.uniform(-lim, lim, M)


def uv_loguniform(rng, M, bmin_m, bmax_m, lam_m):
    """cfg 1: baseline length log-uniform in [bmin, bmax] metres at wavelength lam, azimuth uniform."""
    q = np.exp(rng.uniform(np.log(bmin_m), np.log(bmax_m), M)) / lam_m
    az = rng.uniform(0.0, 2 * np.pi, M)
    return q * np.cos(az), q * np.sin(az)


def antenna_layout(rng, n_ant, median_m=1000.0, sigma_ln=1.0, rmax_m=8000.0):
    """Flat array: radius log-normal (redrawn above rmax), azimuth uniform.  Returns East, North (m)."""
    r = np.empty(n_ant)
    for a in range(n_ant):
        while True:
            x = median_m * np.exp(sigma_ln * rng.standard_normal())
            if x <= rmax_m:
                break
        r[a] = x
    az = rng.uniform(0.0, 2 * np.pi, n_ant)
    return r * np.sin(az), r * np.cos(az)


def uv_tracks_metres(east, north, lat_deg=-23.02, dec_deg=-25.0, ha_hours=4.0, step_s=6.0):
    """Textbook earth-rotation synthesis for a flat array (u, v in METRES, time-major order).

    Equatorial baseline components from local East/North (Up = 0) at latitude ``lat``:
    Lx = -sin(lat) N, Ly = E, Lz = cos(lat) N;  u = sinH Lx + cosH Ly,
    v = -sin(dec) cosH Lx + sin(dec) sinH Ly + cos(dec) Lz.  All n(n-1)/2 baselines, hour angle
    -ha..+ha every ``step_s`` seconds.  Output index = t * n_baselines + b.
    """
    lat, dec = np.deg2rad(lat_deg), np.deg2rad(dec_deg)
    i, j = np.triu_indices(east.size, k=1)
    dE, dN = east[j] - east[i], north[j] - north[i]
    Lx, Ly, Lz = -np.sin(lat) * dN, dE, np.cos(lat) * dN
    nstep = int(round(2 * ha_hours * 3600.0 / step_s)) + 1
    H = np.linspace(-ha_hours, ha_hours, nstep) * (np.pi / 12.0)
    sH, cH = np.sin(H)[:, None], np.cos(H)[:, None]
    uu = sH * Lx[None, :] + cH * Ly[None, :]
    vv = -np.sin(dec) * cH * Lx[None, :] + np.sin(dec) * sH * Ly[None, :] + np.cos(dec) * Lz[None, :]
    return uu.reshape(-1), vv.reshape(-1)


def subset_time_major(rng, total, M):
    """Seeded subset of exactly M of ``total`` samples without replacement, original order kept."""
    if M >= total:
        # more points asked than the track holds (reduced-size tests never do this); tile.
        return np.arange(M) % total
    idx = rng.choice(total, size=M, replace=False)
    idx.sort()
    return idx


def alma_like_uv_metres(rng, n_ant, M, max_baseline_m=None):
    east, north = antenna_layout(rng, n_ant)
    if max_baseline_m is not None:
        i, j = np.triu_indices(n_ant, k=1)
        longest = np.sqrt((east[j] - east[i]) ** 2 + (north[j] - north[i]) ** 2).max()
        east, north = east * (max_baseline_m / longest), north * (max_baseline_m / longest)
    um, vm = uv_tracks_metres(east, north)
    idx = subset_time_major(rng, um.size, M)
    return um[idx], vm[idx]


# -----------------------------------------------------------------------------------------
# synthetic sky: images and their continuous Fourier transforms
# -----------------------------------------------------------------------------------------
def pixel_offsets(nxy, dxy):
    """l (East, per column) and m (North, per row) of the pixel centres (reading A2)."""
    c = (nxy // 2 - np.arange(nxy)) * dxy
    return c, c


def rotate_uv(u, v, PA):
    """Coordinates at which the UNROTATED model is observed (Eq. 11-12)."""
    c, s = np.cos(PA), np.sin(PA)
    return u * c - v * s, u * s + v * c


def translate_phase(u, v, dRA, dDec):
    """exp(+2 pi i (u dRA + v dDec)): the sky moved East by dRA, North by dDec (reading A1)."""
    th = 2 * np.pi * (u * dRA + v * dDec)
    return np.cos(th) + 1j * np.sin(th)


def render_gaussians(nxy, dxy, flux, l0, m0, sig_major, sig_minor, theta, nsig=7.0):
    """Sum of elliptical Gaussians (flux in Jy each), sampled at pixel centres, Jy/pixel.

    ``theta`` is the position angle of the major axis, East of North.  Each source is drawn
    inside a +-nsig*sig_major box only; the truncation is part of the image's definition.
    """
    img = np.zeros((nxy, nxy))
    lc, mc = pixel_offsets(nxy, dxy)
    for F, a, b, sa, sb, th in zip(flux, l0, m0, sig_major, sig_minor, theta):
        half = int(np.ceil(nsig * sa / dxy)) + 1
        jc, ic = nxy // 2 - int(round(a / dxy)), nxy // 2 - int(round(b / dxy))
        j0, j1 = max(0, jc - half), min(nxy, jc + half + 1)
        i0, i1 = max(0, ic - half), min(nxy, ic + half + 1)
        if j0 >= j1 or i0 >= i1:
            continue
        dl = lc[None, j0:j1] - a
        dm = mc[i0:i1, None] - b
        # major axis unit vector in (l, m): (sin th, cos th); minor: (cos th, -sin th)
        p = dl * np.sin(th) + dm * np.cos(th)
        q = dl * np.cos(th) - dm * np.sin(th)
        g = np.exp(-0.5 * ((p / sa) ** 2 + (q / sb) ** 2))
        img[i0:i1, j0:j1] += g * (F * dxy * dxy / (2 * np.pi * sa * sb))
    return img


def gaussians_visibility(u, v, flux, l0, m0, sig_major, sig_minor, theta, chunk=200000):
    """Continuous FT (Appendix-D sign) of the sources of ``render_gaussians`` at (u, v)."""
    out = np.zeros(u.shape, dtype=np.complex128)
    try:  # plumbing only: let torch spread the 500-source sum over cores / the GPU when it is there
        import torch
        dev = torch.device("cuda" if torch.cuda.is_available() else "cpu")
        t = lambda x: torch.as_tensor(np.asarray(x, dtype=np.float64), device=dev)
        F, a, b, sa, sb, th = map(t, (flux, l0, m0, sig_major, sig_minor, theta))
        for s in range(0, u.size, chunk):
            uu, vv = t(u[s:s + chunk])[:, None], t(v[s:s + chunk])[:, None]
            p = uu * torch.sin(th) + vv * torch.cos(th)
            q = uu * torch.cos(th) - vv * torch.sin(th)
            amp = F * torch.exp(-2 * np.pi ** 2 * ((sa * p) ** 2 + (sb * q) ** 2))
            ph = 2 * np.pi * (uu * a + vv * b)
            re, im = (amp * torch.cos(ph)).sum(1), (amp * torch.sin(ph)).sum(1)
            out[s:s + chunk] = re.cpu().numpy() + 1j * im.cpu().numpy()
        return out
    except ImportError:
        pass
    for s in range(0, u.size, chunk):
        uu, vv = u[s:s + chunk, None], v[s:s + chunk, None]
        p = uu * np.sin(theta) + vv * np.cos(theta)
        q = uu * np.cos(theta) - vv * np.sin(theta)
        amp = flux * np.exp(-2 * np.pi ** 2 * ((sig_major * p) ** 2 + (sig_minor * q) ** 2))
        out[s:s + chunk] = (amp * np.exp(2j * np.pi * (uu * l0 + vv * m0))).sum(1)
    return out


def hankel_visibility(profile_fn, rmax, rho, n_r=20000, per_cycle=16):
    """Eq. 25: V(rho) = 2 pi int_0^rmax I(r) J0(2 pi rho r) r dr, tabulated on a
    uniform grid of rho with ``per_cycle`` samples per 1/rmax (trapezoid in r) and evaluated at
    ``rho`` with a cubic spline."""
    from scipy.interpolate import CubicSpline
    from scipy.special import j0
    r = np.linspace(0.0, rmax, n_r + 1)[1:]
    Ir = profile_fn(r) * r
    step = 1.0 / (per_cycle * rmax)
    grid = np.arange(0, int(np.ceil(max(rho.max(), step) / step)) + 4) * step
    tab = np.empty(grid.size)
    dr = r[1] - r[0]
    for s in range(0, grid.size, 64):
        k = j0(2 * np.pi * grid[s:s + 64, None] * r[None, :]) * Ir[None, :]
        tab[s:s + 64] = 2 * np.pi * dr * (k.sum(1) - 0.5 * k[:, -1])
    return CubicSpline(grid, tab)(rho)


def inclined_disc_visibility(profile_fn, rmax, inc, u, v):
    """FT of I(sqrt((l / cos inc)^2 + m^2)): cos(inc) * Hankel at rho = sqrt((u cos inc)^2 + v^2)."""
    rho = np.sqrt((u * np.cos(inc)) ** 2 + v ** 2)
    return np.cos(inc) * hankel_visibility(profile_fn, rmax, rho)


def observe(rng, V_sky, sigma):
    """V_obs = V_sky + N(0, sigma) on Re and Im; ``sigma`` scalar or per point."""
    return (V_sky.real + sigma * rng.standard_normal(V_sky.shape),
            V_sky.imag + sigma * rng.standard_normal(V_sky.shape))


# -----------------------------------------------------------------------------------------
# the five configs
# -----------------------------------------------------------------------------------------
def config0(nxy=256, M=10_000, seed=_SEED0 + 0) -> Workload:
    """chi2Image f64: elliptical Gaussian + 3 point sources, uniform uv (BASELINE.json configs[0])."""
    rng = np.random.default_rng(seed)
    dxy = 0.02 * ARCSEC * (256 / nxy)          # keep the field of view when a test shrinks nxy
    k = 1.0 / (2 * np.sqrt(2 * np.log(2)))
    sig_m, sig_l = 0.5 * ARCSEC * k, 0.3 * ARCSEC * k      # FWHM 0.5" North-South x 0.3" East-West
    g = dict(flux=np.array([1.0]), l0=np.array([0.0]), m0=np.array([0.0]), sig_major=np.array([sig_m]),
             sig_minor=np.array([sig_l]), theta=np.array([0.0]))
    image = render_gaussians(nxy, dxy, nsig=1e9, **g)
    scale = 1.0 / image.sum()                  # "flux 1 Jy" = the pixels sum to 1
    image *= scale
    pf = np.array([0.10, 0.05, 0.02])
    pj = rng.integers(-nxy // 4, nxy // 4 + 1, 3)     # pixels East of centre
    pi_ = rng.integers(-nxy // 4, nxy // 4 + 1, 3)    # pixels North of centre
    for F, a, b in zip(pf, pj, pi_):
        image[nxy // 2 - b, nxy // 2 - a] += F
    u, v = uv_uniform(rng, M, dxy)
    dRA, dDec, PA = 0.05 * ARCSEC, -0.03 * ARCSEC, np.deg2rad(30.0)
    ur, vr = rotate_uv(u, v, PA)
    V = scale * gaussians_visibility(ur, vr, **g)
    for F, a, b in zip(pf, pj, pi_):
        V = V + F * np.exp(2j * np.pi * (ur * a * dxy + vr * b * dxy))
    V = V * translate_phase(u, v, dRA, dDec)
    sigma = 1e-3
    re, im = observe(rng, V, sigma)
    return Workload("cfg0", "chi2Image", nxy, dxy, u, v, re, im, np.full(M, 1.0 / sigma ** 2), dRA, dDec, PA,
                    image=image, meta=dict(sigma=sigma, seed=seed))


def _taper_profile(R_arcsec):
    return R_arcsec ** -0.7 * np.exp(-R_arcsec)


def config1(nxy=1024, M=200_000, nr=2000, seed=_SEED0 + 1) -> Workload:
    """chi2Profile f64 (sweep path): tapered power law, inc 45 deg, PA 60 deg, log-uniform baselines."""
    rng = np.random.default_rng(seed)
    dxy = 0.005 * ARCSEC * (1024 / nxy)
    Rmin, dR = 1e-4 * ARCSEC, 1e-3 * ARCSEC * (2000 / nr)
    inc, PA = np.deg2rad(45.0), np.deg2rad(60.0)
    R = Rmin + dR * np.arange(nr)
    shape = _taper_profile(R / ARCSEC)
    # I0 such that the inclined disc carries ~1 Jy: flux = cos(inc) * 2 pi int I(R) R dR (trapezoid)
    integ = np.sum(0.5 * (shape[1:] * R[1:] + shape[:-1] * R[:-1])) * dR
    I0 = 1.0 / (2 * np.pi * np.cos(inc) * integ)
    profile = I0 * shape                                   # Jy / sr
    u, v = uv_loguniform(rng, M, 15.0, 16000.0, 1.3e-3)
    Rmax = R[-1]
    ur, vr = rotate_uv(u, v, PA)
    fn = lambda r: I0 * np.where((r >= Rmin) & (r <= Rmax), _taper_profile(np.maximum(r, Rmin) / ARCSEC), 0.0)
    V = inclined_disc_visibility(fn, Rmax, inc, ur, vr).astype(np.complex128)
    sigma = 5e-4
    re, im = observe(rng, V, sigma)
    return Workload("cfg1", "chi2Profile", nxy, dxy, u, v, re, im, np.full(M, 1.0 / sigma ** 2), 0.0, 0.0, PA,
                    profile=profile, Rmin=Rmin, dR=dR, inc=inc, meta=dict(sigma=sigma, seed=seed))


def _rings_profile(r_arcsec):
    r = np.maximum(r_arcsec, 1e-4)
    out = 0.2 * (r / 0.1) ** -0.5
    for r0, amp in ((0.2, 1.0), (0.5, 0.6), (0.8, 0.3)):
        out = out + amp * np.exp(-0.5 * ((r - r0) / 0.03) ** 2)
    return np.where(r_arcsec <= 1.2, out, 0.0)


def _seeded_transform(rng):
    return (rng.uniform(-0.1, 0.1) * ARCSEC, rng.uniform(-0.1, 0.1) * ARCSEC, rng.uniform(0.0, np.pi))


def config2(nxy=2048, M=1_000_000, seed=_SEED0 + 2) -> Workload:
    """chi2Image f64: ring+gap disc inclined 35 deg; 43-antenna earth-rotation tracks at 0.87 mm."""
    rng = np.random.default_rng(seed)
    dxy = 0.003 * ARCSEC * (2048 / nxy)
    inc = np.deg2rad(35.0)
    lc, mc = pixel_offsets(nxy, dxy)
    r = np.sqrt((lc[None, :] / np.cos(inc)) ** 2 + mc[:, None] ** 2)
    image = _rings_profile(r / ARCSEC)
    scale = 1.0 / image.sum()
    image = image * scale
    um, vm = alma_like_uv_metres(rng, 43, M)
    lam = 0.87e-3
    u, v = um / lam, vm / lam
    dRA, dDec, PA = _seeded_transform(rng)
    ur, vr = rotate_uv(u, v, PA)
    fn = lambda rr: _rings_profile(rr / ARCSEC) * (scale / dxy ** 2)
    V = inclined_disc_visibility(fn, 1.2 * ARCSEC, inc, ur, vr) * translate_phase(u, v, dRA, dDec)
    sigma = 1e-3
    re, im = observe(rng, V, sigma)
    return Workload("cfg2", "chi2Image", nxy, dxy, u, v, re, im, np.full(M, 1.0 / sigma ** 2), dRA, dDec, PA,
                    image=image, meta=dict(sigma=sigma, seed=seed, inc=inc))


def config3(nxy=4096, M=5_000_000, n_src=500, seed=_SEED0 + 3) -> Workload:
    """sampleImage + chi2Image, f64 (use .as_f32() for fp32): 500 elliptical Gaussians, total 1 Jy;
    50-antenna tracks, longest baseline 16 km, 0.87 mm; log-normal weights (median 1e6)."""
    rng = np.random.default_rng(seed)
    dxy = 0.0015 * ARCSEC * (4096 / nxy)
    k = 1.0 / (2 * np.sqrt(2 * np.log(2)))
    fwhm = np.exp(rng.uniform(np.log(0.005), np.log(0.5), n_src)) * ARCSEC
    ratio = rng.uniform(0.3, 1.0, n_src)
    theta = rng.uniform(0.0, np.pi, n_src)
    fov = nxy * dxy
    l0, m0 = rng.uniform(-fov / 8, fov / 8, n_src), rng.uniform(-fov / 8, fov / 8, n_src)
    flux = np.exp(rng.uniform(0.0, np.log(10.0), n_src))
    flux /= flux.sum()
    g = dict(flux=flux, l0=l0, m0=m0, sig_major=fwhm * k, sig_minor=fwhm * k * ratio, theta=theta)
    image = render_gaussians(nxy, dxy, **g)
    um, vm = alma_like_uv_metres(rng, 50, M, max_baseline_m=16000.0)
    lam = 0.87e-3
    u, v = um / lam, vm / lam
    dRA, dDec, PA = _seeded_transform(rng)
    ur, vr = rotate_uv(u, v, PA)
    V = gaussians_visibility(ur, vr, **g) * translate_phase(u, v, dRA, dDec)
    w = 1e6 * np.exp(0.5 * rng.standard_normal(M))
    re, im = observe(rng, V, 1.0 / np.sqrt(w))
    return Workload("cfg3", "chi2Image", nxy, dxy, u, v, re, im, w, dRA, dDec, PA, image=image,
                    meta=dict(seed=seed, n_src=n_src))


def config4(nxy=1024, M=200_000, C=128, seed=_SEED0 + 4) -> Workload:
    """Batched cube chi2Image f64: C channels of a Keplerian disc (inc 40 deg, 1 Msun, 140 pc),
    channel width 0.2 km/s around 230 GHz; one metre-unit track set scaled by channel frequency."""
    rng = np.random.default_rng(seed)
    dxy = 0.01 * ARCSEC * (1024 / nxy)
    inc = np.deg2rad(40.0)
    GM = 6.674e-11 * 1.989e30
    dist_m = 140.0 * 3.0857e16
    sigma_v = 300.0
    lc, mc = pixel_offsets(nxy, dxy)
    xd = lc[None, :] / np.cos(inc)              # deprojected disc coordinates (rad)
    yd = np.broadcast_to(mc[:, None], (nxy, nxy))
    r = np.maximum(np.sqrt(xd ** 2 + yd ** 2), 0.5 * dxy)
    cosphi = yd / r                              # phi measured from the line of nodes (North-South)
    vlos = np.sqrt(GM / (r * dist_m)) * np.sin(inc) * cosphi
    I0 = (r / (0.5 * ARCSEC)) ** -0.5 * np.exp(-r / (1.5 * ARCSEC))
    vc = (np.arange(C) - (C - 1) / 2.0) * 200.0
    images = np.empty((C, nxy, nxy))
    for c in range(C):
        images[c] = I0 * np.exp(-0.5 * ((vc[c] - vlos) / sigma_v) ** 2)
    images /= images.reshape(C, -1).sum(1).max()
    um, vm = alma_like_uv_metres(rng, 50, M, max_baseline_m=16000.0)
    nu = 230e9 * (1.0 - vc / C_LIGHT)
    u = um[None, :] * (nu[:, None] / C_LIGHT)
    v = vm[None, :] * (nu[:, None] / C_LIGHT)
    dRA, dDec, PA = _seeded_transform(rng)
    # observed sky: a Gaussian surrogate carrying each channel's flux (no closed form exists for
    # a Keplerian channel map; chi2 then measures noise + model mismatch, as early in a real fit)
    flux_c = images.reshape(C, -1).sum(1)
    ur, vr = rotate_uv(u, v, PA)
    s = 0.6 * ARCSEC
    V = flux_c[:, None] * np.exp(-2 * np.pi ** 2 * s ** 2 * ((ur * np.cos(inc)) ** 2 + vr ** 2))
    V = V * translate_phase(u, v, dRA, dDec)
    sigma = 1e-3
    re, im = observe(rng, V, sigma)
    return Workload("cfg4", "chi2ImageBatch", nxy, dxy, np.ascontiguousarray(u), np.ascontiguousarray(v), re, im,
                    np.full((C, M), 1.0 / sigma ** 2), dRA, dDec, PA, image=images,
                    meta=dict(sigma=sigma, seed=seed, C=C))


CONFIGS = (config0, config1, config2, config3, config4)


def config(idx: int, **overrides) -> Workload:
    return CONFIGS[idx](**overrides)
