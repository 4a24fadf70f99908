"""Seeded synthetic channel states shared by the oracle tests, the GPU parity tests and
bench.py.  This module holds NONE of the method's arithmetic: fields are analytic
expressions evaluated on the grid (polynomials in z times trigonometric sums in x, y,
tanh drops), random numbers come from numpy's seeded generator, and the only library
routine used is numpy's inverse FFT to sum band-limited trigonometric series in x, y.
Neither `oracle/` nor the CUDA package is imported here.

The states stand in for the paper's workloads (single-phase turbulent channel, PAPER.md
L231; drop swarm in a 4 pi x 2 pi x 2 channel, L260), whose actual fields are not
available.  Recipes: SURVEY.md section 8(d) / DESIGN.md "Input recipe".
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    nx: int
    ny: int
    nz: int
    re: float
    ch: float
    pe: float
    we: float
    dt: float
    steps: int
    visc_ratio: float = 1.0
    lx: float = 4.0 * math.pi
    ly: float = 2.0 * math.pi
    ndrops: int = 1
    radius: float = 0.4
    band: int = 0            # >0: flat perturbation spectrum on mode indices <= band
    seed: int = 0
    phase_field: int = 1

    @property
    def gradp_x(self) -> float:
        return 2.0 / self.re   # keeps u = 1 - z^2 steady (reading S12)


# BASELINE.json `configs` 1-4 (config 5 = random spectra on the grids in SCALING_GRIDS).
CONFIGS = {
    1: Config("cfg1", 32, 32, 33, re=100.0, ch=0.2, pe=5.0, we=1.0, dt=1e-4, steps=10,
              band=4, seed=1001),
    2: Config("cfg2", 128, 128, 129, re=3000.0, ch=0.05, pe=20.0, we=1.0, dt=5e-5, steps=100,
              seed=1002),
    3: Config("cfg3", 256, 256, 257, re=3000.0, ch=0.025, pe=40.0, we=3.0, dt=2e-5, steps=50,
              ndrops=64, radius=0.2, seed=1003),
    4: Config("cfg4", 512, 256, 257, re=3000.0, ch=0.05, pe=20.0, we=1.0, dt=5e-5, steps=50,
              visc_ratio=0.1, seed=1004),
}
SCALING_GRIDS = {"5a": (256, 128, 129), "5b": (512, 256, 257), "5c": (1024, 512, 513)}


def scaling_config(tag: str) -> Config:
    """Config 5: parameters of the step are not given by BASELINE.json; SURVEY 8(d) proposes
    Re=3000, Ch=0.025, Pe=40, We=1, dt=2e-5."""
    nx, ny, nz = SCALING_GRIDS[tag]
    return Config("cfg" + tag, nx, ny, nz, re=3000.0, ch=0.025, pe=40.0, we=1.0, dt=2e-5,
                  steps=10, seed=1005)


def small_config(nx=16, ny=16, nz=17, **kw) -> Config:
    """A tiny variant of config 1 for fast tests."""
    base = dict(re=100.0, ch=0.25, pe=4.0, we=1.0, dt=1e-4, steps=3, band=3, seed=7)
    base.update(kw)
    return Config("small", nx, ny, nz, **base)


def z_nodes(nz: int) -> np.ndarray:
    """Wall-normal grid the states are sampled on: z_k = cos(pi k/(nz-1)) (reading S1)."""
    return np.cos(np.pi * np.arange(nz) / (nz - 1))


def _signed_index(n: int) -> np.ndarray:
    j = np.arange(n)
    return np.where(j <= n // 2, j, j - n)


def solenoidal_perturbation(c: Config, rng: np.random.Generator):
    """Divergence-free, no-slip velocity perturbation in physical space.

    For every retained (i, j') != (0, 0) (2/3 cut-offs nx//3, ny//3; or |index| <= band):
        w^(z)     = a (1 - z^2)^2 (g0 + g1 z)          -> w = dw/dz = 0 at the walls
        omega^(z) = b (1 - z^2)   (g2 + g3 z)          -> omega_z = 0 at the walls
        u^ = (i kx dw^/dz + i ky omega^) / k^2,  v^ = (i ky dw^/dz - i kx omega^) / k^2
    with complex standard-normal g and envelope a, b ~ |k|^(-4/3) (a k^(-5/3) energy
    spectrum) or flat (band > 0).  dw^/dz is the analytic derivative of the polynomial.
    Summed over x, y with numpy's inverse FFT.  Returns u', v', w' [nz, ny, nx] scaled so
    that max |u'| = 0.1."""
    nx, ny, nz = c.nx, c.ny, c.nz
    nkx = nx // 2 + 1
    z = z_nodes(nz)[:, None, None]
    kx = (2 * np.pi / c.lx) * np.arange(nkx)[None, None, :]
    jp = _signed_index(ny)
    ky = (2 * np.pi / c.ly) * jp[None, :, None]
    ii = np.arange(nkx)[None, None, :]
    jj = jp[None, :, None]
    if c.band > 0:
        keep = (ii <= c.band) & (np.abs(jj) <= c.band)
        env = np.ones((1, ny, nkx))
    else:
        keep = (ii <= nx // 3) & (np.abs(jj) <= ny // 3)
        kmag = np.sqrt(kx ** 2 + ky ** 2)
        env = np.where(kmag > 0, np.maximum(kmag, 1e-30) ** (-4.0 / 3.0), 0.0)
    keep = keep & ~((ii == 0) & (jj == 0))
    env = np.where(keep, env, 0.0)

    def cn():
        return (rng.standard_normal((1, ny, nkx)) + 1j * rng.standard_normal((1, ny, nkx))) * env

    g0, g1, g2, g3 = cn(), cn(), cn(), cn()
    # Hermitian fill of the i = 0 plane: g(-j', 0) = conj(g(j', 0))
    for gcoef in (g0, g1, g2, g3):
        for j in range(1, ny // 2):
            gcoef[0, ny - j, 0] = np.conj(gcoef[0, j, 0])
        gcoef[0, ny // 2, :] = 0.0
    # The z dependence is polynomial and separable: sum the series in x, y once per coefficient field (2-D inverse
    # FFTs), then combine with the polynomials in z (one small matrix product per velocity component).
    k2 = kx ** 2 + ky ** 2
    k2s = np.where(k2 > 0, k2, 1.0)
    scale = nx * ny   # numpy's irfft2 divides by nx*ny; we want plain trigonometric sums

    def xy_sum(a):
        return np.fft.irfft2(a[0], s=(ny, nx), axes=(0, 1)) * scale

    zz = z_nodes(nz)
    q = 1.0 - zz * zz
    # w^ = q^2 (g0 + g1 z);  dw^/dz = -4 z q (g0 + g1 z) + q^2 g1;  omega^ = q (g2 + g3 z)
    pw = np.stack([q * q, q * q * zz], axis=1)                                        # multiplies (g0, g1)
    pdw = np.stack([-4.0 * zz * q, -4.0 * zz * zz * q + q * q], axis=1)               # multiplies (g0, g1)
    pom = np.stack([q, q * zz], axis=1)                                               # multiplies (g2, g3)

    def combine(polys, fields):
        f = np.stack([a.ravel() for a in fields], axis=0)                             # [m, ny*nx]
        return (np.concatenate(polys, axis=1) @ f).reshape(nz, ny, nx)

    w = combine([pw], [xy_sum(g0), xy_sum(g1)])
    u = combine([pdw, pom], [xy_sum(1j * kx * g0 / k2s), xy_sum(1j * kx * g1 / k2s),
                             xy_sum(1j * ky * g2 / k2s), xy_sum(1j * ky * g3 / k2s)])
    v = combine([pdw, -pom], [xy_sum(1j * ky * g0 / k2s), xy_sum(1j * ky * g1 / k2s),
                              xy_sum(1j * kx * g2 / k2s), xy_sum(1j * kx * g3 / k2s)])
    amp = 0.1 / max(np.abs(u).max(), 1e-300)
    return u * amp, v * amp, w * amp


def drop_centres(c: Config, rng: np.random.Generator) -> np.ndarray:
    """Drop centres: one drop -> box centre; several -> seeded rejection sampling with
    separation >= 2R + 6Ch (minimum image in x, y) and wall clearance >= R + 3Ch."""
    if c.ndrops == 1:
        return np.array([[0.5 * c.lx, 0.5 * c.ly, 0.0]])
    pts: list[np.ndarray] = []
    dmin = 2 * c.radius + 6 * c.ch
    zmax = 1.0 - (c.radius + 3 * c.ch)
    tries = 0
    while len(pts) < c.ndrops:
        tries += 1
        if tries > 200000:
            raise RuntimeError("drop placement failed")
        p = np.array([rng.uniform(0, c.lx), rng.uniform(0, c.ly), rng.uniform(-zmax, zmax)])
        ok = True
        for q in pts:
            dx = abs(p[0] - q[0]); dx = min(dx, c.lx - dx)
            dy = abs(p[1] - q[1]); dy = min(dy, c.ly - dy)
            if math.sqrt(dx * dx + dy * dy + (p[2] - q[2]) ** 2) < dmin:
                ok = False
                break
        if ok:
            pts.append(p)
    return np.array(pts)


def drops_phase_field(c: Config, centres: np.ndarray) -> np.ndarray:
    """phi = -1 + sum_d [1 - tanh((r_d - R)/(sqrt2 Ch))], phi = +1 inside drops (Eq. 5 profile
    across each interface; reading S16), minimum-image distance in x, y.  Each drop is evaluated only inside the
    box where its term is not exactly zero in float64 (tanh(t) == 1.0 for t >= 20)."""
    x = (c.lx / c.nx) * np.arange(c.nx)
    y = (c.ly / c.ny) * np.arange(c.ny)
    z = z_nodes(c.nz)
    phi = -np.ones((c.nz, c.ny, c.nx))
    w = math.sqrt(2.0) * c.ch
    reach = c.radius + 20.0 * w
    for (xc, yc, zc) in centres:
        dx = np.abs(x - xc); dx = np.minimum(dx, c.lx - dx)
        dy = np.abs(y - yc); dy = np.minimum(dy, c.ly - dy)
        ix = np.nonzero(dx <= reach)[0]
        iy = np.nonzero(dy <= reach)[0]
        iz = np.nonzero(np.abs(z - zc) <= reach)[0]
        r = np.sqrt(dx[ix][None, None, :] ** 2 + dy[iy][None, :, None] ** 2 + (z[iz][:, None, None] - zc) ** 2)
        phi[np.ix_(iz, iy, ix)] += 1.0 - np.tanh((r - c.radius) / w)
    return phi


def channel_state(c: Config):
    """PHYSICAL-space initial state (u, v, w, phi) of configs 1-4: laminar Poiseuille
    u = 1 - z^2 plus the solenoidal perturbation, and the drop(s)."""
    rng = np.random.default_rng(c.seed)
    up, vp, wp = solenoidal_perturbation(c, rng)
    z = z_nodes(c.nz)[:, None, None]
    u = (1.0 - z * z) + up
    phi = drops_phase_field(c, drop_centres(c, rng)) if c.phase_field else None
    return u, vp, wp, phi


def random_spectrum(nx: int, ny: int, nz: int, rng: np.random.Generator,
                    cut: bool = False, rms: float = 0.3) -> np.ndarray:
    """Config 5 field: SPECTRAL complex [nz, ny, nx/2+1], Gaussian coefficients times a
    (1 + i^2 + j'^2 + n^2)^-1 envelope, Hermitian-consistent on the i = 0 plane, Nyquist
    planes zero; cut=True also zeroes everything outside the 2/3 cut-offs.  Scaled so that
    the root of the summed squared magnitudes is `rms` (no transform needed)."""
    nkx = nx // 2 + 1
    ii = np.arange(nkx)[None, None, :].astype(np.float64)
    jj = _signed_index(ny)[None, :, None].astype(np.float64)
    nn = np.arange(nz)[:, None, None].astype(np.float64)
    a = rng.standard_normal((nz, ny, nkx)) + 1j * rng.standard_normal((nz, ny, nkx))
    a *= 1.0 / (1.0 + ii * ii + jj * jj + nn * nn)
    a[:, ny // 2, :] = 0.0
    a[:, :, nx // 2] = 0.0
    if cut:
        a[:, :, nx // 3 + 1:] = 0.0
        a[:, ny // 3 + 1: ny - ny // 3, :] = 0.0
        a[(2 * (nz - 1)) // 3 + 1:, :, :] = 0.0
    for j in range(1, ny // 2):
        a[:, ny - j, 0] = np.conj(a[:, j, 0])
    a[:, 0, 0] = a[:, 0, 0].real
    a *= rms / math.sqrt(float(np.sum(np.abs(a) ** 2)))
    return a


def random_spectral_state(nx: int, ny: int, nz: int, seed: int, cut: bool = True):
    rng = np.random.default_rng(seed)
    return tuple(random_spectrum(nx, ny, nz, rng, cut=cut) for _ in range(4))


def random_physical_field(nx: int, ny: int, nz: int, seed: int) -> np.ndarray:
    """Plain Gaussian white field in physical space (round-trip tests, dealiasing off)."""
    return np.random.default_rng(seed).standard_normal((nz, ny, nx))
