"""CPU oracle of the iso-surface ray-caster (Fig. 5: "drops are rendered as the
iso-surface phi = 0").  TEST INFRASTRUCTURE ONLY, like psdns_oracle.py: plain numpy float64, one ray per pixel, the
algorithm written out step by step; shares no code with the CUDA path.

The paper renders Fig. 5 off line with a ray tracer it does not describe, so the ALGORITHM here is this project's
reading ("parity unpinned by the paper"); what pins the oracle is geometry (tests/test_oracle_isosurface.py): the depth
and the shading of an analytic sphere and of a plane.

Algorithm (every quantity float64):
  camera   f = unit(target - eye), r = unit(f x up), v = r x f; pixel (px, py), py = 0 the top row:
           sx = (2 (px + 1/2)/W - 1) tan(fov/2) W/H,  sy = (1 - 2 (py + 1/2)/H) tan(fov/2),  d = unit(f + sx r + sy v)
  box      slab intersection of eye + t d with [0, Lx] x [0, Ly] x [-1, 1] -> [t0, t1] (t0 >= 0); miss: intensity 0, depth -1
  field    phi(p): p_z clamped to [-1, 1]; periodic wrap in x, y; trilinear interpolation between the grid values
           (x_i = i Lx/nx, y_j = j Ly/ny, z_k = cos(pi k/N), the Gauss-Lobatto points, k = 0 at z = +1)
  march    g(t) = phi(eye + t d) - iso at t_i = min(t0 + i ds, t1), i = 0 .. ceil((t1 - t0)/ds); the first i >= 1 with
           (g_{i-1} < 0) != (g_i < 0) brackets the surface; NBIS = 24 bisections; depth = midpoint of the last bracket
  shading  n = central differences of phi at the hit point with steps (Lx/nx, Ly/ny, 1/N);
           intensity = 0.2 + 0.8 |unit(n) . unit(light)|  (0.2 where n = 0)
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

NBIS = 24


@dataclass
class Camera:
    eye: tuple
    target: tuple
    up: tuple = (0.0, 0.0, 1.0)
    fov_y_deg: float = 40.0
    width: int = 64
    height: int = 48
    step: float = 0.02
    light: tuple = (0.3, -0.5, 0.8)


def _unit(a):
    a = np.asarray(a, dtype=np.float64)
    return a / np.sqrt(np.sum(a * a, axis=-1, keepdims=True))


def sample_field(phi, lx, ly, p):
    """Trilinear interpolation of phi [nz, ny, nx] at points p [..., 3]."""
    nz, ny, nx = phi.shape
    N = nz - 1
    zn = np.cos(np.pi * np.arange(nz) / N)
    fx = p[..., 0] / (lx / nx)
    fy = p[..., 1] / (ly / ny)
    ix = np.floor(fx)
    iy = np.floor(fy)
    wx = fx - ix
    wy = fy - iy
    i0 = np.mod(ix.astype(np.int64), nx)
    j0 = np.mod(iy.astype(np.int64), ny)
    i1 = np.mod(i0 + 1, nx)
    j1 = np.mod(j0 + 1, ny)
    z = np.clip(p[..., 2], -1.0, 1.0)
    k = np.minimum(np.floor(np.arccos(z) * (N / np.pi)).astype(np.int64), N - 1)
    k = np.maximum(k, 0)
    for _ in range(2):                                   # repair a rounding slip of arccos at a node
        k = np.where((z > zn[k]) & (k > 0), k - 1, k)
        k = np.where((z < zn[k + 1]) & (k < N - 1), k + 1, k)
    wz = (zn[k] - z) / (zn[k] - zn[k + 1])

    def plane(kk):
        a = phi[kk, j0, i0] * (1.0 - wx) + phi[kk, j0, i1] * wx
        b = phi[kk, j1, i0] * (1.0 - wx) + phi[kk, j1, i1] * wx
        return a * (1.0 - wy) + b * wy

    return plane(k) * (1.0 - wz) + plane(k + 1) * wz


def rays(cam: Camera):
    f = _unit(np.subtract(cam.target, cam.eye))
    r = _unit(np.cross(f, np.asarray(cam.up, dtype=np.float64)))
    v = np.cross(r, f)
    th = math.tan(math.radians(cam.fov_y_deg) / 2.0)
    px = np.arange(cam.width)[None, :]
    py = np.arange(cam.height)[:, None]
    sx = (2.0 * (px + 0.5) / cam.width - 1.0) * th * (cam.width / cam.height)
    sy = (1.0 - 2.0 * (py + 0.5) / cam.height) * th
    d = f[None, None, :] + sx[..., None] * r[None, None, :] + sy[..., None] * v[None, None, :]
    return _unit(d)


def render(phi, lx, ly, cam: Camera, iso: float = 0.0):
    """Returns (intensity [H, W], depth [H, W]); depth = -1 where the ray meets no surface."""
    nz, ny, nx = phi.shape
    N = nz - 1
    eye = np.asarray(cam.eye, dtype=np.float64)
    d = rays(cam)
    lo = np.array([0.0, 0.0, -1.0])
    hi = np.array([lx, ly, 1.0])
    with np.errstate(divide="ignore", invalid="ignore"):
        inv = 1.0 / d
        ta = (lo - eye) * inv
        tb = (hi - eye) * inv
    tmin = np.minimum(ta, tb)
    tmax = np.maximum(ta, tb)
    # a ray parallel to a slab and outside it never enters: t-range empty
    par = d == 0.0
    outside = par & ((eye < lo) | (eye > hi))
    tmin = np.where(par, -np.inf, tmin)
    tmax = np.where(par, np.inf, tmax)
    t0 = np.maximum(np.max(tmin, axis=-1), 0.0)
    t1 = np.min(tmax, axis=-1)
    alive = (t1 > t0) & ~np.any(outside, axis=-1)
    H, W = cam.height, cam.width
    intensity = np.zeros((H, W))
    depth = -np.ones((H, W))
    pts = lambda t: eye[None, None, :] + t[..., None] * d
    t_prev = t0.copy()
    g_prev = np.where(alive, sample_field(phi, lx, ly, pts(np.where(alive, t0, 0.0))) - iso, 0.0)
    found = np.zeros((H, W), dtype=bool)
    ta_, tb_ = np.zeros((H, W)), np.zeros((H, W))
    ga_ = np.zeros((H, W))
    nmax = int(np.ceil(np.max(np.where(alive, t1 - t0, 0.0)) / cam.step)) if alive.any() else 0
    for i in range(1, nmax + 1):
        live = alive & ~found & (t_prev < t1)
        if not live.any():
            break
        t = np.minimum(t0 + i * cam.step, t1)
        g = np.where(live, sample_field(phi, lx, ly, pts(np.where(live, t, 0.0))) - iso, 0.0)
        hit = live & ((g_prev < 0.0) != (g < 0.0))
        ta_ = np.where(hit, t_prev, ta_)
        tb_ = np.where(hit, t, tb_)
        ga_ = np.where(hit, g_prev, ga_)
        found |= hit
        g_prev = np.where(live, g, g_prev)
        t_prev = np.where(live, t, t_prev)
    for _ in range(NBIS):
        tm = 0.5 * (ta_ + tb_)
        gm = sample_field(phi, lx, ly, pts(tm)) - iso
        same = (gm < 0.0) == (ga_ < 0.0)
        ta_ = np.where(same, tm, ta_)
        ga_ = np.where(same, gm, ga_)
        tb_ = np.where(same, tb_, tm)
    th = 0.5 * (ta_ + tb_)
    p = pts(th)
    h = np.array([lx / nx, ly / ny, 1.0 / N])
    grad = np.stack([sample_field(phi, lx, ly, p + np.eye(3)[a] * h[a]) - sample_field(phi, lx, ly, p - np.eye(3)[a] * h[a])
                     for a in range(3)], axis=-1) / (2.0 * h)
    gn = np.sqrt(np.sum(grad * grad, axis=-1))
    light = _unit(np.asarray(cam.light, dtype=np.float64))
    with np.errstate(divide="ignore", invalid="ignore"):
        shade = 0.2 + 0.8 * np.abs(np.sum(grad * light, axis=-1) / gn)
    shade = np.where(gn > 0.0, shade, 0.2)
    intensity = np.where(found, shade, 0.0)
    depth = np.where(found, th, -1.0)
    return intensity, depth
