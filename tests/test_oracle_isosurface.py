"""Pins of the iso-surface ray-caster oracle (row f6) against geometry: an analytic sphere and a plane."""
import math

import numpy as np

import isosurface_oracle as R


def sphere_field(nx, ny, nz, lx, ly, centre, radius):
    x = lx / nx * np.arange(nx)[None, None, :]
    y = ly / ny * np.arange(ny)[None, :, None]
    z = np.cos(np.pi * np.arange(nz) / (nz - 1))[:, None, None]
    r = np.sqrt((x - centre[0]) ** 2 + (y - centre[1]) ** 2 + (z - centre[2]) ** 2)
    return radius - r                                     # phi > 0 inside, like a drop (reading S16)


def test_trilinear_sampling_reproduces_linear_fields_and_nodes():
    nx, ny, nz, lx, ly = 8, 8, 9, 2.0, 3.0
    z = np.cos(np.pi * np.arange(nz) / (nz - 1))[:, None, None]
    phi = 2.0 * z + 0.0 * np.zeros((nz, ny, nx))          # linear in z: exact on any (non-uniform) grid
    rng = np.random.default_rng(0)
    p = np.stack([rng.uniform(0, lx, 50), rng.uniform(0, ly, 50), rng.uniform(-1, 1, 50)], axis=-1)
    assert np.abs(R.sample_field(phi, lx, ly, p) - 2.0 * p[:, 2]).max() < 1e-14
    f = rng.standard_normal((nz, ny, nx))
    k, j, i = 3, 5, 2
    node = np.array([[i * lx / nx, j * ly / ny, math.cos(math.pi * k / (nz - 1))]])
    assert abs(R.sample_field(f, lx, ly, node)[0] - f[k, j, i]) < 1e-13
    wrapped = node + np.array([[lx, -ly, 0.0]])           # periodic in x, y
    assert abs(R.sample_field(f, lx, ly, wrapped)[0] - f[k, j, i]) < 1e-12


def test_sphere_depth_and_shading():
    nx, ny, nz, lx, ly = 96, 96, 97, 2.0, 2.0
    c, rad = (1.0, 1.0, 0.0), 0.5
    phi = sphere_field(nx, ny, nz, lx, ly, c, rad)
    cam = R.Camera(eye=(1.0, -3.0, 0.0), target=c, up=(0.0, 0.0, 1.0), fov_y_deg=30.0, width=33, height=33, step=0.01,
                   light=(0.0, -1.0, 0.0))
    inten, depth = R.render(phi, lx, ly, cam)
    mid = 16
    # central ray hits the sphere head on: depth = |eye - centre| - R, normal = -d, |n . l| = 1
    assert abs(depth[mid, mid] - (3.0 + 1.0 - rad)) < 2e-3          # O(h^2) interpolation error of the curved surface
    assert abs(inten[mid, mid] - 1.0) < 1e-3
    # silhouette: rays that pass the sphere at more than R miss, the corners certainly
    assert depth[0, 0] == -1.0 and inten[0, 0] == 0.0
    hit = depth > 0
    d = R.rays(cam)
    eye = np.array(cam.eye)
    # every hit point lies on the sphere to interpolation accuracy, and the shade is |n . l| with n the radial direction
    pts = eye + depth[..., None] * d
    rr = np.sqrt(np.sum((pts - np.array(c)) ** 2, axis=-1))
    assert np.abs(rr[hit] - rad).max() < 3e-3
    nrm = (pts - np.array(c)) / rr[..., None]
    shade = 0.2 + 0.8 * np.abs(nrm[..., 1])
    assert np.abs(inten[hit] - shade[hit]).max() < 2e-2
    # the set of hit pixels is the disc of the analytic sphere (up to one pixel at the rim)
    b = np.sum((eye - np.array(c)) * d, axis=-1)
    disc = b * b - (np.sum((eye - np.array(c)) ** 2) - rad * rad)
    sure_hit = disc > 0.03
    sure_miss = disc < -0.03
    assert hit[sure_hit].all() and not hit[sure_miss].any()


def test_plane_seen_obliquely():
    """phi = z - 0.25: the surface is the plane z = 0.25, exact for the trilinear interpolant; depth is analytic."""
    nx, ny, nz, lx, ly = 16, 16, 33, 4.0, 4.0
    z = np.cos(np.pi * np.arange(nz) / (nz - 1))[:, None, None]
    phi = z - 0.25 + np.zeros((nz, ny, nx))
    cam = R.Camera(eye=(2.0, 2.0, 0.9), target=(2.5, 2.2, -1.0), up=(0.0, 1.0, 0.0), fov_y_deg=20.0, width=9, height=7,
                   step=0.05, light=(0.0, 0.0, 1.0))
    inten, depth = R.render(phi, lx, ly, cam)
    d = R.rays(cam)
    want = (0.25 - 0.9) / d[..., 2]
    assert np.abs(depth - want).max() < 1e-6            # 24 bisections of a 0.05 bracket
    assert np.abs(inten - 1.0).max() < 1e-12            # normal = e_z = light
