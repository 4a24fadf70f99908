"""GPU parity of psdns_render_isosurface (row f6: the phi = 0 iso-surface ray-caster as a CUDA kernel writing into
device buffers, PAPER.md L260 / Fig. 5) against oracle/isosurface_oracle.py, pixel by pixel.
Depth and intensity are float64 on both sides.  A ray that grazes the surface can find its sign change on one side and
miss it on the other when the two fields differ in the last bits, so: the hit masks must agree on all but a handful of
silhouette pixels, and wherever both hit, depth and shade must agree to rounding."""
import numpy as np
import pytest

import isosurface_oracle as R
import psdns_inputs as I
from helpers import oracle_from_config, solver_from_config, to_dev, to_np

pytestmark = pytest.mark.gpu


def compare(gi, gd, oi, od, max_flips):
    ghit, ohit = gd >= 0, od >= 0
    assert (ghit != ohit).sum() <= max_flips, int((ghit != ohit).sum())
    both = ghit & ohit
    assert both.sum() > 50
    assert np.abs(gd[both] - od[both]).max() < 1e-8, np.abs(gd[both] - od[both]).max()
    assert np.abs(gi[both] - oi[both]).max() < 1e-7, np.abs(gi[both] - oi[both]).max()
    assert np.all(gi[~ghit] == 0.0) and np.all(gd[~ghit] == -1.0)


def test_external_field_sphere_and_plane():
    import paper_2406_01322_b200 as P
    nx, ny, nz, lx, ly = 64, 64, 65, 2.0, 2.0
    x = lx / nx * np.arange(nx)[None, None, :]
    y = ly / ny * np.arange(ny)[None, :, None]
    z = np.cos(np.pi * np.arange(nz) / (nz - 1))[:, None, None]
    phi = 0.5 - np.sqrt((x - 1.0) ** 2 + (y - 1.0) ** 2 + (z - 0.1) ** 2)
    s = P.Solver(nx, ny, nz, lx, ly, re=100.0, dt=1e-3, phase_field=0)
    cam = R.Camera(eye=(1.3, -3.0, 0.4), target=(1.0, 1.0, 0.1), up=(0.0, 0.0, 1.0), fov_y_deg=28.0, width=80, height=60,
                   step=0.015, light=(0.3, -0.5, 0.8))
    gi, gd = s.render_isosurface(cam.eye, cam.target, cam.up, cam.fov_y_deg, cam.width, cam.height, cam.step, cam.light,
                                 iso=0.0, field=to_dev(phi))
    oi, od = R.render(phi, lx, ly, cam)
    compare(to_np(gi), to_np(gd), oi, od, max_flips=0)
    # a second iso value and a camera inside the box looking along +x
    cam2 = R.Camera(eye=(0.05, 1.0, 0.0), target=(2.0, 1.1, 0.1), up=(0.0, 0.0, 1.0), fov_y_deg=50.0, width=48, height=48,
                    step=0.02, light=(1.0, 0.0, 0.0))
    gi, gd = s.render_isosurface(cam2.eye, cam2.target, cam2.up, cam2.fov_y_deg, cam2.width, cam2.height, cam2.step,
                                 cam2.light, iso=0.2, field=to_dev(phi))
    oi, od = R.render(phi, lx, ly, cam2, iso=0.2)
    compare(to_np(gi), to_np(gd), oi, od, max_flips=0)
    s.close()


def test_state_phase_field_after_steps():
    """The drop of a small channel state, stepped on both sides, rendered from the STATE (d_field = NULL: the library
    brings phi to physical space itself) against the oracle's render of the oracle's physical phi."""
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=32, ny=32, nz=33)
    st = I.channel_state(c)
    orc, g = oracle_from_config(c)
    orc.set_state("physical", *st)
    orc.step(2)
    s = solver_from_config(c)
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    s.step(2)
    cam = R.Camera(eye=(0.5 * c.lx + 0.4, -1.5, 0.5), target=(0.5 * c.lx, 0.5 * c.ly, 0.0), fov_y_deg=30.0, width=64, height=48,
                   step=0.03, light=(0.2, -0.6, 0.7))
    gi, gd = s.render_isosurface(cam.eye, cam.target, cam.up, cam.fov_y_deg, cam.width, cam.height, cam.step, cam.light)
    oi, od = R.render(orc.get_state("physical")[3], c.lx, c.ly, cam)
    compare(to_np(gi), to_np(gd), oi, od, max_flips=2)
    assert (od >= 0).sum() > 100                              # the drop is in view
    s.close()


def test_render_errors():
    import paper_2406_01322_b200 as P
    s = P.Solver(16, 16, 17, 1.0, 1.0, re=10.0, dt=1e-3, phase_field=0)
    with pytest.raises(P.PsdnsError):
        s.render_isosurface((0, -1, 0), (0.5, 0.5, 0))        # no phase field and no d_field
    with pytest.raises(P.PsdnsError):
        s.render_isosurface((0, -1, 0), (0, 1, 0), up=(0, 1, 0), field=to_dev(np.zeros((17, 16, 16))))   # up || view
    s.close()
