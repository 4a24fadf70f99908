"""GPU parity of the wall variants (row f3; no-slip, free-slip "or a combination of them") against the
oracle: free-slip at both walls, and the two mixed assignments; with the phase field, single-phase, variable viscosity
and on grids that make the column sweeps run several CTAs."""
import numpy as np
import pytest

import psdns_inputs as I
from helpers import assert_parity, oracle_from_config, solver_from_config, to_dev, to_np

pytestmark = pytest.mark.gpu
TOL = 1e-9
NS, FS = 0, 1


def run(c, walls, nsteps, **over):
    import paper_2406_01322_b200 as P
    st = [f for f in I.channel_state(c) if f is not None]
    kw = dict(wall_top=walls[0], wall_bottom=walls[1], **over)
    orc, g = oracle_from_config(c, **kw)
    orc.set_state("physical", *st)
    s = solver_from_config(c, **kw)
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    done = 0
    for n in nsteps:
        orc.step(n - done)
        s.step(n - done)
        done = n
        assert_parity([to_np(t) for t in s.get_state(P.SPECTRAL)], orc.get_state("spectral"), TOL, tag=(c.name, walls, n))
    return s, orc


@pytest.mark.parametrize("walls", [(FS, FS), (FS, NS), (NS, FS)])
def test_walls_small_two_phase(walls):
    s, orc = run(I.small_config(nx=32, ny=32, nz=33), walls, [1, 2, 4])
    # the free wall slips, the other does not: u at the wall from the GPU state
    u = to_np(s.get_state(1)[0])
    top = np.abs(u.sum(axis=0)).max()
    bot = np.abs((u * ((-1.0) ** np.arange(u.shape[0]))[:, None, None]).sum(axis=0)).max()
    assert (top > 1e-3) == (walls[0] == FS) and (bot > 1e-3) == (walls[1] == FS), (top, bot)
    s.close()


@pytest.mark.parametrize("walls", [(FS, FS), (FS, NS)])
def test_walls_single_phase_and_ragged(walls):
    for (nx, ny, nz) in [(16, 64, 17), (64, 16, 65)]:
        s, _ = run(I.small_config(nx=nx, ny=ny, nz=nz, phase_field=0), walls, [3])
        s.close()


def test_walls_variable_viscosity_mixed():
    s, _ = run(I.small_config(nx=32, ny=16, nz=33, visc_ratio=0.3), (NS, FS), [2])
    s.close()


def test_walls_config2_grid_mixed():
    """128x128x129 (config-2 parameters): 7 k columns = look-ahead 4 sweeps, many CTAs per sweep."""
    c = I.CONFIGS[2]
    s, _ = run(c, (FS, NS), [2])
    s.close()


def test_invalid_wall_code_is_rejected():
    import paper_2406_01322_b200 as P
    with pytest.raises(P.PsdnsError):
        P.Solver(16, 16, 17, 1.0, 1.0, re=10.0, dt=1e-3, wall_top=2)
