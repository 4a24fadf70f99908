"""GPU parity of the alternative non-linear form (row f4): the surface tension evaluated as the force
-c_sigma lap(phi) grad(phi) (psdns_params.surface_tension_form = 1) instead of the divergence of the Korteweg tensor,
against the oracle with the same switch."""
import numpy as np
import pytest

import psdns_inputs as I
from helpers import assert_parity, oracle_from_config, solver_from_config, to_dev, to_np

pytestmark = pytest.mark.gpu
TOL = 1e-9


def run(c, nsteps, **over):
    import paper_2406_01322_b200 as P
    st = [f for f in I.channel_state(c) if f is not None]
    over.setdefault("surface_tension_form", 1)
    orc, g = oracle_from_config(c, **over)
    orc.set_state("physical", *st)
    s = solver_from_config(c, **over)
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    done = 0
    for n in nsteps:
        orc.step(n - done)
        s.step(n - done)
        done = n
        assert_parity([to_np(t) for t in s.get_state(P.SPECTRAL)], orc.get_state("spectral"), TOL, tag=(c.name, n))
    return s, orc


def test_force_form_small_and_config1():
    for c in (I.small_config(), I.CONFIGS[1]):
        s, _ = run(c, [1, 2, 5])
        s.close()


def test_force_form_ragged_and_mixed_walls():
    for (nx, ny, nz) in [(16, 64, 17), (64, 16, 65)]:
        s, _ = run(I.small_config(nx=nx, ny=ny, nz=nz), [3])
        s.close()
    s, _ = run(I.small_config(nx=32, ny=32, nz=33), [2], wall_top=1, wall_bottom=0)
    s.close()


def test_force_form_differs_from_the_tensor_form_and_config2_grid():
    """On config 2's grid (128x128x129): parity with the oracle's form 1, and a visible (truncation-level) difference to the
    default form 0 - the switch really selects another discrete operator."""
    import paper_2406_01322_b200 as P
    c = I.CONFIGS[2]
    s, orc = run(c, [2])
    got1 = [to_np(t) for t in s.get_state(P.SPECTRAL)]
    s.close()
    s0 = solver_from_config(c)
    s0.set_state(P.PHYSICAL, *[to_dev(f) for f in I.channel_state(c)])
    s0.step(2)
    got0 = [to_np(t) for t in s0.get_state(P.SPECTRAL)]
    s0.close()
    d = np.sqrt(sum(np.linalg.norm(a - b) ** 2 for a, b in zip(got1[:3], got0[:3]))) / np.sqrt(sum(np.linalg.norm(b) ** 2 for b in got0[:3]))
    assert 1e-13 < d < 1e-3, d


@pytest.mark.parametrize("st_form,phase", [(0, 1), (1, 1), (0, 0)])
def test_rotational_form_of_convection(st_form, phase):
    """convection_form = 1 (u x omega; vorticity spectra from k_prep, three more backward fields), alone, together with the
    force form of the surface tension (then the flux tensor is empty), and single-phase; ragged grid and mixed walls too."""
    for (nx, ny, nz, kw) in [(32, 32, 33, {}), (16, 64, 17, {}), (64, 16, 65, dict(wall_top=1))]:
        c = I.small_config(nx=nx, ny=ny, nz=nz, phase_field=phase)
        s, _ = run(c, [1, 3], convection_form=1, surface_tension_form=st_form, **kw)
        s.close()


def test_force_form_rejects_unsupported_combinations():
    import paper_2406_01322_b200 as P
    with pytest.raises(P.PsdnsError):
        P.Solver(16, 16, 17, 1.0, 1.0, re=10.0, dt=1e-3, phase_field=0, surface_tension_form=1)
    with pytest.raises(P.PsdnsError):
        P.Solver(16, 16, 17, 1.0, 1.0, re=10.0, dt=1e-3, pe=1.0, ch=0.2, we=1.0, visc_ratio=0.5, surface_tension_form=1)
    with pytest.raises(P.PsdnsError):
        P.Solver(16, 16, 17, 1.0, 1.0, re=10.0, dt=1e-3, pe=1.0, ch=0.2, we=1.0, visc_ratio=0.5, convection_form=1)
    for kw in (dict(surface_tension_form=1), dict(convection_form=1)):
        s = P.Solver(16, 16, 17, 1.0, 1.0, re=10.0, dt=1e-3, pe=1.0, ch=0.2, we=1.0, **kw)
        with pytest.raises(P.PsdnsError):
            s.set_option("xfuse", 1)
        s.close()
