"""GPU parity on seeded random COMBINATIONS of grid, physics, walls, non-linear forms and kernel options against the live
oracle: every switch of psdns_params and psdns_set_option is tested on its own elsewhere; this sweep checks that they
compose (variable viscosity with mixed walls, rotational convection with the GEMM-form z pass, capped grids with the
register-fed z pass, ...)."""
import numpy as np
import pytest

import psdns_inputs as I
from helpers import assert_parity, oracle_from_config, solver_from_config, to_dev, to_np

pytestmark = pytest.mark.gpu
TOL = 1e-9


def draw(seed):
    rng = np.random.default_rng(4200 + seed)
    nx = int(rng.choice([16, 32, 64, 128]))
    ny = int(rng.choice([16, 32, 64]))
    nz = int(rng.choice([9, 17, 33, 65])) if nx * ny <= 2048 else int(rng.choice([9, 17, 33]))
    phase = int(rng.random() < 0.8)
    visc = float(rng.choice([1.0, 1.0, 0.2, 3.0])) if phase else 1.0
    forms = dict(surface_tension_form=0, convection_form=0)
    if visc == 1.0 and rng.random() < 0.4:
        forms = dict(surface_tension_form=int(phase and rng.random() < 0.5), convection_form=int(rng.random() < 0.6))
    phys = dict(re=float(rng.choice([50.0, 300.0, 3000.0])), dt=float(rng.choice([1e-3, 1e-4, 2e-5])),
                ch=float(rng.choice([0.15, 0.25, 0.4])), pe=float(rng.choice([2.0, 5.0, 20.0])), we=float(rng.choice([0.5, 1.0, 3.0])))
    walls = dict(wall_top=int(rng.random() < 0.4), wall_bottom=int(rng.random() < 0.4))
    fused = forms["surface_tension_form"] == 0 and forms["convection_form"] == 0
    opts = dict(ztma=int(rng.random() < 0.7), zgemm=int(nz <= 65 and rng.random() < 0.25), grid_cap=int(rng.choice([0, 0, 2, 5])),
                graph=int(rng.random() < 0.7))
    if fused and rng.random() < 0.2:
        opts["xfuse"] = 0
    nsteps = int(rng.integers(1, 4))
    return dict(nx=nx, ny=ny, nz=nz, phase=phase, visc=visc, forms=forms, phys=phys, walls=walls, opts=opts, nsteps=nsteps)


@pytest.mark.parametrize("seed", range(48))
def test_random_combination(seed):
    import paper_2406_01322_b200 as P
    k = draw(seed)
    c = I.small_config(nx=k["nx"], ny=k["ny"], nz=k["nz"], phase_field=k["phase"], visc_ratio=k["visc"], seed=100 + seed,
                       band=int(min(3, k["nx"] // 3 - 1, k["ny"] // 3 - 1)), **k["phys"])
    st = [f for f in I.channel_state(c) if f is not None]
    over = dict(**k["forms"], **k["walls"])
    orc, g = oracle_from_config(c, **over)
    orc.set_state("physical", *st)
    orc.step(k["nsteps"])
    s = solver_from_config(c, unfused_workspace=k["opts"].get("xfuse") == 0, **over)
    for name, v in k["opts"].items():
        s.set_option(name, v)
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    s.step(k["nsteps"])
    assert_parity([to_np(t) for t in s.get_state(P.SPECTRAL)], orc.get_state("spectral"), TOL, tag=k)
    d = dict(zip(P.Solver.DIAG_NAMES, s.diagnostics().cpu().numpy()))
    assert np.isfinite(list(d.values())).all() and d["max_div"] < 1e-9 * k["nz"] ** 2, d
    s.close()
