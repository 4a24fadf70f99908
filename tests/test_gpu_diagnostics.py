"""GPU parity of psdns_diagnostics (row f2: mean phi, max |div u|, kinetic energy, wall shear, bulk velocity computed on
the device from the resident spectra) against the oracle's plain definitions (physical-space quadrature, dense D)."""
import numpy as np
import pytest

import psdns_inputs as I
import psdns_oracle as O
from helpers import oracle_from_config, solver_from_config, to_dev

pytestmark = pytest.mark.gpu


def oracle_diag(g, st):
    u, v, w, phi = st
    top, bot = O.wall_shear(g, u)
    return dict(mean_phi=O.mean_phi(g, phi) if phi is not None else 0.0, max_div=O.max_divergence(g, u, v, w),
                kinetic_energy=O.kinetic_energy(g, u, v, w), shear_top=top, shear_bottom=bot,
                bulk_velocity=O.bulk_velocity(g, u))


def check(got, ref, scale_div):
    for k in ("mean_phi", "kinetic_energy", "shear_top", "shear_bottom", "bulk_velocity"):
        assert abs(got[k] - ref[k]) <= 1e-11 * max(abs(ref[k]), 1.0), (k, got[k], ref[k])
    assert abs(got["max_div"] - ref["max_div"]) <= 1e-11 * scale_div, (got["max_div"], ref["max_div"])


@pytest.mark.parametrize("nx,ny,nz", [(32, 32, 33), (64, 16, 65)])
def test_diagnostics_channel_state_after_steps(nx, ny, nz):
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=nx, ny=ny, nz=nz)
    st = I.channel_state(c)
    orc, g = oracle_from_config(c)
    orc.set_state("physical", *st)
    s = solver_from_config(c)
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    for nsteps in (0, 2):
        orc.step(nsteps)
        s.step(nsteps)
        d = s.diagnostics().cpu().numpy()
        got = dict(zip(P.Solver.DIAG_NAMES, d))
        ref = oracle_diag(g, orc.get_state("spectral"))
        vmax = max(float(np.abs(a).max()) for a in orc.get_state("spectral")[:3])
        check(got, ref, scale_div=vmax * nz * nz)       # after a step div u = 0 algebraically: both sides are rounding
        assert got["kinetic_energy"] > 0.2 and abs(got["shear_top"] + 2.0) < 0.5     # Poiseuille + perturbation
        assert d[6] == 0.0 and d[7] == 0.0
    s.close()


def test_diagnostics_of_a_non_solenoidal_state():
    """Random spectra (no continuity, no no-slip): max |div u| is O(100) and must agree to rounding."""
    import paper_2406_01322_b200 as P
    nx, ny, nz = 64, 32, 33
    st = list(I.random_spectral_state(nx, ny, nz, 11, cut=True))
    g = O.Grid(nx, ny, nz)
    s = P.Solver(nx, ny, nz, g.lx, g.ly, re=100.0, dt=1e-4, pe=4.0, ch=0.25, we=1.0)
    s.set_state(P.SPECTRAL, *[to_dev(a) for a in st])
    got = dict(zip(P.Solver.DIAG_NAMES, s.diagnostics().cpu().numpy()))
    ref = oracle_diag(g, st)
    assert ref["max_div"] > 1e-2
    check(got, ref, scale_div=ref["max_div"])
    s.close()


def test_diagnostics_single_phase_and_errors():
    import torch
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=32, ny=16, nz=17, phase_field=0)
    s = solver_from_config(c)
    with pytest.raises(P.PsdnsError):
        s.diagnostics()                                    # PSDNS_ESTATE
    st = I.channel_state(c)[:3]
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    d = s.diagnostics().cpu().numpy()
    assert d[0] == 0.0 and np.isfinite(d).all()
    assert s.lib.psdns_diagnostics(s.handle, None) == -1
    s.close()


def test_fp64_peak_microbenchmark_is_plausible():
    """psdns_measure_fp64_peak (SURVEY 8(d) FMA-chain microbenchmark): between half and 1.2x of the nominal
    148 SMs x 64 FMA/clk x 2 x 1.965 GHz = 37.2 TFLOP/s on a B200."""
    import paper_2406_01322_b200 as P
    s = P.Solver(32, 32, 33, 12.5, 6.3, re=100.0, dt=1e-3, phase_field=0)
    tf = s.measure_fp64_peak()
    assert 18.0 < tf < 45.0, tf
    s.close()
