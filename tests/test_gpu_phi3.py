"""The two-stage problems in three sweeps (kernels_spectral.cuh, ElimUpNeu / ElimUpDir2: the second Helmholtz solve of the
phi and of the w problem is eliminated UPWARDS inside the up sweep that produces its right-hand side, and back-substituted
by k_finish on its way down) against the five-sweep form of the same solves (`psdns_set_option("phi3" / "w3", 0)`): both
are Gauss eliminations of the same diagonally dominant systems, so the states agree to rounding - on every variant of
the step.  Parity with
the oracle is covered by the ordinary step tests, which run the default (three-sweep) path."""
import numpy as np
import pytest

import psdns_inputs as I
from helpers import solver_from_config, to_dev, to_np

pytestmark = pytest.mark.gpu

CASES = [
    dict(nx=32, ny=32, nz=33),
    dict(nx=16, ny=16, nz=9),                                   # shortest column: rows 2..8 only
    dict(nx=64, ny=16, nz=65),
    dict(nx=128, ny=64, nz=129, over=dict(visc_ratio=0.5)),     # variable viscosity (k_xfusedv)
    dict(nx=32, ny=64, nz=33, over=dict(wall_top=1, wall_bottom=0)),          # mixed walls: 2 x 2 influence closure
    dict(nx=64, ny=32, nz=33, over=dict(wall_top=0, wall_bottom=1)),
    dict(nx=32, ny=32, nz=65, over=dict(wall_top=1, wall_bottom=1)),          # free-slip at both walls
    dict(nx=32, ny=32, nz=33, over=dict(surface_tension_form=1)),             # force form, three-kernel x path
    dict(nx=256, ny=128, nz=129),                               # 11 k columns: the look-ahead depth of small grids
    dict(nx=64, ny=32, nz=65, cfg=dict(phase_field=0)),         # single-phase: the w problem alone
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "%dx%dx%d%s" % (c["nx"], c["ny"], c["nz"], "".join("-" + k for k in {**c.get("over", {}), **c.get("cfg", {})})))
def test_three_sweep_phi_equals_five_sweep(case):
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=case["nx"], ny=case["ny"], nz=case["nz"], **case.get("cfg", {}))
    st = [f for f in I.channel_state(c) if f is not None]
    outs = []
    for opt in (0, 1, 2, 3):         # five sweeps | phi in three | phi and w in three | + lazy theta correction (the default)
        s = solver_from_config(c, **case.get("over", {}))
        s.set_option("phi3", int(opt >= 1))
        s.set_option("w3", int(opt >= 2))
        s.set_option("lazy", int(opt >= 3))
        s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
        s.step(4)
        outs.append([to_np(t) for t in s.get_state(P.SPECTRAL)])
        s.close()
    vel = max(float(np.abs(a).max()) for a in outs[0][:3])
    for other in outs[1:]:
        for name, a, b, scale in zip("uvwp", outs[0], other, (vel, vel, vel, float(np.abs(outs[0][-1]).max()))):
            assert np.all(np.isfinite(b)), name
            assert float(np.abs(a - b).max()) <= 1e-12 * scale, (name, float(np.abs(a - b).max()), scale)


def test_three_sweep_phi_many_columns():
    """Above 60 k columns the sweeps use the shallow register look-ahead (G = 2): 512 x 512 x 17."""
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=512, ny=512, nz=17, band=2)
    st = I.channel_state(c)
    outs = []
    for opt in (0, 1):
        s = solver_from_config(c)
        s.set_option("phi3", opt)
        s.set_option("w3", opt)
        s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
        s.step(3)
        outs.append([to_np(t) for t in s.get_state(P.SPECTRAL)])
        s.close()
    for a, b in zip(*outs):
        assert float(np.abs(a - b).max()) <= 1e-12 * max(float(np.abs(a).max()), 1.0)


def test_lazy_theta_correction_survives_restart_and_option_changes():
    """The three-sweep form leaves theta^ = theta_p + (coefficients of A_par theta_h) between steps.  psdns_get_history must
    hand out the completed theta^ (bit-exact restart), and changing an option in the middle of a run must not lose or
    double the pending correction."""
    import torch
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=64, ny=32, nz=33)
    st = I.channel_state(c)

    def fresh():
        s = solver_from_config(c)
        s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
        return s

    a = fresh()
    a.step(6)
    ref = [to_np(t) for t in a.get_state(P.SPECTRAL)]
    a.close()
    # restart in the middle through the history blob
    b = fresh()
    b.step(3)
    blob = b.get_history()
    mid = [t.clone() for t in b.get_state(P.SPECTRAL)]
    b.step(3)
    cont = [to_np(t) for t in b.get_state(P.SPECTRAL)]
    b.close()
    r = solver_from_config(c)
    r.set_state(P.SPECTRAL, *mid)
    r.set_history(blob)
    r.step(3)
    rest = [to_np(t) for t in r.get_state(P.SPECTRAL)]
    r.close()
    for x, y, z in zip(ref, cont, rest):
        assert np.array_equal(x, y)            # taking the blob does not disturb the run
        assert np.array_equal(y, z)            # and the restart is bit-exact
    # switch the lazy correction off and on again in mid-run: rounding-level agreement with the plain run
    d = fresh()
    d.step(2); d.set_option("lazy", 0); d.step(2); d.set_option("w3", 0); d.step(1); d.set_option("w3", 1); d.set_option("lazy", 1); d.step(1)
    mixed = [to_np(t) for t in d.get_state(P.SPECTRAL)]
    d.close()
    vel = max(float(np.abs(x).max()) for x in ref[:3])
    for x, y, scale in zip(ref, mixed, (vel, vel, vel, float(np.abs(ref[3]).max()))):
        assert float(np.abs(x - y).max()) <= 1e-12 * scale


def test_launches_per_step():
    """One step of the default (three-sweep) path is nine launches in the captured graph: k_begin_step, z / y backward,
    fused x, y / z forward, k_rhs_elim, k_subst3, k_finish; the five-sweep form has two more."""
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=32, ny=32, nz=33)
    st = I.channel_state(c)
    for opts, want in (({}, 9), ({"w3": 0}, 11), ({"w3": 0, "phi3": 0}, 11)):
        s = solver_from_config(c)
        for k, v in opts.items():
            s.set_option(k, v)
        s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
        s.step(2)
        assert int(s.get_info("launches_per_step")) == want, (opts, s.get_info("launches_per_step"))
        s.close()
