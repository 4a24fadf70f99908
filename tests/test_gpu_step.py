"""GPU parity: psdns_step vs the oracle, element by element, through the C ABI.
Tolerance: relative L2 <= 1e-9 on all fields after N steps (BASELINE.json north_star)."""
import os

import numpy as np
import pytest

import psdns_inputs as I
import psdns_oracle as O
from helpers import field_errors, oracle_from_config, solver_from_config, to_dev, to_np

pytestmark = pytest.mark.gpu
TOL = 1e-9


def run_both(c, nsteps, space="physical", **over):
    import paper_2406_01322_b200 as P
    st = I.channel_state(c)
    if not over.get("phase_field", c.phase_field):
        st = st[:3]
    orc, g = oracle_from_config(c, **over)
    orc.set_state("physical", *st)
    s = solver_from_config(c, **over)
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    out = {}
    for n in nsteps:
        done = orc.state.nstep
        orc.step(n - done)
        s.step(n - done)
        ref = orc.get_state("spectral")
        got = [to_np(t) for t in s.get_state(P.SPECTRAL)]
        out[n] = field_errors(got, ref)
    # hidden state via physical space as well
    refp = orc.get_state("physical")
    gotp = [to_np(t) for t in s.get_state(P.PHYSICAL)]
    out["phys"] = field_errors(gotp, refp)
    return out, s, orc


def test_small_config_steps():
    c = I.small_config()
    errs, s, orc = run_both(c, [1, 2, 3])
    for k, (ev, ep) in errs.items():
        assert ev < TOL and ep < TOL, (k, ev, ep)


def test_config1_full():
    """BASELINE.json config 1: 32x32x33, 10 steps."""
    c = I.CONFIGS[1]
    errs, s, orc = run_both(c, [1, 5, 10])
    for k, (ev, ep) in errs.items():
        assert ev < TOL and ep < TOL, (k, ev, ep)
    assert s.launch_count() > 0


def test_single_phase():
    c = I.small_config(nx=32, ny=16, nz=33, phase_field=0)
    errs, *_ = run_both(c, [1, 4], phase_field=0)
    for k, (ev, ep) in errs.items():
        assert ev < TOL, (k, ev)


def test_variable_viscosity():
    """Config-4 physics (lambda = 0.1, reading S14) on a small grid."""
    c = I.small_config(nx=32, ny=32, nz=33, visc_ratio=0.1)
    errs, *_ = run_both(c, [1, 3])
    for k, (ev, ep) in errs.items():
        assert ev < TOL and ep < TOL, (k, ev, ep)


def test_variable_viscosity_wide_and_ragged():
    """The 16-slot fused x kernel of the variable-viscosity step at other radix plans, incl. nx = 1024."""
    for (nx, ny, nz) in [(16, 32, 17), (128, 16, 17), (512, 16, 9), (1024, 16, 9)]:
        c = I.small_config(nx=nx, ny=ny, nz=nz, visc_ratio=0.3)
        errs, *_ = run_both(c, [2])
        for k, (ev, ep) in errs.items():
            assert ev < TOL and ep < TOL, (nx, k, ev, ep)


def test_ragged_shapes():
    """nx != ny != nz-1, padded kx pitch (nkx = 6 -> 8, 22 -> 24) and several column tiles."""
    for (nx, ny, nz) in [(16, 64, 17), (64, 16, 65)]:
        c = I.small_config(nx=nx, ny=ny, nz=nz)
        errs, *_ = run_both(c, [2])
        for k, (ev, ep) in errs.items():
            assert ev < TOL and ep < TOL, (nx, ny, nz, k, ev, ep)


def test_extreme_supported_sizes():
    """Smallest and largest supported line lengths (R4): ny = 1024 (one-CTA-per-SM y pass), nx = ny = 16, nz = 9."""
    for (nx, ny, nz) in [(16, 1024, 9), (16, 16, 9), (1024, 16, 9)]:
        c = I.small_config(nx=nx, ny=ny, nz=nz, band=2)
        errs, *_ = run_both(c, [2])
        for k, (ev, ep) in errs.items():
            assert ev < TOL and ep < TOL, (nx, ny, nz, k, ev, ep)


def test_spectral_set_state_equals_physical():
    import paper_2406_01322_b200 as P
    c = I.small_config()
    st = I.channel_state(c)
    orc, g = oracle_from_config(c)
    orc.set_state("physical", *st)
    spec = orc.get_state("spectral")
    s = solver_from_config(c)
    s.set_state(P.SPECTRAL, *[to_dev(a) for a in spec])
    s.step(2)
    orc.step(2)
    ev, ep = field_errors([to_np(t) for t in s.get_state(P.SPECTRAL)], orc.get_state("spectral"))
    assert ev < TOL and ep < TOL


def test_config2_short():
    """BASELINE.json config 2 (128x128x129) for a few steps; PSDNS_FULL=1 runs all 100."""
    c = I.CONFIGS[2]
    n = c.steps if os.environ.get("PSDNS_FULL") else 3
    errs, *_ = run_both(c, [n])
    for k, (ev, ep) in errs.items():
        assert ev < TOL and ep < TOL, (k, ev, ep)


def test_error_codes():
    import ctypes as C
    import torch
    import paper_2406_01322_b200 as P
    from paper_2406_01322_b200.binding import load_library, psdns_grid, psdns_params
    lib = load_library()
    g = psdns_grid(30, 32, 33, 1.0, 1.0)
    p = psdns_params(100, 1, 1, 1, 1e-3, 0, 1, 1, 1)
    assert lib.psdns_workspace_bytes(C.byref(g), C.byref(p)) == 0
    h = C.c_void_p()
    assert lib.psdns_init(C.byref(g), C.byref(p), None, 0, None, C.byref(h)) == -1
    s = P.Solver(16, 16, 17, 1.0, 1.0, re=10.0, dt=1e-3, phase_field=0)
    with pytest.raises(P.PsdnsError):
        s.step(1)                      # PSDNS_ESTATE: no state yet
    u = torch.zeros(17, 16, 16, dtype=torch.float64, device="cuda")
    assert lib.psdns_set_state(s.handle, 0, u.data_ptr(), None, u.data_ptr(), None) == -1
    ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    g2 = psdns_grid(16, 16, 17, 1.0, 1.0)
    assert lib.psdns_init(C.byref(g2), C.byref(p), ws.data_ptr(), 1024, None, C.byref(h)) == -2


def test_exact_restart_through_history_blob():
    """psdns_get_state + psdns_get_history -> a NEW handle -> psdns_set_state + psdns_set_history: the continued run
    is bit-identical to the uninterrupted one (hidden theta^, omega_z^, D phi^, AB2 history, step counter)."""
    import torch
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=32, ny=16, nz=33)
    st = I.channel_state(c)
    a = solver_from_config(c)
    a.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    a.step(5)
    ref = a.get_state(P.SPECTRAL)
    b = solver_from_config(c)
    b.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    b.step(2)
    state, blob = b.get_state(P.SPECTRAL), b.get_history()
    b.close()
    r = solver_from_config(c)
    with pytest.raises(P.PsdnsError):
        r.set_history(blob)            # PSDNS_ESTATE: set_state first
    r.set_state(P.SPECTRAL, *state)
    r.set_history(blob)
    r.step(3)
    got = r.get_state(P.SPECTRAL)
    for x, y in zip(got, ref):
        assert torch.equal(x, y)
    # without the blob the restart is an Euler start from a re-derived theta: close, but not identical
    r2 = solver_from_config(c)
    r2.set_state(P.SPECTRAL, *state)
    r2.step(3)
    assert not all(torch.equal(x, y) for x, y in zip(r2.get_state(P.SPECTRAL), ref))
    assert r.lib.psdns_set_history(r.handle, None, 0) == -1


def test_nx1024_single_line_x_kernel():
    """nx = 1024 runs the single-line warp-per-field fused x kernel (the one the 1024x512x513 bench runs): element-by-element
    parity on a grid that is wide in x only, with and without the phase field."""
    for phase in (1, 0):
        c = I.small_config(nx=1024, ny=16, nz=9, phase_field=phase)
        errs, *_ = run_both(c, [2], phase_field=phase)
        for k, (ev, ep) in errs.items():
            assert ev < TOL and ep < TOL, (phase, k, ev, ep)


def test_multi_line_x_kernel_plans():
    """nx < 1024 runs the multi-line warp-per-field kernel (k_xfusedwm): 16, 4, 2, 2 lines per CTA iteration and the
    radix plans 16 | 8*4*2 | 8*8*2 | 16*8*2."""
    for (nx, ny, nz) in [(32, 16, 17), (128, 32, 9), (256, 16, 9), (512, 16, 9)]:
        c = I.small_config(nx=nx, ny=ny, nz=nz)
        errs, *_ = run_both(c, [2])
        for k, (ev, ep) in errs.items():
            assert ev < TOL and ep < TOL, (nx, k, ev, ep)


def test_run_host_pipelined_calls_match_device_path():
    """psdns_run_host: three back-to-back calls with different inputs and separate output buffers (the copy-back of one
    call runs on the side stream while the next call uploads and computes) give exactly what set_state / step / get_state
    give on device buffers."""
    import torch
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=32, ny=32, nz=33)
    base = [f for f in I.channel_state(c)]
    s = solver_from_config(c)
    ins, outs, refs = [], [], []
    for k in range(3):
        st = [np.ascontiguousarray(f * (1.0 + 0.1 * k)) for f in base]
        ins.append([torch.from_numpy(a).pin_memory() for a in st])
        outs.append([torch.empty_like(t).pin_memory() for t in ins[-1]])
        s.set_state(P.PHYSICAL, *[t.cuda() for t in ins[-1]])
        s.step(2)
        refs.append([t.cpu() for t in s.get_state(P.PHYSICAL)])
    for k in range(3):
        s.run_host(P.PHYSICAL, 2, ins[k], outs[k])
    s.run_host_wait()
    for k in range(3):
        for a, b in zip(outs[k], refs[k]):
            assert torch.equal(a, b), k
    s.close()
