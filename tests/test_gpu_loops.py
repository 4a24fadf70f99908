"""GPU parity of the PERSISTENT kernels in the mode the full-size bench runs them: every CTA walks several tiles /
lines (stage reuse, mbarrier parity flips, the service warp's bulk prefetch of line + gridDim.x, look-ahead tiles).

Two kinds of test:
  * live-oracle parity on thin slabs that have the FULL line length of the 1024x512x513 bench grid in one direction
    (nx = 1024, ny = 512, nz = 513) and more work items than the one-wave grid, or a grid capped through
    psdns_set_option("grid_cap") so that each CTA iterates many times; states are the bench's random spectra
    (psdns_inputs.random_spectral_state, which satisfies neither no-slip nor continuity) as well as channel states;
  * capped vs uncapped runs of the same step must agree BIT FOR BIT (a tile's arithmetic does not depend on which CTA
    runs it), on grids too large for the live oracle.
Every test asserts grid < work items through psdns_get_info, so the intent cannot rot."""
import numpy as np
import pytest

import psdns_inputs as I
import psdns_oracle as O
from helpers import assert_parity, oracle_from_config, solver_from_config, to_dev, to_np

pytestmark = pytest.mark.gpu
TOL = 1e-9
PERSISTENT = ("zbwd", "ybwd", "xfused", "yfwd", "zfwd")


def scaling_like(nx, ny, nz, **kw):
    """Config-5 step parameters on an arbitrary grid."""
    base = dict(re=3000.0, ch=0.025, pe=40.0, we=1.0, dt=2e-5, steps=2, seed=1005)
    base.update(kw)
    return I.Config(f"cfg5-{nx}x{ny}x{nz}", nx, ny, nz, **base)


def state_of(c, kind):
    if kind == "random":
        st = list(I.random_spectral_state(c.nx, c.ny, c.nz, c.seed, cut=True))
        return "spectral", (st if c.phase_field else st[:3])
    st = I.channel_state(c)
    return "physical", [f for f in st if f is not None]


def run_parity(c, kind, nsteps, cap=0, looping=PERSISTENT, min_iters=2.0):
    import paper_2406_01322_b200 as P
    space, st = state_of(c, kind)
    orc, g = oracle_from_config(c)
    orc.set_state(space, *st)
    orc.step(nsteps)
    s = solver_from_config(c)
    if cap:
        s.set_option("grid_cap", cap)
    s.set_state(P.SPECTRAL if space == "spectral" else P.PHYSICAL, *[to_dev(f) for f in st])
    s.step(nsteps)
    got = [to_np(t) for t in s.get_state(P.SPECTRAL)]
    info = {k: (s.get_info(k + "_grid"), s.get_info(k + "_items")) for k in PERSISTENT}
    for k in looping:
        grid, items = info[k]
        assert grid > 0 and items >= min_iters * grid, (k, grid, items)
    res = assert_parity(got, orc.get_state("spectral"), TOL, tag=(c.name, kind, cap))
    s.close()
    return res, info


@pytest.mark.parametrize("phase,visc", [(1, 1.0), (0, 1.0), (1, 0.3)])
def test_nx1024_x_kernel_loops_uncapped(phase, visc):
    """1024x64x9: 576 lines on a one-wave grid of <= 296 CTAs - the single-line warp-per-field kernel k_xfusedw<1024>
    (and the 16-slot k_xfusedv<1024>) walks 2+ lines per CTA with its natural grid, random-spectra state."""
    c = scaling_like(1024, 64, 9, phase_field=phase, visc_ratio=visc)
    run_parity(c, "random", 2, looping=("xfused",), min_iters=1.9)


@pytest.mark.parametrize("phase", [1, 0])
def test_nx1024_x_kernel_loops_capped(phase):
    """1024x32x17 with 8 CTAs: 68 lines per CTA through every stage buffer and barrier phase."""
    c = scaling_like(1024, 32, 17, phase_field=phase)
    run_parity(c, "random", 2, cap=8, min_iters=3.0)


@pytest.mark.parametrize("nx,ny,nz,phase", [(512, 64, 9, 1), (512, 64, 9, 0), (256, 64, 9, 0), (128, 32, 17, 1)])
def test_multi_line_x_kernel_loops(nx, ny, nz, phase):
    """k_xfusedwm<512 / 256 / 128> (2 / 2 / 4 lines per iteration), both phase settings, capped to 6 CTAs."""
    c = scaling_like(nx, ny, nz, phase_field=phase)
    run_parity(c, "random", 2, cap=6, min_iters=3.0)


def test_ny512_y_pass_pruned_loops():
    """16x512x9: k_ypass<512> with the pruned (341 of 512 rows) spectral side, several tiles per CTA."""
    c = scaling_like(16, 512, 9)
    run_parity(c, "random", 2, cap=2, min_iters=3.0)


@pytest.mark.parametrize("nx,ny,kind", [(16, 16, "random"), (32, 32, "channel")])
def test_nz513_z_pass_truncated_loops(nx, ny, kind):
    """nz = 513: k_zpass<512, .> (radix-8 / 512-thread backward plan that exists only at N = 512) on the truncated path
    (342 of 513 modes in, look-ahead staging of the NEXT tile), many tiles per CTA; the solver sweeps at N = 512."""
    c = scaling_like(nx, ny, 513) if kind == "random" else I.small_config(nx=nx, ny=ny, nz=513, re=3000.0, dt=2e-5, ch=0.05,
                                                                         pe=20.0)
    run_parity(c, kind, 1, cap=4, looping=("zbwd", "zfwd"), min_iters=3.0)


def test_variable_viscosity_loops():
    """k_xfusedv<512> and the 10-field z / 11-field y passes of config 4's step, capped grid, channel state."""
    c = I.small_config(nx=512, ny=32, nz=17, visc_ratio=0.1)
    run_parity(c, "channel", 2, cap=5, min_iters=3.0)


@pytest.mark.parametrize("tag,nx,ny,nz,kw", [
    ("5a", 256, 128, 129, {}),
    ("slab1024", 1024, 64, 65, {}),
    ("slab1024-single", 1024, 64, 33, dict(phase_field=0)),
    ("slab512y", 64, 512, 65, {}),
    ("slabz", 64, 32, 513, {}),
    ("visc", 512, 64, 65, dict(visc_ratio=0.1, ch=0.05, pe=20.0, dt=5e-5)),
])
def test_capped_grid_is_bit_identical(tag, nx, ny, nz, kw):
    """The same 3 steps with the natural one-wave grid and with 7 CTAs: bit-identical states (no oracle needed, so the
    grids are larger: 5a, and slabs with the full 1024 / 512 / 513 line lengths of the bench grid)."""
    import torch
    import paper_2406_01322_b200 as P
    c = scaling_like(nx, ny, nz, **kw)
    space, st = state_of(c, "random")
    dev = [to_dev(f) for f in st]
    outs = []
    for cap in (0, 7):
        s = solver_from_config(c)
        if cap:
            s.set_option("grid_cap", cap)
        s.set_state(P.SPECTRAL, *dev)
        s.step(3)
        outs.append(s.get_state(P.SPECTRAL))
        if cap:
            for k in PERSISTENT:
                assert s.get_info(k + "_items") >= 3 * s.get_info(k + "_grid") > 0, k
        s.close()
    for a, b in zip(*outs):
        assert bool(torch.isfinite(torch.view_as_real(a)).all())
        assert torch.equal(a, b), tag


def test_fused_equals_unfused_x_path():
    """Rows a4-a6 as one fused kernel vs the three-kernel cross-check path through physical-space arrays
    (psdns_set_option "xfuse" 0): same state to rounding after 3 steps, on a grid with nx = 1024 lines and a looping grid."""
    import paper_2406_01322_b200 as P
    c = scaling_like(1024, 64, 33)
    space, st = state_of(c, "random")
    dev = [to_dev(f) for f in st]
    outs = []
    for fuse in (1, 0):
        s = solver_from_config(c, unfused_workspace=True)
        s.set_option("xfuse", fuse)
        s.set_state(P.SPECTRAL, *dev)
        s.step(3)
        outs.append([to_np(t) for t in s.get_state(P.SPECTRAL)])
        s.close()
    assert_parity(outs[0], outs[1], 1e-11, tag="fused vs unfused")
    s = solver_from_config(c)
    with pytest.raises(P.PsdnsError):
        s.set_option("xfuse", 0)          # the lean workspace has no physical-space arrays
    s.close()


@pytest.mark.parametrize("form", [1, 0])
@pytest.mark.parametrize("nx,ny,nz,kind", [(32, 32, 33, "channel"), (16, 16, 513, "random"), (64, 16, 129, "random"),
                                           (16, 64, 17, "channel")])
def test_tma_z_pass_matches_oracle(nx, ny, nz, kind, form):
    """k_zpass_tma (2-D TMA box loads into a two-deep mbarrier stage) against the live oracle, capped grid so that
    both stages and both barrier parities are reused many times; N = 512 takes three boxes (forward) / two (backward)."""
    import paper_2406_01322_b200 as P
    c = scaling_like(nx, ny, nz) if kind == "random" else I.small_config(nx=nx, ny=ny, nz=nz)
    space, st = state_of(c, kind)
    orc, g = oracle_from_config(c)
    orc.set_state(space, *st)
    orc.step(2)
    s = solver_from_config(c)
    s.set_option("ztma", form)               # 1: TMA-fed k_zpass_tma (the default); 0: register-fed k_zpass
    s.set_option("grid_cap", 3)
    s.set_state(P.SPECTRAL if space == "spectral" else P.PHYSICAL, *[to_dev(f) for f in st])
    s.step(2)
    for k in ("zbwd", "zfwd"):
        assert s.get_info(k + "_items") >= 3 * s.get_info(k + "_grid") > 0, k
    assert_parity([to_np(t) for t in s.get_state(P.SPECTRAL)], orc.get_state("spectral"), TOL, tag=("ztma", nx, ny, nz))
    # physical-space get_state runs the full-length backward z pass (nk = nz) through the TMA kernel as well
    ev = [np.abs(to_np(a) - b).max() / np.abs(b).max() for a, b in zip(s.get_state(P.PHYSICAL), orc.get_state("physical"))]
    assert max(ev) < TOL, ev
    s.close()


@pytest.mark.parametrize("nx,ny,nz,phase", [(32, 32, 33, 1), (64, 16, 65, 1), (16, 64, 17, 0)])
def test_gemm_form_chebyshev_matches_oracle(nx, ny, nz, phase):
    """Row f1: the GEMM form of the Chebyshev transform on the FP64 tensor cores (k_zgemm, mma.sync m8n8k4, N <= 64)
    drives the whole step (backward with the i ky phi by-product, forward with truncation) and the physical-space
    get_state (full-length backward)."""
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=nx, ny=ny, nz=nz, phase_field=phase)
    space, st = state_of(c, "channel")
    orc, g = oracle_from_config(c)
    orc.set_state(space, *st)
    orc.step(2)
    s = solver_from_config(c)
    s.set_option("zgemm", 1)
    s.set_option("grid_cap", 3)
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])          # forward z pass with nk = nz
    s.step(2)
    assert_parity([to_np(t) for t in s.get_state(P.SPECTRAL)], orc.get_state("spectral"), TOL, tag=("zgemm", nx, ny, nz))
    ev = [np.abs(to_np(a) - b).max() / np.abs(b).max() for a, b in zip(s.get_state(P.PHYSICAL), orc.get_state("physical"))]
    assert max(ev) < TOL, ev
    s.close()
