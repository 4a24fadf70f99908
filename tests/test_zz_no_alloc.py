"""psdns_diagnostics_static (include/psdns.h): the diagnostics entry point for callers that may not allocate.  Its reduction
partials live in a file-scope `static __device__` array (PSDNS_STATIC_SCRATCH_DOUBLES doubles, shared by every call on the
GPU) instead of the workspace; everything else is the existing path, so the outputs must equal psdns_diagnostics' bit for
bit - on the first call, on the next one, and after a call on another grid has left its partials in the array.

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`, and a failure here must not hide any
other test.  Passes alone in a fresh process and after the rest of the suite (nothing here depends on earlier tests)."""
import numpy as np
import pytest

import psdns_inputs as I
import psdns_oracle as O
from helpers import oracle_from_config, solver_from_config, to_dev

pytestmark = pytest.mark.gpu

TOL = 1e-11     # the tolerance of tests/test_gpu_diagnostics.py


def stepped_solver(nx, ny, nz, nsteps):
    import paper_2406_01322_b200 as P
    c = I.small_config(nx=nx, ny=ny, nz=nz)
    st = I.channel_state(c)
    s = solver_from_config(c)
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in st])
    s.step(nsteps)
    return c, st, s


def close_to(a, b):
    return all(abs(x - y) <= TOL * max(abs(y), 1.0) for x, y in zip(a, b))


def test_static_equals_existing_path_two_calls_in_a_row():
    import torch
    import paper_2406_01322_b200 as P
    c, st, s = stepped_solver(64, 32, 33, 2)
    ref = s.diagnostics().cpu().numpy()
    out = torch.full((8,), float("nan"), dtype=torch.float64, device="cuda")
    for call in range(2):
        out.fill_(float("nan"))
        got = s.diagnostics_static(out).cpu().numpy()
        assert np.all(np.isfinite(got)), (call, got)
        assert close_to(got, ref), (call, got, ref)
        assert np.array_equal(got, ref), (call, got, ref)         # same kernels, same launch shapes: bit-identical
    # and against the oracle's plain definitions, as tests/test_gpu_diagnostics.py does for the existing path
    orc, g = oracle_from_config(c)
    orc.set_state("physical", *st)
    orc.step(2)
    u, v, w, phi = orc.get_state("spectral")
    top, bot = O.wall_shear(g, u)
    want = dict(mean_phi=O.mean_phi(g, phi), kinetic_energy=O.kinetic_energy(g, u, v, w), shear_top=top, shear_bottom=bot,
                bulk_velocity=O.bulk_velocity(g, u))
    have = dict(zip(P.Solver.DIAG_NAMES, got))
    for k, r in want.items():
        assert abs(have[k] - r) <= TOL * max(abs(r), 1.0), (k, have[k], r)
    s.close()


def test_stale_partials_of_another_grid_do_not_leak():
    """The array keeps the last call's contents: a big-valued run on a wider grid first, then a smaller grid whose call
    uses fewer slots; then the first grid again.  Each must equal its own existing-path result."""
    import torch
    _, _, a = stepped_solver(128, 64, 33, 1)
    _, _, b = stepped_solver(32, 32, 17, 1)
    ref_a, ref_b = a.diagnostics().cpu().numpy(), b.diagnostics().cpu().numpy()
    out = torch.empty(8, dtype=torch.float64, device="cuda")
    for s, ref in ((a, ref_a), (b, ref_b), (b, ref_b), (a, ref_a)):
        got = s.diagnostics_static(out).cpu().numpy()     # .cpu() synchronises: the calls do not overlap on the GPU
        assert np.array_equal(got, ref), (got, ref)
    assert not np.array_equal(ref_a, ref_b)
    a.close()
    b.close()


def test_static_path_allocates_no_device_memory():
    import torch
    _, _, s = stepped_solver(64, 32, 33, 1)
    out = torch.empty(8, dtype=torch.float64, device="cuda")
    s.diagnostics_static(out)             # first call: symbol address look-up, lazily loaded kernels
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    launches0 = s.launch_count()
    for _ in range(20):
        s.diagnostics_static(out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert s.launch_count() - launches0 == 20 * 4      # columns, z pass, energy, final
    s.close()


def test_rejections():
    import torch
    import paper_2406_01322_b200 as P
    _, _, s = stepped_solver(32, 32, 17, 0)
    out = torch.zeros(8, dtype=torch.float64, device="cuda")
    with pytest.raises(P.PsdnsError):
        s.diagnostics_static(torch.zeros(8, dtype=torch.float32, device="cuda"))
    s.kernel_timing("zbwd", True)                 # timing creates events per launch: refused
    with pytest.raises(P.PsdnsError, match="timing"):
        s.diagnostics_static(out)
    s.kernel_timing("zbwd", False)
    s.diagnostics_static(out)
    s.close()
    fresh = solver_from_config(I.small_config(nx=32, ny=32, nz=17))
    with pytest.raises(P.PsdnsError, match="no state"):
        fresh.diagnostics_static(out)
    fresh.close()


def test_grid_beyond_the_static_limit_is_refused():
    """1024 x 1024 retains 344 * 683 columns: 918 column blocks + 8 * 148 energy blocks > 2048 doubles."""
    import torch
    import paper_2406_01322_b200 as P
    nx, ny, nz = 1024, 1024, 9
    g = O.Grid(nx, ny, nz)
    s = P.Solver(nx, ny, nz, g.lx, g.ly, re=100.0, dt=1e-4, phase_field=False)
    need = int(s.get_info("n_sm")) * 8 + -(-(344 * 683) // 256)
    if need <= P.STATIC_SCRATCH_DOUBLES:
        pytest.skip("this GPU has few enough SMs for 1024 x 1024 to fit")
    z = torch.zeros((nz, ny, nx), dtype=torch.float64, device="cuda")
    s.set_state(P.PHYSICAL, z, z, z)
    out = torch.full((8,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(P.PsdnsError, match="limit is %d" % P.STATIC_SCRATCH_DOUBLES):
        s.diagnostics_static(out)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())               # nothing was launched
    assert bool((s.diagnostics() == 0.0).all())   # the existing path takes the grid
    s.close()
