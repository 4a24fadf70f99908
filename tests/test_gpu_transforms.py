"""GPU parity: transforms of libpsdns vs the oracle's dense matrix transforms (through the C ABI).
Tolerance: relative L2 <= 1e-11 per transform round trip (BASELINE.json north_star)."""
import numpy as np
import pytest

import psdns_inputs as I
import psdns_oracle as O
from helpers import to_dev, to_np

pytestmark = pytest.mark.gpu
TOL = 1e-11

GRIDS = [(16, 16, 9), (32, 32, 33), (64, 32, 17), (32, 128, 65), (128, 64, 129), (256, 16, 9)]


def make_solver(nx, ny, nz):
    import paper_2406_01322_b200 as P
    return P.Solver(nx, ny, nz, 4 * np.pi, 2 * np.pi, re=100.0, dt=1e-3, phase_field=0)


@pytest.mark.parametrize("nx,ny,nz", GRIDS)
def test_roundtrip_from_physical(nx, ny, nz):
    import paper_2406_01322_b200 as P
    s = make_solver(nx, ny, nz)
    g = O.Grid(nx, ny, nz)
    f = I.random_physical_field(nx, ny, nz, seed=nx + ny + nz)
    out, mid = s.transform_roundtrip(P.PHYSICAL, to_dev(f), want_mid=True)
    import torch
    assert torch.equal(out, s.transform_roundtrip(P.PHYSICAL, to_dev(f)))   # without d_mid: private layout in between, same bits
    out, mid = to_np(out), to_np(mid)
    ref_mid = O.forward_transform(f, g)
    assert O.rel_l2(mid, ref_mid) < TOL          # forward transform, element by element
    assert O.rel_l2(out, f) < TOL                # round trip = identity
    assert O.rel_l2(out, O.backward_transform(ref_mid, g)) < TOL


@pytest.mark.parametrize("nx,ny,nz", GRIDS[:4])
def test_roundtrip_from_spectral(nx, ny, nz):
    import paper_2406_01322_b200 as P
    s = make_solver(nx, ny, nz)
    g = O.Grid(nx, ny, nz)
    a = I.random_spectrum(nx, ny, nz, np.random.default_rng(5), cut=False, rms=1.0)
    out, mid = s.transform_roundtrip(P.SPECTRAL, to_dev(a), want_mid=True)
    out, mid = to_np(out), to_np(mid)
    ref_mid = O.backward_transform(a, g)
    assert O.rel_l2(mid, ref_mid) < TOL
    assert O.rel_l2(out, a) < TOL                # Hermitian-consistent, Nyquist-free input


def test_roundtrip_drops_inconsistent_imaginary_parts():
    """Reading S20: imaginary parts on the i = 0 / Nyquist planes that violate Hermitian symmetry are dropped
    the same way by both sides."""
    import paper_2406_01322_b200 as P
    nx, ny, nz = 32, 16, 9
    s = make_solver(nx, ny, nz)
    g = O.Grid(nx, ny, nz)
    rng = np.random.default_rng(9)
    a = rng.standard_normal((nz, ny, nx // 2 + 1)) + 1j * rng.standard_normal((nz, ny, nx // 2 + 1))
    out, mid = s.transform_roundtrip(P.SPECTRAL, to_dev(a), want_mid=True)
    ref_mid = O.backward_transform(a, g)
    assert O.rel_l2(to_np(mid), ref_mid) < TOL
    assert O.rel_l2(to_np(out), O.forward_transform(ref_mid, g)) < TOL


def test_set_get_state_physical_projection():
    """set_state(PHYSICAL) then get_state: P_xy projection of the field (retained kx, ky; all nz modes)."""
    import paper_2406_01322_b200 as P
    nx, ny, nz = 64, 32, 33
    s = make_solver(nx, ny, nz)
    g = O.Grid(nx, ny, nz)
    fs = [I.random_physical_field(nx, ny, nz, seed=k) for k in range(3)]
    s.set_state(P.PHYSICAL, *[to_dev(f) for f in fs])
    spec = [to_np(t) for t in s.get_state(P.SPECTRAL)]
    phys = [to_np(t) for t in s.get_state(P.PHYSICAL)]
    Pxy = O.truncation_mask(g, 1, z=False)
    for f, a, b in zip(fs, spec, phys):
        ref = np.where(Pxy, O.forward_transform(f, g), 0)
        assert O.rel_l2(a, ref) < TOL
        assert np.all(a[~Pxy] == 0)
        assert O.rel_l2(b, O.backward_transform(ref, g)) < TOL
