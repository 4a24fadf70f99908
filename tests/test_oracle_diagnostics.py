"""Pins of the diagnostics functions of the oracle (row f2: mean phi, max |div u|, kinetic energy, wall shear)
against closed forms."""
import numpy as np

import psdns_oracle as O


def poiseuille_hat(g, amp=1.0):
    u = np.zeros((g.nz, g.ny, g.nkx), dtype=np.complex128)
    u[0, 0, 0], u[2, 0, 0] = 0.5 * amp, -0.5 * amp        # 1 - z^2 = T0/2 - T2/2
    return u


def test_clenshaw_curtis_weights_integrate_polynomials():
    for N in (8, 16, 33 - 1, 64):
        w = O.clenshaw_curtis_weights(N)
        z = O.cheb_nodes(N)
        assert abs(w.sum() - 2.0) < 1e-14
        assert abs(w @ z ** 2 - 2.0 / 3.0) < 1e-14
        assert abs(w @ z ** 3) < 1e-14
        assert abs(w @ z ** N - 2.0 / (N + 1)) < 1e-13          # highest even degree still exact
        assert np.all(w > 0) and np.allclose(w, w[::-1])


def test_poiseuille_energy_shear_bulk():
    g = O.Grid(16, 8, 17)
    u = poiseuille_hat(g)
    zero = np.zeros_like(u)
    # (1/2)(1/2) int (1 - z^2)^2 dz = (1/4)(16/15)
    assert abs(O.kinetic_energy(g, u, zero, zero) - 4.0 / 15.0) < 1e-14
    top, bot = O.wall_shear(g, u)
    assert abs(top + 2.0) < 1e-13 and abs(bot - 2.0) < 1e-13   # d(1 - z^2)/dz = -2 z
    assert abs(O.bulk_velocity(g, u) - 2.0 / 3.0) < 1e-14


def test_energy_of_a_wave_adds_in_quadrature():
    """u = (1 - z^2) + a cos(kx x + ky y) (1 - z^2): the cross term averages out, <cos^2> = 1/2."""
    g = O.Grid(16, 16, 17)
    a = 0.3
    u = poiseuille_hat(g)
    for (i, j) in [(3, 2)]:
        u[0, j, i] += 0.5 * a * 0.5
        u[2, j, i] += -0.5 * a * 0.5                           # real cos = (e^{i.} + c.c.)/2: half-spectrum keeps one half
    v = np.zeros_like(u)
    want = 0.25 * (16.0 / 15.0) * (1.0 + 0.5 * a * a)
    assert abs(O.kinetic_energy(g, u, v, v) - want) < 1e-14


def test_max_divergence_of_solenoidal_and_compressive_modes():
    g = O.Grid(16, 16, 17)
    kx, ky = O.wavenumbers(g)
    u = np.zeros((g.nz, g.ny, g.nkx), dtype=np.complex128)
    v, w = np.zeros_like(u), np.zeros_like(u)
    u[1, 2, 3] = ky[2]; v[1, 2, 3] = -kx[3]                   # (ky, -kx, 0) T_1(z): divergence free
    assert O.max_divergence(g, u, v, w) < 1e-15
    w[2, 2, 3] = 1.0                                           # D T_2 = 4 T_1
    assert abs(O.max_divergence(g, u, v, w) - 4.0) < 1e-14
