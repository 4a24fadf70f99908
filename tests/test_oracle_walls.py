"""Pins of the oracle's wall variants (row f3; "no-slip or free-slip, or a combination of them"):
free-slip w = 0, du/dz = dv/dz = 0  =>  d omega_z/dz = 0 and, through continuity, d^2 w/dz^2 = 0.
 * the boundary rows against numpy's Chebyshev class;
 * free-slip Stokes modes decay by the Crank-Nicolson factor: cos(pi z) cos(ky y) in omega_z (Neumann walls),
   cos(pi z / 2) cos(kx x + ky y) in w (w = w'' = 0 at the walls: an eigenfunction of the laplacian);
 * mixed walls: the steady mean flow u = 3 + 2z - z^2 (no-slip at z = -1, free-slip at z = +1, G = 2/Re) and its mirror
   image stay steady; a manufactured polynomial of the coupled theta / w problem is reproduced exactly;
 * after a step from a generic state every wall condition holds and the velocity is divergence-free."""
import math

import numpy as np
import pytest
from numpy.polynomial import chebyshev as C

import psdns_inputs as I
import psdns_oracle as O

NS, FS = O.NO_SLIP, O.FREE_SLIP


def test_wall_rows_against_numpy_chebyshev():
    N = 12
    for n in range(N + 1):
        T = C.Chebyshev.basis(n)
        for wall in (+1, -1):
            for kind, f in ((O.DIRICHLET, T), (O.NEUMANN, T.deriv(1)), (O.SECOND_DERIVATIVE, T.deriv(2))):
                assert abs(O.wall_row(N, kind, wall)[n] - f(float(wall))) < 1e-9 * max(1.0, abs(f(float(wall))))
    rows = O.boundary_rows(N, (O.NEUMANN, O.DIRICHLET))
    assert np.allclose(rows[0], O.wall_row(N, O.NEUMANN, +1)) and np.allclose(rows[1], O.wall_row(N, O.DIRICHLET, -1))


def test_free_slip_stokes_mode_in_omega_z():
    g = O.Grid(8, 8, 33)
    p = O.Params(re=50.0, dt=2e-3, phase_field=0, wall_top=FS, wall_bottom=FS)
    z = O.cheb_nodes(g.N)[:, None, None]
    y = g.ly / g.ny * np.arange(g.ny)[None, :, None]
    ky = 2 * np.pi / g.ly * 2
    u = 0.7 * np.cos(np.pi * z) * np.cos(ky * y) * np.ones((1, 1, g.nx))     # du/dz = 0 at z = +-1, (u . grad) u = 0
    zero = np.zeros_like(u)
    orc = O.Oracle(g, p)
    orc.set_state("physical", u, zero, zero)
    gam = p.dt / (2 * p.re)
    kap2 = ky ** 2 + np.pi ** 2
    fac = (1 - gam * kap2) / (1 + gam * kap2)
    for n in range(1, 4):
        orc.step(1)
        un, vn, wn = orc.get_state("physical")
        assert np.abs(un - fac ** n * u).max() < 1e-12
        assert np.abs(vn).max() < 1e-13 and np.abs(wn).max() < 1e-13
    # the same mode between no-slip walls violates u = 0 there: the first solve must change it at O(1)
    ns = O.Oracle(g, O.Params(re=50.0, dt=2e-3, phase_field=0))
    ns.set_state("physical", u, zero, zero)
    ns.step(1)
    assert np.abs(ns.get_state("physical")[0] - fac * u).max() > 0.1


def test_free_slip_stokes_mode_in_w():
    g = O.Grid(8, 8, 33)
    p = O.Params(re=50.0, dt=2e-3, phase_field=0, wall_top=FS, wall_bottom=FS)
    ii, jj = 2, 1
    kx, ky = 2 * np.pi / g.lx * ii, 2 * np.pi / g.ly * jj
    k2 = kx * kx + ky * ky
    z = O.cheb_nodes(g.N)[:, None, None]
    x = g.lx / g.nx * np.arange(g.nx)[None, None, :]
    y = g.ly / g.ny * np.arange(g.ny)[None, :, None]
    A, m = 1e-3, np.pi / 2
    ph = kx * x + ky * y
    w = A * np.cos(m * z) * np.cos(ph)                                   # w = w'' = 0 at the walls
    u = (kx / k2) * A * m * np.sin(m * z) * np.sin(ph)                   # continuity with omega_z = 0
    v = (ky / k2) * A * m * np.sin(m * z) * np.sin(ph)
    orc = O.Oracle(g, p)
    orc.set_state("physical", u, v, w)
    s0 = orc.state
    assert np.abs(O.divergence_spectrum(g, s0.u, s0.v, s0.w)).max() < 1e-13 * A * 100
    w0, u0, v0 = (f[:, jj, ii].copy() for f in (s0.w, s0.u, s0.v))
    gam = p.dt / (2 * p.re)
    kap2 = k2 + m * m
    fac = (1 - gam * kap2) / (1 + gam * kap2)
    for n in range(1, 4):
        orc.step(1)
        s = orc.state
        for got, ref in ((s.w, w0), (s.u, u0), (s.v, v0)):
            assert np.abs(got[:, jj, ii] - fac ** n * ref).max() < 1e-11 * np.abs(ref).max(), n


@pytest.mark.parametrize("top,bottom,sign", [(FS, NS, +1.0), (NS, FS, -1.0)])
def test_mixed_walls_mean_flow_is_steady(top, bottom, sign):
    """u'' = -G Re = -2 with u = 0 at the no-slip wall and u' = 0 at the free-slip wall: u = 3 + 2 s z - z^2."""
    g = O.Grid(8, 8, 17)
    p = O.Params(re=100.0, dt=1e-3, gradp_x=2.0 / 100.0, phase_field=0, wall_top=top, wall_bottom=bottom)
    z = O.cheb_nodes(g.N)[:, None, None]
    u = (3.0 + 2.0 * sign * z - z * z) * np.ones((1, g.ny, g.nx))
    orc = O.Oracle(g, p)
    orc.set_state("physical", u, 0 * u, 0 * u)
    orc.step(5)
    un, vn, wn = orc.get_state("physical")
    assert np.abs(un - u).max() < 1e-12
    assert np.abs(vn).max() < 1e-13 and np.abs(wn).max() < 1e-13
    # with no-slip at both walls the same profile is not steady
    ns = O.Oracle(g, O.Params(re=100.0, dt=1e-3, gradp_x=2.0 / 100.0, phase_field=0))
    ns.set_state("physical", u, 0 * u, 0 * u)
    ns.step(1)
    assert np.abs(ns.get_state("physical")[0] - u).max() > 1e-2


def test_mixed_walls_manufactured_w():
    """w = (1 + z - z^2 - z^3)(2 - z): w(+-1) = 0, w'(-1) = 0, w''(+1) = 0.  theta = (D^2 - k^2) w, hw = -gamma (D^2 - beta^2) theta."""
    N = 16
    z = C.Chebyshev([0, 1])
    wpoly = (1 + z - z ** 2 - z ** 3) * (2 - z)
    assert abs(wpoly(1.0)) < 1e-14 and abs(wpoly(-1.0)) < 1e-14
    assert abs(wpoly.deriv(1)(-1.0)) < 1e-13 and abs(wpoly.deriv(2)(1.0)) < 1e-13
    k2, gamma = 2.3, 1e-3
    beta2 = k2 + 1.0 / gamma
    th = wpoly.deriv(2) - k2 * wpoly
    hw = -gamma * (th.deriv(2) - beta2 * th)
    pad = lambda c: np.concatenate([c.coef, np.zeros(N + 1 - len(c.coef))])
    theta, w = O.coupled_w_solve(pad(hw)[:, None].astype(np.complex128), np.array([beta2]), np.array([k2]), gamma,
                                 walls=(FS, NS))
    assert np.abs(w[:, 0] - pad(wpoly)).max() < 1e-11
    assert np.abs(theta[:, 0] - pad(th)).max() < 1e-9
    # the other assignment of the walls does NOT reproduce it
    _, w2 = O.coupled_w_solve(pad(hw)[:, None].astype(np.complex128), np.array([beta2]), np.array([k2]), gamma, walls=(NS, FS))
    assert np.abs(w2[:, 0] - pad(wpoly)).max() > 1e-3


@pytest.mark.parametrize("top,bottom", [(FS, FS), (FS, NS), (NS, FS)])
def test_wall_conditions_and_continuity_after_steps(top, bottom):
    c = I.small_config()
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    p = O.Params(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x, wall_top=top, wall_bottom=bottom)
    orc = O.Oracle(g, p)
    orc.set_state("physical", *I.channel_state(c))
    orc.step(2)
    s = orc.state
    assert np.abs(O.divergence_spectrum(g, s.u, s.v, s.w)).max() < 1e-12
    scale = max(np.abs(f).max() for f in (s.u, s.v, s.w))

    def at(f, kind, wall):
        return np.abs(np.tensordot(O.wall_row(g.N, kind, wall), f, axes=(0, 0))).max()

    for wall, kind in ((+1, top), (-1, bottom)):
        assert at(s.w, O.DIRICHLET, wall) < 1e-12 * scale
        if kind == NS:
            assert at(s.u, O.DIRICHLET, wall) < 1e-11 * scale and at(s.v, O.DIRICHLET, wall) < 1e-11 * scale
            assert at(s.w, O.NEUMANN, wall) < 1e-10 * scale
        else:
            assert at(s.u, O.NEUMANN, wall) < 1e-9 * scale and at(s.v, O.NEUMANN, wall) < 1e-9 * scale
            assert at(s.w, O.SECOND_DERIVATIVE, wall) < 1e-8 * scale
            assert at(s.u, O.DIRICHLET, wall) > 1e-3            # the wall really slips
