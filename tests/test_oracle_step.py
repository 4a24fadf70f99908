"""Pins for the oracle's time step (not gpu): closed forms of the scheme and invariants.
 * Stokes mode decays by the Crank-Nicolson factor (channel version of exp(-nu k^2 t)), both for a mode that
   lives in omega_z (w = 0) and for the clamped eigenmodes of the 4th-order w equation (w != 0: pins H_w, Eq. 15);
 * laminar Poiseuille flow is steady with G = 2/Re;
 * the new velocity is divergence-free algebraically;
 * the split Cahn-Hilliard solve satisfies the 4th-order operator identity (S8) and the
   wall conditions; the tanh profile of Eq. 5 is stationary to truncation level;
   mean(phi) is conserved for a z-odd profile;
 * the explicit terms N_omega, N_w, S_phi, S_x-bar equal the continuous formulas of
   Eqs. 1, 4, 7, 8, 14, 15, 17 differentiated symbolically (sympy) on a manufactured state;
 * second-order convergence in time of the Navier-Stokes part (AB2 + CN, S7)."""
import math

import numpy as np
import pytest

import psdns_oracle as O
import psdns_inputs as I


def test_stokes_mode_crank_nicolson_factor():
    g = O.Grid(8, 8, 33)
    p = O.Params(re=50.0, dt=2e-3, phase_field=0)
    z = O.cheb_nodes(g.N)[:, None, None]
    y = g.ly / g.ny * np.arange(g.ny)[None, :, None]
    ky = 2 * np.pi / g.ly * 2
    A = 0.7
    u = A * np.cos(np.pi * z / 2) * np.cos(ky * y) * np.ones((1, 1, g.nx))
    zero = np.zeros_like(u)
    orc = O.Oracle(g, p)
    orc.set_state("physical", u, zero, zero)
    gam = p.dt / (2 * p.re)
    kap2 = ky ** 2 + np.pi ** 2 / 4
    fac = (1 - gam * kap2) / (1 + gam * kap2)
    for n in range(1, 4):
        orc.step(1)
        un, vn, wn = orc.get_state("physical")
        assert np.abs(un - fac ** n * u).max() < 1e-12
        assert np.abs(vn).max() < 1e-13 and np.abs(wn).max() < 1e-13
    # and it approaches the viscous decay exp(-kappa^2 t / Re)
    assert abs(fac ** 3 - math.exp(-kap2 * 3 * p.dt / p.re)) < 1e-9


@pytest.mark.parametrize("parity", ["even", "odd"])
def test_stokes_eigenmode_of_the_w_equation(parity):
    """Pins the Crank-Nicolson right-hand side of Eq. 15, H_w = theta + gamma (D^2 - k^2) theta + dt NL_w
    (reading S13), with w != 0.  Linearised Eq. 15: d/dt lap(w) = (1/Re) lap(lap(w)), w = dw/dz = 0 at z = +-1.  Eigenmodes:
        even: W = cosh(kz)/cosh k - cos(mu z)/cos mu,  k tanh k + mu tan mu = 0
        odd : W = sinh(kz)/sinh k - sin(mu z)/sin mu,  k coth k - mu cot mu = 0
    (both give W(+-1) = W'(+-1) = 0; lap W = (k^2 + mu^2) x the trigonometric part, an eigenfunction of lap with
    eigenvalue -(k^2 + mu^2)).  One step of the scheme multiplies w, theta = lap w and (through Eqs. 6, 16) u, v by
    g = (1 - gamma kappa^2)/(1 + gamma kappa^2), kappa^2 = k^2 + mu^2, exactly in time and to spectral accuracy in z.
    A single Fourier mode of amplitude A feeds back on itself only at O(A^3 dt), so A = 1e-3 leaves the non-linear
    terms below rounding.  A wrong sign or factor on gamma lap(theta) gives g = 1 or worse: off by 4e-4 per step."""
    from scipy.optimize import brentq
    g = O.Grid(8, 8, 33)
    p = O.Params(re=50.0, dt=2e-3, phase_field=0)
    ii, jj = 2, 1
    kx, ky = 2 * np.pi / g.lx * ii, 2 * np.pi / g.ly * jj
    k = math.hypot(kx, ky)
    if parity == "even":
        mu = brentq(lambda m: k * math.tanh(k) + m * math.tan(m), math.pi / 2 + 1e-9, math.pi - 1e-9)
        W = lambda z: np.cosh(k * z) / math.cosh(k) - np.cos(mu * z) / math.cos(mu)
        dW = lambda z: k * np.sinh(k * z) / math.cosh(k) + mu * np.sin(mu * z) / math.cos(mu)
    else:
        mu = brentq(lambda m: k / math.tanh(k) - m / math.tan(m), math.pi + 1e-9, 1.5 * math.pi - 1e-9)
        W = lambda z: np.sinh(k * z) / math.sinh(k) - np.sin(mu * z) / math.sin(mu)
        dW = lambda z: k * np.cosh(k * z) / math.sinh(k) - mu * np.cos(mu * z) / math.sin(mu)
    assert abs(W(1.0)) < 1e-12 and abs(dW(1.0)) < 1e-10 and abs(W(-1.0)) < 1e-12 and abs(dW(-1.0)) < 1e-10
    z = O.cheb_nodes(g.N)[:, None, None]
    x = g.lx / g.nx * np.arange(g.nx)[None, None, :]
    y = g.ly / g.ny * np.arange(g.ny)[None, :, None]
    A = 1e-3
    ph = kx * x + ky * y
    w = A * W(z) * np.cos(ph)
    u = -(kx / k ** 2) * A * dW(z) * np.sin(ph)        # continuity (Eq. 6) with omega_z = 0 (Eq. 16)
    v = -(ky / k ** 2) * A * dW(z) * np.sin(ph)
    orc = O.Oracle(g, p)
    orc.set_state("physical", u, v, w)
    s0 = orc.state
    w0, th0, u0, v0 = (f[:, jj, ii].copy() for f in (s0.w, s0.theta, s0.u, s0.v))
    gam = p.dt / (2 * p.re)
    kap2 = k * k + mu * mu
    fac = (1 - gam * kap2) / (1 + gam * kap2)
    assert 1e-4 < 1 - fac < 1e-2
    for n in range(1, 4):
        orc.step(1)
        s = orc.state
        for got, ref, tol in ((s.w, w0, 1e-12), (s.theta, th0, 1e-10), (s.u, u0, 1e-12), (s.v, v0, 1e-12)):
            assert np.abs(got[:, jj, ii] - fac ** n * ref).max() < tol * np.abs(ref).max(), (parity, n)
    assert abs(fac ** 3 - math.exp(-kap2 * 3 * p.dt / p.re)) < 1e-9


def test_poiseuille_is_steady():
    g = O.Grid(8, 8, 17)
    p = O.Params(re=100.0, dt=1e-3, gradp_x=2.0 / 100.0, phase_field=0)
    z = O.cheb_nodes(g.N)[:, None, None]
    u = (1 - z * z) * np.ones((1, g.ny, g.nx))
    orc = O.Oracle(g, p)
    orc.set_state("physical", u, 0 * u, 0 * u)
    orc.step(5)
    un, vn, wn = orc.get_state("physical")
    assert np.abs(un - u).max() < 1e-13
    assert np.abs(vn).max() < 1e-14 and np.abs(wn).max() < 1e-14


def test_divergence_free_and_no_slip_after_steps():
    c = I.small_config()
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    p = O.Params(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x)
    orc = O.Oracle(g, p)
    orc.set_state("physical", *I.channel_state(c))
    orc.step(2)
    s = orc.state
    div = O.divergence_spectrum(g, s.u, s.v, s.w)
    assert np.abs(div).max() < 1e-13
    for f in (s.u, s.v, s.w):
        assert np.abs(f.sum(axis=0)).max() < 1e-12                     # value at z = +1
        sgn = ((-1.0) ** np.arange(g.nz))[:, None, None]
        assert np.abs((f * sgn).sum(axis=0)).max() < 1e-12             # value at z = -1
    n2 = (np.arange(g.nz) ** 2.0)[:, None, None]
    assert np.abs((n2 * s.w).sum(axis=0)).max() < 1e-10                # dw/dz at z = +1
    # hidden state consistent with w: rows 0..N-2 of (D^2 - k^2) w = theta
    lap = orc._lap(s.w)
    assert np.abs((lap - s.theta)[: g.N - 1]).max() < 1e-8 * max(1.0, np.abs(s.theta).max())


def test_cahn_hilliard_two_stage_identity_and_wall_conditions():
    """Eq. 17 split into two Helmholtz problems (L142, S8): with L = D^2 - k^2 - lambda_phi,
    psi is rebuilt from phi^{n+1} alone (rows 0..N-2 of L phi, last two coefficients from
    D psi(+-1) = 0) and must satisfy gamma_phi L psi = H_phi in rows 0..N-2, so that
    gamma_phi (lap - lambda)^2 = 1 - dt (s Ch^2/Pe) lap + dt (Ch^2/Pe) lap^2 acts on phi^{n+1}
    up to the tau rows.  Also D phi(+-1) = 0 (S10).
    (SURVEY 8(c) S8 states the one-shot 4th-order identity holds in rows <= N-4; it cannot:
    D^2 is dense upper triangular, so psi's tau residual enters every row.  See DESIGN.md.)"""
    c = I.small_config(nz=33)
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    p = O.Params(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x)
    orc = O.Oracle(g, p)
    orc.set_state("physical", *I.channel_state(c))
    s0 = orc.state
    NL = orc.explicit_terms()["phi"]
    H = s0.phi + p.dt * NL
    orc.step(1)
    ph = orc.state.phi
    N = g.N
    lam = math.sqrt(p.pe / (p.dt * p.ch ** 2))
    gphi = p.dt * p.ch ** 2 / p.pe
    assert abs(gphi * lam * lam - 1.0) < 1e-14 and abs(2 * lam - 2 * math.sqrt(p.pe / (p.dt * p.ch ** 2))) < 1e-9
    Lop = lambda a: orc._lap(a) - lam * a
    psi = Lop(ph)
    # last two coefficients of psi from the two Neumann rows
    bn = O.boundary_rows(N, O.NEUMANN)
    A2 = bn[:, N - 1:]
    rhs = -np.einsum("rn,nji->rji", bn[:, : N - 1].astype(complex), psi[: N - 1])
    psi[N - 1:] = np.einsum("rs,sji->rji", np.linalg.inv(A2).astype(complex), rhs)
    res = gphi * Lop(psi) - H
    err = np.abs(np.where(orc.Pxy[: N - 1], res[: N - 1], 0)).max()
    assert err < 1e-10 * max(1.0, np.abs(H).max())
    # D phi(+-1) = 0 exactly (boundary rows).  D^3 phi(+-1) = 0 is only enforced through
    # D psi(+-1) = 0, i.e. up to psi's tau residual, so it is not asserted here.
    n2 = (np.arange(g.nz) ** 2.0)[:, None, None]
    sgn = ((-1.0) ** np.arange(g.nz))[:, None, None]
    assert np.abs((n2 * ph).sum(axis=0)).max() < 1e-11
    assert np.abs((n2 * sgn * ph).sum(axis=0)).max() < 1e-11


def _ch_1d(N, ch, steps, profile):
    g = O.Grid(4, 4, N + 1)
    p = O.Params(re=100.0, dt=1e-4, pe=1.0 / ch, ch=ch, we=1.0)
    z = O.cheb_nodes(N)[:, None, None]
    phi = profile(z) * np.ones((1, g.ny, g.nx))
    zero = np.zeros_like(phi)
    orc = O.Oracle(g, p)
    orc.set_state("physical", zero, zero, zero, phi)
    m0 = O.mean_phi(g, orc.state.phi)
    orc.step(steps)
    return phi, orc.get_state("physical")[3], m0, O.mean_phi(g, orc.state.phi), orc


def test_tanh_equilibrium_profile_is_stationary():
    """Eq. 5: phi = tanh(z / (sqrt2 Ch)) has mu = const; stationary to truncation level
    (~5e-10 per step at N = 256, Ch = 0.07)."""
    ch = 0.07
    phi0, phi1, m0, m1, orc = _ch_1d(256, ch, 4, lambda z: np.tanh(z / (math.sqrt(2) * ch)))
    assert O.rel_l2(phi1, phi0) < 4 * 2e-9
    u, v, w, _ = orc.get_state("physical")
    assert max(np.abs(u).max(), np.abs(v).max(), np.abs(w).max()) < 1e-9   # no spurious flow in x,y; 1-D
    assert abs(m1 - m0) < 1e-13                                           # z-odd profile: mean conserved


def test_mean_phi_of_an_off_centre_interface():
    """mean(phi) (Eq. 1 is a conservation law: d/dt int phi = (1/Pe) [d mu/dz] at the walls = 0 with the no-flux
    conditions of reading S10) for an interface at z0 = 0.2, which is NOT z-odd:
      * `mean_phi` equals the closed form (1/2) int tanh((z - z0)/w) dz = (w/2) ln[cosh((1 - z0)/w)/cosh((1 + z0)/w)];
      * the tau scheme conserves it only up to the tau residual of the psi problem, which falls spectrally with
        resolution (SURVEY 8(c) "mean(phi)": measured there 4e-5 at N = 128, Ch = 0.05 ... 2e-9 at N = 256, Ch = 0.07 over
        10 steps): drift over 10 steps < 1e-8 at N = 256, Ch = 0.07, and >= 1000 x smaller than at N = 128."""
    ch, z0 = 0.07, 0.2
    w = math.sqrt(2) * ch
    drift = {}
    for N in (128, 256):
        phi0, phi1, m0, m1, orc = _ch_1d(N, ch, 10, lambda z: np.tanh((z - z0) / w))
        exact = 0.5 * w * (np.log(np.cosh((1 - z0) / w)) - np.log(np.cosh((1 + z0) / w)))
        assert abs(m0 - exact) < 1e-12, (N, m0, exact)
        drift[N] = abs(m1 - m0)
    assert drift[256] < 1e-8 and drift[256] < 1e-3 * drift[128] and drift[128] < 1e-4, drift


def test_non_equilibrium_profile_relaxes_towards_tanh():
    """A too-wide interface sharpens: the distance to the Eq. 5 profile must decrease."""
    ch = 0.07
    eq = lambda z: np.tanh(z / (math.sqrt(2) * ch))
    wide = lambda z: np.tanh(z / (math.sqrt(2) * ch * 1.3))
    phi0, phi1, *_ = _ch_1d(128, ch, 20, wide)
    z = O.cheb_nodes(128)[:, None, None]
    d0 = np.linalg.norm((phi0 - eq(z))[:, 0, 0]); d1 = np.linalg.norm((phi1 - eq(z))[:, 0, 0])
    assert d1 < d0


@pytest.mark.parametrize("form,conv", [(0, 0), (1, 0), (0, 1), (1, 1)])
def test_explicit_terms_match_symbolic_continuous_formulas(form, conv):
    """form 0: Korteweg tensor (Eq. 8 as written); form 1: the force -c_sigma lap(phi) grad(phi); conv 0: -div(u u) (S4);
    conv 1: the rotational form u x omega - each against ITS OWN continuous expression."""
    import sympy as sp
    g = O.Grid(16, 16, 65)
    p = O.Params(re=80.0, dt=1e-3, pe=3.0, ch=0.3, we=1.3, gradp_x=0.04, visc_ratio=0.3, surface_tension_form=form,
                 convection_form=conv)
    x, y, z = sp.symbols("x y z", real=True)
    kx, ky = sp.Rational(1, 2), 1                         # fundamental wavenumbers of 4pi x 2pi
    q = 1 - z ** 2
    A = sp.Matrix([q ** 3 * sp.sin(ky * y) * sp.cos(kx * x) * sp.Rational(3, 10),
                   q ** 3 * sp.cos(2 * ky * y) * sp.sin(kx * x) * sp.Rational(2, 10),
                   q ** 2 * (1 + z / 2) * sp.sin(kx * x + sp.Rational(1, 3)) * sp.sin(ky * y)])
    X = (x, y, z)
    curl = lambda F: sp.Matrix([sp.diff(F[2], y) - sp.diff(F[1], z),
                                sp.diff(F[0], z) - sp.diff(F[2], x),
                                sp.diff(F[1], x) - sp.diff(F[0], y)])
    U = curl(A) + sp.Matrix([q * sp.Rational(1, 2), 0, 0])        # plus a mean flow
    phi = sp.Rational(3, 10) * q ** 4 * sp.cos(kx * x) * sp.cos(ky * y) + sp.Rational(1, 5) * z * sp.sin(ky * y) - sp.Rational(1, 10)
    grad = lambda f: sp.Matrix([sp.diff(f, s) for s in X])
    lap = lambda f: sum(sp.diff(f, s, 2) for s in X)
    gp = grad(phi)
    cs = 3 / sp.sqrt(8) * sp.Float(p.ch) / sp.Float(p.we)
    eta1 = (sp.Float(p.visc_ratio) - 1) * (phi + 1) / 2 / sp.Float(p.re)
    T = sp.zeros(3, 3)
    for a in range(3):
        for b in range(3):
            T[a, b] = ((-U[a] * U[b] if conv == 0 else 0) + (cs * ((gp.dot(gp) if a == b else 0) - gp[a] * gp[b]) if form == 0 else 0)
                       + eta1 * (sp.diff(U[b], X[a]) + sp.diff(U[a], X[b])))
    S = sp.Matrix([sum(sp.diff(T[a, b], X[b]) for b in range(3)) for a in range(3)])
    if form == 1:
        S = S - cs * lap(phi) * gp
    if conv == 1:
        S = S + U.cross(curl(U))
    S[0] = S[0] + sp.Float(p.gradp_x)
    divS = sum(sp.diff(S[a], X[a]) for a in range(3))
    N_om = curl(S)[2]                                              # Eq. 14
    N_w = lap(S[2]) - sp.diff(divS, z)                             # Eq. 15
    sco = 2 * math.sqrt(p.pe / (p.dt * p.ch ** 2))
    S_phi = (-U.dot(gp) + lap(phi ** 3) / sp.Float(p.pe)
             - (1 + sco * p.ch ** 2) / sp.Float(p.pe) * lap(phi))  # Eq. 17 with S8/S9

    xs = g.lx / g.nx * np.arange(g.nx)[None, None, :]
    ys = g.ly / g.ny * np.arange(g.ny)[None, :, None]
    zs = O.cheb_nodes(g.N)[:, None, None]
    ev = lambda e: np.broadcast_to(sp.lambdify(X, e, "numpy")(xs, ys, zs), (g.nz, g.ny, g.nx)).astype(float)

    orc = O.Oracle(g, p)
    orc.set_state("physical", ev(U[0]), ev(U[1]), ev(U[2]), ev(phi))
    N = orc.explicit_terms()
    P = orc.P
    for key, expr in (("om", N_om), ("w", N_w), ("phi", S_phi)):
        ref = np.where(P, O.forward_transform(ev(expr), g), 0)
        got = np.where(P, N[key], 0)
        assert O.rel_l2(got, ref) < 2e-9, key
    refx = O.forward_transform(ev(S[0]), g)[:, 0, 0]
    K = O.retained_counts(g)[2]
    assert np.abs(N["ubar"][: K + 1] - refx[: K + 1]).max() < 1e-10 * max(1, np.abs(refx).max())


def test_lambda_one_reproduces_matched_viscosity():
    c = I.small_config()
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    st = I.channel_state(c)
    res = []
    for lam in (1.0, 1.0 + 1e-300):
        p = O.Params(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x, visc_ratio=lam)
        orc = O.Oracle(g, p); orc.set_state("physical", *st); orc.step(2)
        res.append(orc.state)
    assert np.array_equal(res[0].u, res[1].u) and np.array_equal(res[0].phi, res[1].phi)


def test_navier_stokes_part_is_second_order_in_time():
    """AB2 (Euler start-up) + Crank-Nicolson (S7): halving dt must cut the error ~4x."""
    c = I.small_config(nx=8, ny=8, nz=17, re=20.0, phase_field=0, band=2)
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    u, v, w, _ = I.channel_state(c)
    z = O.cheb_nodes(g.N)[:, None, None]
    base = (1 - z * z) * np.ones_like(u)
    u, v, w = base + 8 * (u - base), 8 * v, 8 * w     # stronger (still solenoidal) perturbation
    Tend = 0.04
    sols = {}
    for n in (8, 16, 32, 256):
        p = O.Params(re=c.re, dt=Tend / n, gradp_x=c.gradp_x, phase_field=0)
        orc = O.Oracle(g, p); orc.set_state("physical", u, v, w); orc.step(n)
        sols[n] = np.concatenate([f.ravel() for f in orc.get_state("spectral")])
    e = {n: np.linalg.norm(sols[n] - sols[256]) for n in (8, 16, 32)}
    assert 3.3 < e[8] / e[16] < 4.8 and 3.3 < e[16] / e[32] < 4.9, e


def test_variable_viscosity_steady_layered_flow():
    """Reading S14 (eta(phi) = 1 + (lambda - 1)(phi + 1)/2, viscous term split into implicit (1/Re) lap u and explicit
    (1/Re) div[(eta - 1)(grad u + grad u^T)]) pinned against a closed form that does not use the split: for the layered
    state phi = tanh(z/(sqrt2 Ch)) (Eq. 5), u = u(z), the x-momentum balance is d/dz(eta u') = -G Re, i.e.
    eta u' = -G Re z + c with u(+-1) = 0 -- a quadrature.  That state must be steady under the scheme up to the
    truncation error, which falls spectrally with resolution; a wrong sign or factor in the split leaves a tendency
    of order G (lambda - 1) ~ 3e-2."""
    from scipy.integrate import quad
    re, lam, G, dt = 50.0, 0.3, 2.0 / 50.0, 1e-3

    def tendency(nz, ch):
        g = O.Grid(8, 8, nz, 4 * math.pi, 2 * math.pi)
        z = O.cheb_nodes(g.N)
        eta = lambda s: 1.0 + (lam - 1.0) * (math.tanh(s / (math.sqrt(2.0) * ch)) + 1.0) / 2.0
        q = dict(epsabs=1e-13, epsrel=1e-13, limit=200)
        c = -quad(lambda s: -G * re * s / eta(s), -1, 1, **q)[0] / quad(lambda s: 1.0 / eta(s), -1, 1, **q)[0]
        u1 = np.array([quad(lambda s: (-G * re * s + c) / eta(s), -1, zz, **q)[0] for zz in z])
        u = np.broadcast_to(u1[:, None, None], (nz, 8, 8)).copy()
        phi = np.broadcast_to(np.tanh(z / (math.sqrt(2.0) * ch))[:, None, None], (nz, 8, 8)).copy()
        orc = O.Oracle(g, O.Params(re=re, dt=dt, pe=1.0 / ch, ch=ch, we=1.0, gradp_x=G, visc_ratio=lam))
        orc.set_state("physical", u, np.zeros_like(u), np.zeros_like(u), phi)
        orc.step(2)
        un, vn, wn, _ = orc.get_state("physical")
        assert np.abs(vn).max() < 1e-12 and np.abs(wn).max() < 1e-12
        return np.abs(un - u).max() / (2 * dt), np.abs(u1).max()

    import warnings
    with warnings.catch_warnings():
        warnings.simplefilter("ignore")          # quad reports round-off at the 1e-13 request
        t_coarse, umax = tendency(129, 0.1)
        t_fine, _ = tendency(257, 0.07)
    assert umax > 1.5                            # the low-viscosity layer speeds the flow up (lambda = 1: max u = 1)
    assert t_coarse < 5e-6 and t_fine < 5e-8, (t_coarse, t_fine)


def test_surface_tension_forms_differ_by_a_gradient_only():
    """Korteweg divergence (form 0) and the force -c lap(phi) grad(phi) (form 1) differ by grad(c |grad phi|^2 / 2), which
    the curl (Eq. 14) and the lap S_z - d/dz div S combination (Eq. 15) annihilate: N_omega and N_w of the two forms agree
    to truncation error on a resolved state - but not to rounding (they are different discrete operators), which is why
    the form is a switch of the oracle and not a free choice of the kernels.  S_phi does not contain the term at all."""
    g = O.Grid(16, 16, 49)
    z = O.cheb_nodes(g.N)[:, None, None]
    x = g.lx / g.nx * np.arange(g.nx)[None, None, :]
    y = g.ly / g.ny * np.arange(g.ny)[None, :, None]
    q = 1 - z * z
    phi = 0.3 * q ** 4 * np.cos(0.5 * x) * np.cos(y) + 0.2 * z * np.sin(y) - 0.1 + 0 * x
    u = 0.5 * q * np.ones_like(phi)
    zero = np.zeros_like(phi)
    out = []
    for form in (0, 1):
        p = O.Params(re=80.0, dt=1e-3, pe=3.0, ch=0.3, we=1.3, surface_tension_form=form)
        orc = O.Oracle(g, p)
        orc.set_state("physical", u, zero, zero, phi)
        out.append(orc.explicit_terms())
    for key in ("om", "w"):
        d = O.rel_l2(out[1][key], out[0][key])
        assert 1e-15 < d < 1e-7, (key, d)
    assert np.array_equal(out[0]["phi"], out[1]["phi"])
    # the mean-flow forcing S-bar_x differs by d/dx of a mean: nothing
    assert np.abs(out[0]["ubar"] - out[1]["ubar"]).max() < 1e-12


def test_convection_forms_differ_by_a_gradient_only():
    """Divergence form -div(u u) and rotational form u x omega differ by grad(|u|^2 / 2) for a solenoidal field: N_omega,
    N_w and the mean-flow forcing agree to truncation error on a resolved solenoidal state, not to rounding."""
    c = I.small_config(nx=16, ny=16, nz=49, band=2, phase_field=0)
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    st = I.channel_state(c)[:3]
    out = []
    for conv in (0, 1):
        orc = O.Oracle(g, O.Params(re=c.re, dt=c.dt, gradp_x=c.gradp_x, phase_field=0, convection_form=conv))
        orc.set_state("physical", *st)
        out.append(orc.explicit_terms())
    for key in ("om", "w"):
        d = O.rel_l2(out[1][key], out[0][key])
        assert 1e-16 < d < 1e-8, (key, d)
    assert np.abs(out[0]["ubar"] - out[1]["ubar"]).max() < 1e-10 * np.abs(out[0]["ubar"]).max() + 1e-13
