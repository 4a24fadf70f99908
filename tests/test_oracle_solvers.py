"""Pins for the oracle's Chebyshev-tau Helmholtz / biharmonic solves (not gpu):
manufactured polynomial solutions, residual check, the classical quasi-tridiagonal
recurrence (an independent algorithm for the same tau system) and the
influence-matrix route to the coupled w problem."""
import numpy as np
import pytest
from numpy.polynomial import Polynomial as Poly

import psdns_oracle as O


def cheb_coeffs(p: Poly, N):
    z = O.cheb_nodes(N)
    return O.cheb_fwd_matrix(N) @ p(z)


@pytest.mark.parametrize("sigma", [0.25, 37.0, 1.2e8])
def test_helmholtz_poiseuille_profile(sigma):
    """u = 1 - z^2  =>  u'' - sigma u = -2 - sigma (1 - z^2)."""
    N = 16
    u = Poly([1, 0, -1])
    f = u.deriv(2) - sigma * u
    a = O.helmholtz_solve(cheb_coeffs(f, N)[:, None].astype(complex), np.array([sigma]), O.DIRICHLET)
    ref = np.zeros(N + 1); ref[0], ref[2] = 0.5, -0.5
    assert np.abs(a[:, 0] - ref).max() < 1e-13


@pytest.mark.parametrize("bc", [O.DIRICHLET, O.NEUMANN])
@pytest.mark.parametrize("sigma", [0.0 + 1.0, 250.0, 3.3e5])
def test_helmholtz_manufactured_with_boundary_values(bc, sigma):
    N = 24
    rng = np.random.default_rng(11)
    u = Poly(rng.standard_normal(12))
    f = u.deriv(2) - sigma * u
    if bc == O.DIRICHLET:
        bp, bm = u(1.0), u(-1.0)
    else:
        bp, bm = u.deriv()(1.0), u.deriv()(-1.0)
    rhs = (cheb_coeffs(f, N) * (1 + 0.5j))[:, None]
    a = O.helmholtz_solve(rhs, np.array([sigma]), bc, bp * (1 + 0.5j), bm * (1 + 0.5j))
    ref = cheb_coeffs(u, N) * (1 + 0.5j)
    assert np.abs(a[:, 0] - ref).max() < 1e-9 * max(1.0, np.abs(ref).max())


def quasi_tridiagonal_solve(f, sigma, bc, bp, bm):
    """Independent algorithm: the classical recurrence for u'' - sigma u = f in Chebyshev
    coefficients (rows k = 2..N):
      -sigma p_k u_{k-2} + (1 - sigma q_k) u_k - sigma r_k u_{k+2} = p_k f_{k-2} + q_k f_k + r_k f_{k+2}
    p_k = ct_{k-2}/(4k(k-1)), q_k = -e_{k+2}/(2(k^2-1)), r_k = e_{k+4}/(4k(k+1)),
    plus the two boundary rows; assembled as a dense matrix and solved in one go."""
    N = f.size - 1
    A = np.zeros((N + 1, N + 1)); b = np.zeros(N + 1, dtype=complex)
    e = lambda j: 1.0 if j <= N else 0.0
    ct = lambda j: 2.0 if j == 0 else 1.0
    for k in range(2, N + 1):
        p = ct(k - 2) / (4.0 * k * (k - 1)); q = -e(k + 2) / (2.0 * (k * k - 1)); r = e(k + 4) / (4.0 * k * (k + 1))
        A[k, k - 2] = -sigma * p; A[k, k] = 1 - sigma * q
        b[k] = p * f[k - 2] + q * f[k]
        if k + 2 <= N:
            A[k, k + 2] = -sigma * r; b[k] += r * f[k + 2]
    A[:2] = O.boundary_rows(N, bc); b[0], b[1] = bp, bm
    return np.linalg.solve(A, b)


@pytest.mark.parametrize("N", [16, 64, 128])
@pytest.mark.parametrize("sigma", [0.25, 1.0e3, 1.2e8])
@pytest.mark.parametrize("bc", [O.DIRICHLET, O.NEUMANN])
def test_dense_tau_equals_quasi_tridiagonal(N, sigma, bc):
    rng = np.random.default_rng(N)
    f = rng.standard_normal(N + 1) + 1j * rng.standard_normal(N + 1)
    a = O.helmholtz_solve(f[:, None], np.array([sigma]), bc, 0.3, -0.2)[:, 0]
    b = quasi_tridiagonal_solve(f, sigma, bc, 0.3, -0.2)
    assert np.abs(a - b).max() < 1e-11 * max(1.0, np.abs(a).max())


def test_tau_residual_rows():
    N = 32
    rng = np.random.default_rng(5)
    f = rng.standard_normal((N + 1, 3)) + 0j
    sig = np.array([2.0, 50.0, 4000.0])
    a = O.helmholtz_solve(f, sig, O.DIRICHLET)
    D = O.cheb_deriv_matrix(N).astype(np.longdouble)
    D2 = D @ D
    for m in range(3):
        r = D2 @ a[:, m].real.astype(np.longdouble) - sig[m] * a[:, m].real - f[:, m].real
        assert np.abs(np.asarray(r[: N - 1], float)).max() < 1e-9
        assert abs(a[:, m].sum()) < 1e-13 and abs((a[:, m] * (-1.0) ** np.arange(N + 1)).sum()) < 1e-13


def test_w_manufactured_biharmonic():
    """w = (1 - z^2)^2 : w = Dw = 0 at both walls."""
    N = 24
    k2, gamma = 3.7, 1e-3
    beta2 = k2 + 1 / gamma
    w = Poly([1, 0, -1]) ** 2
    theta = w.deriv(2) - k2 * w
    f = theta.deriv(2) - beta2 * theta           # (D^2 - beta2) theta = f = -hw/gamma
    hw = (-gamma * cheb_coeffs(f, N))[:, None].astype(complex)
    th, ww = O.coupled_w_solve(hw, np.array([beta2]), np.array([k2]), gamma)
    assert np.abs(ww[:, 0] - cheb_coeffs(w, N)).max() < 1e-11
    assert np.abs(th[:, 0] - cheb_coeffs(theta, N)).max() < 1e-9
    n = np.arange(N + 1.0)
    assert abs((n * n * ww[:, 0]).sum()) < 1e-10
    assert abs(((-1.0) ** (n + 1) * n * n * ww[:, 0]).sum()) < 1e-10


@pytest.mark.parametrize("N,k2,gamma", [(16, 0.25, 1e-3), (64, 40.0, 8.3e-9), (128, 900.0, 8.3e-9)])
def test_coupled_w_equals_influence_matrix(N, k2, gamma):
    """theta = theta_p + A theta_1 + B theta_2 with A, B from Dw(+-1) = 0 solves the same
    linear system as the coupled (2N+2) dense problem."""
    rng = np.random.default_rng(N + 1)
    hw = (rng.standard_normal(N + 1) + 1j * rng.standard_normal(N + 1))[:, None]
    beta2 = np.array([k2 + 1 / gamma]); k2a = np.array([k2])
    th, w = O.coupled_w_solve(hw, beta2, k2a, gamma)
    zero = np.zeros((N + 1, 1), complex)
    thp = O.helmholtz_solve(-hw / gamma, beta2, O.DIRICHLET)
    th1 = O.helmholtz_solve(zero, beta2, O.DIRICHLET, 1.0, 0.0)
    th2 = O.helmholtz_solve(zero, beta2, O.DIRICHLET, 0.0, 1.0)
    wp, w1, w2 = (O.helmholtz_solve(t, k2a, O.DIRICHLET) for t in (thp, th1, th2))
    bn = O.boundary_rows(N, O.NEUMANN)
    M = np.array([[bn[0] @ w1[:, 0], bn[0] @ w2[:, 0]], [bn[1] @ w1[:, 0], bn[1] @ w2[:, 0]]])
    AB = np.linalg.solve(M, -np.array([bn[0] @ wp[:, 0], bn[1] @ wp[:, 0]]))
    w_im = wp + AB[0] * w1 + AB[1] * w2
    th_im = thp + AB[0] * th1 + AB[1] * th2
    assert np.abs(w_im - w).max() < 1e-10 * max(1.0, np.abs(w).max())
    assert np.abs(th_im - th).max() < 1e-8 * max(1.0, np.abs(th).max())
