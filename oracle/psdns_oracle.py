"""CPU oracle for the pseudo-spectral channel-flow step of arXiv 2406.01322.

TEST INFRASTRUCTURE ONLY.  This file is the slow, plain definition that the CUDA library
(`libpsdns`) is compared against.  Only `tests/`, `__graft_entry__.smoke()` and the
`cpu_baseline` / `--impl reference` legs of `bench.py` may import it.  It shares no code,
table or constant with the CUDA path and imports nothing from the product package.

Everything is float64 / complex128 numpy.  Transforms are dense matrix products with the
DFT / cosine matrices written out from their definitions (no FFT), derivatives are dense
coefficient-space matrices, every Helmholtz problem is assembled densely (Chebyshev tau)
and solved by LAPACK LU with partial pivoting (`numpy.linalg.solve`).  No blocking, no
fusion, no re-ordering beyond what the definitions state.

What the paper fixes and where (PAPER.md line numbers):
  * equations: Cahn-Hilliard Eq. 1 (L58), chemical potential Eq. 4 (L72), Navier-Stokes
    Eqs. 6-7 (L84-86), Korteweg surface-tension force Eq. 8 (L90-92);
  * formulation: wall-normal vorticity Eq. 14 (L120), 4th-order w equation Eq. 15 (L122),
    vorticity definition Eq. 16 (L126), split Cahn-Hilliard Eq. 17 (L130-132);
  * discretisation: Fourier x Fourier x Chebyshev, non-linear terms in physical space,
    Adams-Bashforth / Crank-Nicolson / implicit Euler (L134);
  * time-step algorithm i)-v) (L136-142); Chebyshev transform = DCT-I (L178);
  * "series of 1D Helmholtz independent problems" per (kx, ky) (L134, L200).
Where the paper is silent the readings S1-S21 of SURVEY.md section 8(c) / DESIGN.md are
used; each is named where it enters.

Array conventions (identical to the C-ABI boundary, include/psdns.h):
  PHYSICAL  real    [nz][ny][nx]        z index k <-> z_k = cos(pi k / N), N = nz-1  (S1)
  SPECTRAL  complex [nz][ny][nx//2+1]   n = Chebyshev mode, ky in FFT order, kx = 0..nx/2

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Chebyshev transform of T_m and of z^3,
D T_3 = 3 T_0 + 6 T_2, equality with the length-2N DFT of the even extension (L178),
plane waves / Parseval / shift theorem, dealiased product == exact truncated convolution,
manufactured Helmholtz and biharmonic solutions, coupled-vs-influence-matrix w solve,
Crank-Nicolson decay factor of Stokes modes (omega_z mode with w = 0; clamped eigenmodes of the
4th-order w equation, which pin H_w of Eq. 15), steady Poiseuille flow, algebraic
divergence-freeness, the split-CH operator identity, the tanh equilibrium profile (Eq. 5),
mean(phi) of an off-centre interface (closed form; drift falling spectrally with N),
an independent sympy-differentiated manufactured RHS, and a brute-force all-dense
re-formulation of the step on tiny grids (tests/test_oracle_bruteforce.py).
Parity unpinned (no statement in the paper to pin against): the variable-viscosity term
(reading S14) beyond its lambda=1 limit and the 1-D steady-state quadrature check.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# --------------------------------------------------------------------------------------
# grid, wavenumbers, transform matrices
# --------------------------------------------------------------------------------------


@dataclass(frozen=True)
class Grid:
    """Channel grid: nx, ny equispaced periodic points, nz Chebyshev-Gauss-Lobatto points
    on z in [-1, 1] (domain Lx x Ly x 2h)."""
    nx: int
    ny: int
    nz: int
    lx: float = 4.0 * math.pi
    ly: float = 2.0 * math.pi

    @property
    def N(self) -> int:
        return self.nz - 1

    @property
    def nkx(self) -> int:
        return self.nx // 2 + 1


@dataclass
class Params:
    """Dimensionless groups of Eqs. 2, 9, 10 and the Cahn number (L70), plus the readings
    S12 (mean forcing), S14 (viscosity ratio), S3 (dealiasing)."""
    re: float
    dt: float
    pe: float = 1.0
    ch: float = 1.0
    we: float = 1.0
    gradp_x: float = 0.0
    visc_ratio: float = 1.0
    phase_field: int = 1
    dealias: int = 1
    # "no-slip or free-slip [walls], or a combination of them".  0 = no-slip (u = v = w = 0),
    # 1 = free-slip (w = 0, du/dz = dv/dz = 0), for the wall z = +1 (top) and z = -1 (bottom); reading S10b of DESIGN.md
    wall_top: int = 0
    wall_bottom: int = 0
    # Form of the surface-tension term (reading S5): 0 = divergence of the Korteweg tensor, Eq. 8 as
    # written (tensor in physical space, divergence in spectral space); 1 = the force -c_sigma lap(phi) grad(phi), which
    # differs from Eq. 8 by the gradient c_sigma grad(|grad phi|^2)/2 - annihilated by the curl formulation of Eqs. 14-15
    # in the continuous problem, to truncation error in the discrete one
    surface_tension_form: int = 0
    # Form of the convective term (reading S4): 0 = divergence form -div(u u); 1 = rotational form u x omega
    # (the two differ by grad(|u|^2 / 2), which Eqs. 14-15 annihilate - to truncation error in the discrete problem)
    convection_form: int = 0


NO_SLIP, FREE_SLIP = 0, 1


def cheb_nodes(N: int) -> np.ndarray:
    """S1: z_k = cos(pi k / N), k = 0..N (k = 0 is the wall z = +1)."""
    return np.cos(np.pi * np.arange(N + 1) / N)


def wavenumbers(g: Grid):
    """kx_i = 2 pi i / Lx (i = 0..nx/2); ky_j = 2 pi j' / Ly with j' = j for j <= ny/2,
    j - ny otherwise (FFT order)."""
    kx = 2.0 * np.pi * np.arange(g.nkx) / g.lx
    jp = np.arange(g.ny)
    jp = np.where(jp <= g.ny // 2, jp, jp - g.ny)
    ky = 2.0 * np.pi * jp / g.ly
    return kx, ky


def dft_matrix(n: int, sign: int) -> np.ndarray:
    """F[k, j] = exp(sign * 2 pi i j k / n): the definition of the DFT (S2: sign = -1 and a
    1/n factor on the forward transform, sign = +1 unnormalised on the backward one)."""
    j = np.arange(n)
    return np.exp(sign * 2j * np.pi * np.outer(j, j) / n)


def cheb_bwd_matrix(N: int) -> np.ndarray:
    """Cb[k, n] = T_n(z_k) = cos(pi n k / N): f(z_k) = sum_n a_n T_n(z_k)."""
    k = np.arange(N + 1)
    return np.cos(np.pi * np.outer(k, k) / N)


def cheb_fwd_matrix(N: int) -> np.ndarray:
    """Cf[n, k] = 2 / (N c_n c_k) cos(pi n k / N), c_0 = c_N = 2, else 1 (S2): the discrete
    Chebyshev (Gauss-Lobatto) transform, a DCT-I."""
    k = np.arange(N + 1)
    c = np.ones(N + 1)
    c[0] = c[N] = 2.0
    return (2.0 / N) * np.cos(np.pi * np.outer(k, k) / N) / np.outer(c, c)


def cheb_deriv_matrix(N: int) -> np.ndarray:
    """Coefficient-space derivative, b = D a for d/dz of sum a_n T_n:
    D[n, p] = 2 p / ctilde_n for p > n and p + n odd (ctilde_0 = 2, else 1)."""
    D = np.zeros((N + 1, N + 1))
    for n in range(N + 1):
        for p in range(n + 1, N + 1, 2):
            D[n, p] = 2.0 * p
    D[0, :] *= 0.5
    return D


def apply_along(M: np.ndarray, a: np.ndarray, axis: int) -> np.ndarray:
    """out[..., r, ...] = sum_c M[r, c] a[..., c, ...] along `axis`: one dense matrix product."""
    M = M.astype(np.result_type(M.dtype, a.dtype), copy=False)
    a = a.astype(M.dtype, copy=False)
    return np.moveaxis(np.tensordot(M, a, axes=(1, axis)), 0, axis)


# --------------------------------------------------------------------------------------
# 3-D transforms (x first, then y, then z on the way forward)
# --------------------------------------------------------------------------------------


def forward_transform(f: np.ndarray, g: Grid) -> np.ndarray:
    """PHYSICAL -> SPECTRAL.  fhat(i, j, n) = (1/(nx ny)) sum_xy f e^{-i(kx x + ky y)},
    then the Chebyshev transform of every (kx, ky) column (S2).  x is real-to-half-complex
    (D2Z, L176)."""
    f = np.asarray(f, dtype=np.float64)
    assert f.shape == (g.nz, g.ny, g.nx)
    Fx = dft_matrix(g.nx, -1)[: g.nkx, :] / g.nx          # [i, x]
    Fy = dft_matrix(g.ny, -1) / g.ny                      # [j, y]
    Cf = cheb_fwd_matrix(g.N)                             # [n, k]
    a = apply_along(Fx, f, 2)                             # [k, y, i]
    a = apply_along(Fy, a, 1)                             # [k, j, i]
    a = apply_along(Cf, a, 0)                             # [n, j, i]
    return a


def backward_transform(a: np.ndarray, g: Grid) -> np.ndarray:
    """SPECTRAL -> PHYSICAL: f = sum_{i,j',n} fhat T_n(z_k) e^{i(kx x + ky y)} with the
    conjugate half of the x spectrum implied.  The i = 0 and i = nx/2 planes contribute
    only the real part after the y transform (S20)."""
    a = np.asarray(a, dtype=np.complex128)
    assert a.shape == (g.nz, g.ny, g.nkx)
    Cb = cheb_bwd_matrix(g.N)
    By = dft_matrix(g.ny, +1)                             # [y, j]
    b = apply_along(Cb, a, 0)                             # [k, j, i]
    b = apply_along(By, b, 1)                             # [k, y, i]
    i = np.arange(g.nkx)
    x = np.arange(g.nx)
    w = np.full(g.nkx, 2.0)
    w[0] = 1.0
    if g.nx % 2 == 0:
        w[-1] = 1.0
    ang = 2.0 * np.pi * np.outer(i, x) / g.nx             # [i, x]
    # f(x) = sum_i w_i Re( b_i e^{+i ang} )
    return b.real @ (w[:, None] * np.cos(ang)) - b.imag @ (w[:, None] * np.sin(ang))


# --------------------------------------------------------------------------------------
# dealiasing (reading S3: the paper gives no rule)
# --------------------------------------------------------------------------------------


def retained_counts(g: Grid, dealias: int = 1):
    """S3: 2/3 rule in all three directions: keep i <= nx//3, |j'| <= ny//3, n <= (2N)//3.
    Returns (I, J, K) = the three cut-offs."""
    if dealias:
        return g.nx // 3, g.ny // 3, (2 * g.N) // 3
    # no dealiasing: everything except the x / y Nyquist planes, all Chebyshev modes
    return g.nx // 2 - 1, g.ny // 2 - 1, g.N


def truncation_mask(g: Grid, dealias: int = 1, z: bool = True) -> np.ndarray:
    """Boolean mask [nz, ny, nkx] of the retained coefficients (operator P of S3);
    z=False gives the (kx, ky)-only mask P_xy."""
    I, J, K = retained_counts(g, dealias)
    jp = np.arange(g.ny)
    jp = np.where(jp <= g.ny // 2, jp, jp - g.ny)
    mi = np.arange(g.nkx) <= I
    mj = np.abs(jp) <= J
    mn = (np.arange(g.nz) <= K) if z else np.ones(g.nz, dtype=bool)
    return mn[:, None, None] & mj[None, :, None] & mi[None, None, :]


# --------------------------------------------------------------------------------------
# Chebyshev-tau Helmholtz problems (reading S11)
# --------------------------------------------------------------------------------------

DIRICHLET = 0
NEUMANN = 1
SECOND_DERIVATIVE = 2


def wall_row(N: int, kind: int, wall: int) -> np.ndarray:
    """Row acting on Chebyshev coefficients that evaluates, at the wall z = wall (+1 or -1):
    the value T_n(+-1) = (+-1)^n (DIRICHLET), the first derivative T_n'(+-1) = (+-1)^(n+1) n^2 (NEUMANN) or the
    second derivative T_n''(+-1) = (+-1)^n n^2 (n^2 - 1) / 3 (SECOND_DERIVATIVE)."""
    n = np.arange(N + 1, dtype=np.float64)
    sgn = np.ones(N + 1) if wall > 0 else np.where(np.arange(N + 1) % 2 == 0, 1.0, -1.0)
    if kind == DIRICHLET:
        return sgn
    if kind == NEUMANN:
        return (sgn if wall > 0 else -sgn) * n * n
    return sgn * n * n * (n * n - 1.0) / 3.0


def boundary_rows(N: int, bc) -> np.ndarray:
    """Two rows acting on Chebyshev coefficients, first the wall z = +1, then z = -1.  bc: one kind for both walls, or a
    pair (kind at z = +1, kind at z = -1) for mixed walls."""
    bp, bm = (bc, bc) if np.isscalar(bc) else bc
    return np.stack([wall_row(N, bp, +1), wall_row(N, bm, -1)])


def helmholtz_solve(f: np.ndarray, sigma: np.ndarray, bc: int,
                    bplus=0.0, bminus=0.0, chunk: int = 256) -> np.ndarray:
    """Solve (D^2 - sigma_m) a_m = f_m (rows 0..N-2) with boundary values/derivatives
    bplus at z=+1 and bminus at z=-1, for a batch m of independent columns.
    f: complex [N+1, M]; sigma: real [M].  Dense assembly + LU per column."""
    N = f.shape[0] - 1
    M = f.shape[1]
    D = cheb_deriv_matrix(N)
    D2 = D @ D
    rows = boundary_rows(N, bc)
    bplus = np.broadcast_to(np.asarray(bplus, dtype=np.complex128), (M,))
    bminus = np.broadcast_to(np.asarray(bminus, dtype=np.complex128), (M,))
    out = np.empty_like(f, dtype=np.complex128)
    eye = np.eye(N + 1)
    for s in range(0, M, chunk):
        e = min(M, s + chunk)
        A = D2[None, :, :] - sigma[s:e, None, None] * eye[None, :, :]
        A[:, N - 1:, :] = rows[None, :, :]
        rhs = f[:, s:e].T.copy()                         # [m, N+1]
        rhs[:, N - 1] = bplus[s:e]
        rhs[:, N] = bminus[s:e]
        b = np.stack([rhs.real, rhs.imag], axis=-1)      # [m, N+1, 2]
        x = np.linalg.solve(A, b)
        out[:, s:e] = (x[..., 0] + 1j * x[..., 1]).T
    return out


def coupled_w_solve(hw: np.ndarray, beta2: np.ndarray, k2: np.ndarray, gamma: float,
                    chunk: int = 64, walls=(NO_SLIP, NO_SLIP)):
    """The 4th-order wall-normal velocity problem as two coupled Helmholtz problems
    (readings S10, S11, S13):
        (D^2 - beta2) theta = -hw / gamma     rows 0..N-2, no condition on theta
        (D^2 - k2) w - theta = 0              rows 0..N-2
        w(+-1) = 0, and per wall Dw = 0 (no-slip) or D^2 w = 0 (free-slip: du/dz = dv/dz = 0 and continuity,
        PAPER.md L52; walls = (kind at z = +1, kind at z = -1))
    assembled as one (2N+2)x(2N+2) dense system per column.  Returns (theta, w)."""
    N = hw.shape[0] - 1
    M = hw.shape[1]
    D = cheb_deriv_matrix(N)
    D2 = D @ D
    eye = np.eye(N + 1)
    bd = boundary_rows(N, DIRICHLET)
    bn = boundary_rows(N, tuple(SECOND_DERIVATIVE if k == FREE_SLIP else NEUMANN for k in walls))
    theta = np.empty((N + 1, M), dtype=np.complex128)
    w = np.empty((N + 1, M), dtype=np.complex128)
    n1 = N + 1
    for s in range(0, M, chunk):
        e = min(M, s + chunk)
        m = e - s
        A = np.zeros((m, 2 * n1, 2 * n1))
        # unknown vector = [theta (N+1), w (N+1)]
        A[:, : N - 1, :n1] = (D2[None] - beta2[s:e, None, None] * eye[None])[:, : N - 1, :]
        A[:, N - 1: 2 * N - 2, :n1] = -eye[None, : N - 1, :]
        A[:, N - 1: 2 * N - 2, n1:] = (D2[None] - k2[s:e, None, None] * eye[None])[:, : N - 1, :]
        A[:, 2 * N - 2: 2 * N, n1:] = bd[None]
        A[:, 2 * N: 2 * N + 2, n1:] = bn[None]
        rhs = np.zeros((m, 2 * n1), dtype=np.complex128)
        rhs[:, : N - 1] = (-hw[: N - 1, s:e] / gamma).T
        b = np.stack([rhs.real, rhs.imag], axis=-1)
        x = np.linalg.solve(A, b)
        xc = x[..., 0] + 1j * x[..., 1]
        theta[:, s:e] = xc[:, :n1].T
        w[:, s:e] = xc[:, n1:].T
    return theta, w


# --------------------------------------------------------------------------------------
# pointwise non-linear terms (row a5; Eqs. 1, 4, 7, 8; L182-196)
# --------------------------------------------------------------------------------------


def pointwise_terms(p: Params, u, v, w, phi=None, phx=None, phy=None, phz=None, strain=None, lap_phi=None, vort=None):
    """Physical-space products.  Returns dict with the symmetric flux tensor
    T_ij = -u_i u_j + c_sigma ( |grad phi|^2 delta_ij - phi_i phi_j ) [+ (eta-1)/Re E_ij]
    (divergence form of Eq. 7's convective term, reading S4; Korteweg tensor of Eq. 8,
    c_sigma = 3/sqrt(8) Ch/We, reading S5; variable viscosity reading S14) and, with the
    phase field on, Q = u . grad phi (Eq. 1) and C = phi^3 (Eq. 4)."""
    if p.convection_form == 0:
        T = {
            "xx": -u * u, "xy": -u * v, "xz": -u * w,
            "yy": -v * v, "yz": -v * w, "zz": -w * w,
        }
        out = {"T": T}
    else:
        # rotational form: -(u . grad) u = u x omega - grad(|u|^2 / 2); the gradient is dropped, u x omega is a force vector
        zero = np.zeros_like(u)
        T = {k: zero.copy() for k in ("xx", "xy", "xz", "yy", "yz", "zz")}
        ox, oy, oz = vort
        out = {"T": T, "F": {"x": v * oz - w * oy, "y": w * ox - u * oz, "z": u * oy - v * ox}}
    if p.phase_field:
        cs = 3.0 / math.sqrt(8.0) * p.ch / p.we
        if p.surface_tension_form == 0:
            g2 = phx * phx + phy * phy + phz * phz
            T["xx"] = T["xx"] + cs * (g2 - phx * phx)
            T["yy"] = T["yy"] + cs * (g2 - phy * phy)
            T["zz"] = T["zz"] + cs * (g2 - phz * phz)
            T["xy"] = T["xy"] - cs * phx * phy
            T["xz"] = T["xz"] - cs * phx * phz
            T["yz"] = T["yz"] - cs * phy * phz
        else:
            # force form: f = -c_sigma lap(phi) grad(phi), a vector added to S = div T (not a divergence itself)
            fs = {"x": -cs * lap_phi * phx, "y": -cs * lap_phi * phy, "z": -cs * lap_phi * phz}
            out["F"] = {k: out["F"][k] + fs[k] for k in fs} if "F" in out else fs
        out["Q"] = u * phx + v * phy + w * phz
        out["C"] = phi * phi * phi
        if p.visc_ratio != 1.0:
            # S14: eta(phi) = 1 + (lambda-1)(phi+1)/2; explicit part (eta-1)/Re * E_ij,
            # E_ij = d_i u_j + d_j u_i, E_zz = -E_xx - E_yy (continuity, Eq. 6)
            eta1 = (p.visc_ratio - 1.0) * (phi + 1.0) * 0.5 / p.re
            exx, eyy, exy, exz, eyz = strain
            T["xx"] = T["xx"] + eta1 * exx
            T["yy"] = T["yy"] + eta1 * eyy
            T["zz"] = T["zz"] + eta1 * (-exx - eyy)
            T["xy"] = T["xy"] + eta1 * exy
            T["xz"] = T["xz"] + eta1 * exz
            T["yz"] = T["yz"] + eta1 * eyz
    return out


# --------------------------------------------------------------------------------------
# the solver
# --------------------------------------------------------------------------------------


@dataclass
class State:
    u: np.ndarray
    v: np.ndarray
    w: np.ndarray
    phi: np.ndarray | None
    theta: np.ndarray               # hidden: (D^2 - k^2) w  (S13)
    hist: dict = field(default_factory=dict)   # N^{n-1} terms for AB2 (S7)
    nstep: int = 0


class Oracle:
    """psdns_init / set_state / step / get_state, the slow way."""

    def __init__(self, g: Grid, p: Params):
        assert g.nx % 2 == 0 and g.ny % 2 == 0 and g.nz >= 5
        self.g, self.p = g, p
        self.kx, self.ky = wavenumbers(g)
        self.KX = self.kx[None, None, :]
        self.KY = self.ky[None, :, None]
        self.K2 = (self.KX ** 2 + self.KY ** 2)              # [1, ny, nkx]
        self.D = cheb_deriv_matrix(g.N)
        self.D2 = self.D @ self.D
        self.P = truncation_mask(g, p.dealias, z=True)
        self.Pxy = truncation_mask(g, p.dealias, z=False)
        self.state: State | None = None

    # -- helpers ------------------------------------------------------------------------
    def _Dz(self, a):
        return apply_along(self.D, a, 0)

    def _D2z(self, a):
        return apply_along(self.D2, a, 0)

    def _lap(self, a):
        return self._D2z(a) - self.K2 * a

    # -- state --------------------------------------------------------------------------
    def set_state(self, space: str, u, v, w, phi=None):
        """Step i) of the time-step algorithm.  PHYSICAL input is forward
        transformed in full; the (kx, ky) modes outside the retained set are then dropped
        (P_xy, S3) because the step only ever solves retained wavenumbers.  Derives the
        hidden theta = (D^2 - k^2) w (S13) and clears the AB2 history (S7)."""
        g = self.g
        if space == "physical":
            u, v, w = (forward_transform(f, g) for f in (u, v, w))
            if self.p.phase_field:
                phi = forward_transform(phi, g)
        u, v, w = (np.where(self.Pxy, np.asarray(f, dtype=np.complex128), 0.0) for f in (u, v, w))
        if self.p.phase_field:
            phi = np.where(self.Pxy, np.asarray(phi, dtype=np.complex128), 0.0)
        else:
            phi = None
        theta = self._lap(w)
        self.state = State(u, v, w, phi, theta)

    def get_state(self, space: str):
        s = self.state
        fields = [s.u, s.v, s.w] + ([s.phi] if self.p.phase_field else [])
        if space == "physical":
            fields = [backward_transform(f, self.g) for f in fields]
        return fields

    # -- non-linear terms in spectral space (rows a1-a8) -------------------------------------
    def nonlinear_spectra(self):
        """Rows a1-a8: truncated copies -> backward transforms -> pointwise products ->
        forward transforms -> truncation.  Returns dict of the 6 T_ij spectra (+Q, C)."""
        g, p, s = self.g, self.p, self.state
        P = self.P
        uP, vP, wP = (np.where(P, f, 0.0) for f in (s.u, s.v, s.w))
        spec = [uP, vP, wP]
        if p.phase_field:
            phP = np.where(P, s.phi, 0.0)
            spec += [phP, 1j * self.KX * phP, 1j * self.KY * phP, self._Dz(phP)]
            if p.surface_tension_form == 1:
                lap_spec = np.where(P, self._lap(phP), 0.0)      # lap of the truncated phi, truncated again (operator P)
            if p.visc_ratio != 1.0:
                spec += [2j * self.KX * uP, 2j * self.KY * vP,
                         1j * self.KY * uP + 1j * self.KX * vP,
                         self._Dz(uP) + 1j * self.KX * wP,
                         self._Dz(vP) + 1j * self.KY * wP]
        phys = [backward_transform(a, g) for a in spec]
        vort = None
        if p.convection_form == 1:   # vorticity of the truncated velocity, in spectral space, then to physical space
            vs = [1j * self.KY * wP - self._Dz(vP), self._Dz(uP) - 1j * self.KX * wP, 1j * self.KX * vP - 1j * self.KY * uP]
            vort = [backward_transform(a, g) for a in vs]
        if p.phase_field:
            strain = phys[7:12] if p.visc_ratio != 1.0 else None
            lap_phys = backward_transform(lap_spec, g) if p.surface_tension_form == 1 else None
            pw = pointwise_terms(p, phys[0], phys[1], phys[2], phys[3], phys[4], phys[5], phys[6], strain, lap_phys, vort)
        else:
            pw = pointwise_terms(p, phys[0], phys[1], phys[2], vort=vort)
        out = {k: np.where(P, forward_transform(t, g), 0.0) for k, t in pw["T"].items()}
        if p.phase_field:
            out["Q"] = np.where(P, forward_transform(pw["Q"], g), 0.0)
            out["C"] = np.where(P, forward_transform(pw["C"], g), 0.0)
            out["phP"] = phP
        if "F" in pw:
            for k, t in pw["F"].items():
                out["F" + k] = np.where(P, forward_transform(t, g), 0.0)
        return out

    def explicit_terms(self):
        """Row a9: S = div T (+G), N_omega (Eq. 14), N_w (Eq. 15), S_phi (Eq. 17, S8, S9)."""
        p = self.p
        t = self.nonlinear_spectra()
        ikx, iky = 1j * self.KX, 1j * self.KY
        Sx = ikx * t["xx"] + iky * t["xy"] + self._Dz(t["xz"])
        Sy = ikx * t["xy"] + iky * t["yy"] + self._Dz(t["yz"])
        Sz = ikx * t["xz"] + iky * t["yz"] + self._Dz(t["zz"])
        if "Fx" in t:                                              # force form of the surface tension (8(f)-4)
            Sx, Sy, Sz = Sx + t["Fx"], Sy + t["Fy"], Sz + t["Fz"]
        Sx[0, 0, 0] += p.gradp_x                                   # S12
        N = {}
        N["om"] = ikx * Sy - iky * Sx                              # Eq. 14
        N["w"] = -self.K2 * Sz - self._Dz(ikx * Sx + iky * Sy)     # Eq. 15
        N["ubar"] = Sx[:, 0, 0].copy()                             # S12: mean-flow equations
        N["vbar"] = Sy[:, 0, 0].copy()
        if p.phase_field:
            s_coef = 2.0 * math.sqrt(p.pe / (p.dt * p.ch ** 2))    # S8
            N["phi"] = (-t["Q"] + (1.0 / p.pe) * self._lap(t["C"])
                        - ((1.0 + s_coef * p.ch ** 2) / p.pe) * self._lap(t["phP"]))   # S9
        return N

    # -- one step ------------------------------------------------------
    def step(self, nsteps: int = 1):
        for _ in range(nsteps):
            self._step_once()

    def _step_once(self):
        g, p, s = self.g, self.p, self.state
        Nn = self.explicit_terms()
        if s.nstep == 0 or not s.hist:
            NL = Nn                                                 # S7: Euler start-up
        else:
            NL = {k: 1.5 * Nn[k] - 0.5 * s.hist[k] for k in Nn}     # AB2
        dt = p.dt
        gamma = dt / (2.0 * p.re)
        ikx, iky = 1j * self.KX, 1j * self.KY

        # retained (kx, ky) columns
        ret = np.argwhere(self.Pxy[0])                             # [(j, i)]
        nz = g.nz
        jj, ii = ret[:, 0], ret[:, 1]
        k2 = (self.kx[ii] ** 2 + self.ky[jj] ** 2)
        nonzero = ~((jj == 0) & (ii == 0))
        jn, in_ = jj[nonzero], ii[nonzero]
        k2n = k2[nonzero]
        beta2 = k2n + 1.0 / gamma

        # -- wall-normal vorticity, Eq. 14, Crank-Nicolson
        om = ikx * s.v - iky * s.u                                   # Eq. 16
        H_om = om + gamma * self._lap(om) + dt * NL["om"]
        # walls: no-slip u = v = 0 gives omega_z = 0; free-slip du/dz = dv/dz = 0 gives d omega_z/dz = 0
        walls = (p.wall_top, p.wall_bottom)
        bc_h = tuple(NEUMANN if k == FREE_SLIP else DIRICHLET for k in walls)
        om_new = helmholtz_solve(-H_om[:, jn, in_] / gamma, beta2, bc_h)

        # -- wall-normal velocity, Eq. 15, Crank-Nicolson, two Helmholtz problems (L140)
        H_w = s.theta + gamma * self._lap(s.theta) + dt * NL["w"]
        th_new, w_new = coupled_w_solve(H_w[:, jn, in_], beta2, k2n, gamma, walls=walls)

        # -- u, v from continuity (Eq. 6) and the vorticity definition (Eq. 16): row a11
        Dcol = self.D.astype(np.complex128)
        Dw = Dcol @ w_new
        ikxc, ikyc = 1j * self.kx[in_][None, :], 1j * self.ky[jn][None, :]
        u_new = (ikxc * Dw + ikyc * om_new) / k2n[None, :]
        v_new = (ikyc * Dw - ikxc * om_new) / k2n[None, :]

        U = np.zeros((nz, g.ny, g.nkx), dtype=np.complex128)
        V = np.zeros_like(U)
        W = np.zeros_like(U)
        TH = np.zeros_like(U)
        U[:, jn, in_] = u_new
        V[:, jn, in_] = v_new
        W[:, jn, in_] = w_new
        TH[:, jn, in_] = th_new

        # -- mean flow (kx, ky) = (0, 0), reading S12
        for name, F in (("ubar", s.u), ("vbar", s.v)):
            m = F[:, 0, 0]
            H = m + gamma * (self.D2 @ m) + dt * NL[name]
            sol = helmholtz_solve((-H / gamma)[:, None], np.array([1.0 / gamma]), bc_h)
            (U if name == "ubar" else V)[:, 0, 0] = sol[:, 0]

        # -- Cahn-Hilliard, Eq. 17, implicit Euler, two Helmholtz problems (L142)
        PHI = None
        if p.phase_field:
            gphi = dt * p.ch ** 2 / p.pe
            lam = math.sqrt(p.pe / (dt * p.ch ** 2))
            H_phi = s.phi + dt * NL["phi"]
            sig = k2 + lam
            psi = helmholtz_solve(H_phi[:, jj, ii] / gphi, sig, NEUMANN)
            ph = helmholtz_solve(psi, sig, NEUMANN)
            PHI = np.zeros_like(U)
            PHI[:, jj, ii] = ph

        self.state = State(U, V, W, PHI, TH, hist=Nn, nstep=s.nstep + 1)


# --------------------------------------------------------------------------------------
# diagnostics used by tests
# --------------------------------------------------------------------------------------


def divergence_spectrum(g: Grid, u, v, w):
    kx, ky = wavenumbers(g)
    D = cheb_deriv_matrix(g.N).astype(np.complex128)
    return 1j * kx[None, None, :] * u + 1j * ky[None, :, None] * v + apply_along(D, w, 0)


def mean_phi(g: Grid, phi_hat):
    """Volume mean of phi: (1/2) int_{-1}^{1} of the (0,0) column = (1/2) sum_{n even}
    a_n * 2 / (1 - n^2)."""
    n = np.arange(0, g.nz, 2)
    return float(np.real(np.sum(phi_hat[n, 0, 0] * (2.0 / (1.0 - n.astype(np.float64) ** 2)))) * 0.5)


def clenshaw_curtis_weights(N: int) -> np.ndarray:
    """Quadrature weights on z_k = cos(pi k/N) that integrate every polynomial of degree <= N exactly over
    [-1, 1]: int f dz = sum_{n even} a_n 2/(1 - n^2) with a = forward Chebyshev transform of f, hence
    w_k = sum_{n even} 2/(1 - n^2) Cf[n, k]."""
    n = np.arange(0, N + 1, 2)
    return (2.0 / (1.0 - n.astype(np.float64) ** 2)) @ cheb_fwd_matrix(N)[n, :]


def kinetic_energy(g: Grid, u_hat, v_hat, w_hat) -> float:
    """Volume-averaged kinetic energy (1/2) <u^2 + v^2 + w^2> of the diagnostics row,
    evaluated the plain way: fields in physical space, mean over the periodic x, y points, Clenshaw-Curtis quadrature
    over the collocation points in z, divided by the channel height 2."""
    e = sum(backward_transform(a, g) ** 2 for a in (u_hat, v_hat, w_hat))
    return float(0.25 * np.sum(clenshaw_curtis_weights(g.N) * e.mean(axis=(1, 2))))


def wall_shear(g: Grid, u_hat):
    """d u-bar/dz of the mean streamwise velocity (the (0,0) column) at z = +1 and z = -1:
    T_n'(+-1) = (+-1)^(n+1) n^2."""
    n = np.arange(g.nz, dtype=np.float64)
    a = np.real(u_hat[:, 0, 0])
    return float(np.sum(n * n * a)), float(np.sum(np.where(np.arange(g.nz) % 2 == 0, -1.0, 1.0) * n * n * a))


def bulk_velocity(g: Grid, u_hat) -> float:
    """(1/2) int u-bar dz, same quadrature as mean_phi."""
    return mean_phi(g, u_hat)


def max_divergence(g: Grid, u, v, w) -> float:
    """max over the spectrum of |i kx u^ + i ky v^ + D w^|."""
    return float(np.abs(divergence_spectrum(g, u, v, w)).max())


def rel_l2(a, b):
    """||a - b||_2 / ||b||_2 over all entries."""
    a, b = np.asarray(a), np.asarray(b)
    den = np.linalg.norm(b.ravel())
    return float(np.linalg.norm((a - b).ravel()) / (den if den > 0 else 1.0))
