"""Pin for the oracle's full step (not gpu): an independent ALL-DENSE re-formulation of psdns_step on tiny grids
(8x8x9, 16x8x17), SURVEY 8(c) "full step: brute force on tiny grids against an independent all-dense formulation".

Nothing below calls a helper of `psdns_oracle` except to run the oracle itself for the comparison.  The
re-formulation differs from the oracle in construction wherever the mathematics allows a second route:
  * spectra are kept on the FULL signed wavenumber set (i', j' of both signs, Hermitian pairs explicit) and fields are
    summed directly, f = sum a T_n(z) e^{i(kx x + ky y)}: no half-spectrum weights, no real/imaginary split (oracle:
    backward_transform);
  * the z derivative is the ANALYTIC derivative of the basis, T_n'(z) = n sin(n t)/sin t (n^2 (+-1)^(n+1) at the walls),
    evaluated at the nodes and transformed back, D = Cf T' (oracle: the 2p/c_n upper-triangular recurrence matrix);
    grad(phi) is evaluated in physical space from the differentiated series, not from derived spectra;
  * Eq. 15's explicit term is taken in the continuous form N_w = lap(S_z) - d/dz div(S) (oracle:
    -k^2 S_z - D(ikx S_x + iky S_y));
  * every implicit problem is ONE dense linear system over all wavenumbers and Chebyshev modes at once (block diagonal
    in exact arithmetic, assembled as a full matrix and solved by one LU), the w problem as the coupled theta-w system
    with the four wall conditions written with T_n(+-1), T_n'(+-1).
Conventions (readings S1-S13 of DESIGN.md) are restated from PAPER.md Eqs. 1-17, L134-142."""
import math

import numpy as np
import pytest

import psdns_inputs as I
import psdns_oracle as O


class DenseStep:
    def __init__(self, nx, ny, nz, lx, ly, re, dt, pe, ch, we, gradp):
        self.nx, self.ny, self.N = nx, ny, nz - 1
        N = self.N
        self.re, self.dt, self.pe, self.ch, self.we, self.gradp = re, dt, pe, ch, we, gradp
        self.x = lx / nx * np.arange(nx)
        self.y = ly / ny * np.arange(ny)
        t = np.pi * np.arange(N + 1) / N
        self.z = np.cos(t)                                                   # S1
        I3, J3, self.K3 = nx // 3, ny // 3, (2 * N) // 3                     # S3
        self.ip = np.arange(-I3, I3 + 1)                                     # signed retained wavenumber indices
        self.jp = np.arange(-J3, J3 + 1)
        self.kx = 2 * np.pi / lx * self.ip
        self.ky = 2 * np.pi / ly * self.jp
        n = np.arange(N + 1)
        self.T = np.cos(np.outer(t, n))                                      # T[k, n] = T_n(z_k)
        with np.errstate(divide="ignore", invalid="ignore"):
            Tp = n[None, :] * np.sin(np.outer(t, n)) / np.sin(t)[:, None]
        Tp[0, :] = n ** 2.0                                                  # T_n'(+1) = n^2
        Tp[N, :] = n ** 2.0 * (-1.0) ** (n + 1)                              # T_n'(-1) = (-1)^(n+1) n^2
        self.Tp = Tp
        c = np.ones(N + 1); c[0] = c[N] = 2.0
        self.Cf = (2.0 / N) * self.T.T / np.outer(c, c)                      # S2: a_n = 2/(N c_n) sum_k f_k T_n(z_k)/c_k
        self.D = self.Cf @ Tp                                                # coefficient-space d/dz
        self.Ex = np.exp(1j * np.outer(self.x, self.kx))                     # [x, i']
        self.Ey = np.exp(1j * np.outer(self.y, self.ky))                     # [y, j']

    # physical real [k, y, x]  ->  coefficients [n, j', i'] on the signed retained set
    def fwd(self, f):
        a = np.einsum("kyx,xi->kyi", f, self.Ex.conj()) / self.nx
        a = np.einsum("kyi,yj->kji", a, self.Ey.conj()) / self.ny
        return np.einsum("nk,kji->nji", self.Cf, a)

    def bwd(self, a, zmat=None):
        zmat = self.T if zmat is None else zmat
        f = np.einsum("kn,nji->kji", zmat, a)
        f = np.einsum("kji,yj->kyi", f, self.Ey)
        f = np.einsum("kyi,xi->kyx", f, self.Ex)
        assert np.abs(f.imag).max() <= 1e-9 * max(1.0, np.abs(f.real).max())   # Hermitian pairs make the sum real
        return f.real

    def cut(self, a):                                                        # operator P in z
        b = a.copy(); b[self.K3 + 1:] = 0.0
        return b

    def dz(self, a):
        return np.einsum("nm,mji->nji", self.D, a)

    def lap(self, a):
        KX, KY = self.kx[None, None, :], self.ky[None, :, None]
        return self.dz(self.dz(a)) - (KX ** 2 + KY ** 2) * a

    def explicit(self, u, v, w, ph):
        KX, KY = 1j * self.kx[None, None, :], 1j * self.ky[None, :, None]
        uP, vP, wP, pP = (self.cut(a) for a in (u, v, w, ph))
        U, V, W, PH = (self.bwd(a) for a in (uP, vP, wP, pP))
        px, py, pz = self.bwd(KX * pP), self.bwd(KY * pP), self.bwd(pP, self.Tp)
        cs = 3.0 / math.sqrt(8.0) * self.ch / self.we                        # Eq. 8
        vel, gp = (U, V, W), (px, py, pz)
        g2 = px * px + py * py + pz * pz
        T = [[self.cut(self.fwd(-vel[a] * vel[b] + cs * ((g2 if a == b else 0.0) - gp[a] * gp[b])))
              for b in range(3)] for a in range(3)]                          # Eq. 7 (divergence form, S4) + Eq. 8
        d = (lambda a: KX * a, lambda a: KY * a, self.dz)
        S = [sum(d[b](T[a][b]) for b in range(3)) for a in range(3)]
        j0, i0 = len(self.jp) // 2, len(self.ip) // 2
        S[0][0, j0, i0] += self.gradp                                        # S12
        divS = sum(d[a](S[a]) for a in range(3))
        out = {"om": KX * S[1] - KY * S[0],                                  # Eq. 14
               "w": self.lap(S[2]) - self.dz(divS),                          # Eq. 15, continuous form
               "ubar": S[0][:, j0, i0].copy(), "vbar": S[1][:, j0, i0].copy()}
        Q = self.cut(self.fwd(U * px + V * py + W * pz))                     # Eq. 1
        C = self.cut(self.fwd(PH ** 3))                                      # Eq. 4
        s_coef = 2.0 * math.sqrt(self.pe / (self.dt * self.ch ** 2))         # S8
        out["phi"] = -Q + self.lap(C) / self.pe - (1.0 + s_coef * self.ch ** 2) / self.pe * self.lap(pP)   # Eq. 17, S9
        return out

    def big_solve(self, sig, rhs, brow, btarget=0.0):
        """All columns at once: unknown x[(col, n)], rows n <= N-2 of (D^2 - sig_col) x = rhs, two wall rows per column."""
        N, ncol = self.N, len(sig)
        n1 = N + 1
        D2 = self.D @ self.D
        A = np.zeros((ncol * n1, ncol * n1)); b = np.zeros(ncol * n1, dtype=complex)
        for c in range(ncol):
            blk = D2 - sig[c] * np.eye(n1)
            blk[N - 1:] = brow
            A[c * n1:(c + 1) * n1, c * n1:(c + 1) * n1] = blk
            b[c * n1:c * n1 + N - 1] = rhs[: N - 1, c]
            b[c * n1 + N - 1:(c + 1) * n1] = btarget
        x = np.linalg.solve(A, b)
        return x.reshape(ncol, n1).T

    def step(self, st, hist):
        u, v, w, ph, th = st
        N, dt = self.N, self.dt
        n1 = N + 1
        Nn = self.explicit(u, v, w, ph)
        NL = Nn if hist is None else {k: 1.5 * Nn[k] - 0.5 * hist[k] for k in Nn}      # S7
        gam = dt / (2.0 * self.re)
        KX, KY = self.kx[None, None, :], self.ky[None, :, None]
        K2 = (KX ** 2 + KY ** 2) * np.ones((1, len(self.jp), len(self.ip)))
        nj, ni = len(self.jp), len(self.ip)
        j0, i0 = nj // 2, ni // 2
        cols = [(j, i) for j in range(nj) for i in range(ni) if not (j == j0 and i == i0)]
        jj, ii = np.array([c[0] for c in cols]), np.array([c[1] for c in cols])
        k2 = K2[0, jj, ii]
        dir_rows = np.stack([self.T[0], self.T[N]])                          # values at z = +1, -1
        neu_rows = np.stack([self.Tp[0], self.Tp[N]])                        # derivatives at z = +1, -1
        om = 1j * KX * v - 1j * KY * u                                       # Eq. 16
        H_om = om + gam * self.lap(om) + dt * NL["om"]
        om_new = self.big_solve(k2 + 1.0 / gam, -H_om[:, jj, ii] / gam, dir_rows)
        # w: coupled (theta, w) system, all columns at once
        H_w = th + gam * self.lap(th) + dt * NL["w"]
        ncol = len(cols)
        D2 = self.D @ self.D
        A = np.zeros((ncol * 2 * n1, ncol * 2 * n1)); b = np.zeros(ncol * 2 * n1, dtype=complex)
        for c in range(ncol):
            o = c * 2 * n1
            A[o:o + N - 1, o:o + n1] = (D2 - (k2[c] + 1.0 / gam) * np.eye(n1))[: N - 1]
            b[o:o + N - 1] = -H_w[: N - 1, jj[c], ii[c]] / gam
            A[o + N - 1:o + 2 * N - 2, o + n1:o + 2 * n1] = (D2 - k2[c] * np.eye(n1))[: N - 1]
            A[o + N - 1:o + 2 * N - 2, o:o + n1] = -np.eye(n1)[: N - 1]
            A[o + 2 * N - 2:o + 2 * N, o + n1:o + 2 * n1] = dir_rows
            A[o + 2 * N:o + 2 * N + 2, o + n1:o + 2 * n1] = neu_rows
        x = np.linalg.solve(A, b).reshape(ncol, 2 * n1)
        th_new, w_new = x[:, :n1].T, x[:, n1:].T
        dw = self.D @ w_new
        ikx, iky = 1j * self.kx[ii][None, :], 1j * self.ky[jj][None, :]
        u_new = (ikx * dw + iky * om_new) / k2[None, :]                      # Eqs. 6, 16
        v_new = (iky * dw - ikx * om_new) / k2[None, :]
        U, V, W, TH = (np.zeros_like(u) for _ in range(4))
        U[:, jj, ii], V[:, jj, ii], W[:, jj, ii], TH[:, jj, ii] = u_new, v_new, w_new, th_new
        for name, F, OUT in (("ubar", u, U), ("vbar", v, V)):                # S12
            m = F[:, j0, i0]
            H = m + gam * (D2 @ m) + dt * NL[name]
            OUT[:, j0, i0] = self.big_solve(np.array([1.0 / gam]), (-H / gam)[:, None], dir_rows)[:, 0]
        gphi = dt * self.ch ** 2 / self.pe
        lam = math.sqrt(self.pe / (dt * self.ch ** 2))
        allj, alli = np.meshgrid(np.arange(nj), np.arange(ni), indexing="ij")
        aj, ai = allj.ravel(), alli.ravel()
        sig = K2[0, aj, ai] + lam
        H_phi = ph + dt * NL["phi"]
        psi = self.big_solve(sig, H_phi[:, aj, ai] / gphi, neu_rows)         # Eq. 17 as two Helmholtz problems (L142)
        PHI = np.zeros_like(ph)
        PHI[:, aj, ai] = self.big_solve(sig, psi, neu_rows)
        return (U, V, W, PHI, TH), Nn


def half_spectrum(a_signed, ds, nx, ny):
    """signed [n, j', i'] -> boundary SPECTRAL layout [nz, ny, nx//2+1] (zeros outside the retained set)."""
    out = np.zeros((a_signed.shape[0], ny, nx // 2 + 1), dtype=complex)
    for bj, j in enumerate(ds.jp):
        for bi, i in enumerate(ds.ip):
            if i >= 0:
                out[:, j % ny, i] = a_signed[:, bj, bi]
    return out


@pytest.mark.parametrize("shape,nsteps", [((8, 8, 9), 3), ((16, 8, 17), 2)])
def test_full_step_matches_independent_dense_formulation(shape, nsteps):
    nx, ny, nz = shape
    c = I.small_config(nx=nx, ny=ny, nz=nz, band=2)
    st = I.channel_state(c)
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    orc = O.Oracle(g, O.Params(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x))
    orc.set_state("physical", *st)
    ds = DenseStep(nx, ny, nz, c.lx, c.ly, c.re, c.dt, c.pe, c.ch, c.we, c.gradp_x)
    u, v, w, ph = (ds.fwd(f) for f in st)                                    # step i) (L138); retained (kx, ky) only
    state, hist = (u, v, w, ph, ds.lap(w)), None                             # S13: theta = lap(w)
    for n in range(1, nsteps + 1):
        orc.step(1)
        state, hist = ds.step(state, hist)
        ref = orc.get_state("spectral") + [orc.state.theta]
        got = [half_spectrum(a, ds, nx, ny) for a in state]
        vel = math.sqrt(sum(np.linalg.norm(r) ** 2 for r in ref[:3]))
        for name, a, r, den in zip("uvwpt", got, ref, (vel, vel, vel, np.linalg.norm(ref[3]), np.linalg.norm(ref[4]))):
            err = np.linalg.norm(a - r) / den
            assert err < 1e-10, (shape, n, name, err)
        # the Hermitian partner modes (i' < 0) the oracle never stores are consistent in the dense run
        for a in state[:4]:
            assert np.abs(a - np.conj(a[:, ::-1, ::-1])).max() < 1e-10 * max(1.0, np.abs(a).max())
