"""Pins for the oracle's transforms, derivative and dealiasing (not gpu).
Each test checks the oracle against something other than itself: textbook Chebyshev
identities (tests/golden), numpy/scipy library transforms, the length-2N DFT of the even
extension, brute-force sums and convolutions."""
import os

import numpy as np
import pytest
import scipy.fft

import psdns_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden", "chebyshev_identities.txt")


def _golden():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        name, poly, cheb = [s.strip() for s in line.split(";")]
        out[name] = (np.array(poly.split(), float), np.array(cheb.split(), float))
    return out


@pytest.mark.parametrize("N", [8, 16, 33])
def test_chebyshev_of_Tm_is_delta(N):
    z = O.cheb_nodes(N)
    Cf = O.cheb_fwd_matrix(N)
    for m in range(N + 1):
        a = Cf @ np.cos(m * np.arccos(z))
        e = np.zeros(N + 1); e[m] = 1.0
        assert np.abs(a - e).max() < 1e-13


def test_golden_polynomials():
    N = 12
    z = O.cheb_nodes(N)
    Cf, Cb = O.cheb_fwd_matrix(N), O.cheb_bwd_matrix(N)
    gold = _golden()
    for name, (poly, cheb) in gold.items():
        f = np.polyval(poly[::-1], z)
        a = Cf @ f
        ref = np.zeros(N + 1); ref[: len(cheb)] = cheb
        assert np.abs(a - ref).max() < 1e-14, name
        assert np.abs(Cb @ ref - f).max() < 1e-14, name
    # derivative: D(T3) = 3 T0 + 6 T2  (golden 'dT3' is d/dz of 4z^3-3z)
    D = O.cheb_deriv_matrix(N)
    e3 = np.zeros(N + 1); e3[3] = 1
    ref = np.zeros(N + 1); ref[:3] = gold["dT3"][1]
    assert np.abs(D @ e3 - ref).max() < 1e-14


def test_derivative_matches_polynomial_derivative():
    N = 20
    rng = np.random.default_rng(0)
    z = O.cheb_nodes(N)
    p = np.polynomial.Polynomial(rng.standard_normal(15))
    a = O.cheb_fwd_matrix(N) @ p(z)
    da = O.cheb_deriv_matrix(N) @ a
    assert np.abs(O.cheb_bwd_matrix(N) @ da - p.deriv()(z)).max() < 1e-10
    # equals numpy's own Chebyshev-series derivative
    assert np.abs(da[:-1] - np.polynomial.chebyshev.chebder(a)).max() < 1e-10


@pytest.mark.parametrize("N", [8, 32])
def test_dct_equals_dft_of_even_extension(N):
    """Chebyshev transform of an N-point signal = DFT of its 2N even extension."""
    rng = np.random.default_rng(1)
    f = rng.standard_normal(N + 1)
    ext = np.concatenate([f, f[-2:0:-1]])
    assert ext.size == 2 * N
    F = np.fft.fft(ext)
    assert np.abs(F.imag).max() < 1e-12
    c = np.ones(N + 1); c[0] = c[N] = 2
    a_ref = F.real[: N + 1] / (N * c)
    assert np.abs(O.cheb_fwd_matrix(N) @ f - a_ref).max() < 1e-14
    # and against scipy's DCT-I
    a_sc = scipy.fft.dct(f, type=1) / (N * c)
    assert np.abs(O.cheb_fwd_matrix(N) @ f - a_sc).max() < 1e-14
    # backward = DCT-I too ("the backward transform of a DCT-I is a DCT-I")
    a = rng.standard_normal(N + 1)
    h = a.copy(); h[1:N] *= 0.5
    assert np.abs(O.cheb_bwd_matrix(N) @ a - scipy.fft.dct(h, type=1)).max() < 1e-12


def test_forward_matches_library_fft():
    g = O.Grid(16, 8, 9)
    rng = np.random.default_rng(2)
    f = rng.standard_normal((g.nz, g.ny, g.nx))
    a = O.forward_transform(f, g)
    ref = np.fft.rfft2(f, axes=(1, 2)) / (g.nx * g.ny)
    c = np.ones(g.nz); c[0] = c[-1] = 2
    ref = scipy.fft.dct(ref.real, type=1, axis=0) + 1j * scipy.fft.dct(ref.imag, type=1, axis=0)
    ref = ref / (g.N * c[:, None, None])
    assert O.rel_l2(a, ref) < 1e-14


def test_roundtrip_identity():
    g = O.Grid(16, 12, 11)
    rng = np.random.default_rng(3)
    f = rng.standard_normal((g.nz, g.ny, g.nx))
    assert O.rel_l2(O.backward_transform(O.forward_transform(f, g), g), f) < 1e-13
    a = O.forward_transform(f, g)          # Hermitian-consistent by construction
    assert O.rel_l2(O.forward_transform(O.backward_transform(a, g), g), a) < 1e-13


def test_plane_wave_single_coefficient_and_shift():
    g = O.Grid(16, 8, 9, lx=4 * np.pi, ly=2 * np.pi)
    x = g.lx / g.nx * np.arange(g.nx)[None, None, :]
    y = g.ly / g.ny * np.arange(g.ny)[None, :, None]
    z = O.cheb_nodes(g.N)[:, None, None]
    kx, ky = O.wavenumbers(g)
    i, j, n = 3, 6, 2        # j = 6 -> j' = -2
    f = np.cos(kx[i] * x + ky[j] * y + 0.3) * np.cos(n * np.arccos(z))
    a = O.forward_transform(f, g)
    ref = np.zeros_like(a)
    ref[n, j, i] = 0.5 * np.exp(0.3j)
    assert np.abs(a - ref).max() < 1e-14
    # shift theorem: f(x - d) -> a * exp(-i kx d)
    d = 2 * g.lx / g.nx
    f2 = np.cos(kx[i] * (x - d) + ky[j] * y + 0.3) * np.cos(n * np.arccos(z))
    assert np.abs(O.forward_transform(f2, g)[n, j, i] - ref[n, j, i] * np.exp(-1j * kx[i] * d)) < 1e-14


def test_parseval_xy():
    g = O.Grid(8, 8, 5)
    rng = np.random.default_rng(4)
    f = rng.standard_normal((g.nz, g.ny, g.nx))
    # x,y-only check at every z: mean(f^2) = sum over full spectrum |f^|^2
    Fx = O.dft_matrix(g.nx, -1)[: g.nkx] / g.nx
    Fy = O.dft_matrix(g.ny, -1) / g.ny
    a = np.einsum("jy,kyi->kji", Fy, f @ Fx.T)
    wts = np.full(g.nkx, 2.0); wts[0] = wts[-1] = 1.0
    lhs = (f ** 2).mean(axis=(1, 2))
    rhs = (np.abs(a) ** 2 * wts[None, None, :]).sum(axis=(1, 2))
    assert np.abs(lhs - rhs).max() < 1e-13


def test_backward_is_brute_force_sum():
    g = O.Grid(8, 6, 5)
    rng = np.random.default_rng(5)
    a = O.forward_transform(rng.standard_normal((g.nz, g.ny, g.nx)), g)
    kx, ky = O.wavenumbers(g)
    f = O.backward_transform(a, g)
    z = O.cheb_nodes(g.N)
    for (k, yy, xx) in [(0, 0, 0), (2, 3, 5), (4, 5, 7), (1, 2, 1)]:
        x = g.lx / g.nx * xx
        y = g.ly / g.ny * yy
        s = 0.0
        for n in range(g.nz):
            Tn = np.cos(n * np.arccos(z[k]))
            for j in range(g.ny):
                for i in range(g.nkx):
                    wgt = 1.0 if (i == 0 or i == g.nx // 2) else 2.0
                    s += wgt * (a[n, j, i] * Tn * np.exp(1j * (kx[i] * x + ky[j] * y))).real
        assert abs(s - f[k, yy, xx]) < 1e-12


def test_truncation_mask_counts():
    g = O.Grid(32, 32, 33)
    I, J, K = O.retained_counts(g)
    assert (I, J, K) == (10, 10, 21)
    m = O.truncation_mask(g)
    assert m.sum() == (I + 1) * (2 * J + 1) * (K + 1) == 11 * 21 * 22
    g = O.Grid(1024, 512, 513)
    I, J, K = O.retained_counts(g)
    assert (I + 1, 2 * J + 1, K + 1) == (342, 341, 342)


def test_dealiased_product_is_exact_truncated_convolution():
    """S3: with the 2/3 cut-offs a quadratic product evaluated pseudo-spectrally equals the
    exact convolution of the truncated spectra, truncated (brute force on 8x8x9)."""
    g = O.Grid(8, 8, 9)
    rng = np.random.default_rng(6)
    P = O.truncation_mask(g)
    a = np.where(P, O.forward_transform(rng.standard_normal((g.nz, g.ny, g.nx)), g), 0)
    b = np.where(P, O.forward_transform(rng.standard_normal((g.nz, g.ny, g.nx)), g), 0)
    pa, pb = O.backward_transform(a, g), O.backward_transform(b, g)
    c = np.where(P, O.forward_transform(pa * pb, g), 0)

    # exact convolution: expand to full signed (i, j') Fourier spectra and Chebyshev series
    I, J, K = O.retained_counts(g)
    def full(s):
        d = {}
        for n in range(K + 1):
            for jp in range(-J, J + 1):
                for i in range(-I, I + 1):
                    v = s[n, jp % g.ny, abs(i)]
                    if i < 0:
                        v = np.conj(s[n, (-jp) % g.ny, -i])
                    if i == 0:
                        v = 0.5 * (s[n, jp % g.ny, 0] + np.conj(s[n, (-jp) % g.ny, 0]))
                    d[(n, jp, i)] = v
        return d
    A, B = full(a), full(b)
    ref = np.zeros_like(c)
    for (n1, j1, i1), va in A.items():
        if va == 0:
            continue
        for (n2, j2, i2), vb in B.items():
            i, jp = i1 + i2, j1 + j2
            if i < 0 or i > I or abs(jp) > J:
                continue
            # T_n1 T_n2 = (T_{n1+n2} + T_{|n1-n2|}) / 2
            for n in (n1 + n2, abs(n1 - n2)):
                if n <= K:
                    ref[n, jp % g.ny, i] += 0.5 * va * vb
    # i = 0 plane of c is the Hermitian-symmetrised one as well
    assert np.abs(c - ref).max() < 1e-13
