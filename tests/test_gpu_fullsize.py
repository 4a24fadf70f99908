"""GPU checks at BASELINE.json's full size (config 5c, 1024x512x513), in the launch configuration bench.py times.

The oracle needs about an hour for one dense step at this size, so (tier rule 3):
  * the transform is compared with the oracle on SAMPLED output coefficients, each computed one by one from the
    oracle's own dense matrices (definition sums over the whole 2.7e8-point field);
  * the time step is checked through properties that hold at any size and that a wrong kernel breaks:
    exactly-zero dealiased modes, no-slip (u = v = w = dw/dz = 0 at both walls), the Neumann conditions on phi,
    the algebraic continuity equation i kx u^ + i ky v^ + D w^ = 0 and Hermitian symmetry of the kx = 0 plane.
Element-by-element parity of the same kernels is covered at the smaller sizes in test_gpu_step.py /
test_gpu_transforms.py (several tiles and ragged tails)."""
import numpy as np
import pytest

import psdns_inputs as I
import psdns_oracle as O

pytestmark = pytest.mark.gpu

NX, NY, NZ = I.SCALING_GRIDS["5c"]


def _skip_if_small_gpu(nbytes):
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()          # blocks cached by earlier tests are not "in use"
    free, _ = torch.cuda.mem_get_info()
    if free < nbytes:
        pytest.skip(f"needs {nbytes / 2**30:.0f} GiB of free device memory")


def test_fullsize_roundtrip_and_sampled_forward():
    """psdns_transform_roundtrip at 1024x512x513: identity to 1e-11 (north_star) and 12 forward coefficients
    against the oracle's definition a^(i,j,n) = sum_k Cf[n,k] sum_y Fy[j,y] sum_x Fx[i,x] f[k,y,x]."""
    import torch
    import paper_2406_01322_b200 as P
    _skip_if_small_gpu(90 * 2**30)
    s = P.Solver(NX, NY, NZ, 4 * np.pi, 2 * np.pi, re=3000.0, dt=2e-5, phase_field=0)
    f = I.random_physical_field(NX, NY, NZ, seed=5)
    fd = torch.from_numpy(f).cuda()
    out, mid = s.transform_roundtrip(P.PHYSICAL, fd, want_mid=True)
    err = float(torch.linalg.vector_norm(out - fd) / torch.linalg.vector_norm(fd))
    assert err < 1e-11, err
    rms = float(torch.linalg.vector_norm(mid)) / np.sqrt(mid.numel())
    N = NZ - 1
    Fx = O.dft_matrix(NX, -1) / NX
    Fy = O.dft_matrix(NY, -1) / NY
    Cf = O.cheb_fwd_matrix(N)
    samples = {0: [(0, 0), (3, 1), (NY - 1, N), (200, 300)],
               341: [(0, 2), (170, 341), (NY - 170, 5), (17, N - 1)],
               NX // 2: [(0, 0), (NY // 2, 7), (1, N), (300, 100)]}
    worst = 0.0
    for i, jn in samples.items():
        gx = f @ Fx[i].real + 1j * (f @ Fx[i].imag)   # [nz, ny]: the x sum of the definition, whole field
        for (j, n) in jn:
            ref = Cf[n] @ (gx @ Fy[j])
            got = complex(mid[n, j, i].item())
            worst = max(worst, abs(got - ref) / rms)
    assert worst < 1e-11, worst
    s.close()


def _deriv_coeffs(a):
    """Chebyshev derivative recurrence along axis 0 (torch, on the device): test-side restatement of
    SURVEY 8(c) 'b_N = 0, b_{N-1} = 2N a_N, c_n b_n = b_{n+2} + 2(n+1) a_{n+1}'."""
    import torch
    N = a.shape[0] - 1
    b = torch.zeros_like(a)
    for n in range(N - 1, -1, -1):
        b[n] = 2.0 * (n + 1) * a[n + 1]
        if n + 2 <= N:
            b[n] += b[n + 2]
    b[0] *= 0.5
    return b


def test_fullsize_step_properties():
    """Two psdns_step calls on the bench workload (config 5c random spectra), then invariants of the scheme."""
    import torch
    import paper_2406_01322_b200 as P
    _skip_if_small_gpu(110 * 2**30)
    c = I.scaling_config("5c")
    host = I.random_spectral_state(c.nx, c.ny, c.nz, c.seed, cut=True)
    s = P.Solver(c.nx, c.ny, c.nz, c.lx, c.ly, re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x)
    dev = [torch.from_numpy(a).cuda() for a in host]
    del host
    s.set_state(P.SPECTRAL, *dev)
    del dev
    s.step(2)
    u, v, w, phi = s.get_state(P.SPECTRAL)
    assert s.launch_count() > 0
    for t in (u, v, w, phi):
        assert bool(torch.isfinite(torch.view_as_real(t)).all())
    N = c.nz - 1
    I3, J3 = c.nx // 3, c.ny // 3
    scale = max(float(t.abs().max()) for t in (u, v, w))
    # dealiased (kx, ky) modes are exactly zero (reading R1 / S3)
    for t in (u, v, w, phi):
        assert float(t[:, :, I3 + 1:].abs().max()) == 0.0
        assert float(t[:, J3 + 1: c.ny - J3, :].abs().max()) == 0.0
    n = torch.arange(c.nz, device="cuda", dtype=torch.float64)
    sgn = torch.where(torch.arange(c.nz, device="cuda") % 2 == 0, 1.0, -1.0).to(torch.float64)
    wall = {"+1": torch.ones_like(n), "-1": sgn}

    def functional(t, weights):   # sum_n weights_n t_n for every (ky, kx)
        return torch.einsum("n,njk->jk", weights.to(t.dtype), t)

    for name, sg in wall.items():
        for t in (u, v, w):       # no-slip: T_n(+-1) = (+-1)^n
            assert float(functional(t, sg).abs().max()) < 1e-11 * scale * c.nz, name
        # dw/dz = 0 and dphi/dz = 0: T_n'(+-1) = (+-1)^(n+1) n^2
        assert float(functional(w, sg * n * n).abs().max()) < 1e-10 * scale * c.nz ** 2, name
        assert float(functional(phi, sg * n * n).abs().max()) < 1e-10 * float(phi.abs().max()) * c.nz ** 2, name
    # continuity, algebraically exact after row a11 for every (kx, ky) != (0, 0)
    kx = (2 * np.pi / c.lx) * torch.arange(c.nx // 2 + 1, device="cuda", dtype=torch.float64)
    jj = torch.arange(c.ny, device="cuda")
    ky = (2 * np.pi / c.ly) * torch.where(jj <= c.ny // 2, jj, jj - c.ny).to(torch.float64)
    div = 1j * kx[None, None, :] * u + 1j * ky[None, :, None] * v + _deriv_coeffs(w)
    div[:, 0, 0] = 0.0            # the mean mode carries u-bar, v-bar (reading S12); w^(0,0) = 0
    assert float(w[:, 0, 0].abs().max()) == 0.0
    assert float(div.abs().max()) < 1e-10 * scale * c.nz, float(div.abs().max())
    # Hermitian symmetry of the kx = 0 plane (real fields): a(0, -j) = conj a(0, j)
    for t in (u, v, w, phi):
        p = t[:, :, 0]
        m = torch.conj(torch.roll(torch.flip(p, dims=[1]), shifts=1, dims=1))
        assert float((p - m).abs().max()) < 1e-10 * max(float(p.abs().max()), 1e-300)
    s.close()


def test_fullsize_cross_checks_between_kernel_variants():
    """1024x512x513, two steps of the bench workload's grid, three ways: the product path (fused x kernel, TMA-fed z
    passes), the three-kernel x path through physical-space arrays (psdns_set_option "xfuse" 0) and the register-fed z
    passes ("ztma" 0).  Different kernels, different radix plans and summation orders, same discretisation: the states
    must agree to rounding, field by field, in relative L2 AND in max-abs - garbage from any of the full-size
    instantiations (k_xfusedw<1024>, k_zpass_tma<512>, k_ypass<512>, the > 60 k-column sweeps) cannot pass all three."""
    import gc
    import torch
    import paper_2406_01322_b200 as P
    gc.collect()
    torch.cuda.empty_cache()
    _skip_if_small_gpu(105 * 2**30)
    c = I.scaling_config("5c")
    host = I.random_spectral_state(c.nx, c.ny, c.nz, c.seed, cut=True)
    dev = [torch.from_numpy(a).cuda() for a in host]
    del host
    results = []
    for opts in ({}, {"xfuse": 0}, {"ztma": 0}):
        s = P.Solver(c.nx, c.ny, c.nz, c.lx, c.ly, re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x,
                     unfused_workspace="xfuse" in opts)
        for k, v in opts.items():
            s.set_option(k, v)
        s.set_state(P.SPECTRAL, *dev)
        s.step(2)
        results.append(s.get_state(P.SPECTRAL))
        s.close()
        del s
        torch.cuda.empty_cache()
    ref = results[0]
    vnorm = float(torch.sqrt(sum(torch.linalg.vector_norm(t) ** 2 for t in ref[:3])))
    vmax = max(float(torch.view_as_real(t).abs().max()) for t in ref[:3])
    for other in results[1:]:
        for f, (a, b) in enumerate(zip(other, ref)):
            den_l2 = vnorm if f < 3 else float(torch.linalg.vector_norm(b))
            den_mx = vmax if f < 3 else float(torch.view_as_real(b).abs().max())
            assert float(torch.linalg.vector_norm(a - b)) < 1e-11 * den_l2, f
            assert float(torch.view_as_real(a - b).abs().max()) < 1e-11 * den_mx, f
