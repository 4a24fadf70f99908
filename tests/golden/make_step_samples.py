"""Writes tests/golden/<tag>_step<n>_samples.txt: the ORACLE's state after n steps of a BASELINE.json config on its
full grid, reduced to what a parity test can check in seconds (the dense oracle needs 20 s .. 10 min per step on
these grids, too long for the default test run):

  * `norm f v`, `maxabs f v`   l2 norm and max |Re|,|Im| of every full spectrum (f = 0..3 = u v w phi);
  * `proj p f v`               NPROJ seeded random projections sum_e (r_e Re a_e + q_e Im a_e) over the WHOLE boundary
                               spectrum (first-order sensitive to an error anywhere; weights: projection_weights());
  * `i j n  u v w phi`         NSAMPLES coefficients (re im of each field) drawn UNIFORMLY over the whole retained
                               (kx, ky) set and all Chebyshev modes: every kx tile of 8, both signs of ky, n up to N
                               (the state is not truncated in z), plus fixed corner cases.

    python tests/golden/make_step_samples.py 3 1 3        # config 3 (256x256x257): fixtures after 1 and after 3 steps
    python tests/golden/make_step_samples.py 5a 1 3 25    # config 5 random spectra on 256x128x129
    python tests/golden/make_step_samples.py 2 100

Calls only oracle/ and the seeded input generators (psdns_inputs); nothing here comes from the CUDA path."""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for p in (ROOT, os.path.join(ROOT, "oracle")):
    if p not in sys.path:
        sys.path.insert(0, p)

import psdns_inputs as I  # noqa: E402
import psdns_oracle as O  # noqa: E402

NSAMPLES = 2048
NPROJ = 2


def config_of(tag: str):
    """tag '1'..'4' -> BASELINE.json configs 1-4 (channel states, PHYSICAL); '5a' / '5b' / '5c' -> config 5 (random
    spectra, SPECTRAL).  Returns (Config, space, fields)."""
    if tag in I.SCALING_GRIDS:
        c = I.scaling_config(tag)
        return c, "spectral", list(I.random_spectral_state(c.nx, c.ny, c.nz, c.seed, cut=True))
    c = I.CONFIGS[int(tag)]
    return c, "physical", list(I.channel_state(c))


def sample_indices(c, seed: int):
    """Seeded (i, j, n) triples, uniform over i <= nx//3, |j'| <= ny//3, n <= N, after a fixed list of corners."""
    rng = np.random.default_rng(seed)
    N = c.nz - 1
    I3, J3, K3 = c.nx // 3, c.ny // 3, (2 * N) // 3
    out = [(0, 0, 0), (0, 0, 2), (0, 0, N), (1, 0, 1), (0, 1, 3), (1, c.ny - 1, 2), (I3, J3, 0), (I3, c.ny - J3, 5),
           (2, 3, K3), (5, 7, N), (I3, J3, N), (I3, c.ny - J3, N - 1), (0, J3, K3 + 1), (I3 - 1, 0, N)]
    while len(out) < NSAMPLES:
        out.append((int(rng.integers(0, I3 + 1)), int(rng.integers(-J3, J3 + 1)) % c.ny, int(rng.integers(0, N + 1))))
    return out


def projection_weights(c, p: int):
    """Weights of projection p: two standard-normal arrays [nz, ny, nx//2+1] (for Re and Im), seed 77000 + p.
    The GPU test regenerates them with the same call."""
    rng = np.random.default_rng(77000 + p)
    shape = (c.nz, c.ny, c.nx // 2 + 1)
    return rng.standard_normal(shape), rng.standard_normal(shape)


def write_fixture(tag, c, nsteps, spec):
    idx = sample_indices(c, 9000 + sum(ord(ch) for ch in tag))
    path = os.path.join(HERE, f"cfg{tag}_step{nsteps}_samples.txt")
    with open(path, "w") as f:
        f.write(f"# oracle/psdns_oracle.py, BASELINE.json config {tag} ({c.nx}x{c.ny}x{c.nz}), state after {nsteps} step(s)\n")
        f.write("# written by tests/golden/make_step_samples.py (calls only oracle/ and psdns_inputs); format: see that file\n")
        for fi, a in enumerate(spec):
            f.write(f"norm {fi} {float(np.linalg.norm(a.ravel()))!r}\n")
            f.write(f"maxabs {fi} {float(max(np.abs(a.real).max(), np.abs(a.imag).max()))!r}\n")
        for p in range(NPROJ):
            r, q = projection_weights(c, p)
            for fi, a in enumerate(spec):
                f.write(f"proj {p} {fi} {float(np.sum(r * a.real) + np.sum(q * a.imag))!r}\n")
        for (i, j, n) in idx:
            vals = " ".join(f"{complex(a[n, j, i]).real!r} {complex(a[n, j, i]).imag!r}" for a in spec)
            f.write(f"{i} {j} {n} {vals}\n")
    return path


def main():
    tag = sys.argv[1]
    steps = sorted(int(s) for s in sys.argv[2:])
    t0 = time.time()
    c, space, st = config_of(tag)
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    orc = O.Oracle(g, O.Params(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x, visc_ratio=c.visc_ratio,
                               phase_field=c.phase_field))
    orc.set_state(space, *st)
    for n in steps:
        while orc.state.nstep < n:
            orc.step(1)
            print(f"cfg{tag}: step {orc.state.nstep} done at {time.time() - t0:.0f} s", flush=True)
        path = write_fixture(tag, c, n, orc.get_state("spectral"))
        print(f"wrote {path} at {time.time() - t0:.0f} s", flush=True)


if __name__ == "__main__":
    main()
