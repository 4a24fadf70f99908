"""Writes tests/golden/cfg<k>_step<n>_samples.txt: sampled spectral coefficients of the state after n oracle steps
of BASELINE.json config k, for the full-grid GPU parity tests of configs 3 and 4 (the dense oracle needs minutes
per step on these grids, too long for the default test run).

    python tests/golden/make_step_samples.py 3 1        # config 3 (256x256x257), 1 step
    python tests/golden/make_step_samples.py 4 1        # config 4 (512x256x257, visc_ratio 0.1), 1 step

Calls only oracle/ and the seeded input generators (psdns_inputs); nothing here comes from the CUDA path.
Line format: field i j n re im   (field 0..3 = u v w phi; boundary SPECTRAL indices), preceded by the l2 norms of
the four full spectra (rows 'norm field value')."""
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

NSAMPLES = 160


def sample_indices(c, rng):
    """Seeded (i, j, n) triples inside the retained set, plus fixed low modes and the (0,0) column."""
    N = c.nz - 1
    I3, J3, K3 = c.nx // 3, c.ny // 3, (2 * N) // 3
    out = [(0, 0, 0), (0, 0, 2), (1, 0, 1), (0, 1, 3), (1, c.ny - 1, 2), (I3, J3, 0), (I3, c.ny - J3, 5), (2, 3, K3), (5, 7, N)]
    while len(out) < NSAMPLES:
        i = int(rng.integers(0, min(I3, 24) + 1))
        jp = int(rng.integers(-min(J3, 24), min(J3, 24) + 1))
        n = int(rng.integers(0, min(N, 96) + 1))
        out.append((i, jp % c.ny, n))
    return out


def main():
    k, nsteps = int(sys.argv[1]), int(sys.argv[2])
    c = I.CONFIGS[k]
    t0 = time.time()
    st = I.channel_state(c)
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    orc = O.Oracle(g, O.Params(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x, visc_ratio=c.visc_ratio,
                               phase_field=c.phase_field))
    orc.set_state("physical", *st)
    orc.step(nsteps)
    spec = orc.get_state("spectral")
    idx = sample_indices(c, np.random.default_rng(9000 + k))
    path = os.path.join(HERE, f"cfg{k}_step{nsteps}_samples.txt")
    with open(path, "w") as f:
        f.write(f"# oracle/psdns_oracle.py, BASELINE.json config {k} ({c.nx}x{c.ny}x{c.nz}), state after {nsteps} step(s)\n")
        f.write("# written by tests/golden/make_step_samples.py (calls only oracle/ and psdns_inputs)\n")
        for fi, a in enumerate(spec):
            f.write(f"norm {fi} {float(np.linalg.norm(a.ravel()))!r}\n")
        for fi, a in enumerate(spec):
            for (i, j, n) in idx:
                v = complex(a[n, j, i])
                f.write(f"{fi} {i} {j} {n} {v.real!r} {v.imag!r}\n")
    print(f"wrote {path} in {time.time() - t0:.0f} s")


if __name__ == "__main__":
    main()
