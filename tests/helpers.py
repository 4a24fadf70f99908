"""Shared helpers for the parity tests: build the oracle and the CUDA solver from one Config."""
import numpy as np

import psdns_inputs as I
import psdns_oracle as O


def oracle_from_config(c, **over):
    g = O.Grid(c.nx, c.ny, c.nz, c.lx, c.ly)
    kw = dict(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x, visc_ratio=c.visc_ratio,
              phase_field=c.phase_field)
    kw.update(over)
    return O.Oracle(g, O.Params(**kw)), g


def solver_from_config(c, **over):
    import paper_2406_01322_b200 as P
    kw = dict(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x, visc_ratio=c.visc_ratio,
              phase_field=c.phase_field)
    kw.update(over)
    return P.Solver(c.nx, c.ny, c.nz, c.lx, c.ly, **kw)


def to_dev(a):
    import torch
    if a is None:
        return None
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def to_np(t):
    return t.detach().cpu().numpy()


def field_errors(got, ref):
    """Reading S17: velocity error normalised by the joint norm of (u, v, w); phi by its own."""
    vel_den = np.sqrt(sum(np.linalg.norm(r.ravel()) ** 2 for r in ref[:3]))
    vel_err = np.sqrt(sum(np.linalg.norm((a - r).ravel()) ** 2 for a, r in zip(got[:3], ref[:3]))) / vel_den
    phi_err = 0.0
    if len(ref) > 3 and ref[3] is not None:
        phi_err = np.linalg.norm((got[3] - ref[3]).ravel()) / np.linalg.norm(ref[3].ravel())
    return float(vel_err), float(phi_err)
