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


def solver_from_config(c, unfused_workspace=False, **over):
    import paper_2406_01322_b200 as P
    kw = dict(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x, visc_ratio=c.visc_ratio,
              phase_field=c.phase_field)
    kw.update(over)
    return P.Solver(c.nx, c.ny, c.nz, c.lx, c.ly, unfused_workspace=unfused_workspace, **kw)


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


# Floor of the per-column check below, as a fraction of the largest column norm of the group: the non-linear terms
# spread rounding errors of size eps * max|field| into every wavenumber, so a column whose own norm is far below the
# largest one cannot be held to a relative error of 1e-9 of ITSELF.
COLUMN_FLOOR = 1e-3


def detailed_errors(got, ref):
    """Sharper companions of the relative-L2 norm (which the mean flow dominates).  For the velocity group (u, v, w
    jointly, reading S17) and for phi, on SPECTRAL arrays [nz, ny, nkx]:
      max-abs error / max-abs of the reference group, and
      the worst (kx, ky) column: ||err column||_2 / max(||ref column||_2, COLUMN_FLOOR * largest ref column norm).
    Returns ((vel_maxabs, vel_column), (phi_maxabs, phi_column))."""
    def group(gs, rs):
        err2 = sum(np.abs(a - r) ** 2 for a, r in zip(gs, rs))
        ref2 = sum(np.abs(r) ** 2 for r in rs)
        maxabs = float(np.sqrt(err2.max()) / np.sqrt(ref2.max()))
        ecol = np.sqrt(err2.sum(axis=0))
        rcol = np.sqrt(ref2.sum(axis=0))
        col = float((ecol / np.maximum(rcol, COLUMN_FLOOR * rcol.max())).max())
        return maxabs, col
    vel = group(got[:3], ref[:3])
    phi = (0.0, 0.0)
    if len(ref) > 3 and ref[3] is not None:
        phi = group(got[3:4], ref[3:4])
    return vel, phi


def assert_parity(got, ref, tol, tag=""):
    """relative L2 (north_star tolerance) AND max-abs AND worst-column error, all <= tol."""
    ev, ep = field_errors(got, ref)
    (vm, vc), (pm, pc) = detailed_errors(got, ref)
    assert ev < tol and ep < tol, (tag, "rel-l2", ev, ep)
    assert vm < tol and pm < tol, (tag, "max-abs", vm, pm)
    assert vc < tol and pc < tol, (tag, "worst column", vc, pc)
    return dict(l2=(ev, ep), maxabs=(vm, pm), column=(vc, pc))
