"""Helpers shared by the GPU parity tests: run the fp64 oracle and the CUDA path on the same
seeded fp32 inputs and compare element by element.  Test infrastructure only."""
import numpy as np

W19 = np.array([12] + [2] * 6 + [1] * 12) / 36.0
C19 = np.array([[0, 0, 0], [1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1],
                [1, 1, 0], [-1, -1, 0], [1, -1, 0], [-1, 1, 0], [1, 0, 1], [-1, 0, -1], [1, 0, -1],
                [-1, 0, 1], [0, 1, 1], [0, -1, -1], [0, 1, -1], [0, -1, 1]])

POP_TOL = 1e-5      # north_star: max relative error on the populations after 1 step,
                    # measured against the natural scale w_i * rho_0 (G15)
MACRO_TOL = 1e-4    # north_star: max abs error on rho_r, rho_b, u after many steps
DRIFT_TOL = 1e-6    # north_star: relative drift of total mass per component


def make_oracle(lbo, w):
    o = lbo.Oracle(w.nx, w.ny, w.nz, *w.params)
    if w.solid is not None:
        o.set_geometry(w.solid)
    o.set_body_force(*w.g)
    o.set_nc_cutoff(w.phi_c)
    from paper_2005_12764_b200 import workloads
    workloads.configure_walls(o, w)            # wall groups, particles
    o.init(w.rho_r, w.rho_b, w.u)
    return o


def make_gpu(lbmod, w, storage="ab"):
    sim = lbmod.from_workload(w, storage=storage)
    sim.init(np.ascontiguousarray(w.rho_r), None if w.rho_b is None else np.ascontiguousarray(w.rho_b),
             np.ascontiguousarray(w.u))
    return sim


def pop_error(sim, o, two=True):
    """max over components, directions and sites of |f_gpu - f_oracle| / (w_i rho_0), as an
    array [nz, ny, nx] of per-site maxima."""
    err = None
    for k in range(2 if two else 1):
        fg = sim.get_populations(k).astype(np.float64)
        fo = o.get_populations(k)
        e = (np.abs(fg - fo) / W19[:, None, None, None]).max(0)
        err = e if err is None else np.maximum(err, e)
    return err


def dilate(mask, n=1):
    """Grow a boolean site mask by n D3Q19 neighbour shells (periodic)."""
    out = mask.copy()
    for _ in range(n):
        cur = out.copy()
        for c in C19[1:]:
            out |= np.roll(cur, shift=(c[2], c[1], c[0]), axis=(0, 1, 2))
    return out


def macro_errors(sim, o):
    rr, rb, u = sim.get_macros()
    orr, orb, ou = o.get_macros()
    out = dict(rho_r=np.abs(rr - orr).max(), u=np.abs(u - ou).max())
    if rb is not None and orb is not None:
        out["rho_b"] = np.abs(rb - orb).max()
    return out, (rr, rb, u), (orr, orb, ou)


def masses(rr, rb):
    return (float(np.sum(rr, dtype=np.float64)), float(np.sum(rb, dtype=np.float64)) if rb is not None else 0.0)
