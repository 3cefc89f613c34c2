"""GPU parity of the second model (the paper's section 3.1 as printed: Shan-Chen force, Eq. 10,
through the exact-difference source, Eq. 9, in Eq. 5-6) against the fp64 oracle."""
import numpy as np
import pytest

import parity_util as pu
from paper_2005_12764_b200 import workloads as W
from test_gpu_edges import _random_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lbmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2005_12764_b200 import lb
    return lb


def _pair(lbmod, lbo, w, G_C, storage="ab"):
    o = lbo.Oracle(w.nx, w.ny, w.nz, *w.params)
    o.set_model("sc", G_C)
    if w.solid is not None:
        o.set_geometry(w.solid)
    o.set_body_force(*w.g)
    o.init(w.rho_r, w.rho_b, w.u)
    sim = lbmod.LB(w.nx, w.ny, w.nz, w.tau_r, w.tau_b, w.A, w.beta, w.A_nc)
    sim.set_storage(storage)
    sim.set_model("sc", G_C)
    if w.solid is not None:
        sim.set_geometry(np.ascontiguousarray(w.solid, dtype=np.uint8))
    sim.set_body_force(*w.g)
    sim.init(np.ascontiguousarray(w.rho_r), np.ascontiguousarray(w.rho_b), np.ascontiguousarray(w.u))
    return o, sim


@pytest.mark.parametrize("shape", [(4, 4, 4), (36, 13, 7), (68, 9, 21)])
@pytest.mark.parametrize("walls", [False, True])
@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_sc_parity_ragged(lbmod, lbo, shape, walls, storage):
    """Populations after 1, 2 and 5 steps, phi and macroscopic fields: two taus, body force,
    walls, boxes that are not multiples of the tile."""
    w = _random_workload(*shape, seed=sum(shape) + 3 * walls, walls=walls)
    fluid = np.ones(w.shape, bool) if w.solid is None else (w.solid == 0)
    o, sim = _pair(lbmod, lbo, w, 1.6, storage)
    assert pu.pop_error(sim, o).max() < pu.POP_TOL
    done = 0
    for n in (1, 2, 5):
        o.step(n - done); sim.step(n - done)
        done = n
        e = pu.pop_error(sim, o)
        assert e.max() < pu.POP_TOL, (n, e.max())
    assert np.abs(sim.get_phi() - o.get_fields()["phi"])[fluid].max() < 2e-6
    errs, (rr, rb, u), _ = pu.macro_errors(sim, o)
    assert max(errs.values()) < 1e-5, errs
    if w.solid is not None:
        solid = w.solid != 0
        assert rr[solid].max() == 0 and np.abs(u[:, solid]).max() == 0


def test_sc_demixing_run(lbmod, lbo):
    """64^3 spinodal noise with G_C = 3 > 2/rho_0: the mixture separates; masses are conserved,
    momentum stays zero, and after 100 steps the fields still agree with the oracle within the
    divergence of an oracle run whose input was perturbed by 1e-7 (the state is unstable)."""
    w = W.get("c3-mini")
    o, sim = _pair(lbmod, lbo, w, 3.0)
    o2 = lbo.Oracle(w.nx, w.ny, w.nz, *w.params)
    o2.set_model("sc", 3.0)
    pert = 1e-7 * np.random.default_rng(5).uniform(-1, 1, w.shape)
    o2.init(w.rho_r.astype(np.float64) + pert, w.rho_b.astype(np.float64) - pert, w.u)
    o.step(1); sim.step(1); o2.step(1)
    assert pu.pop_error(sim, o).max() < pu.POP_TOL
    o.step(99); sim.step(99); o2.step(99)
    errs, (rr, rb, u), (orr, orb, ou) = pu.macro_errors(sim, o)
    c_rr, c_rb, c_u = o2.get_macros()
    control = max(np.abs(c_rr - orr).max(), np.abs(c_rb - orb).max(), np.abs(c_u - ou).max())
    assert max(errs.values()) < max(3 * control, pu.MACRO_TOL), (errs, control)
    m0, m1 = pu.masses(w.rho_r, w.rho_b), pu.masses(rr, rb)
    assert abs(m1[0] - m0[0]) / m0[0] < pu.DRIFT_TOL and abs(m1[1] - m0[1]) / m0[1] < pu.DRIFT_TOL
    mom = np.abs([(u[a].astype(np.float64) * (rr + rb)).sum() for a in range(3)]).max() / w.sites
    assert mom < 1e-5
    sim.step(900)
    phi = sim.get_phi()
    assert np.isfinite(phi).all() and np.std(phi) > 5 * np.std((w.rho_r - w.rho_b) / (w.rho_r + w.rho_b))


def test_sc_AA_equals_AB_bitwise(lbmod, lbo):
    w = _random_workload(36, 13, 10, seed=41, walls=True)
    _, a = _pair(lbmod, lbo, w, 1.6, "ab")
    _, b = _pair(lbmod, lbo, w, 1.6, "aa")
    for n in (3, 1):
        a.step(n); b.step(n)
        for k in (0, 1):
            assert np.array_equal(a.get_populations(k), b.get_populations(k))


def test_sc_errors(lbmod):
    lb = lbmod
    sim = lb.LB(8, 8, 8)
    sim.set_model("sc", 1.0)
    with pytest.raises(lb.LBError) as ei:
        sim.init(np.ones((8, 8, 8), np.float32), None, np.zeros((3, 8, 8, 8), np.float32))
    assert ei.value.code == lb.LB_EINVAL
    sim.init(np.ones((8, 8, 8), np.float32), np.ones((8, 8, 8), np.float32), np.zeros((3, 8, 8, 8), np.float32))
    with pytest.raises(lb.LBError) as ei:
        sim.set_model("cg")
    assert ei.value.code == lb.LB_ESTATE


def test_sc_full_size_sampled_blocks_and_conservation(lbmod, lbo):
    """The configuration bench.py --model sc times (C3 at 256^3, G_C = 3): one step checked on
    sampled 28^3 blocks against the oracle run on a cut-out of the input, then 200 more steps:
    finite, masses conserved, zero net momentum, the mixture has started to separate."""
    w = W.get("c3")
    _, sim = None, lbmod.LB(w.nx, w.ny, w.nz, *w.params)
    sim.set_model("sc", 3.0)
    sim.init(np.ascontiguousarray(w.rho_r), np.ascontiguousarray(w.rho_b), np.ascontiguousarray(w.u))
    sim.step(1)
    f = [sim.get_populations(k) for k in (0, 1)]
    rng = np.random.default_rng(19)
    centres = [(0, 0, 0), (w.nx - 1, w.ny // 2, w.nz - 1)] + \
        [tuple(int(v) for v in rng.integers(0, [w.nx, w.ny, w.nz])) for _ in range(4)]
    half, margin = 14, 3
    n = 2 * half
    worst = 0.0
    for (cx, cy, cz) in centres:
        ix = np.arange(cx - half, cx + half) % w.nx
        iy = np.arange(cy - half, cy + half) % w.ny
        iz = np.arange(cz - half, cz + half) % w.nz
        sel = np.ix_(iz, iy, ix)
        o = lbo.Oracle(n, n, n, *w.params)
        o.set_model("sc", 3.0)
        o.init(w.rho_r[sel], w.rho_b[sel], w.u[(slice(None),) + sel])
        o.step(1)
        inner = np.zeros((n, n, n), bool)
        inner[margin:-margin, margin:-margin, margin:-margin] = True
        for k in (0, 1):
            e = np.abs(f[k][(slice(None),) + sel].astype(np.float64) - o.get_populations(k)) / pu.W19[:, None, None, None]
            worst = max(worst, e[:, inner].max())
    assert worst < pu.POP_TOL, worst
    del f
    sim.step(200)
    rr, rb, u = sim.get_macros()
    assert np.isfinite(u).all()
    m0, m1 = pu.masses(w.rho_r, w.rho_b), pu.masses(rr, rb)
    assert abs(m1[0] - m0[0]) / m0[0] < pu.DRIFT_TOL and abs(m1[1] - m0[1]) / m0[1] < pu.DRIFT_TOL
    mom = np.abs([(u[a].astype(np.float64) * (rr + rb)).sum() for a in range(3)]).max() / w.sites
    assert mom < 1e-5
    assert np.std((rr - rb) / (rr + rb)) > 3 * np.std((w.rho_r - w.rho_b) / (w.rho_r + w.rho_b))
