"""Rigid spherical particles on the CUDA path (NEXT-4; the paper's section 6, Eq. 15)
against the fp64 oracle: populations, node map and particle states step by step while the particles
cross the box, spin, push each other and cross a red / blue interface; on the CUDA path itself:
momentum of fluid + particles, and the drag on a held sphere against Stokes' law."""
import numpy as np
import pytest

import parity_util as pu
from test_oracle_colloids import particle, C

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lbmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2005_12764_b200 import lb
    return lb


def _pair(lbmod, lbo, shape, params, parts, rr, rb, u=None, g=(0, 0, 0), opts=None, solid=None, forces=None):
    nx, ny, nz = shape
    u = np.zeros((3, nz, ny, nx), np.float32) if u is None else u
    o = lbo.Oracle(nx, ny, nz, *params)
    sim = lbmod.LB(nx, ny, nz, *params)
    for obj in (o, sim):
        if solid is not None:
            obj.set_geometry(solid)
        obj.set_body_force(*g)
        obj.set_particles(parts)
        if opts:
            obj.set_particle_options(**opts)
        for i, (F, T) in (forces or {}).items():
            obj.set_particle_force(i, F=F, T=T)
    rr32 = np.ascontiguousarray(rr, np.float32)
    rb32 = None if rb is None else np.ascontiguousarray(rb, np.float32)
    o.init(rr32, rb32, u)
    sim.init(rr32, rb32, u)
    return o, sim


def _compare(o, sim, two, tol_state=2e-6):
    sol_o, pid_o = o.get_node_map()
    fluid = sol_o == 0
    # the node map is the oracle's: the CUDA path returns zeros exactly on the solid nodes
    rr, rb, u = sim.get_macros()
    orr, orb, ou = o.get_macros()
    assert np.array_equal(rr == 0, ~fluid), "node maps differ"
    e = 0.0
    for k in range(2 if two else 1):
        d = np.abs(sim.get_populations(k).astype(np.float64) - o.get_populations(k)) / pu.W19[:, None, None, None]
        e = max(e, d[:, fluid].max())
    st, fo = sim.get_particles()
    so, fo_o = o.get_particles()
    return e, np.abs(st - so).max(), np.abs(fo - fo_o).max(), max(np.abs(rr - orr).max(), np.abs(u - ou).max())


@pytest.mark.parametrize("two", [True, False])
def test_particles_parity_with_oracle_step_by_step(lbmod, lbo, two):
    """Two particles (different radii and densities) fly through a 40 x 24 x 20 box, spin, repel each
    other (pair force and lubrication on) and, in the two-component case, cross a flat interface with
    the near-contact force on.  After every one of 30 steps: identical node map, populations within
    1e-5 (G15 norm), particle states (r, u, w, q) within 2e-6, forces within 1e-5."""
    nx, ny, nz = 40, 24, 20
    parts = [particle((9.3, 12.1, 9.7), u=(0.04, -0.01, 0.015), w=(0.003, 0.001, -0.002), R=4.5, density=2.0),
             particle((22.2, 11.6, 10.4), u=(-0.05, 0.004, 0.01), w=(0.0, -0.004, 0.001), R=3.6, density=4.0)]
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    phi = np.tanh((x - 16.3) / 2.0) * np.tanh((30.2 - np.abs(x - 16.3)) / 2.0)
    rr, rb = ((1 + phi) / 2, (1 - phi) / 2) if two else (np.ones((nz, ny, nx)), None)
    params = (0.9, 1.1, 0.01, 0.7, 0.02) if two else (0.8, 0.8, 0.0, 0.0, 0.0)
    o, sim = _pair(lbmod, lbo, (nx, ny, nz), params, parts, rr, rb, g=(1e-5, 0, -2e-5),
                   opts=dict(mobile=True, K=0.02, h_c=2.5, lubrication=True))
    e, ds, df, dm = _compare(o, sim, two)
    assert e < pu.POP_TOL and ds == 0.0
    changed = 0
    prev = o.get_node_map()[0]
    fluid = np.ones((nz, ny, nx), bool)
    risky = np.zeros((nz, ny, nx), bool)
    for n in range(1, 31):
        if two:
            risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & (prev == 0), 1)
        o.step(1); sim.step(1)
        cur = o.get_node_map()[0]
        changed += int((cur != prev).sum())
        prev = cur
        if n in (1, 2, 3, 5, 10, 20, 30):
            sol_o = cur
            rr_g, rb_g, u_g = sim.get_macros()
            assert np.array_equal(rr_g == 0, sol_o != 0), (n, "node maps differ")
            if n <= 3 or not two:
                # populations; with the near-contact force the G12 set is carried along and covers this
                # small box after a few steps, so the later steps are held by the fields below
                ok = (sol_o == 0) & ~risky
                assert ok.sum() > 0.3 * ok.size
                worst = 0.0
                for k in range(2 if two else 1):
                    d = np.abs(sim.get_populations(k).astype(np.float64) - o.get_populations(k)) / pu.W19[:, None, None, None]
                    worst = max(worst, d[:, ok].max())
                assert worst < (pu.POP_TOL if n <= 5 else 5 * pu.POP_TOL), (n, worst)
            orr, orb, ou = o.get_macros()
            assert max(np.abs(rr_g - orr).max(), np.abs(u_g - ou).max()) < pu.MACRO_TOL, n
            st, fo = sim.get_particles()
            so, fo_o = o.get_particles()
            assert np.abs(st - so).max() < 2e-6 * max(1, n / 5), (n, np.abs(st - so).max())
            assert np.abs(fo - fo_o).max() < 1e-5 * max(1.0, np.abs(fo_o).max()), (n, np.abs(fo - fo_o).max())
    assert changed > 60                       # nodes did enter and leave the particles


def test_particles_momentum_conservation_on_gpu(lbmod):
    """On the CUDA path itself: sum_x sum_i f_i c_i + sum_p m_p u_p stays constant over 200 steps of two
    moving, spinning particles (to the rounding of fp32 populations: the sum is ~1e1, the bound 2e-4)."""
    n = 32
    parts = [particle((9.3, 16.1, 15.7), u=(0.04, -0.01, 0.015), w=(0.003, 0.001, -0.002), R=4.5, density=3.0),
             particle((22.6, 15.8, 16.4), u=(-0.05, 0.0, 0.01), w=(0.0, -0.004, 0.001), R=3.6, density=5.0)]
    sim = lbmod.LB(n, n, n, 1.0, 1.0, 0.0, 0.0, 0.0)
    sim.set_particles(parts)
    sim.set_particle_options(mobile=True, K=0.02, h_c=2.0, lubrication=True)
    sim.init(np.ones((n, n, n), np.float32), None, np.zeros((3, n, n, n), np.float32))

    def total():
        rr, _, u = sim.get_macros()               # zeros on the particle nodes; u = m / rho (no force)
        st, _ = sim.get_particles()
        return (u.astype(np.float64) * rr).sum(axis=(1, 2, 3)) + (st[:, 14:15] * st[:, 3:6]).sum(0)
    p0 = total()
    for _ in range(4):
        sim.step(50)
        assert np.abs(total() - p0).max() < 2e-4, np.abs(total() - p0).max()
    assert np.abs(p0).max() > 1.0


def test_held_sphere_drag_on_gpu(lbmod, lbo):
    """A held sphere in a driven fluid (pin PC4's set-up) on the CUDA path: the force on it after 3000
    steps against the oracle's (1e-4 relative) and against Stokes' law for a periodic array (10 %)."""
    n, R, g = 24, 3.5, 1e-6
    parts = [particle((11.5, 11.5, 11.5), R=R)]
    o, sim = _pair(lbmod, lbo, (n, n, n), (1.0, 1.0, 0.0, 0.0, 0.0), parts, np.ones((n, n, n)), None, g=(g, 0, 0), opts=dict(mobile=False))
    o.step(3000); sim.step(3000)
    fg, fo = sim.get_particles()[1], o.get_particles()[1]
    assert abs(fg[0, 0] / fo[0, 0] - 1.0) < 1e-4, (fg[0, 0], fo[0, 0])
    _, _, u = sim.get_macros()
    U = u[0].sum(dtype=np.float64) / n ** 3
    c = 4.0 / 3.0 * np.pi * R ** 3 / n ** 3
    K = 1.0 / (1.0 - 1.7601 * c ** (1 / 3) + c - 1.5593 * c ** 2)
    assert abs(fg[0, 0] / (6 * np.pi * (1.0 / 6.0) * R * U * K) - 1.0) < 0.10


def test_particles_need_ab_storage_and_no_slab(lbmod):
    sim = lbmod.LB(16, 16, 16, 1.0, 1.0, 0.0, 0.0, 0.0)
    sim.set_storage("aa")
    sim.set_particles([particle((8, 8, 8), R=3.0)])
    with pytest.raises(lbmod.LBError) as ei:
        sim.init(np.ones((16, 16, 16), np.float32), None, np.zeros((3, 16, 16, 16), np.float32))
    assert ei.value.code == lbmod.LB_ESTATE
    with pytest.raises(lbmod.LBError):
        lbmod.LB(16, 16, 16).set_particles([particle((8, 8, 8), R=7.0)])        # does not fit the box
    with pytest.raises(lbmod.LBError):
        lbmod.LB(16, 16, 16).set_particles([particle((8, 8, 8), R=3.0, mass=-1.0)])


def test_bijel_mini_workload_parity(lbmod, lbo):
    """The bench's colloid workload in small (48^3 spinodal mixture, 6 neutrally wetting colloids of
    R = 4.5): through lb.from_workload / make_oracle, 1 and 40 steps."""
    from paper_2005_12764_b200 import workloads as W
    w = W.get("bijel-mini")
    assert w.info["colloids"] == 6
    o, sim = pu.make_oracle(lbo, w), pu.make_gpu(lbmod, w)
    o.step(1); sim.step(1)
    fluid = o.get_node_map()[0] == 0
    assert pu.pop_error(sim, o)[fluid].max() < pu.POP_TOL
    o.step(39); sim.step(39)
    rr, rb, u = sim.get_macros()
    orr, orb, ou = o.get_macros()
    assert np.array_equal(rr == 0, o.get_node_map()[0] != 0)
    assert max(np.abs(rr - orr).max(), np.abs(rb - orb).max(), np.abs(u - ou).max()) < pu.MACRO_TOL
    st, fo = sim.get_particles()
    so, _ = o.get_particles()
    assert np.abs(st - so).max() < 1e-5
    assert np.abs(st[:, 3:6]).max() > 1e-6          # the demixing fluid does push the colloids


@pytest.mark.parametrize("two,wet", [(True, False), (True, True), (False, False)])
def test_particles_between_sliding_walls_parity(lbmod, lbo, two, wet):
    """A particle in a channel whose y walls slide in opposite directions (wall groups 2 and 3, G28:
    the wall-group instantiations of the fused kernel, to which a particle's node is a wall at rest)
    against the oracle: node map, populations, fields and particle state over 20 steps.  wet: walls and
    particle alike carry a prescribed phi in the colour stencil (G30: a wetting colloid)."""
    nx, ny, nz = 40, 20, 16
    solid = np.zeros((nz, ny, nx), np.uint8)
    solid[:, 0, :] = 2
    solid[:, ny - 1, :] = 3
    parts = [particle((14.2, 8.7, 8.1), u=(0.03, 0.02, -0.01), w=(0.0, 0.002, 0.004), R=4.2, density=2.0)]
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    phi = np.tanh((x - 20.3) / 2.0) * np.tanh((15.2 - np.abs(x - 20.3)) / 2.0)
    rr, rb = ((1 + phi) / 2, (1 - phi) / 2) if two else (np.ones((nz, ny, nx)), None)
    rr = np.where(solid > 0, 0.0, rr)
    rb = None if rb is None else np.where(solid > 0, 0.0, rb)
    params = (0.9, 1.1, 0.01, 0.7, 0.0) if two else (0.8, 0.8, 0.0, 0.0, 0.0)
    o, sim = _pair(lbmod, lbo, (nx, ny, nz), params, parts, rr, rb, solid=solid, opts=dict(mobile=True, K=0.0, h_c=0.0, lubrication=False))
    # (wall velocities may be set at any time: they act from the next step)
    for obj in (o, sim):
        obj.set_wall_velocity(2, -0.02, 0.0, 0.0)
        obj.set_wall_velocity(3, 0.02, 0.0, 0.003)
        if wet:
            obj.set_wall_phi(0.3)
    for n in range(1, 21):
        o.step(1); sim.step(1)
        if n in (1, 2, 5, 10, 20):
            e, ds, df, dm = _compare(o, sim, two)
            assert e < pu.POP_TOL * max(1, n / 2), (n, e)
            assert ds < 2e-6 and dm < pu.MACRO_TOL, (n, ds, dm)
            assert df < 1e-5 * max(1.0, np.abs(o.get_particles()[1]).max()), (n, df)


def test_particles_step_graph_is_bit_identical(lbmod):
    """lb_step replays a CUDA graph of 16 steps for small boxes, with particles too (the particle
    kernels take no decision on the host): same bits as plain launches, fluid and particles."""
    from paper_2005_12764_b200 import workloads as W
    w = W.get("bijel-mini")
    out = []
    for graph in (0, 1):
        sim = lbmod.from_workload(w)
        sim.set_tuning(graph=graph)
        sim.init(w.rho_r, w.rho_b, w.u)
        sim.step(3); sim.step(70); sim.step(1000)
        out.append((sim.get_populations(0), sim.get_populations(1), sim.get_phi(), sim.get_particles(), sim.launch_count()))
    a, b = out
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    assert np.array_equal(a[3][0], b[3][0]) and np.array_equal(a[3][1], b[3][1])
    assert a[4] == b[4]
