"""z-slab decomposition on ONE GPU: the slabs of a box
as several handles of one process, halo messages moved by device copies (paper_2005_12764_b200.slab.
LocalRing), against the undivided box.  With the bricks of both runs cut at the same planes the two
must agree BIT FOR BIT (the slab faces are brick faces of the undivided run; a ghost plane holds a copy
of what the neighbour stored); with the automatic brick depth they agree to the rounding of the
forwarded sums.  The undivided box itself is held against the oracle in test_gpu_parity.py; one case
here goes to the oracle directly."""
import numpy as np
import pytest

import parity_util as pu
from paper_2005_12764_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lbmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2005_12764_b200 import lb
    return lb


@pytest.fixture(scope="module")
def slabmod(lbmod):
    from paper_2005_12764_b200 import slab
    return slab


def _same_bits(ring, sim, two=True):
    for k in range(2 if two else 1):
        assert np.array_equal(ring.gather("get_populations", k), sim.get_populations(k)), "populations of component %d" % k
    a, b = ring.gather("get_macros"), sim.get_macros()
    for x, y in zip(a, b):
        assert (x is None and y is None) or np.array_equal(x, y)
    if two:
        assert np.array_equal(ring.gather("get_phi"), sim.get_phi())


# (workload, cuts, zc): the cuts are multiples of zc, so both runs have the same bricks
CASES = [("c3-mini", (32, 32), 16), ("c3-mini", (16, 32, 16), 16), ("c4-mini", (16, 16), 8), ("c4-mini", (8, 24), 8),
         ("c5-mini", (40, 56), 8), ("c5-mini", (96,), 12)]


@pytest.mark.parametrize("storage", ["ab", "aa"])
@pytest.mark.parametrize("name,cuts,zc", CASES)
def test_slabs_equal_undivided_box_bitwise(lbmod, slabmod, name, cuts, zc, storage):
    """C3-mini (periodic), C4-mini (walls and body force: the wall planes z = 0, nz - 1 sit on both
    sides of the periodic cut, the y walls cross every cut) and C5-mini (near contact: the probe and
    its 4-plane phi halo cross the cuts), A/B and in-place storage, after 1, 2, 3 and 5 steps (both
    in-place parities are packed and unpacked differently)."""
    w = W.get(name)
    sim = pu.make_gpu(lbmod, w, storage)
    sim.set_tuning(zc=zc)
    ring = slabmod.LocalRing(w, cuts, storage, zc=zc)
    ring.init()
    _same_bits(ring, sim)
    m_ring = [sum(s.sim.check_state()[k] for s in ring.slabs) for k in (0, 1)]
    m_box = sim.check_state()
    assert abs(m_ring[0] - m_box[0]) / m_box[0] < 1e-12 and abs(m_ring[1] - m_box[1]) / m_box[1] < 1e-12    # at t = 0 too
    done = 0
    for n in (1, 2, 3, 5):
        ring.step(n - done); sim.step(n - done)
        done = n
        _same_bits(ring, sim)
    mr = sum(s.sim.check_state()[0] for s in ring.slabs)
    assert abs(mr - sim.check_state()[0]) / mr < 1e-12          # the slabs' own planes, no ghost plane counted


def test_slabs_single_component(lbmod, slabmod):
    w = W.get("c2-mini")
    for storage in ("ab", "aa"):
        sim = pu.make_gpu(lbmod, w, storage)
        sim.set_tuning(zc=16)
        ring = slabmod.LocalRing(w, (32, 16, 16), storage, zc=16)
        ring.init()
        ring.step(4); sim.step(4)
        _same_bits(ring, sim, two=False)
        assert ring.slabs[0].halo_bytes == (5 * 64 * 64 * 4, 0)


def _walled_random(nx, ny, nz, seed, model=None):
    rng = np.random.default_rng(seed)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    phi = np.zeros((nz, ny, nx))
    for _ in range(6):
        k = rng.integers(1, 3, 3)
        ph = rng.uniform(0, 2 * np.pi, 3)
        phi += rng.normal() * np.cos(2 * np.pi * k[0] * x / nx + ph[0]) * np.cos(2 * np.pi * k[1] * y / ny + ph[1]) \
            * np.cos(2 * np.pi * k[2] * z / nz + ph[2])
    phi = np.tanh(1.5 * phi)
    rho = 1.0 + 0.02 * rng.uniform(-1, 1, phi.shape)
    solid = np.zeros((nz, ny, nx), np.uint8)
    solid[:, 0, :] = 1
    # obstacles on both sides of the cuts at z = 10 and z = 20, and one that spans a cut
    solid[9, 3:6, 4:9] = 1
    solid[10, 7:9, 20:30] = 1
    solid[19:22, 5, 2:5] = 1
    solid[0, :, 10:14] = 1
    solid[nz - 1, 2:4, :] = 1
    return W.Workload("walled-random", nx, ny, nz, 0.8, 1.2, 0.01, 0.7, 0.02,
                      (rho * (1 + phi) / 2).astype(np.float32), (rho * (1 - phi) / 2).astype(np.float32),
                      (0.02 * rng.normal(size=(3, nz, ny, nx))).astype(np.float32), solid=solid, g=(1e-4, -5e-5, 2e-5))


@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_slabs_ragged_box_with_obstacles_on_the_cuts(lbmod, lbo, slabmod, storage):
    """A box whose extents are no multiples of the tile (36 x 13 x 30), two relaxation times, body
    force, near contact, obstacles that touch and span the cuts: three slabs of 10 planes against the
    undivided box (bit for bit) and against the oracle (populations, G12 exclusion)."""
    w = _walled_random(36, 13, 30, seed=3)
    sim = pu.make_gpu(lbmod, w, storage)
    sim.set_tuning(zc=10)
    ring = slabmod.LocalRing(w, (10, 10, 10), storage, zc=10)
    ring.init()
    o = pu.make_oracle(lbo, w)
    fluid = w.solid == 0
    risky = np.zeros(w.shape, bool)
    for n in range(1, 5):
        risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1)
        ring.step(1); sim.step(1); o.step(1)
        _same_bits(ring, sim)
        ok = fluid & ~risky
        assert ok.any()
        for k in (0, 1):
            e = np.abs(ring.gather("get_populations", k).astype(np.float64) - o.get_populations(k)) / pu.W19[:, None, None, None]
            assert e.max(0)[ok].max() < pu.POP_TOL, (n, k)


def test_slabs_automatic_bricks_agree_to_rounding(lbmod, slabmod):
    """Without the brick depth pinned the two runs cut their bricks differently; the forwarded sums
    then differ in summation order only (no near contact here: no decision can flip)."""
    w = W.get("c3-mini")
    sim = pu.make_gpu(lbmod, w)
    ring = slabmod.LocalRing(w, (24, 40))
    ring.init()
    ring.step(5); sim.step(5)
    for k in (0, 1):
        d = np.abs(ring.gather("get_populations", k).astype(np.float64) - sim.get_populations(k)) / pu.W19[:, None, None, None]
        assert d.max() < 1e-5
    assert np.abs(ring.gather("get_phi") - sim.get_phi()).max() < 1e-6


def test_slab_calls_out_of_order_and_bad_buffers(lbmod, slabmod):
    import torch
    w = W.get("c3-mini")
    s = slabmod.Slab.from_workload(w, 0, 32)
    with pytest.raises(lbmod.LBError) as ei:
        s.sim.slab_halo_bytes()                                    # before lb_init
    assert ei.value.code == lbmod.LB_ESTATE
    s.init_from(w)
    with pytest.raises(lbmod.LBError) as ei:
        s.sim.step(1)                                              # a slab is not stepped by lb_step
    assert ei.value.code == lbmod.LB_ESTATE
    with pytest.raises(lbmod.LBError) as ei:
        s.begin()                                                  # phi ghost planes not exchanged yet
    assert ei.value.code == lbmod.LB_ESTATE
    s.pack_phi(); s.buf["f_recv_lo"].copy_(s.buf["f_send_hi"]); s.buf["f_recv_hi"].copy_(s.buf["f_send_lo"]); s.unpack_phi()
    with pytest.raises(lbmod.LBError) as ei:
        s.interior()                                               # before lb_slab_begin
    assert ei.value.code == lbmod.LB_ESTATE
    with pytest.raises(lbmod.LBError) as ei:
        s.sim.slab_begin(np.zeros(16, np.float32), np.zeros(16, np.float32))    # host buffers
    assert ei.value.code == lbmod.LB_EINVAL
    t = torch.zeros(s.halo_bytes[0] // 4 + 4, dtype=torch.float32, device="cuda")
    with pytest.raises(lbmod.LBError) as ei:
        s.sim.slab_begin(t[1:], t)                                 # misaligned
    assert ei.value.code == lbmod.LB_EINVAL
    plain = lbmod.LB(32, 32, 32)
    with pytest.raises(lbmod.LBError):
        plain.set_slab(0, 16)                                      # does not fit
    with pytest.raises(lbmod.LBError):
        lbmod.LB(32, 32, 4).set_slab(0, 64)                        # thinner than twice the phi halo


@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_distributed_slab_world1_two_streams(lbmod, slabmod, storage):
    """The per-rank driver (side stream for the population exchange, events between the phases) with
    a world of one rank, whose neighbours are itself: bit-identical to the undivided box."""
    w = W.get("c5-mini")
    sim = pu.make_gpu(lbmod, w, storage)
    sim.set_tuning(zc=12)
    ds = slabmod.DistributedSlab(slabmod.Slab.from_workload(w, 0, w.nz, storage, zc=12), rank=0, world=1)
    ds.init_from(w)
    ds.step(4); sim.step(4)
    for k in (0, 1):
        assert np.array_equal(ds.slab.sim.get_populations(k), sim.get_populations(k))


# ------------------------------------------------------------------------------- particles over slabs
def _particle_workload(two, walls=False):
    """A 40 x 24 x 32 box with three particles: one astride the cut at z = 16 and moving along z, one
    crossing the periodic z boundary (the ring's wrap), one inside a slab; pair force on; in the
    two-component case a flat interface that the first particle sits in and the near-contact force."""
    from test_oracle_colloids import particle
    nx, ny, nz = 40, 24, 32
    parts = np.array([particle((11.3, 12.1, 15.6), u=(0.01, -0.01, 0.05), w=(0.003, 0.001, -0.002), R=4.5, density=2.0),
                      particle((27.2, 11.6, 30.9), u=(-0.02, 0.004, 0.045), w=(0.0, -0.004, 0.001), R=3.6, density=3.0),
                      particle((26.0, 10.9, 21.3), u=(0.0, 0.01, -0.04), w=(0.002, 0.0, 0.0), R=3.2, density=2.5)])
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    phi = np.tanh((x - 12.3) / 2.0) * np.tanh((30.2 - np.abs(x - 12.3)) / 2.0)
    rr = ((1 + phi) / 2 if two else np.ones((nz, ny, nx))).astype(np.float32)
    rb = ((1 - phi) / 2).astype(np.float32) if two else None
    solid = None
    if walls:
        solid = np.zeros((nz, ny, nx), np.uint8)
        solid[:, 0, :] = 1
        solid[:, ny - 1, :] = 1
    params = (0.9, 1.1, 0.01, 0.7, 0.02) if two else (0.8, 0.8, 0.0, 0.0, 0.0)
    return W.Workload("slab-particles", nx, ny, nz, *params, rr, rb, np.zeros((3, nz, ny, nx), np.float32), solid=solid,
                      g=(1e-5, 0.0, -2e-5),
                      info={"particles": parts, "particle_options": dict(mobile=True, K=0.02, h_c=2.5, lubrication=True)})


@pytest.mark.parametrize("cuts", [(16, 16), (8, 16, 8), (12, 20), (32,)])
@pytest.mark.parametrize("two,walls", [(True, False), (False, False), (True, True)])
def test_slabs_with_replicated_particles(lbmod, slabmod, two, walls, cuts):
    """Replicated data: every slab holds all particles; the link sums and the
    impulses of the node changes are added over the slabs.  Against the undivided box over 40
    steps, in which nodes enter and leave the particles on both sides of the cuts: the same node
    map, particle states to the rounding of the two sums, populations and fields to the rounding
    that follows from it; and all slabs hold the same particle states bit for bit.  (32,): a ring of
    one slab, which holds the planes next to its faces twice, as own and as ghost planes."""
    w = _particle_workload(two, walls)
    sim = lbmod.from_workload(w)
    sim.set_tuning(zc=8)
    sim.init(w.rho_r, w.rho_b, w.u)
    ring = slabmod.LocalRing(w, cuts, "ab", zc=8)
    ring.init()
    solid0 = sim.get_macros()[0] == 0
    changed = 0
    # cuts at brick faces of the undivided run: the fluid agrees bit for bit and only the order of the
    # two sums differs; other cuts: the forwarded phi sums round differently (fp32), and the forces follow
    aligned = all(c % 8 == 0 for c in cuts)
    tol_state, tol_force = (1e-9, 1e-9) if aligned else (1e-7, 1e-5)
    for n in range(1, 41):
        ring.step(1); sim.step(1)
        if n in (1, 2, 3, 5, 10, 20, 30, 40):
            st, fo = sim.get_particles()
            for s in ring.slabs:
                st_s, fo_s = s.sim.get_particles()
                assert np.array_equal(st_s, ring.slabs[0].sim.get_particles()[0])      # replicated: the same bits everywhere
                assert np.abs(st_s - st).max() < tol_state, (n, np.abs(st_s - st).max())
                assert np.abs(fo_s - fo).max() < tol_force * max(1.0, np.abs(fo).max()), (n, np.abs(fo_s - fo).max())
            a, b = ring.gather("get_macros"), sim.get_macros()
            assert np.array_equal(a[0] == 0, b[0] == 0), (n, "node maps differ")
            changed += int(((b[0] == 0) != solid0).sum())
            solid0 = b[0] == 0
            for x, y in zip(a, b):
                assert (x is None and y is None) or np.abs(x - y).max() < 1e-6, n
            for k in range(2 if two else 1):
                d = np.abs(ring.gather("get_populations", k).astype(np.float64) - sim.get_populations(k)) / pu.W19[:, None, None, None]
                assert d.max() < 1e-6, (n, k, d.max())
            if two:
                fluid = b[0] != 0
                assert np.abs(ring.gather("get_phi") - sim.get_phi())[fluid].max() < 2e-6, n
    assert changed > 40                       # nodes did enter and leave the particles
