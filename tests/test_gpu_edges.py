"""GPU edge cases, accessors, error behaviour and full-size checks of the CUDA path."""
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


def _random_workload(nx, ny, nz, seed, walls=False, A_nc=0.02, tau=(0.8, 1.2), g=(1e-4, -5e-5, 2e-5)):
    rng = np.random.default_rng(seed)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    # smooth random phase field so that interfaces, probes and bulk all occur
    phi = np.zeros((nz, ny, nx))
    for _ in range(6):
        k = rng.integers(1, 3, 3)
        ph = rng.uniform(0, 2 * np.pi, 3)
        phi += rng.normal() * np.cos(2 * np.pi * k[0] * x / nx + ph[0]) * np.cos(2 * np.pi * k[1] * y / ny + ph[1]) \
            * np.cos(2 * np.pi * k[2] * z / nz + ph[2])
    phi = np.tanh(1.5 * phi)
    rho = 1.0 + 0.02 * rng.uniform(-1, 1, phi.shape)
    solid = None
    if walls:
        solid = np.zeros((nz, ny, nx), np.uint8)
        solid[:, 0, :] = 1
        solid[0, :, :] = 1
        solid[nz // 2, ny // 2, nx // 3] = 1
        solid[1:3, 2:4, nx - 1] = 1
    return W.Workload("random", nx, ny, nz, tau[0], tau[1], 0.01, 0.7, A_nc,
                      (rho * (1 + phi) / 2).astype(np.float32), (rho * (1 - phi) / 2).astype(np.float32),
                      (0.02 * rng.normal(size=(3, nz, ny, nx))).astype(np.float32), solid=solid, g=g)


@pytest.mark.parametrize("shape", [(4, 4, 4), (36, 13, 7), (68, 9, 21), (32, 8, 16)])
@pytest.mark.parametrize("walls", [False, True])
@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_ragged_boxes_all_features(lbmod, lbo, shape, walls, storage):
    """Smallest box, extents that are not multiples of the 32 x 8 tile or of the z chunk, two
    taus, body force, walls, near contact: populations after 1, 2 and 5 steps.  The 4 x 4 x 4 box runs
    without the near-contact force (its probe of 4 sites wraps around the whole box and the G12
    exclusion set would cover it), so that every one of its sites is checked at every step; on the
    other boxes the set of checked sites may never be empty."""
    tiny = shape == (4, 4, 4)
    w = _random_workload(*shape, seed=sum(shape) + walls, walls=walls, A_nc=0.0 if tiny else 0.02)
    o, sim = pu.make_oracle(lbo, w), pu.make_gpu(lbmod, w, storage)
    fluid = np.ones(w.shape, bool) if w.solid is None else (w.solid == 0)
    assert pu.pop_error(sim, o).max() < pu.POP_TOL
    phi_g = sim.get_phi()
    assert np.abs(phi_g - o.get_fields()["phi"])[fluid].max() < 1e-5
    risky = np.zeros(w.shape, bool)
    done = 0
    for n in (1, 2, 5):
        for _ in range(n - done):
            risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1)
            o.step(1); sim.step(1)
        done = n
        e = pu.pop_error(sim, o)
        ok = ~risky & fluid
        assert ok.any(), (n, risky.mean())
        assert e[ok].max() < pu.POP_TOL, (n, e[ok].max())
        if tiny:
            assert not risky.any()
        elif n == 1 or w.sites >= 5000:
            assert risky.mean() < 0.5, (n, risky.mean())     # small boxes: the dilated set grows by a shell per step
    errs, _, _ = pu.macro_errors(sim, o)
    if not risky.any():
        assert max(errs.values()) < pu.MACRO_TOL


def test_no_near_contact_no_force_paths(lbmod, lbo):
    """A_nc = 0 (H = 1 ring), equal taus, g = 0, with and without walls."""
    for walls in (False, True):
        w = _random_workload(40, 12, 10, seed=77, walls=walls, A_nc=0.0, tau=(1.0, 1.0), g=(0, 0, 0))
        o, sim = pu.make_oracle(lbo, w), pu.make_gpu(lbmod, w)
        o.step(3); sim.step(3)
        assert pu.pop_error(sim, o).max() < pu.POP_TOL


def test_poiseuille_single_component_walls(lbmod, lbo):
    """Single-component kernel with the bit-packed mask and a body force (pin P7's setup)."""
    nx, ny, nz = 4, 34, 4
    solid = np.zeros((nz, ny, nx), np.uint8)
    solid[:, 0, :] = solid[:, -1, :] = 1
    w = W.Workload("poiseuille", nx, ny, nz, 1.0, 1.0, 0, 0, 0, np.ones((nz, ny, nx), np.float32), None,
                   np.zeros((3, nz, ny, nx), np.float32), solid=solid, g=(1e-6, 0, 0))
    for storage in ("ab", "aa"):
        o, sim = pu.make_oracle(lbo, w), pu.make_gpu(lbmod, w, storage)
        o.step(2001); sim.step(2001)
        errs, (rr, _, u), (orr, _, ou) = pu.macro_errors(sim, o)
        assert errs["u"] < 1e-7 and errs["rho_r"] < 1e-5, errs
        assert u[0].max() > 1e-4


def test_set_get_populations_roundtrip(lbmod, lbo):
    w = _random_workload(36, 9, 6, seed=5, walls=True)
    o = pu.make_oracle(lbo, w)
    o.step(2)
    for storage in ("ab", "aa"):
        sim = pu.make_gpu(lbmod, w, storage)
        sim.step(1)          # AA: leave the buffer in the swapped state first
        fr, fb = o.get_populations(0).astype(np.float32), o.get_populations(1).astype(np.float32)
        sim.set_populations(0, fr)
        sim.set_populations(1, fb)
        fluid = w.solid == 0
        assert np.abs(sim.get_populations(0) - fr)[:, fluid].max() < 1e-7
        assert np.abs(sim.get_populations(1) - fb)[:, fluid].max() < 1e-7
        o2 = pu.make_oracle(lbo, w)
        o2.set_populations(0, fr); o2.set_populations(1, fb)
        o2.step(1); sim.step(1)
        assert pu.pop_error(sim, o2).max() < pu.POP_TOL


def test_device_pointers_and_stream(lbmod, lbo):
    """Device-resident inputs/outputs (torch tensors) and a non-default torch stream."""
    import torch
    w = W.get("c1")
    o = pu.make_oracle(lbo, w)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        rr = torch.from_numpy(w.rho_r).cuda()
        rb = torch.from_numpy(w.rho_b).cuda()
        u = torch.from_numpy(w.u).cuda()
        sim = lbmod.from_workload(w)
        sim.init(rr, rb, u)
        sim.step(10)
        out_r, out_b, out_u = torch.empty_like(rr), torch.empty_like(rb), torch.empty_like(u)
        sim.get_macros(out_r, out_b, out_u)
    s.synchronize()
    o.step(10)
    orr, orb, ou = o.get_macros()
    assert np.abs(out_r.cpu().numpy() - orr).max() < pu.MACRO_TOL
    assert np.abs(out_u.cpu().numpy() - ou).max() < pu.MACRO_TOL
    assert sim.launch_count() >= 11 and sim.device_bytes() > 2 * 38 * w.sites * 4


def test_error_codes(lbmod):
    lb = lbmod
    for bad in [(30, 8, 8), (2, 8, 8), (8, 3, 8)]:
        with pytest.raises(lb.LBError) as ei:
            lb.LB(*bad)
        assert ei.value.code == lb.LB_EINVAL
    with pytest.raises(lb.LBError) as ei:
        lb.LB(8, 8, 8, tau_r=0.5)
    assert ei.value.code == lb.LB_EINVAL
    sim = lb.LB(8, 8, 8)
    with pytest.raises(lb.LBError) as ei:
        sim.step(1)
    assert ei.value.code == lb.LB_ESTATE
    sim.init(np.ones((8, 8, 8), np.float32), np.ones((8, 8, 8), np.float32), np.zeros((3, 8, 8, 8), np.float32))
    with pytest.raises(lb.LBError) as ei:
        sim.set_geometry(np.zeros((8, 8, 8), np.uint8))
    assert ei.value.code == lb.LB_ESTATE
    with pytest.raises(lb.LBError) as ei:
        sim.set_storage("aa")
    assert ei.value.code == lb.LB_ESTATE
    sim.step(0)
    sim.destroy()
    sim.destroy()


# ------------------------------------------------------------------------------- full size
def _block_oracle_check(lbmod, lbo, w, sim, centres, half=14, margin=7):
    """Sampled outputs at full size: around each centre cut a (2*half)^3 block of the INPUT,
    run the oracle on it as a periodic box for one step and compare the block's interior, whose
    domain of dependence (1 stream + 1 gradient + 4 probe + 1 slack) lies inside the block."""
    f = [sim.get_populations(k) for k in (0, 1)]
    worst = 0.0
    for (cx, cy, cz) in centres:
        ix = np.arange(cx - half, cx + half) % w.nx
        iy = np.arange(cy - half, cy + half) % w.ny
        iz = np.arange(cz - half, cz + half) % w.nz
        sel = np.ix_(iz, iy, ix)
        n = 2 * half
        o = lbo.Oracle(n, n, n, *w.params)
        if w.solid is not None:
            o.set_geometry(w.solid[sel])
        o.set_body_force(*w.g)
        o.set_nc_cutoff(w.phi_c)
        o.init(w.rho_r[sel], w.rho_b[sel], w.u[(slice(None),) + sel])
        marg = o.get_fields()["margin"]
        o.step(1)
        inner = np.zeros((n, n, n), bool)
        inner[margin:-margin, margin:-margin, margin:-margin] = True
        if w.solid is not None:
            inner &= w.solid[sel] == 0
        inner &= ~pu.dilate(marg < 1e-5, 1)
        for k in (0, 1):
            e = np.abs(f[k][(slice(None),) + sel].astype(np.float64) - o.get_populations(k)) / pu.W19[:, None, None, None]
            worst = max(worst, e[:, inner].max())
    return worst


@pytest.mark.parametrize("name", ["c3", "c4"])
def test_full_size_sampled_blocks_and_conservation(lbmod, lbo, name):
    """Full-size configs in the launch configuration bench.py times: one step checked on
    sampled blocks against the oracle, then conservation over more steps."""
    w = W.get(name)
    sim = pu.make_gpu(lbmod, w)
    rr0, rb0, _ = sim.get_macros()
    m0 = pu.masses(rr0, rb0)
    sim.step(1)
    rng = np.random.default_rng(9)
    centres = [(0, 0, 0), (w.nx - 1, w.ny // 2, w.nz - 1)] + \
        [tuple(int(v) for v in rng.integers(0, [w.nx, w.ny, w.nz])) for _ in range(4)]
    worst = _block_oracle_check(lbmod, lbo, w, sim, centres)
    assert worst < pu.POP_TOL, worst
    sim.step(199)
    rr, rb, u = sim.get_macros()
    assert np.isfinite(u).all()
    m1 = pu.masses(rr, rb)
    assert abs(m1[0] - m0[0]) / m0[0] < pu.DRIFT_TOL and abs(m1[1] - m0[1]) / m0[1] < pu.DRIFT_TOL
    if name == "c3":
        mom = np.abs([(u[a].astype(np.float64) * (rr + rb)).sum() for a in range(3)]).max() / w.sites
        assert mom < 1e-5


# ------------------------------------------------------------------------------- moment forwarding
@pytest.mark.parametrize("storage", ["ab", "aa"])
@pytest.mark.parametrize("walls", [False, True])
def test_forwarded_phi_matches_oracle_and_full_sweep(lbmod, lbo, storage, walls):
    """phi(t+1) that k_fused forwards (+ k_phase_fwd for the brick faces) against the oracle's phi
    and against the full phase-field sweep (forward = 0), over several steps, on a box whose
    extents are not multiples of the 32 x 8 tile and with bricks of 3 planes so that every kind
    of brick face, edge and box wrap occurs many times."""
    w = _random_workload(68, 21, 13, seed=11 + walls, walls=walls)
    fluid = np.ones(w.shape, bool) if w.solid is None else (w.solid == 0)
    o = pu.make_oracle(lbo, w)
    a, b = pu.make_gpu(lbmod, w, storage), pu.make_gpu(lbmod, w, storage)
    a.set_tuning(forward=1, zc=3)
    b.set_tuning(forward=0)
    risky = np.zeros(w.shape, bool)
    for n in range(1, 5):
        risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1)
        o.step(1); a.step(1); b.step(1)
        pa, pb, po = a.get_phi(), b.get_phi(), o.get_fields()["phi"]
        ok = fluid & ~risky
        assert np.abs(pa - po)[ok].max() < 2e-6, (n, np.abs(pa - po)[ok].max())
        # the two phi paths differ only in summation order
        assert np.abs(pa - pb)[ok].max() < 2e-6, (n, np.abs(pa - pb)[ok].max())
        e = pu.pop_error(a, o)
        assert e[ok].max() < pu.POP_TOL, (n, e[ok].max())


def test_forwarding_brick_sizes_agree(lbmod):
    """The forwarded sums may not depend on how the box is cut into bricks beyond rounding."""
    w = W.get("c5-mini")
    ref = None
    for zc in (0, 1, 5, 96):
        sim = pu.make_gpu(lbmod, w)
        sim.set_tuning(zc=zc, forward=2)              # (2: also with one plane per brick, where lb_step would sweep)
        sim.step(3)
        phi = sim.get_phi()
        if ref is None:
            ref = phi
        else:
            assert np.abs(phi - ref).max() < 1e-6, (zc, np.abs(phi - ref).max())


def test_single_plane_bricks_take_the_full_sweep(lbmod):
    """A box far smaller than one wave of CTAs gets bricks of one plane, and lb_step then forms phi
    by the full sweep instead of forwarding (lb_set_tuning "forward"): one launch per step more
    than the count of k_fused launches either way, and the same phi as forwarding to rounding."""
    w = W.get("c1")
    phis, launches = [], []
    for fwd in (1, 2, 0):
        sim = pu.make_gpu(lbmod, w)
        sim.set_tuning(forward=fwd, graph=0)
        sim.step(1)
        l0 = sim.launch_count()
        sim.step(20)
        launches.append(sim.launch_count() - l0)
        phis.append(sim.get_phi())
    assert launches[0] == launches[1] == launches[2] == 40
    assert np.array_equal(phis[0], phis[2])           # default on this box = the full sweep
    assert np.abs(phis[0] - phis[1]).max() < 2e-6


def test_full_size_c5_sampled_macros_and_conservation(lbmod, lbo):
    """Config C5 at its full 640^3 (near contact, periodic, A/B, the launch configuration that
    bench.py times): rho_r, rho_b, u after one step on sampled blocks against the oracle run on
    a cut-out of the input (the populations of 2.6e8 sites are too many to bring back), then
    mass conservation and finiteness over 50 steps."""
    w = W.get("c5")
    sim = pu.make_gpu(lbmod, w)
    m0 = pu.masses(w.rho_r, w.rho_b)
    sim.step(1)
    rr, rb, u = sim.get_macros()
    rng = np.random.default_rng(17)
    centres = [(0, 0, 0), (w.nx - 1, w.ny // 2, w.nz - 1)] + \
        [tuple(int(v) for v in rng.integers(0, [w.nx, w.ny, w.nz])) for _ in range(4)]
    # two centres on droplet surfaces so that the probe and the recolouring are exercised
    zz, yy, xx = np.nonzero(np.abs(w.rho_r[::40, ::40, ::40] - 0.5) < 0.3)
    centres += [(int(xx[i]) * 40, int(yy[i]) * 40, int(zz[i]) * 40) for i in (0, len(xx) // 2)] if len(xx) else []
    half, margin = 14, 7
    n = 2 * half
    worst = 0.0
    for (cx, cy, cz) in centres:
        ix = np.arange(cx - half, cx + half) % w.nx
        iy = np.arange(cy - half, cy + half) % w.ny
        iz = np.arange(cz - half, cz + half) % w.nz
        sel = np.ix_(iz, iy, ix)
        o = lbo.Oracle(n, n, n, *w.params)
        o.set_nc_cutoff(w.phi_c)
        o.init(w.rho_r[sel], w.rho_b[sel], w.u[(slice(None),) + sel])
        risky = o.get_fields()["margin"] < 1e-5
        o.step(1)
        risky |= o.get_fields()["margin"] < 1e-5       # get_macros evaluates the force again
        orr, orb, ou = o.get_macros()
        inner = np.zeros((n, n, n), bool)
        inner[margin:-margin, margin:-margin, margin:-margin] = True
        inner &= ~pu.dilate(risky, 2)
        worst = max(worst, np.abs(rr[sel] - orr)[inner].max(), np.abs(rb[sel] - orb)[inner].max(),
                    np.abs(u[(slice(None),) + sel] - ou)[:, inner].max())
    assert worst < 5e-6, worst
    sim.step(49)
    rr, rb, u = sim.get_macros()
    assert np.isfinite(u).all()
    m1 = pu.masses(rr, rb)
    assert abs(m1[0] - m0[0]) / m0[0] < pu.DRIFT_TOL and abs(m1[1] - m0[1]) / m0[1] < pu.DRIFT_TOL
    mom = np.abs([(u[a].astype(np.float64) * (rr + rb)).sum() for a in range(3)]).max() / w.sites
    assert mom < 1e-5


@pytest.mark.parametrize("name,steps", [("c2", 1000), ("c3", 5000), ("c4", 10000), ("c5", 1000)])
def test_whole_run_conservation(lbmod, name, steps):
    """The run lengths BASELINE.json asks for, at full size: no NaN, per-component mass drift
    below 1e-6 relative over the whole run, momentum per site constant where no force acts."""
    w = W.get(name)
    sim = pu.make_gpu(lbmod, w)
    rr0, rb0, u0 = sim.get_macros()
    m0 = pu.masses(rr0, rb0)
    sim.step(steps)
    rr, rb, u = sim.get_macros()
    assert np.isfinite(u).all() and np.isfinite(rr).all()
    m1 = pu.masses(rr, rb)
    assert abs(m1[0] - m0[0]) / m0[0] < pu.DRIFT_TOL, (m0, m1)
    if rb is not None:
        assert abs(m1[1] - m0[1]) / m0[1] < pu.DRIFT_TOL, (m0, m1)
    rho = rr if rb is None else rr + rb
    mom = np.array([(u[a].astype(np.float64) * rho).sum() for a in range(3)]) / w.sites
    if name in ("c3", "c5"):
        assert np.abs(mom).max() < 1e-5, mom
    if name == "c3":
        # the mixture has separated: phi is bimodal now, it was +-0.1 noise at t = 0
        phi = (rr - rb) / rho
        assert np.mean(np.abs(phi) > 0.5) > 0.5
    if name == "c2":
        assert np.abs(mom).max() < 1e-5, mom
        ke0 = float((u0.astype(np.float64) ** 2).sum())
        ke = float((u.astype(np.float64) ** 2).sum())
        assert 0.5 < ke / ke0 < 1.0, ke / ke0       # decays (0.886 for pure viscous decay, G19/P13)
    if name == "c4":
        fluid = w.solid == 0
        assert u[0][fluid].mean() > 0 and np.abs(u[:, ~fluid]).max() == 0


# ------------------------------------------------------------------------------- exact-difference forcing
@pytest.mark.parametrize("storage", ["ab", "aa"])
@pytest.mark.parametrize("walls", [False, True])
def test_exact_difference_forcing_parity(lbmod, lbo, storage, walls):
    """The paper's own forcing (Eq. 9) on the CUDA path against the oracle: body
    force, near contact, two taus, with and without walls; populations after 1, 2 and 5 steps."""
    w = _random_workload(36, 13, 10, seed=31 + walls, walls=walls)
    fluid = np.ones(w.shape, bool) if w.solid is None else (w.solid == 0)
    o, sim = pu.make_oracle(lbo, w), pu.make_gpu(lbmod, w, storage)
    o.set_forcing("edm"); sim.set_forcing("edm")
    risky = np.zeros(w.shape, bool)
    done = 0
    for n in (1, 2, 5):
        for _ in range(n - done):
            risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1)
            o.step(1); sim.step(1)
        done = n
        e = pu.pop_error(sim, o)
        assert e[~risky].max() < pu.POP_TOL, (n, e[~risky].max())
    # the two forcings are different schemes: the Guo run must differ from this one
    g = pu.make_gpu(lbmod, w, storage)
    g.step(5)
    assert np.abs(g.get_populations(0) - sim.get_populations(0)).max() > 1e-7
    errs, _, _ = pu.macro_errors(sim, o)
    assert errs["u"] < 5e-3


def test_exact_difference_poiseuille_single_component(lbmod, lbo):
    nx, ny, nz = 4, 34, 4
    solid = np.zeros((nz, ny, nx), np.uint8)
    solid[:, 0, :] = solid[:, -1, :] = 1
    w = W.Workload("poiseuille", nx, ny, nz, 1.0, 1.0, 0, 0, 0, np.ones((nz, ny, nx), np.float32), None,
                   np.zeros((3, nz, ny, nx), np.float32), solid=solid, g=(1e-6, 0, 0))
    o, sim = pu.make_oracle(lbo, w), pu.make_gpu(lbmod, w)
    o.set_forcing("edm"); sim.set_forcing("edm")
    o.step(2001); sim.step(2001)
    errs, (rr, _, u), _ = pu.macro_errors(sim, o)
    assert errs["u"] < 1e-7 and errs["rho_r"] < 1e-5, errs
    assert u[0].max() > 1e-4


# ------------------------------------------------------------------------------- handle life cycle
def test_handles_are_independent_and_reusable(lbmod, lbo):
    """Two handles of different boxes and models stepping alternately; re-init of a handle (also
    with a different component count); create/destroy cycles return the device memory."""
    import torch
    lb = lbmod
    w1 = _random_workload(36, 13, 7, seed=3, walls=True)
    w2 = _random_workload(40, 12, 10, seed=4, walls=False, A_nc=0.0)
    o1, s1 = pu.make_oracle(lbo, w1), pu.make_gpu(lb, w1, "aa")
    o2 = lbo.Oracle(w2.nx, w2.ny, w2.nz, *w2.params); o2.set_model("sc", 1.5); o2.set_body_force(*w2.g); o2.init(w2.rho_r, w2.rho_b, w2.u)
    s2 = lb.LB(w2.nx, w2.ny, w2.nz, *w2.params); s2.set_model("sc", 1.5); s2.set_body_force(*w2.g)
    s2.init(w2.rho_r, w2.rho_b, w2.u)
    risky = np.zeros(w1.shape, bool)
    fluid = w1.solid == 0
    for _ in range(3):
        risky = pu.dilate(risky, 1) | pu.dilate((o1.get_fields()["margin"] < 1e-5) & fluid, 1)
        s1.step(1); s2.step(1); o1.step(1); o2.step(1)
    assert pu.pop_error(s1, o1)[~risky].max() < pu.POP_TOL
    assert pu.pop_error(s2, o2).max() < pu.POP_TOL
    # re-init the same handle: two components again, then a single component, then two again
    s2.init(w2.rho_r, w2.rho_b, w2.u)
    o2.init(w2.rho_r, w2.rho_b, w2.u)
    s2.step(2); o2.step(2)
    assert pu.pop_error(s2, o2).max() < pu.POP_TOL
    s3 = lb.LB(w2.nx, w2.ny, w2.nz, 0.8, 0.8)
    s3.init(w2.rho_r + w2.rho_b, None, w2.u)
    s3.step(2)
    s3.init(w2.rho_r, w2.rho_b, w2.u)
    o3 = lbo.Oracle(w2.nx, w2.ny, w2.nz, 0.8, 0.8); o3.init(w2.rho_r, w2.rho_b, w2.u)
    s3.step(2); o3.step(2)
    assert pu.pop_error(s3, o3).max() < pu.POP_TOL
    # memory comes back
    torch.cuda.synchronize()
    for s in (s1, s2, s3):
        s.destroy()
    base = torch.cuda.memory_allocated()
    for _ in range(5):
        s = pu.make_gpu(lb, w1)
        s.step(1)
        s.destroy()
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == base


def test_set_populations_then_forwarded_steps(lbmod, lbo):
    """After lb_set_populations the forwarded phi is stale: the next step must take the full
    phase-field sweep, the ones after it the forwarded path, in both models."""
    w = _random_workload(36, 9, 6, seed=9, walls=True)
    for model in ("cg", "sc"):
        o = lbo.Oracle(w.nx, w.ny, w.nz, *w.params); o.set_model(model, 1.4); o.set_geometry(w.solid); o.init(w.rho_r, w.rho_b, w.u)
        o.step(3)
        fr, fb = o.get_populations(0).astype(np.float32), o.get_populations(1).astype(np.float32)
        o2 = lbo.Oracle(w.nx, w.ny, w.nz, *w.params); o2.set_model(model, 1.4); o2.set_geometry(w.solid); o2.init(w.rho_r, w.rho_b, w.u)
        o2.set_populations(0, fr); o2.set_populations(1, fb)
        sim = lbmod.LB(w.nx, w.ny, w.nz, *w.params); sim.set_model(model, 1.4)
        sim.set_geometry(np.ascontiguousarray(w.solid, dtype=np.uint8))
        sim.init(w.rho_r, w.rho_b, w.u)
        sim.step(2)
        sim.set_populations(0, fr); sim.set_populations(1, fb)
        risky = np.zeros(w.shape, bool)
        for n in range(3):
            risky = pu.dilate(risky, 1) | pu.dilate((o2.get_fields()["margin"] < 1e-5) & (w.solid == 0), 1)
            sim.step(1); o2.step(1)
            assert pu.pop_error(sim, o2)[~risky].max() < pu.POP_TOL, (model, n)


# ------------------------------------------------------------------------------- randomised configurations
@pytest.mark.parametrize("seed", list(range(12)))
def test_randomised_configurations(lbmod, lbo, seed):
    """Random box shapes (incl. extents of 4 and long thin boxes) with random combinations of walls,
    near contact, body force, equal / unequal taus, forcing, model, storage and brick size:
    populations after 1 and 4 steps against the oracle."""
    rng = np.random.default_rng(1000 + seed)
    nx = int(rng.choice([4, 8, 12, 36, 64, 100, 132]))
    ny = int(rng.choice([4, 5, 8, 9, 16, 23]))
    nz = int(rng.choice([4, 6, 11, 16, 33]))
    if nx * ny * nz > 60000:
        nz = 4
    walls = bool(rng.integers(2))
    model = "sc" if rng.integers(3) == 0 else "cg"
    A_nc = 0.0 if (model == "sc" or rng.integers(2)) else 0.02
    tau = (0.8, 1.2) if rng.integers(2) else (1.0, 1.0)
    g = (1e-4, -5e-5, 2e-5) if rng.integers(2) else (0.0, 0.0, 0.0)
    forcing = "edm" if rng.integers(2) else "guo"
    storage = "aa" if rng.integers(2) else "ab"
    zc = int(rng.choice([0, 1, 2, 5]))
    w = _random_workload(nx, ny, nz, seed=2000 + seed, walls=walls, A_nc=A_nc, tau=tau, g=g)
    if walls and (ny < 5 or nz < 5 or nx < 8):
        w.solid[:] = 0
        w.solid[0, :, :] = 1                    # one wall plane is all a tiny box has room for
    fluid = w.solid == 0 if w.solid is not None else np.ones(w.shape, bool)
    o = lbo.Oracle(w.nx, w.ny, w.nz, *w.params)
    sim = lbmod.LB(w.nx, w.ny, w.nz, *w.params)
    sim.set_storage(storage)
    if model == "sc":
        o.set_model("sc", 1.5); sim.set_model("sc", 1.5)
    else:
        o.set_forcing(forcing); sim.set_forcing(forcing)
    if w.solid is not None:
        o.set_geometry(w.solid); sim.set_geometry(np.ascontiguousarray(w.solid, dtype=np.uint8))
    o.set_body_force(*g); sim.set_body_force(*g)
    o.init(w.rho_r, w.rho_b, w.u); sim.init(w.rho_r, w.rho_b, w.u)
    sim.set_tuning(zc=zc)
    tag = dict(shape=(nx, ny, nz), walls=walls, model=model, A_nc=A_nc, tau=tau, g=g, forcing=forcing, storage=storage, zc=zc)
    risky = np.zeros(w.shape, bool)
    for n in range(1, 5):
        risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1)
        o.step(1); sim.step(1)
        if n in (1, 4):
            e = pu.pop_error(sim, o)
            ok = ~risky & fluid
            if ok.any():
                assert e[ok].max() < pu.POP_TOL, (tag, n, e[ok].max())
    rr, rb, u = sim.get_macros()
    assert np.isfinite(u).all(), tag


# ------------------------------------------------------------------------------- moving walls
def _couette_workload(two, ny=34, nx=8, nz=4):
    solid = np.zeros((nz, ny, nx), np.uint8)
    solid[:, 0, :] = 2
    solid[:, -1, :] = 3
    ones = np.ones((nz, ny, nx), np.float32)
    return W.Workload("couette", nx, ny, nz, 0.9, 1.3 if two else 0.9, 0.0, 0.0, 0.0,
                      0.4 * ones if two else ones, 0.6 * ones if two else None,
                      np.zeros((3, nz, ny, nx), np.float32), solid=solid)


@pytest.mark.parametrize("two", [False, True])
@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_couette_between_sliding_walls(lbmod, two, storage):
    """"solid walls with opposite speeds +-U = 0.01" (G28): the steady profile
    between half-way moving walls is the straight line u_x = U (2 (y - 1/2)/H - 1), on the CUDA
    path itself (closed form, no oracle), one and two components."""
    w = _couette_workload(two)
    sim = lbmod.from_workload(w, storage=storage)
    sim.set_wall_velocity(2, -0.01, 0.0, 0.0)
    sim.set_wall_velocity(3, 0.01, 0.0, 0.0)
    sim.init(w.rho_r, w.rho_b, w.u)
    sim.step(30000)
    rr, rb, u = sim.get_macros()
    y = np.arange(w.ny)
    exact = 0.01 * (2 * (y - 0.5) / (w.ny - 2.0) - 1.0)
    prof = u[0][2, :, 3]
    assert np.abs(prof[1:-1] - exact[1:-1]).max() < 1e-5, np.abs(prof[1:-1] - exact[1:-1]).max()
    rho = rr if rb is None else rr + rb
    assert abs(float(rho[:, 1:-1, :].mean()) - 1.0) < 1e-5


@pytest.mark.parametrize("model", ["cg", "sc"])
@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_moving_walls_parity(lbmod, lbo, model, storage):
    """Sliding and pushing walls of both groups (and a wall at rest) against the oracle:
    populations after 1, 2 and 5 steps, both models, near contact and body force on."""
    w = _random_workload(36, 13, 10, seed=51, walls=True, A_nc=0.0 if model == "sc" else 0.02)
    w.solid[:, 0, :] = 2                  # the y = 0 plane slides and pushes
    w.solid[0, :, :] = 1                  # the z = 0 plane is at rest
    w.solid[w.nz // 2, w.ny // 2, w.nx // 3] = 3
    fluid = w.solid == 0
    o = lbo.Oracle(w.nx, w.ny, w.nz, *w.params)
    sim = lbmod.LB(w.nx, w.ny, w.nz, *w.params)
    sim.set_storage(storage)
    if model == "sc":
        o.set_model("sc", 1.5); sim.set_model("sc", 1.5)
    for obj in (o, sim):
        obj.set_geometry(w.solid)
        obj.set_body_force(*w.g)
        obj.set_wall_velocity(2, 0.01, 0.002, -0.003)
        obj.set_wall_velocity(3, -0.004, 0.0, 0.006)
        obj.init(w.rho_r, w.rho_b, w.u)
    risky = np.zeros(w.shape, bool)
    done = 0
    for n in (1, 2, 5):
        for _ in range(n - done):
            risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1)
            o.step(1); sim.step(1)
        done = n
        e = pu.pop_error(sim, o)
        assert e[~risky & fluid].max() < pu.POP_TOL, (n, e[~risky & fluid].max())
    # the moving walls do change the result
    ref = lbmod.LB(w.nx, w.ny, w.nz, *w.params)
    ref.set_storage(storage)
    if model == "sc":
        ref.set_model("sc", 1.5)
    ref.set_geometry(w.solid); ref.set_body_force(*w.g); ref.init(w.rho_r, w.rho_b, w.u)
    ref.step(5)
    assert np.abs(ref.get_populations(0) - sim.get_populations(0)).max() > 1e-6


@pytest.mark.parametrize("forcing", ["guo", "edm"])
@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_symmetric_probe_and_wetting_parity(lbmod, lbo, storage, forcing):
    """Colour-symmetric near-contact probe (G29) and prescribed phi at solid nodes (G30) against the
    oracle: populations after 1, 2 and 5 steps and the velocity of lb_get_macros (which repeats
    the probe), walls, body force and two taus on; both options change the result."""
    w = _random_workload(36, 13, 10, seed=61, walls=True, A_nc=0.05)
    fluid = w.solid == 0
    o = lbo.Oracle(w.nx, w.ny, w.nz, *w.params)
    sim = lbmod.LB(w.nx, w.ny, w.nz, *w.params)
    sim.set_storage(storage)
    for obj in (o, sim):
        obj.set_geometry(w.solid)
        obj.set_body_force(*w.g)
        obj.set_forcing(forcing)
        obj.set_nc_symmetric(True)
        obj.set_wall_phi(0.4)
        obj.init(w.rho_r, w.rho_b, w.u)
    h = o.get_fields()["h"]
    assert ((h & 15) > 0).sum() > 20 and ((h >> 4) > 0).sum() > 20          # both probes fire
    risky = np.zeros(w.shape, bool)
    done = 0
    for n in (1, 2, 5):
        for _ in range(n - done):
            risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1)
            o.step(1); sim.step(1)
        done = n
        e = pu.pop_error(sim, o)
        assert e[~risky & fluid].max() < pu.POP_TOL, (n, e[~risky & fluid].max())
    now_risky = pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1) | risky
    _, _, u_o = o.get_macros()
    _, _, u_g = sim.get_macros()
    assert np.abs(u_g - u_o)[:, ~now_risky & fluid].max() < 1e-5
    assert risky[fluid].mean() < 0.5
    # each option alone changes the result
    for kw in ({"sym": False, "wet": 0.4}, {"sym": True, "wet": None}):
        ref = lbmod.LB(w.nx, w.ny, w.nz, *w.params)
        ref.set_storage(storage)
        ref.set_geometry(w.solid); ref.set_body_force(*w.g); ref.set_forcing(forcing)
        ref.set_nc_symmetric(kw["sym"]); ref.set_wall_phi(kw["wet"])
        ref.init(w.rho_r, w.rho_b, w.u)
        ref.step(5)
        assert np.abs(ref.get_populations(0) - sim.get_populations(0)).max() > 1e-6, kw


@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_colour_exchange_invariance_on_gpu(lbmod, storage):
    """With the symmetric probe and phi_wall -> -phi_wall the CUDA path is invariant under the
    exchange of the two fluids up to fp32 rounding (the stored pair {f - w, f^r} is not symmetric
    in r and b); with the one-sided probe it is not."""
    n = 16
    z, y, x = np.meshgrid(*(np.arange(n),) * 3, indexing="ij")
    k = 2 * np.pi / n
    s = (np.sin(2 * k * x + 0.3) * np.cos(k * y) + np.sin(2 * k * y + 1.1) * np.cos(2 * k * z + 0.5)
         + 0.7 * np.sin(3 * k * z + k * x))
    phi = 0.98 * np.tanh(2.0 * s)
    u0 = (0.01 * np.stack([np.sin(k * y), np.sin(k * z), np.sin(k * x)])).astype(np.float32)
    solid = np.zeros((n, n, n), np.uint8)
    solid[:, 0, :] = 1
    fluid = solid == 0

    def run(swap, sym):
        tr, tb = (1.2, 0.8) if swap else (0.8, 1.2)
        sim = lbmod.LB(n, n, n, tr, tb, 0.01, 0.7, 0.05)
        sim.set_storage(storage)
        sim.set_geometry(solid)
        sim.set_nc_symmetric(sym)
        sim.set_wall_phi(-0.3 if swap else 0.3)
        p = -phi if swap else phi
        sim.init(((1 + p) / 2).astype(np.float32), ((1 - p) / 2).astype(np.float32), u0)
        sim.step(20)
        return sim.get_macros()

    a_r, a_b, a_u = run(False, True)
    b_r, b_b, b_u = run(True, True)
    assert np.abs(a_r - b_b)[fluid].max() < 2e-5 and np.abs(a_b - b_r)[fluid].max() < 2e-5
    assert np.abs(a_u - b_u)[:, fluid].max() < 2e-5
    c_r, _, _ = run(False, False)
    _, d_b, _ = run(True, False)
    assert np.abs(c_r - d_b)[fluid].max() > 1e-3


# ---------------------------------------------------------------------------------- open boundaries (G31)
def _open_mask(nx, ny, nz, walls):
    solid = np.zeros((nz, ny, nx), np.uint8)
    if walls:
        solid[:, 1:-1, 0] = 2
        solid[:, 1:-1, -1] = 3
        solid[:, 0, :] = 1
        solid[:, -1, :] = 1
    else:
        solid[:, :, 0] = 2
        solid[:, :, -1] = 3
    return solid


@pytest.mark.parametrize("model", ["cg", "sc", "single"])
@pytest.mark.parametrize("storage", ["ab", "aa"])
@pytest.mark.parametrize("kinds", [("inlet", "outlet"), ("reservoir", "reservoir"), ("outlet", "inlet")])
def test_open_boundaries_parity(lbmod, lbo, model, storage, kinds):
    """Velocity inlet, reservoir and pressure outlet (G31; the flow focuser's open ends,
    PAPER.md:207-219) on wall groups 2 and 3 against the oracle: populations after 1, 2 and 5
    steps on a random state with a wall at rest, body force and (colour gradient) near contact."""
    two = model != "single"
    w = _random_workload(36, 13, 10, seed=77, walls=True, A_nc=0.02 if model == "cg" else 0.0)
    w.solid[:, :, 0] = 2                  # the x = 0 plane is open (group 2)
    w.solid[:, :, -1] = 3                 # so is x = nx-1 (group 3)
    w.solid[0, :, 1:-1] = 1               # the z = 0 plane is at rest
    w.solid[w.nz // 2, w.ny // 2, w.nx // 3] = 3
    fluid = w.solid == 0
    params = list(w.params)
    if not two:
        params[1] = params[0]
    o = lbo.Oracle(w.nx, w.ny, w.nz, *params)
    sim = lbmod.LB(w.nx, w.ny, w.nz, *params)
    sim.set_storage(storage)
    if model == "sc":
        o.set_model("sc", 1.5); sim.set_model("sc", 1.5)
    rho_r = w.rho_r + (0 if two else w.rho_b)

    def dens(kind, a, b):
        # one component: the density of an inlet / reservoir is rho_r alone (rho_b is ignored), that
        # of an outlet rho_r + rho_b; keep either near the fluid's (a 40 % jump is a shock whose
        # fp32 rounding differences grow by orders of magnitude within a few steps)
        return (a, b) if two or kind == "outlet" else (a + b, 0.5)
    for obj in (o, sim):
        obj.set_geometry(w.solid)
        obj.set_body_force(*w.g)
        obj.set_wall_velocity(2, 0.012, 0.002, -0.003)
        obj.set_wall_velocity(3, -0.008, 0.001, 0.002)
        obj.set_wall_type(2, kinds[0], *dens(kinds[0], 0.62, 0.41))
        obj.set_wall_type(3, kinds[1], *dens(kinds[1], 0.35, 0.63))
        obj.init(rho_r, w.rho_b if two else None, w.u)
    risky = np.zeros(w.shape, bool)
    done = 0
    for n in (1, 2, 5):
        for _ in range(n - done):
            if model == "cg":
                risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1)
            o.step(1); sim.step(1)
        done = n
        e = pu.pop_error(sim, o, two=two)
        assert e[~risky & fluid].max() < pu.POP_TOL, (n, e[~risky & fluid].max())
    errs, _, _ = pu.macro_errors(sim, o)
    assert max(errs.values()) < pu.MACRO_TOL, errs
    # the open boundaries do change the result (against the same groups as moving walls)
    ref = lbmod.LB(w.nx, w.ny, w.nz, *params)
    ref.set_storage(storage)
    if model == "sc":
        ref.set_model("sc", 1.5)
    ref.set_geometry(w.solid); ref.set_body_force(*w.g)
    ref.set_wall_velocity(2, 0.012, 0.002, -0.003); ref.set_wall_velocity(3, -0.008, 0.001, 0.002)
    ref.init(rho_r, w.rho_b if two else None, w.u)
    ref.step(5)
    assert np.abs(ref.get_populations(0) - sim.get_populations(0)).max() > 1e-4


@pytest.mark.parametrize("exit_kind", ["reservoir", "outlet"])
@pytest.mark.parametrize("two", [False, True])
@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_open_plug_flow_is_a_fixed_point_on_gpu(lbmod, two, exit_kind, storage):
    """A uniform flow at the prescribed densities is an exact fixed point of velocity inlet +
    pressure boundary (f^eq_i -+ f^eq_opp(i) of Eq. 2): closed form on the CUDA
    path itself, no oracle.  fp32: the state stays within rounding of the plug flow."""
    nx, ny, nz, U = 36, 9, 12, 0.03
    solid = _open_mask(nx, ny, nz, walls=False)
    rr0, rb0 = (0.7, 0.4) if two else (1.1, 0.0)
    sim = lbmod.LB(nx, ny, nz, 0.8, 1.1 if two else 0.8, 0.0, 0.0, 0.0)
    sim.set_storage(storage)
    sim.set_geometry(solid)
    sim.set_wall_velocity(2, U, 0.0, 0.0)
    sim.set_wall_type(2, "inlet", rr0, rb0)
    sim.set_wall_type(3, exit_kind, rr0, rb0)
    ones = np.ones((nz, ny, nx), np.float32)
    u0 = np.zeros((3, nz, ny, nx), np.float32)
    u0[0] = U
    sim.init(rr0 * ones, rb0 * ones if two else None, u0)
    sim.step(500)
    rr, rb, u = sim.get_macros()
    fl = solid == 0
    assert np.abs(rr[fl] - rr0).max() < 2e-5 and np.abs(u[0][fl] - U).max() < 2e-5
    assert np.abs(u[1:]).max() < 2e-5
    if two:
        assert np.abs(rb[fl] - rb0).max() < 2e-5


@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_open_inlet_outlet_mass_balance_on_gpu(lbmod, storage):
    """Velocity inlet (red-rich plug U) and pressure outlet in a walled channel, on the CUDA path
    itself: the steady mass flux through every cross-section is what the inlet links inject,
    rho_in U (H - 1/3) (each inlet link adds 6 w_i rho_in U; the two corner nodes lack one diagonal
    each); the red share of the flux tends to the inlet's 0.7; the profile develops into the
    parabola (the oracle's pin P18, here in fp32)."""
    nx, ny, nz, U = 52, 14, 4, 0.02
    solid = _open_mask(nx, ny, nz, walls=True)
    sim = lbmod.LB(nx, ny, nz, 0.9, 0.9, 0.0, 0.0, 0.0)
    sim.set_storage(storage)
    sim.set_geometry(solid)
    sim.set_wall_velocity(2, U, 0.0, 0.0)
    sim.set_wall_type(2, "inlet", 0.7, 0.3)
    sim.set_wall_type(3, "outlet", 0.5, 0.5)
    sim.set_wall_type(4, "reservoir", 0.5, 0.5)
    sim.set_wall_velocity(4, 0.01, 0.0, 0.0)
    with pytest.raises(RuntimeError):
        sim.set_wall_velocity(5, 0.01, 0.0, 0.0)
    ones = np.ones((nz, ny, nx), np.float32)
    sim.init(0.5 * ones, 0.5 * ones, np.zeros((3, nz, ny, nx), np.float32))
    sim.step(12000)
    rr, rb, u = sim.get_macros()
    rr, rb, u = rr.astype(np.float64), rb.astype(np.float64), u.astype(np.float64)
    rho = rr + rb
    H = ny - 2
    flux = (rho * u[0])[1, 1:-1, 1:-1].sum(axis=0)
    assert np.abs(flux / (U * (H - 1.0 / 3.0)) - 1.0).max() < 1e-4, np.abs(flux / (U * (H - 1.0 / 3.0)) - 1.0).max()
    red = (rr * u[0])[1, 1:-1, 1:-1].sum(axis=0)
    assert np.abs(red / (0.7 * U * (H - 1.0 / 3.0)) - 1.0).max() < 5e-3
    y = np.arange(ny) - 0.5
    x = nx - 8
    umean = flux[x - 1] / H / rho[1, 1:-1, x].mean()
    para = 6.0 * umean * y[1:-1] * (H - y[1:-1]) / H ** 2
    assert np.abs(u[0][1, 1:-1, x] / para - 1.0).max() < 0.025


def test_open_boundary_error_codes(lbmod):
    sim = lbmod.LB(8, 8, 8, 1.0, 1.0, 0.0, 0.0, 0.0)
    for args in ((1, 1, 1.0, 0.0), (5, 1, 1.0, 0.0), (2, 4, 1.0, 0.0), (2, -1, 1.0, 0.0), (2, 1, -0.5, 0.0),
                 (3, 2, 0.5, float("nan"))):
        with pytest.raises(RuntimeError):
            sim.set_wall_type(*args)
    sim.set_wall_type(2, 0)
    sim.set_wall_type(3, "outlet", 0.5, 0.5)
    sim.set_wall_type(4, "reservoir", 0.5, 0.5)
    sim.set_wall_velocity(4, 0.01, 0.0, 0.0)
    with pytest.raises(RuntimeError):
        sim.set_wall_velocity(5, 0.01, 0.0, 0.0)


# ---------------------------------------------------------------------------------- flow focuser (three wall groups)
def _focuser_pair(lbmod, lbo, w, storage):
    o = lbo.Oracle(w.nx, w.ny, w.nz, *w.params)
    sim = lbmod.LB(w.nx, w.ny, w.nz, *w.params)
    sim.set_storage(storage)
    for obj in (o, sim):
        obj.set_geometry(w.solid)
        W.configure_walls(obj, w)
        obj.init(w.rho_r, w.rho_b, w.u)
    return o, sim


@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_focuser_parity(lbmod, lbo, storage):
    """The flow-focusing device (stand-in dimensions, G31) with its
    dispersed inlet, continuous inlets and outlet on wall groups 2, 3, 4, in 3-D with walls in z
    and the near-contact force on: populations after 1, 2 and 5 steps and macroscopic fields after
    300 steps against the oracle."""
    w = W.focuser(72, 40, 12, wd=8, wc=8, t=3, li=16, wo=8, lo=6, u_d=0.02, u_c=0.015, A_nc=0.02, walls_z=True)
    o, sim = _focuser_pair(lbmod, lbo, w, storage)
    fluid = w.solid == 0
    risky = np.zeros(w.shape, bool)
    done = 0
    for n in (1, 2, 5):
        for _ in range(n - done):
            risky = pu.dilate(risky, 1) | pu.dilate((o.get_fields()["margin"] < 1e-5) & fluid, 1)
            o.step(1); sim.step(1)
        done = n
        e = pu.pop_error(sim, o)
        assert e[~risky & fluid].max() < pu.POP_TOL, (n, e[~risky & fluid].max())
    o.step(295); sim.step(295)
    errs, (rr, rb, u), _ = pu.macro_errors(sim, o)
    assert max(errs.values()) < pu.MACRO_TOL, errs
    assert np.abs(u).max() > 5e-3                       # the inlets do drive a flow


@pytest.mark.parametrize("storage", ["ab", "aa"])
def test_focuser_relabelled_groups_and_exact_injection_on_gpu(lbmod, storage):
    """On the CUDA path itself (no oracle): (a) permuting the labels of the three wall groups
    together with their settings changes nothing, bit for bit; (b) while no red fluid has reached
    the outlet the red mass grows per step by what the links out of the dispersed inlet inject,
    u_d (w_d - 1/3) per plane (oracle pin P19, here to fp32 rounding)."""
    w = W.focuser(96, 48, 4)
    sims = []
    for perm in ({2: 2, 3: 3, 4: 4}, {2: 4, 4: 3, 3: 2}):
        solid = w.solid.copy()
        for a, b in perm.items():
            solid[w.solid == a] = b
        sim = lbmod.LB(w.nx, w.ny, w.nz, *w.params)
        sim.set_storage(storage)
        sim.set_geometry(solid)
        for g, d in w.info["wall_groups"].items():
            sim.set_wall_velocity(perm[g], *d["u"])
            sim.set_wall_type(perm[g], d["kind"], *d["rho"])
        sim.init(w.rho_r, w.rho_b, w.u)
        sims.append(sim)
    fl = w.solid == 0
    m0 = float(sims[0].get_macros()[0][fl].sum(dtype=np.float64))
    for s in sims:
        s.step(1500)
    a, b = sims[0].get_macros(), sims[1].get_macros()
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    rr = a[0]
    assert rr[:, :, -8:].max() < 1e-7
    rate = w.info["wall_groups"][2]["u"][0] * (w.info["wd"] - 1.0 / 3.0) * w.nz
    gain = float(rr[fl].sum(dtype=np.float64)) - m0
    assert abs(gain / (1500 * rate) - 1.0) < 1e-4, gain / (1500 * rate)


def test_focuser_3d_run(lbmod):
    """The 3-D device (256 x 96 x 48, walls in z, near contact on) for 6000 steps: the dispersed
    phase is pushed through the orifice, everything stays finite and within the lattice's Mach
    range, the total mass stays bounded (the outlet passes what the inlets inject) and the wall
    groups reach the kernel (the inlet columns move at the prescribed speeds)."""
    w = W.get("focuser-3d")
    sim = lbmod.LB(w.nx, w.ny, w.nz, *w.params)
    sim.set_geometry(w.solid)
    W.configure_walls(sim, w)
    sim.init(w.rho_r, w.rho_b, w.u)
    fl = w.solid == 0
    rr0, rb0, _ = sim.get_macros()
    m0 = float((rr0 + rb0)[fl].sum(dtype=np.float64))
    front0 = np.where((rr0 > rb0) & fl)[2].max()
    sim.step(6000)
    rr, rb, u = sim.get_macros()
    assert np.isfinite(u).all() and np.abs(u).max() < 0.15
    front = np.where((rr > rb) & fl)[2].max()
    assert front > front0 + 20, (front0, front)
    assert abs(float((rr + rb)[fl].sum(dtype=np.float64)) / m0 - 1.0) < 0.03
    zc, yc = w.nz // 2, w.ny // 2
    ud = w.info["wall_groups"][2]["u"][0]
    assert 0.5 * ud < u[0][zc, yc, 4] < 2.5 * ud           # between the plug speed and the developed peak
    assert u[0][zc, 6 + 12, 4] > 0


def test_focuser_pinches_off_a_droplet(lbmod):
    """The device in the dripping regime (Ca = rho nu u_c / sigma = 0.125, alpha = u_d / 2 u_c = 0.15;
    "focuser-drip"): behind the orifice the continuous phase squeezes the dispersed thread until a
    droplet pinches off, the mechanism of the paper's Fig. 4.  After 12000 steps
    the red phase consists of the thread and at least one separate droplet of more than 5000
    sites; the thread was one piece at 3000 steps."""
    from scipy import ndimage
    w = W.get("focuser-drip")
    sim = lbmod.from_workload(w)
    sim.init(w.rho_r, w.rho_b, w.u)
    fl = w.solid == 0

    def pieces():
        rr, rb, u = sim.get_macros()
        assert np.isfinite(u).all()
        lab, n = ndimage.label((rr > rb) & fl)
        return sorted(np.bincount(lab.ravel())[1:].tolist(), reverse=True)

    sim.step(3000)
    assert len([s for s in pieces() if s > 1000]) == 1
    sim.step(9000)
    big = [s for s in pieces() if s > 5000]
    assert len(big) >= 2, big


def test_state_check_reports_nan_and_masses(lbmod):
    """G23 (fault tolerance is named at PAPER.md:154): lb_check_state sums the
    component masses on the device and reports a non-finite state with LB_ESTATE; lb_step runs the
    same check by itself every 1000 steps and then stops stepping."""
    w = W.get("c1")
    for storage in ("ab", "aa"):
        sim = pu.make_gpu(lbmod, w, storage)
        m0 = pu.masses(w.rho_r, w.rho_b)
        mr, mb = sim.check_state()
        assert abs(mr - m0[0]) / m0[0] < 1e-6 and abs(mb - m0[1]) / m0[1] < 1e-6
        sim.step(1001)                              # crosses one automatic check: healthy state, no error
        mr, mb = sim.check_state()
        assert abs(mr - m0[0]) / m0[0] < pu.DRIFT_TOL and abs(mb - m0[1]) / m0[1] < pu.DRIFT_TOL
        fr, fb = sim.get_populations(0), sim.get_populations(1)
        fr[3, 5, 6, 7] = np.nan
        sim.set_populations(0, fr)
        sim.set_populations(1, fb)
        with pytest.raises(lbmod.LBError) as ei:
            sim.check_state()
        assert ei.value.code == lbmod.LB_ESTATE and "non-finite" in str(ei.value)
        sim.step(999)                               # below the check interval: the NaN spreads silently
        with pytest.raises(lbmod.LBError) as ei:
            sim.step(2)                             # 1001 steps since the last check: lb_step reports it
        assert ei.value.code == lbmod.LB_ESTATE
    # single component
    w2 = W.get("c2-mini")
    sim = pu.make_gpu(lbmod, w2)
    sim.step(3)
    mr, mb = sim.check_state()
    assert abs(mr - w2.sites) / w2.sites < 1e-6 and mb == 0.0


@pytest.mark.parametrize("name,storage", [("c1", "ab"), ("c1", "aa"), ("c4-mini", "ab"), ("c4-mini", "aa"), ("c2-mini", "ab")])
def test_step_graph_is_bit_identical_to_plain_launches(lbmod, name, storage):
    """lb_set_tuning("graph"): lb_step replays a CUDA graph of 16 steps for small boxes.  Same bits,
    same launch count and the same state check as plain launches; a changed parameter (here the
    body force) between two calls rebuilds the graph."""
    w = W.get(name)
    two = w.rho_b is not None
    sims = {}
    for graph in (0, 1):
        sim = pu.make_gpu(lbmod, w, storage)
        sim.set_tuning(graph=graph)
        sim.step(3)                                   # plain in both (the first steps), odd parity next
        sim.step(37)                                  # 2 replays + 5 plain steps
        sim.set_body_force(2e-5, -1e-5, 3e-5)
        sim.step(64)                                  # new key: rebuilt, 4 replays
        sim.step(1000)                                # crosses the state check at 1000 steps
        sims[graph] = sim
    assert sims[0].launch_count() == sims[1].launch_count()
    for k in range(2 if two else 1):
        assert np.array_equal(sims[0].get_populations(k), sims[1].get_populations(k))
    if two:
        assert np.array_equal(sims[0].get_phi(), sims[1].get_phi())
        a, b = sims[0].check_state(), sims[1].check_state()
        assert abs(a[0] - b[0]) <= 1e-12 * a[0] and abs(a[1] - b[1]) <= 1e-12 * a[1]


def test_host_device_and_mixed_arrays_agree(lbmod):
    """lb_init and lb_get_macros take host or device arrays; host arrays cross the bus in pieces on a
    copy stream of the handle's own while the kernel treats the piece before (a ragged last piece
    here: 36 x 13 x 10 sites).  All-host, all-device and mixed calls must give the same bits."""
    import torch
    w = _random_workload(36, 13, 10, seed=77, walls=True)
    ref = None
    for mode in ("host", "device", "mixed"):
        sim = lbmod.from_workload(w)
        rr, rb, u = w.rho_r, w.rho_b, w.u
        if mode != "host":
            rr = torch.from_numpy(w.rho_r).cuda()
            u = torch.from_numpy(w.u).cuda()
        if mode == "device":
            rb = torch.from_numpy(w.rho_b).cuda()
        sim.init(rr, rb, u)
        sim.step(3)
        o_rr = np.empty(w.shape, np.float32) if mode != "device" else torch.empty(w.shape, dtype=torch.float32, device="cuda")
        o_rb = np.empty(w.shape, np.float32) if mode == "host" else torch.empty(w.shape, dtype=torch.float32, device="cuda")
        o_u = np.empty((3,) + w.shape, np.float32) if mode == "host" else torch.empty((3,) + w.shape, dtype=torch.float32, device="cuda")
        sim.get_macros(o_rr, o_rb, o_u)
        torch.cuda.synchronize()
        got = [x if isinstance(x, np.ndarray) else x.cpu().numpy() for x in (o_rr, o_rb, o_u)]
        if ref is None:
            ref = got
            assert np.isfinite(got[2]).all() and got[0][w.solid == 0].min() > 0
        else:
            for a, b in zip(ref, got):
                assert np.array_equal(a, b), mode
