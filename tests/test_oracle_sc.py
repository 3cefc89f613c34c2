"""Pins of the oracle's second model: the paper's section 3.1 as printed, two components coupled
by the Shan-Chen force (Eq. 10) through the exact-difference source (Eq. 9,
PAPER.md:131) in Eq. 5-6.  CPU only.  Expected values are invariants, a
closed-form stability bound and the independent numpy restatement in tests/np_twin.py."""
import numpy as np
import pytest

import np_twin as tw


def _sc(lbo, nx, ny, nz, tau_r, tau_b, G_C, rho_r, rho_b, u, solid=None, g=(0, 0, 0)):
    o = lbo.Oracle(nx, ny, nz, tau_r, tau_b, 0.0, 0.0, 0.0)
    o.set_model("sc", G_C)
    if solid is not None:
        o.set_geometry(solid)
    o.set_body_force(*g)
    o.init(rho_r, rho_b, u)
    return o


def test_SC1_uniform_mixture_is_fixed_point(lbo):
    """A uniform mixture at uniform velocity feels no force (sum_i w_i c_i = 0) and stays put."""
    nx, ny, nz = 8, 6, 4
    u = np.zeros((3, nz, ny, nx)); u[0], u[1], u[2] = 0.03, -0.02, 0.01
    o = _sc(lbo, nx, ny, nz, 0.8, 1.3, 2.5, np.full((nz, ny, nx), 0.3), np.full((nz, ny, nx), 0.7), u)
    f0 = [o.get_populations(k) for k in (0, 1)]
    o.step(3)
    for k in (0, 1):
        assert np.abs(o.get_populations(k) - f0[k]).max() < 1e-14


def test_SC2_mass_and_momentum(lbo):
    """Eq. 9 carries no mass (per-component mass is conserved exactly, also with walls and g); the
    pair forces of Eq. 10 cancel in the sum over a periodic box, so the total momentum is
    conserved when g = 0."""
    rng = np.random.default_rng(3)
    nx, ny, nz = 12, 10, 8
    rr = rng.uniform(0.2, 0.8, (nz, ny, nx)); rb = rng.uniform(0.2, 0.8, (nz, ny, nx))
    u = 0.02 * rng.normal(size=(3, nz, ny, nx))
    c = np.array(lbo.constants()[0], float)
    o = _sc(lbo, nx, ny, nz, 0.9, 1.1, 1.7, rr, rb, u)
    f = o.get_populations(0) + o.get_populations(1)
    p0 = np.einsum("ia,izyx->a", c, f)
    o.step(50)
    f = o.get_populations(0) + o.get_populations(1)
    assert abs(o.get_populations(0).sum() - rr.sum()) / rr.sum() < 1e-13
    assert abs(o.get_populations(1).sum() - rb.sum()) / rb.sum() < 1e-13
    assert np.abs(np.einsum("ia,izyx->a", c, f) - p0).max() / rr.size < 1e-15
    # walls + body force: masses still exact
    solid = np.zeros((nz, ny, nx), bool); solid[:, 0, :] = True; solid[2, 4, 5] = True
    o = _sc(lbo, nx, ny, nz, 0.9, 1.1, 1.7, rr, rb, u, solid=solid, g=(1e-4, 0, -2e-5))
    m0 = [o.get_populations(k).sum() for k in (0, 1)]
    o.step(50)
    for k in (0, 1):
        assert abs(o.get_populations(k).sum() - m0[k]) / m0[k] < 1e-13


@pytest.mark.parametrize("shape,walls", [((4, 4, 4), False), ((6, 5, 4), True)])
def test_SC3_brute_force_numpy_twin(lbo, shape, walls):
    nx, ny, nz = shape
    rng = np.random.default_rng(21 + nx)
    solid = np.zeros((nz, ny, nx), bool)
    if walls:
        solid[:, 0, :] = True
        solid[1, 2, 3] = True
    g = (1e-4, -5e-5, 2e-5)
    rr = rng.uniform(0.2, 0.8, (nz, ny, nx)); rb = rng.uniform(0.2, 0.8, (nz, ny, nx))
    u = 0.02 * rng.normal(size=(3, nz, ny, nx))
    o = _sc(lbo, nx, ny, nz, 0.8, 1.2, 1.9, rr, rb, u, solid=solid, g=g)
    fr = tw.equilibrium(rr, u) * ~solid
    fb = tw.equilibrium(rb, u) * ~solid
    for _ in range(10):
        fr, fb = tw.step_sc(fr, fb, solid, 0.8, 1.2, 1.9, g=g)
        o.step(1)
        assert np.abs(o.get_populations(0) - fr).max() < 1e-13
        assert np.abs(o.get_populations(1) - fb).max() < 1e-13


def test_SC4_sign_and_demixing_threshold(lbo):
    """"G_C ... takes positive values for repulsive interactions".  With
    F^r = -G_C rho^r c_s^2 grad rho^b to leading order, a symmetric mixture of total density rho_0
    is linearly unstable to demixing iff G_C > 2 / rho_0 (d(mu_r - mu_b)/d rho_r =
    c_s^2 (4 / rho_0 - 2 G_C) < 0).  rho_0 = 1: noise grows for G_C = 3, decays for G_C = 1 and
    for the attractive G_C = -1 (at -3 the total density itself is unstable, dp/drho =
    c_s^2 (1 + G_C rho_0 / 2) < 0).  A flipped sign in Eq. 10 fails the first case: it would turn
    G_C = 3 into an attraction, under which a mixture never demixes."""
    rng = np.random.default_rng(8)
    n = 24
    xi = 0.01 * rng.uniform(-1, 1, (4, n, n))
    out = {}
    for G in (3.0, 1.0, -1.0):
        o = _sc(lbo, n, n, 4, 1.0, 1.0, G, 0.5 + xi, 0.5 - xi, np.zeros((3, 4, n, n)))
        o.step(400)
        rr, rb, _ = o.get_macros()
        out[G] = np.std((rr - rb) / (rr + rb)) / np.std(2 * xi)
    assert out[3.0] > 5.0, out
    assert out[1.0] < 0.5 and out[-1.0] < 0.5, out


def test_SC5_velocity_is_half_step(lbo):
    """get_macros returns (m + F/2)/rho with F = F^r + F^b; under a uniform body force on a uniform
    mixture at rest that is (t + 1/2) g after t steps."""
    n = 4
    g = np.array([2e-4, -1e-4, 3e-4])
    o = _sc(lbo, n, n, n, 0.8, 1.2, 2.0, np.full((n, n, n), 0.4), np.full((n, n, n), 0.6), np.zeros((3, n, n, n)), g=g)
    for t in range(1, 4):
        o.step(1)
        _, _, u = o.get_macros()
        assert np.abs(u - ((t + 0.5) * g)[:, None, None, None]).max() < 1e-15
