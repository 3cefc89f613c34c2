"""Pins of the oracle's rigid-particle part (NEXT-4; the paper's section 6, Eq. 15)
against what the mathematics fixes: exact conservation of the momentum of fluid + particles (also
through node changes), exact absence of force and torque in a fluid at rest, the closed forms of the
leapfrog / quaternion integrator, Stokes' drag on a periodic array of spheres (Hasimoto) and the torque
on a spinning sphere, Newton's third law and the closed form of the pair force.  CPU only.

Readings G32-G37: the paper gives Eq. 15 and names leapfrog + quaternions and "interactions
with the fluid and the inter-particle forces, including the lubrication term"; the
link rule, the node changes and the pair force are this build's."""
import numpy as np
import pytest

C = np.array([[0, 0, 0], [1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1], [1, 1, 0], [-1, -1, 0],
              [1, -1, 0], [-1, 1, 0], [1, 0, 1], [-1, 0, -1], [1, 0, -1], [-1, 0, 1], [0, 1, 1], [0, -1, -1], [0, 1, -1], [0, -1, 1]])


def particle(r, u=(0, 0, 0), w=(0, 0, 0), R=4.5, density=1.0, mass=None):
    m = density * 4.0 / 3.0 * np.pi * R ** 3 if mass is None else mass
    return list(r) + list(u) + list(w) + [1.0, 0.0, 0.0, 0.0, R, m]


def fluid_momentum(o, two):
    f = o.get_populations(0) + (o.get_populations(1) if two else 0.0)
    f = f * (o.get_node_map()[0] == 0)[None]
    return np.array([(f * C[:, a][:, None, None, None]).sum() for a in range(3)]), f.sum()


def total_momentum(o, two):
    st, _ = o.get_particles()
    return fluid_momentum(o, two)[0] + (st[:, 14:15] * st[:, 3:6]).sum(0)


@pytest.mark.parametrize("two", [False, True])
def test_PC1_momentum_of_fluid_and_particles_is_conserved_exactly(lbo, two):
    """Two spinning particles crossing a box (one across the periodic boundary and through a red /
    blue interface), pair repulsion and lubrication on: sum_x sum_i f_i c_i + sum_p m_p u_p is
    constant to rounding at every step, although nodes enter and leave the particles all the time
    (the link exchange G33, the node changes G36 and the pair force G37 all conserve it)."""
    n = 24
    o = lbo.Oracle(n, n, n, 0.9, 1.1, 0.01 if two else 0.0, 0.7 if two else 0.0, 0.0)
    o.set_particles([particle((5.3, 12.1, 11.7), u=(0.04, -0.01, 0.015), w=(0.003, 0.001, -0.002), R=4.5, density=3.0),
                     particle((16.6, 11.8, 12.4), u=(-0.05, 0.0, 0.01), w=(0.0, -0.004, 0.001), R=3.6, density=5.0)])
    o.set_particle_options(mobile=True, K=0.02, h_c=2.0, lubrication=True)
    z, y, x = np.meshgrid(*(np.arange(n),) * 3, indexing="ij")
    phi = np.tanh((x - 12) / 2.0) * np.tanh((18 - np.abs(x - 12)) / 2.0)
    rr, rb = ((1 + phi) / 2, (1 - phi) / 2) if two else (np.ones((n, n, n)), None)
    o.init(rr, rb, np.zeros((3, n, n, n)))
    p0 = total_momentum(o, two)
    changed = 0
    prev = o.get_node_map()[0]
    for _ in range(60):
        o.step(1)
        assert np.abs(total_momentum(o, two) - p0).max() < 1e-10
        cur = o.get_node_map()[0]
        changed += int((cur != prev).sum())
        prev = cur
    assert changed > 100                      # nodes did enter and leave
    st, fo = o.get_particles()
    assert np.abs(np.linalg.norm(st[:, 9:13], axis=1) - 1.0).max() < 1e-12      # unit quaternions
    assert np.abs(fo[0, 6:9] + fo[1, 6:9]).max() < 1e-15                          # pair force: actio = reactio


@pytest.mark.parametrize("centre", [(8.0, 8.0, 8.0), (8.5, 8.5, 8.5), (7.31, 8.77, 8.02)])
def test_PC2_no_force_and_no_torque_in_a_fluid_at_rest(lbo, centre):
    """A uniform fluid at rest presses equally on every link of the closed staircase surface: the sum
    over the links of 2 w_j rho c_j and its moment vanish identically, wherever the centre sits."""
    n = 16
    for two in (False, True):
        o = lbo.Oracle(n, n, n, 1.0, 1.0, 0.0, 0.0, 0.0)
        o.set_particles([particle(centre, R=4.2)])
        o.init(0.7 * np.ones((n, n, n)), 0.4 * np.ones((n, n, n)) if two else None, np.zeros((3, n, n, n)))
        o.step(3)
        st, fo = o.get_particles()
        assert np.abs(fo[0, :6]).max() < 1e-13 and np.abs(st[0, 3:9]).max() < 1e-15
        rr, rb, u = o.get_macros()
        assert np.abs(u).max() < 1e-15


def test_PC3_leapfrog_and_quaternion_closed_forms(lbo):
    """Eq. 15 by leapfrog with quaternions, on a particle so heavy that
    the fluid does not matter: u_n = n F/m, r_n = r_0 + n (n + 1)/2 F/m (leapfrog: the velocity is
    updated first), w constant under no torque, q_n = rotation by n |w| about w."""
    n = 12
    o = lbo.Oracle(n, n, n, 1.0, 1.0, 0.0, 0.0, 0.0)
    m = 1e15
    w = np.array([0.01, -0.02, 0.015])
    o.set_particles([particle((5.5, 6.0, 6.2), w=w, R=3.0, mass=m)])
    F = np.array([2e10, -1e10, 3e10])
    o.set_particle_force(0, F=F)
    o.init(np.ones((n, n, n)), None, np.zeros((3, n, n, n)))
    steps = 25
    o.step(steps)
    st, _ = o.get_particles()
    assert np.abs(st[0, 3:6] - steps * F / m).max() < 1e-12
    assert np.abs(st[0, :3] - (np.array([5.5, 6.0, 6.2]) + steps * (steps + 1) / 2 * F / m)).max() < 1e-9
    assert np.abs(st[0, 6:9] - w).max() < 1e-12
    th = steps * np.linalg.norm(w)
    q = np.concatenate([[np.cos(th / 2)], np.sin(th / 2) * w / np.linalg.norm(w)])
    assert np.abs(st[0, 9:13] - q).max() < 1e-10
    # a torque spins it up: w_n = n T / I, I = 2/5 m R^2
    o2 = lbo.Oracle(n, n, n, 1.0, 1.0, 0.0, 0.0, 0.0)
    o2.set_particles([particle((5.5, 6.0, 6.2), R=3.0, mass=m)])
    T = np.array([0.0, 0.0, 4e12])
    o2.set_particle_force(0, T=T)
    o2.init(np.ones((n, n, n)), None, np.zeros((3, n, n, n)))
    o2.step(10)
    st2, _ = o2.get_particles()
    assert np.abs(st2[0, 6:9] - 10 * T / (0.4 * m * 9.0)).max() < 1e-12


def test_PC4_stokes_drag_on_a_periodic_array(lbo):
    """A held sphere in a fluid pushed by a body force.  (a) Momentum balance of one step, exact: the
    fluid's momentum changes by the body force minus what the links hand to the sphere.  (b) Once the
    flow around the sphere has formed (R^2 / nu = 70 steps; the mean flow itself relaxes over ~800
    steps), the drag follows Stokes' law for a simple cubic array of spheres (Hasimoto 1959):
    F = 6 pi mu R U / (1 - 1.7601 c^(1/3) + c - 1.5593 c^2), c the volume fraction, U the mean velocity
    over the whole cell.  The staircase sphere's hydrodynamic radius differs from the nominal one by a
    fraction of a lattice unit: 10 %."""
    n, R, g = 24, 3.5, 1e-6
    o = lbo.Oracle(n, n, n, 1.0, 1.0, 0.0, 0.0, 0.0)
    o.set_particles([particle((11.5, 11.5, 11.5), R=R)])
    o.set_particle_options(mobile=False)
    o.set_body_force(g, 0, 0)
    o.init(np.ones((n, n, n)), None, np.zeros((3, n, n, n)))
    o.step(4000)
    p_before, mass = fluid_momentum(o, False)
    o.step(1)
    p_after, _ = fluid_momentum(o, False)
    st, fo = o.get_particles()
    assert np.abs((p_after - p_before) - (np.array([g * mass, 0, 0]) - fo[0, :3])).max() < 1e-12
    _, _, u = o.get_macros()
    U = u[0].sum() / n ** 3                               # superficial velocity (zero inside the sphere)
    assert abs(fo[0, 0] / (g * mass) - 1.0) < 0.02        # close to steady: drag ~ body force on the fluid
    c = 4.0 / 3.0 * np.pi * R ** 3 / n ** 3
    K = 1.0 / (1.0 - 1.7601 * c ** (1 / 3) + c - 1.5593 * c ** 2)
    mu = 1.0 / 6.0
    assert abs(fo[0, 0] / (6 * np.pi * mu * R * U * K) - 1.0) < 0.10, fo[0, 0] / (6 * np.pi * mu * R * U * K)
    assert np.abs(fo[0, 1:6]).max() < 1e-3 * abs(fo[0, 0])             # no lift, no torque


def test_PC5_torque_on_a_spinning_sphere(lbo):
    """A sphere spinning at w in a fluid at rest feels T = -8 pi mu R^3 w (the periodic images add a
    correction of the order of the volume fraction): sign and size of the rotational part of u_b."""
    n, R, w = 32, 5.5, 1e-3
    o = lbo.Oracle(n, n, n, 1.0, 1.0, 0.0, 0.0, 0.0)
    o.set_particles([particle((16.0, 16.0, 16.0), w=(0, 0, w), R=R)])
    o.set_particle_options(mobile=False)
    o.init(np.ones((n, n, n)), None, np.zeros((3, n, n, n)))
    o.step(3000)
    st, fo = o.get_particles()
    mu = 1.0 / 6.0
    ratio = fo[0, 5] / (-8 * np.pi * mu * R ** 3 * w)
    assert 0.95 < ratio < 1.25, ratio
    assert np.abs(fo[0, :5]).max() < 1e-6 * abs(fo[0, 5])


def test_PC6_pair_force_closed_form(lbo):
    """G37: K (h_c - h)^(3/2) along the line of centres for gaps below h_c, nothing beyond; the
    lubrication term opposes the approach and vanishes for tangential motion."""
    n = 24
    def run(gap, u1=(0, 0, 0), lub=False, K=0.05):
        o = lbo.Oracle(n, n, n, 1.0, 1.0, 0.0, 0.0, 0.0)
        o.set_particles([particle((8.0, 12, 12), u=u1, R=3.0), particle((8.0 + 6.0 + gap, 12, 12), R=3.0)])
        o.set_particle_options(mobile=True, K=K, h_c=2.0, lubrication=lub)
        o.init(np.ones((n, n, n)), None, np.zeros((3, n, n, n)))
        o.step(1)
        return o.get_particles()[1][:, 6:9]
    f = run(1.2)
    assert abs(f[0, 0] + 0.05 * 0.8 ** 1.5) < 1e-14 and abs(f[1, 0] - 0.05 * 0.8 ** 1.5) < 1e-14 and np.abs(f[:, 1:]).max() == 0
    assert np.abs(run(2.5)).max() == 0
    mu, Reff, h = 1.0 / 6.0, 1.5, 1.2
    fl = run(1.2, u1=(0.01, 0, 0), lub=True, K=0.0)
    assert abs(fl[0, 0] + 6 * np.pi * mu * Reff ** 2 * (1 / h - 1 / 2.0) * 0.01) < 1e-14        # approach: pushed back
    assert np.abs(run(1.2, u1=(0, 0.01, 0), lub=True, K=0.0)).max() < 1e-15                      # sliding past: nothing
