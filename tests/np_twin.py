"""Brute-force numpy restatement of one colour-gradient LB step (pin P12).

Independent of oracle/lbo.cpp: whole-array operations with np.roll, streaming in PUSH form
with masks for walls, near-contact probe by Python loops.  Written from the equations
(Eq. 1-8, Eq. 11) and the readings in DESIGN.md, not from
the oracle's source.  Test infrastructure only.
"""
import numpy as np

C = np.array([[0, 0, 0], [1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1],
              [1, 1, 0], [-1, -1, 0], [1, -1, 0], [-1, 1, 0], [1, 0, 1], [-1, 0, -1], [1, 0, -1],
              [-1, 0, 1], [0, 1, 1], [0, -1, -1], [0, 1, -1], [0, -1, 1]])
WT = np.array([12] + [2] * 6 + [1] * 12) / 36.0
BB = np.array([-12] + [2] * 6 + [1] * 12) / 36.0


def opposite(i):
    return int(np.where((C == -C[i]).all(1))[0][0])


def shift(a, c):
    """result(x) = a(x - c) for arrays indexed [z, y, x]."""
    return np.roll(a, shift=(int(c[2]), int(c[1]), int(c[0])), axis=(0, 1, 2))


def half_away(v):
    return np.sign(v) * np.floor(np.abs(v) + 0.5)


def step(fr, fb, solid, tau_r, tau_b, A, beta, A_nc=0.0, g=(0.0, 0.0, 0.0), phi_c=0.9,
         h_min=3, h_max=4, eps=1e-12, forcing="guo", wall_group=None, wall_u=None):
    """One time step. fr, fb: [19, nz, ny, nx] pre-collision; solid: bool [nz, ny, nx]."""
    nz, ny, nx = solid.shape
    fluid = ~solid
    rr, rb = fr.sum(0), fb.sum(0)
    rho = np.where(fluid, rr + rb, 1.0)
    phi = np.where(fluid, (rr - rb) / rho, 0.0)
    ftot = fr + fb
    m = np.stack([(ftot * C[:, a, None, None, None]).sum(0) for a in range(3)])
    G = np.zeros((3, nz, ny, nx))
    for i in range(1, 19):
        ph_n = shift(phi, -C[i])
        so_n = shift(solid, -C[i])
        ph_n = np.where(so_n, phi, ph_n)
        for a in range(3):
            G[a] += 3.0 * WT[i] * C[i, a] * ph_n
    Gn = np.sqrt((G ** 2).sum(0))
    Fnc = np.zeros_like(G)
    if A_nc != 0.0:
        for z in range(nz):
            for y in range(ny):
                for x in range(nx):
                    if solid[z, y, x] or not (abs(phi[z, y, x]) < phi_c and Gn[z, y, x] > eps):
                        continue
                    n = -G[:, z, y, x] / Gn[z, y, x]
                    h = 0
                    for k in range(1, h_max + 1):
                        d = half_away(k * n).astype(int)
                        p = ((z + d[2]) % nz, (y + d[1]) % ny, (x + d[0]) % nx)
                        if solid[p]:
                            break
                        if k >= 2 and phi[p] >= phi[z, y, x]:
                            h = k
                            break
                    if h:
                        Ah = A_nc if h <= h_min else A_nc * (h_min / h) ** 3
                        Fnc[:, z, y, x] = 0.5 * Ah * G[:, z, y, x]
    F = np.stack([rho * g[a] + Fnc[a] for a in range(3)])
    edm = forcing == "edm"       # exact difference, Eq. 9: bare velocity in f^eq
    u = m / rho if edm else (m + 0.5 * F) / rho
    if tau_r == tau_b:
        omega = np.full(rho.shape, 1.0 / tau_r)
    else:
        nur, nub = (tau_r - 0.5) / 3, (tau_b - 0.5) / 3
        nubar = 1.0 / ((rr / rho) / nur + (rb / rho) / nub)
        omega = 1.0 / (3.0 * nubar + 0.5)
    uu = (u ** 2).sum(0)
    aniso = Gn > eps
    Gs = np.where(aniso, Gn, 1.0)
    post_r = np.zeros_like(fr)
    post_b = np.zeros_like(fb)
    for i in range(19):
        cu = sum(C[i, a] * u[a] for a in range(3))
        feq = WT[i] * rho * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * uu)
        guo = (1 - 0.5 * omega) * WT[i] * sum((3 * (C[i, a] - u[a]) + 9 * cu * C[i, a]) * F[a] for a in range(3))
        if edm:
            v = u + F / rho
            cv = sum(C[i, a] * v[a] for a in range(3))
            guo = WT[i] * rho * (1 + 3 * cv + 4.5 * cv ** 2 - 1.5 * (v ** 2).sum(0)) - feq
        fs = ftot[i] - omega * (ftot[i] - feq) + guo
        cg = sum(C[i, a] * G[a] for a in range(3))
        fs = fs + np.where(aniso, A * (WT[i] * cg ** 2 / Gs - BB[i] * Gn), 0.0)
        r = (rr / rho) * fs
        if i > 0:
            r = r + np.where(aniso, beta * (rr * rb / rho) * WT[i] * cg / (np.sqrt((C[i] ** 2).sum()) * Gs), 0.0)
        post_r[i] = r
        post_b[i] = fs - r
    # streaming, push form: what leaves x along c_i lands on x + c_i, or comes back reversed
    new_r = np.zeros_like(fr)
    new_b = np.zeros_like(fb)
    for i in range(19):
        o = opposite(i)
        dest_solid = shift(solid, -C[i])          # is x + c_i solid?
        for post, new, rk in ((post_r, new_r, rr), (post_b, new_b, rb)):
            go = np.where(fluid & ~dest_solid, post[i], 0.0)
            new[i] += shift(go, C[i])
            back = post[i]
            if wall_group is not None:
                # moving wall (G28): the reflected population loses 6 w_i rho^k (c_i . u_w)
                grp = shift(wall_group, -C[i])            # group of the site x + c_i
                cuw = sum(C[i, a] * np.asarray(wall_u)[grp, a] for a in range(3))
                back = back - 6.0 * WT[i] * rk * cuw
            new[o] += np.where(fluid & dest_solid, back, 0.0)
    new_r *= fluid
    new_b *= fluid
    return new_r, new_b


def equilibrium(rho, u):
    """[19, nz, ny, nx] equilibrium of Eq. 2."""
    uu = (u ** 2).sum(0)
    out = []
    for i in range(19):
        cu = sum(C[i, a] * u[a] for a in range(3))
        out.append(WT[i] * rho * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * uu))
    return np.stack(out)


def step_sc(fr, fb, solid, tau_r, tau_b, G_C, g=(0.0, 0.0, 0.0), wall_group=None, wall_u=None):
    """One time step of the paper's section 3.1 as printed: Eq. 5-6 with the exact-difference
    source of Eq. 9 and the Shan-Chen force of Eq. 10, repulsive for G_C > 0
    (G27).  Whole-array form, push streaming."""
    fluid = ~solid
    rr = fr.sum(0)
    rb = fb.sum(0)
    rho = np.where(fluid, rr + rb, 1.0)
    m = np.stack([sum(C[i, a] * (fr[i] + fb[i]) for i in range(19)) for a in range(3)])
    u = m / rho
    # accelerations a^k = F^k / rho^k = -G_C sum_i w_i rho^kbar(x + c_i) c_i (+ g); a solid
    # neighbour contributes the centre value
    ar = np.zeros((3,) + rr.shape)
    ab = np.zeros((3,) + rr.shape)
    for i in range(1, 19):
        nb_solid = shift(solid, -C[i])                 # is x + c_i solid?
        pb = np.where(nb_solid, rb, shift(rb, -C[i]))  # rho^b(x + c_i)
        pr = np.where(nb_solid, rr, shift(rr, -C[i]))
        for a in range(3):
            ar[a] += -G_C * WT[i] * pb * C[i, a]
            ab[a] += -G_C * WT[i] * pr * C[i, a]
    for a in range(3):
        ar[a] += g[a]
        ab[a] += g[a]
    if tau_r == tau_b:
        omega = np.full(rho.shape, 1.0 / tau_r)
    else:
        nur, nub = (tau_r - 0.5) / 3, (tau_b - 0.5) / 3
        with np.errstate(divide="ignore", invalid="ignore"):
            omega = 1.0 / (3.0 / ((rr / rho) / nur + (rb / rho) / nub) + 0.5)
    post_r = (1 - omega) * fr + omega * equilibrium(rr, u) + equilibrium(rr, u + ar) - equilibrium(rr, u)
    post_b = (1 - omega) * fb + omega * equilibrium(rb, u) + equilibrium(rb, u + ab) - equilibrium(rb, u)
    new_r = np.zeros_like(fr)
    new_b = np.zeros_like(fb)
    for i in range(19):
        o = opposite(i)
        dest_solid = shift(solid, -C[i])
        for post, new, rk in ((post_r, new_r, rr), (post_b, new_b, rb)):
            go = np.where(fluid & ~dest_solid, post[i], 0.0)
            new[i] += shift(go, C[i])
            back = post[i]
            if wall_group is not None:
                # moving wall (G28): the reflected population loses 6 w_i rho^k (c_i . u_w)
                grp = shift(wall_group, -C[i])            # group of the site x + c_i
                cuw = sum(C[i, a] * np.asarray(wall_u)[grp, a] for a in range(3))
                back = back - 6.0 * WT[i] * rk * cuw
            new[o] += np.where(fluid & dest_solid, back, 0.0)
    new_r *= fluid
    new_b *= fluid
    return new_r, new_b
