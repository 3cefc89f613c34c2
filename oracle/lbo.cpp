// oracle/lbo.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, fp64 CPU oracle for the two-component colour-gradient D3Q19 lattice
// Boltzmann step with near-contact repulsion (arxiv 2005.12764).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
// It shares no code with the CUDA path (paper_2005_12764_b200/csrc) and neither includes
// the other.
//
// What it follows, step by step, in the paper's order (PAPER.md = /root/reference/PAPER.md):
//   S0 init         Eq. 2 per component with the common u
//   S1 moments      rho_k = sum_i f^k_i, m = sum_i c_i f_i         PAPER.md:96 (Eq. 3)
//   S2 gradient     G = 3 sum_i w_i c_i phi(x+c_i)                 stencil of Eq. 10
//   S3 near contact F_rep = -A_h[h] n delta_I                      PAPER.md:221-223 (Eq. 11)
//   S4 force, u     Guo half-force shift (north_star; S_i role PAPER.md:92); variant: exact
//                   difference, the paper's own Eq. 9, lbo_set_forcing(h, 1)
//   S5 omega_eff    Eq. 7-8, sign of Eq. 7 fixed by Eq. 4
//   S6 BGK + source Eq. 1 on the total f = f^r + f^b
//   S7 perturbation colour-gradient surface tension (north_star; not in the paper's text)
//   S8 recolouring  Latva-Kokko (north_star; not in the paper's text)
//   S9 streaming    exact shift + link-wise bounce-back
// Second model (lbo_set_model(h, 1, G_C)): the paper's section 3.1 as printed, Shan-Chen force
// (Eq. 10) with exact-difference forcing (Eq. 9) in Eq. 5-6; S1, S5, S9 are shared.
// Readings of everything the paper leaves open are G1-G24 of SURVEY.md section 8(c), restated
// in DESIGN.md.
//
// Pins (tests/test_oracle_*.py): P1 constants, P2 equilibrium fixed point, P3 mass, P4 momentum,
// P5 shear-wave viscosity (Eq. 4), P6 mixture viscosity (Eq. 8), P7 Poiseuille, P8 Laplace,
// P9 near-contact sign/size, P10 film table A_h(h), P11 lattice symmetry, P12 brute-force numpy
// twin, P13 Taylor-Green decay.
// P14 exact-difference forcing, P15 Couette flow between sliding walls (G28), P16 colour-exchange
// symmetry of the symmetric probe (G29), P17 wetting: symmetry, neutrality and monotone contact
// angle (G30), P18 open boundaries: plug flow fixed point, pressure-driven Poiseuille, mass balance
// (G31); SC1-SC5 for the second model; P20 interface width of the recolouring operator (closed form).
// Rigid particles (the paper's section 6; readings G32-G37 further down): PC1 exact
// momentum of fluid + particles, PC2 no force in a fluid at rest, PC3 leapfrog / quaternion closed
// forms, PC4 Stokes drag (Hasimoto), PC5 torque on a spinning sphere, PC6 pair force
// (tests/test_oracle_colloids.py).
// PARITY UNPINNED against the paper (pinned only against DESIGN.md's reading): the discrete
// contact search (G10), H_MAX, the wall rule for phi (G8, G30), the guard eps (G7).
//
// Deliberately nothing clever: loops over sites and over the 19 directions, two full
// population arrays, OpenMP on the outermost site loop only.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

namespace {

constexpr int Q = 19;
// Velocity order; the paper numbers i = 1..19 and fixes no order.
const int CX[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
const int CY[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
const int CZ[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
const int OPP[Q] = {0, 2, 1, 4, 3, 6, 5, 8, 7, 10, 9, 12, 11, 14, 13, 16, 15, 18, 17};
// "weights normalized to unity" PAPER.md:90; values are the standard D3Q19 ones (G2).
const double W[Q] = {1.0 / 3, 1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18,
                     1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36,
                     1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36};
// Perturbation constants B_i (G5): sum B_i = 1/3, sum B_i c_ia c_ib = delta_ab / 3.
const double B[Q] = {-1.0 / 3, 1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18,
                     1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36,
                     1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36};
constexpr double EPS_G = 1e-12;  // guard on |G| (G7)
constexpr int H_MIN = 3;         // "h_min = 3-4 lattice units" PAPER.md:223 (G10)
constexpr int H_MAX = 4;         // outer cut-off of the probe (G10)

struct Oracle {
  int nx = 0, ny = 0, nz = 0;
  size_t S = 0;
  double tau_r = 1, tau_b = 1, A = 0, beta = 0, A_nc = 0;
  double g[3] = {0, 0, 0};
  double phi_c = 0.9;
  int nc_mode = 0;  // 0 = probe (S3), 1 = test hook: every |phi|<phi_c site in contact with A_h = A_nc
  int nc_sym = 0;   // 1 = colour-symmetric probe (G29): the rule plus its image under r <-> b
  int wet = 0;      // 1 = prescribed phi at solid nodes (G30): a solid neighbour contributes phi_wall
  double phi_wall = 0.0;
  int model = 0;    // 0 = colour gradient (north_star), 1 = Shan-Chen, the paper's own Eq. 5-10
  double G_C = 0.0; // strength of the inter-component force of Eq. 10, positive = repulsive
  int forcing = 0;  // 0 = Guo (north_star; S4, S6), 1 = exact difference, the paper's own Eq. 9
  bool two = true;
  bool inited = false;
  bool any_solid = false;
  std::vector<uint8_t> solid;            // S, 0 = fluid, 1 = wall at rest, 2 / 3 / 4 = walls moving with uw[2] / uw[3] / uw[4],
                                         // 5 = node inside a rigid particle (NEXT-4; pid[s] says which)
  double uw[6][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}, {0, 0, 0}, {0, 0, 0}, {0, 0, 0}};   // wall velocities by group (G28); [5] stays 0
  int wtype[6] = {0, 0, 0, 0, 0, 0};     // group 2 / 3 / 4: 0 = moving wall, 1 = velocity inlet, 2 = reservoir, 3 = pressure outlet (G31)
  double wrho[6][2] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}, {0, 0}, {0, 0}};     // prescribed rho_r, rho_b of an inlet / outlet
  std::vector<double> uex, uey, uez;     // velocity that entered f^eq in the last collision (outlet rule, G31)
  std::vector<double> f[2], fpost[2];    // [k][site*19 + i], pre- and post-collision
  std::vector<double> rho_r, rho_b, phi; // per site (S1)
  std::vector<double> mx, my, mz;        // bare momentum (S1)
  std::vector<double> Fx, Fy, Fz;        // total force of the last evaluation (S4)
  std::vector<double> Gx, Gy, Gz;        // colour gradient of the last evaluation (S2)
  std::vector<int> hcontact;             // contact distance found by the probe, 0 = none
  std::vector<double> margin;            // smallest margin of any discrete decision (G12)
  std::string err;
  // ---- rigid spherical particles (the paper's section 6; readings G32-G37 below)
  struct Particle {
    double r[3], u[3], w[3], q[4];   // centre, velocity, angular velocity, orientation quaternion (w, x, y, z)
    double R, mass, inertia;         // radius, m_p, I_p = 2/5 m_p R^2 (solid sphere)
    double F[3], T[3];               // force and torque from the fluid links of the last step
    double Fext[3], Text[3];         // constant external force / torque
    double Fpp[3];                   // inter-particle force of the last step
  };
  std::vector<Particle> parts;
  std::vector<int> pid;              // S, particle index of a particle node, else -1
  int p_mobile = 1;                  // 0: particles are held (infinite inertia): links exchange momentum, nothing moves
  double p_K = 0.0, p_hc = 0.0;      // soft repulsion K (h_c - h)^(3/2) for gaps h < h_c (G37)
  int p_lub = 0;                     // 1: normal lubrication force for gaps h < h_c (G37)

  size_t idx(int x, int y, int z) const { return (size_t)x + (size_t)nx * ((size_t)y + (size_t)ny * (size_t)z); }
  static int wrap(int a, int n) {  // periodic image; loops so that boxes with n = 1 work (G22)
    while (a < 0) a += n;
    while (a >= n) a -= n;
    return a;
  }
  size_t nbr(int x, int y, int z, int dx, int dy, int dz) const {
    return idx(wrap(x + dx, nx), wrap(y + dy, ny), wrap(z + dz, nz));
  }
};

double feq(int i, double rho, double ux, double uy, double uz) {
  // Eq. 2 PAPER.md:87-90 with c_s^2 = 1/3: w_i rho (1 + 3 c.u + 4.5 (c.u)^2 - 1.5 u.u)
  double cu = CX[i] * ux + CY[i] * uy + CZ[i] * uz;
  double uu = ux * ux + uy * uy + uz * uz;
  return W[i] * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * uu);
}

// S1 for every fluid site.
void moments(Oracle& o) {
  const size_t S = o.S;
#pragma omp parallel for schedule(static)
  for (long long sll = 0; sll < (long long)S; ++sll) {
    size_t s = (size_t)sll;
    if (o.solid[s]) {
      o.rho_r[s] = o.rho_b[s] = o.phi[s] = 0.0;
      o.mx[s] = o.my[s] = o.mz[s] = 0.0;
      continue;
    }
    double rr = 0, rb = 0, mx = 0, my = 0, mz = 0;
    for (int i = 0; i < Q; ++i) {
      double fr = o.f[0][s * Q + i];
      double fb = o.two ? o.f[1][s * Q + i] : 0.0;
      rr += fr;
      rb += fb;
      mx += CX[i] * (fr + fb);
      my += CY[i] * (fr + fb);
      mz += CZ[i] * (fr + fb);
    }
    o.rho_r[s] = rr;
    o.rho_b[s] = rb;
    o.phi[s] = (rr - rb) / (rr + rb);
    o.mx[s] = mx;
    o.my[s] = my;
    o.mz[s] = mz;
  }
}

// S2-S4 at one fluid site: gradient, near-contact force, total force. Returns via refs.
void force_at(Oracle& o, int x, int y, int z, double& Gx, double& Gy, double& Gz, double& Fx,
              double& Fy, double& Fz) {
  const size_t s = o.idx(x, y, z);
  const double rho = o.rho_r[s] + o.rho_b[s];
  Gx = Gy = Gz = 0.0;
  double Fncx = 0, Fncy = 0, Fncz = 0;
  int hfound = 0;
  double marg = 1e300;
  if (o.two) {
    const double phi0 = o.phi[s];
    // S2: G = 3 sum_{i>=1} w_i c_i phi~(x+c_i); a solid neighbour contributes phi(x) (G8), or
    // the prescribed wall value phi_wall when wetting is on (G30).
    for (int i = 1; i < Q; ++i) {
      size_t n = o.nbr(x, y, z, CX[i], CY[i], CZ[i]);
      double p = o.solid[n] ? (o.wet ? o.phi_wall : phi0) : o.phi[n];
      Gx += 3.0 * W[i] * CX[i] * p;
      Gy += 3.0 * W[i] * CY[i] * p;
      Gz += 3.0 * W[i] * CZ[i] * p;
    }
    const double Gn = std::sqrt(Gx * Gx + Gy * Gy + Gz * Gz);
    // S3: near-contact force, Eq. 11 PAPER.md:221 with delta_I = |G|/2 (G9), n = -G/|G| (G10).
    if (o.A_nc != 0.0) {
      marg = std::fabs(std::fabs(phi0) - o.phi_c);
      if (std::fabs(phi0) < o.phi_c && Gn > EPS_G) {
        double Ah = 0.0;
        if (o.nc_mode == 1) {
          Ah = o.A_nc;
          hfound = 1;
        } else {
          const double n[3] = {-Gx / Gn, -Gy / Gn, -Gz / Gn};
          for (int k = 1; k <= H_MAX; ++k) {
            int d[3];
            for (int a = 0; a < 3; ++a) {
              double v = k * n[a];
              d[a] = (int)std::lround(v);  // round half away from zero
              double fr = std::fabs(v) - std::floor(std::fabs(v));
              marg = std::fmin(marg, std::fabs(fr - 0.5));
            }
            size_t p = o.nbr(x, y, z, d[0], d[1], d[2]);
            if (o.solid[p]) break;  // wall in the way: no contact
            if (k >= 2) {
              marg = std::fmin(marg, std::fabs(o.phi[p] - phi0));
              if (o.phi[p] >= phi0) {
                hfound = k;
                break;
              }
            }
          }
          if (hfound > 0) {
            // A_h = A for h <= h_min, decays as h^-3 beyond.
            Ah = hfound <= H_MIN ? o.A_nc
                                 : o.A_nc * std::pow((double)H_MIN / (double)hfound, 3.0);
          }
          if (o.nc_sym) {
            // G29: Fig. 5 is symmetric in the two fluids.  The image of the rule
            // above under r <-> b (phi -> -phi, G -> -G): march along +G/|G| and stop at the first
            // k >= 2 with phi(probe) <= phi(x) (two blue interfaces across a red film); its force
            // is -A_h(h+) G / 2.  Both are applied: F = (A_h(h-) - A_h(h+)) G / 2.
            int hplus = 0;
            for (int k = 1; k <= H_MAX; ++k) {
              int d[3];
              for (int a = 0; a < 3; ++a) {
                double v = -k * n[a];
                d[a] = (int)std::lround(v);
              }
              size_t p = o.nbr(x, y, z, d[0], d[1], d[2]);
              if (o.solid[p]) break;
              if (k >= 2) {
                marg = std::fmin(marg, std::fabs(o.phi[p] - phi0));
                if (o.phi[p] <= phi0) {
                  hplus = k;
                  break;
                }
              }
            }
            if (hplus > 0) {
              Ah -= hplus <= H_MIN ? o.A_nc : o.A_nc * std::pow((double)H_MIN / (double)hplus, 3.0);
              hfound |= hplus << 4;   // reported as h- + 16 h+
            }
          }
        }
        // -A_h n delta_I = -A_h (-G/|G|) (|G|/2) = +A_h G / 2
        Fncx = 0.5 * Ah * Gx;
        Fncy = 0.5 * Ah * Gy;
        Fncz = 0.5 * Ah * Gz;
      }
    }
  }
  // S4: F = rho g + F_nc (G13).
  Fx = rho * o.g[0] + Fncx;
  Fy = rho * o.g[1] + Fncy;
  Fz = rho * o.g[2] + Fncz;
  o.Gx[s] = Gx; o.Gy[s] = Gy; o.Gz[s] = Gz;
  o.Fx[s] = Fx; o.Fy[s] = Fy; o.Fz[s] = Fz;
  o.hcontact[s] = hfound;
  o.margin[s] = marg;
}

// S5-S8 at one fluid site; writes fpost.
void collide_at(Oracle& o, int x, int y, int z) {
  const size_t S = o.S;
  const size_t s = o.idx(x, y, z);
  double Gx, Gy, Gz, Fx, Fy, Fz;
  force_at(o, x, y, z, Gx, Gy, Gz, Fx, Fy, Fz);
  const double rr = o.rho_r[s], rb = o.rho_b[s];
  const double rho = rr + rb;
  // S4: u = (m + F/2)/rho with Guo forcing.  With exact-difference forcing (Eq. 9)
  // the equilibrium is taken at the bare velocity m/rho (Eq. 3) and the source is
  // f^eq(rho, u + F dt/rho) - f^eq(rho, u), dt = 1.
  const bool edm = o.forcing == 1;
  const double hs = edm ? 0.0 : 0.5;
  const double ux = (o.mx[s] + hs * Fx) / rho;
  const double uy = (o.my[s] + hs * Fy) / rho;
  const double uz = (o.mz[s] + hs * Fz) / rho;
  o.uex[s] = ux; o.uey[s] = uy; o.uez[s] = uz;
  // S5: relaxation rate. Eq. 8, then omega = 1/(3 nu + 1/2) which is Eq. 4
  // PAPER.md:102 inverted (the minus sign printed in Eq. 7 contradicts Eq. 4: G1).
  double omega;
  if (!o.two || o.tau_r == o.tau_b) {
    omega = 1.0 / o.tau_r;
  } else {
    double nu_r = (o.tau_r - 0.5) / 3.0, nu_b = (o.tau_b - 0.5) / 3.0;
    double inv_nu = (rr / rho) / nu_r + (rb / rho) / nu_b;
    double nu = 1.0 / inv_nu;
    omega = 1.0 / (3.0 * nu + 0.5);
  }
  const double Gn = std::sqrt(Gx * Gx + Gy * Gy + Gz * Gz);
  const bool aniso = o.two && Gn > EPS_G;
  double fstar[Q];
  for (int i = 0; i < Q; ++i) {
    // S6: collide the total (G3), Eq. 1 PAPER.md:78 with S_i the Guo term (G4).
    double fi = o.f[0][s * Q + i] + (o.two ? o.f[1][s * Q + i] : 0.0);
    double fe = feq(i, rho, ux, uy, uz);
    double cu = CX[i] * ux + CY[i] * uy + CZ[i] * uz;
    double sx = 3.0 * (CX[i] - ux) + 9.0 * cu * CX[i];
    double sy = 3.0 * (CY[i] - uy) + 9.0 * cu * CY[i];
    double sz = 3.0 * (CZ[i] - uz) + 9.0 * cu * CZ[i];
    double guo = (1.0 - 0.5 * omega) * W[i] * (sx * Fx + sy * Fy + sz * Fz);
    if (edm) guo = feq(i, rho, ux + Fx / rho, uy + Fy / rho, uz + Fz / rho) - fe;   // Eq. 9
    double v = fi - omega * (fi - fe) + guo;
    // S7: colour-gradient perturbation (G5).
    if (aniso) {
      double cg = CX[i] * Gx + CY[i] * Gy + CZ[i] * Gz;
      v += o.A * (W[i] * cg * cg / Gn - B[i] * Gn);
    }
    fstar[i] = v;
  }
  if (!o.two) {
    for (int i = 0; i < Q; ++i) o.fpost[0][s * Q + i] = fstar[i];
    return;
  }
  // S8: Latva-Kokko recolouring (G6); blue by subtraction so that f^r + f^b = f* exactly.
  for (int i = 0; i < Q; ++i) {
    double fr = (rr / rho) * fstar[i];
    if (aniso && i > 0) {
      double cg = CX[i] * Gx + CY[i] * Gy + CZ[i] * Gz;
      double cnorm = std::sqrt((double)(CX[i] * CX[i] + CY[i] * CY[i] + CZ[i] * CZ[i]));
      fr += o.beta * (rr * rb / rho) * W[i] * cg / (cnorm * Gn);
    }
    o.fpost[0][s * Q + i] = fr;
    o.fpost[1][s * Q + i] = fstar[i] - fr;
  }
}

// S9: f^k_i(x,t+1) = f^k*_i(x-c_i) if x-c_i is fluid, else f^k*_opp(i)(x) (G21).
void stream(Oracle& o) {
  const size_t S = o.S;
  const int nk = o.two ? 2 : 1;
#pragma omp parallel for schedule(static)
  for (int z = 0; z < o.nz; ++z)
    for (int y = 0; y < o.ny; ++y)
      for (int x = 0; x < o.nx; ++x) {
        size_t s = o.idx(x, y, z);
        if (o.solid[s]) continue;
        for (int i = 0; i < Q; ++i) {
          size_t n = o.nbr(x, y, z, -CX[i], -CY[i], -CZ[i]);
          for (int k = 0; k < nk; ++k) {
            if (!o.solid[n]) {
              o.f[k][s * Q + i] = o.fpost[k][n * Q + i];
            } else {
              // half-way bounce-back at a wall moving with u_w ("solid walls with opposite speeds
              // +-U"; rule: reading G28): the reflected population gains
              // 2 w_i rho^k (c_i . u_w) / c_s^2 = 6 w_i rho^k (c_i . u_w), rho^k the site's density
              const int g = o.solid[n];
              const double* uw = o.uw[g];
              const double cu = CX[i] * uw[0] + CY[i] * uw[1] + CZ[i] * uw[2];
              if (o.wtype[g] >= 2) {
                // open boundaries (G31; the flow focuser's outlet, rule not given):
                // pressure outlet by anti-bounce-back,
                // f^k_i(x, t+1) = -f^k*_opp(i)(x, t) + 2 w_i rho^k_out [1 + 4.5 (c_i.u)^2 - 1.5 u.u],
                // u = the velocity that entered f^eq at x in this step
                const double vx = o.uex[s], vy = o.uey[s], vz = o.uez[s];
                const double cv = CX[i] * vx + CY[i] * vy + CZ[i] * vz;
                const double E = 1.0 + 4.5 * cv * cv - 1.5 * (vx * vx + vy * vy + vz * vz);
                // type 2 (reservoir): rho^k_out as prescribed.  Type 3 (outflow): only the total is
                // prescribed, the composition is the boundary node's own,
                // rho^k_out = (rho_r + rho_b)_prescribed rho^k(x) / rho(x)
                double rk_out = o.wrho[g][k];
                if (o.wtype[g] == 3) {
                  const double rk = k == 0 ? o.rho_r[s] : o.rho_b[s];
                  const double rho = o.two ? o.rho_r[s] + o.rho_b[s] : o.rho_r[s];
                  rk_out = (o.wrho[g][0] + o.wrho[g][1]) * rk / rho;
                }
                o.f[k][s * Q + i] = -o.fpost[k][s * Q + OPP[i]] + 2.0 * W[i] * rk_out * E;
              } else {
                // type 1, velocity inlet: the same rule with the prescribed densities of the
                // incoming fluid in place of the site's own (G31)
                const double rk = o.wtype[g] == 1 ? o.wrho[g][k] : (k == 0 ? o.rho_r[s] : o.rho_b[s]);
                o.f[k][s * Q + i] = o.fpost[k][s * Q + OPP[i]] + 6.0 * W[i] * rk * cu;
              }
            }
          }
        }
      }
}

// ---- Shan-Chen model, the paper's section 3.1 as printed (model = 1) --------------------------
// Eq. 10: F^r(x) = rho^r(x) G_C sum_i w_i rho^b(x + c_i) c_i, and the same with r, b
// swapped.  "G_C ... takes positive values for repulsive interactions", which needs a
// minus sign in front (reading G27 in DESIGN.md): a^k = F^k / rho^k = -G_C sum_i w_i rho^kbar(x + c_i) c_i.
// A solid neighbour contributes the centre value (neutral wall, as G8).  The body acceleration g is
// added to both.  Returns the accelerations a^r, a^b.
void sc_accel_at(const Oracle& o, int x, int y, int z, double ar[3], double ab[3]) {
  const size_t s = o.idx(x, y, z);
  for (int a = 0; a < 3; ++a) ar[a] = ab[a] = 0.0;
  for (int i = 1; i < Q; ++i) {
    size_t n = o.nbr(x, y, z, CX[i], CY[i], CZ[i]);
    const double pb = o.solid[n] ? o.rho_b[s] : o.rho_b[n];
    const double pr = o.solid[n] ? o.rho_r[s] : o.rho_r[n];
    const int c[3] = {CX[i], CY[i], CZ[i]};
    for (int a = 0; a < 3; ++a) {
      ar[a] += -o.G_C * W[i] * pb * c[a];
      ab[a] += -o.G_C * W[i] * pr * c[a];
    }
  }
  for (int a = 0; a < 3; ++a) { ar[a] += o.g[a]; ab[a] += o.g[a]; }
}

// Eq. 5-9 at one fluid site: each component relaxes to f^eq(rho^k, u) with the
// common bare velocity u = m / rho (Eq. 3) and the common omega_eff (Eq. 7-8, sign G1), plus the
// exact-difference source S^k_i = f^eq_i(rho^k, u + F^k dt / rho^k) - f^eq_i(rho^k, u), dt = 1.
void collide_sc_at(Oracle& o, int x, int y, int z) {
  const size_t s = o.idx(x, y, z);
  double ar[3], ab[3];
  sc_accel_at(o, x, y, z, ar, ab);
  const double rr = o.rho_r[s], rb = o.rho_b[s], rho = rr + rb;
  o.Fx[s] = rr * ar[0] + rb * ab[0];   // total force, for the velocity that get_macros returns
  o.Fy[s] = rr * ar[1] + rb * ab[1];
  o.Fz[s] = rr * ar[2] + rb * ab[2];
  const double ux = o.mx[s] / rho, uy = o.my[s] / rho, uz = o.mz[s] / rho;
  o.uex[s] = ux; o.uey[s] = uy; o.uez[s] = uz;
  double omega;
  if (o.tau_r == o.tau_b) {
    omega = 1.0 / o.tau_r;
  } else {
    double nu_r = (o.tau_r - 0.5) / 3.0, nu_b = (o.tau_b - 0.5) / 3.0;
    double nu = 1.0 / ((rr / rho) / nu_r + (rb / rho) / nu_b);
    omega = 1.0 / (3.0 * nu + 0.5);
  }
  for (int i = 0; i < Q; ++i) {
    const double fer = feq(i, rr, ux, uy, uz), feb = feq(i, rb, ux, uy, uz);
    const double Sr = feq(i, rr, ux + ar[0], uy + ar[1], uz + ar[2]) - fer;
    const double Sb = feq(i, rb, ux + ab[0], uy + ab[1], uz + ab[2]) - feb;
    o.fpost[0][s * Q + i] = (1.0 - omega) * o.f[0][s * Q + i] + omega * fer + Sr;
    o.fpost[1][s * Q + i] = (1.0 - omega) * o.f[1][s * Q + i] + omega * feb + Sb;
  }
}

// ---- Rigid particles: the paper's section 6 ------------------------------
// "colloidal particles are represented as rigid spheres of radius R, moving under the effect of a
// total force F_p and torque T_p ... Newton's equations of motion (Eq. 15) ... solved by a leapfrog
// approach, using quaternion algebra for the rotational component".  How the
// fluid acts on a particle is only cited (refs [61, 62], Ladd).  Readings (G32-G37):
//  G32 nodes: a lattice node x belongs to particle p if |x - r_p| < R_p (minimum image).  A link
//      from a fluid node s along c_j into such a node meets the surface at its midpoint
//      x_b = s + c_j / 2, which moves with u_b = u_p + w_p x (x_b - r_p).
//  G33 link rule, applied right after the collision with the node map of time t: the population
//      that leaves s towards the particle is stored as what comes back,
//      g^k_j(s) = f^k*_j(s) - 6 w_j rho^k(s) (c_j . u_b)   (half-way bounce-back at a moving wall, as
//      G28; rho^k the component's density at s), and the particle receives the momentum
//      dP = sum_k (f^k*_j + g^k_j) c_j and the torque (x_b - r_p) x dP.
//  G35 Eq. 15 by leapfrog: u_p += (F_p + F_pp + F_ext)/m_p, r_p += u_p, w_p += (T_p + T_ext)/I_p,
//      q <- dq(w_p) q with dq the rotation by the angle |w_p| about w_p (unit time step).
//  G36 node changes after the move.  A node that leaves the particle is filled with the equilibrium
//      (Eq. 2) at the mean densities of its fluid neighbours and the surface velocity there; what it
//      holds is taken from the particle's momentum.  A node that enters the particle gives its
//      populations' momentum to the particle.  Links whose far end changed are put right so that
//      momentum is conserved exactly: a link into a node that is fluid now gets its population
//      f^k*_j back (the exchange of G33 is undone); a link into a node that is solid now is
//      reflected by G33 with the particle's new state.  Streaming then uses the new node map.
//  G37 particle-particle forces ("including the lubrication term", forms not given): for a
//      gap h = |r_ij| - R_i - R_j < h_c a repulsion K (h_c - h)^(3/2) along the line of centres and,
//      if switched on, the normal lubrication force -6 pi mu R_eff^2 (1/h - 1/h_c) (u_ij . n) n with
//      R_eff = R_i R_j / (R_i + R_j), mu = rho_0 nu, rho_0 = 1, nu from tau_r; h is floored at 0.1.
double min_image(double d, int n) { return d - n * std::floor(d / n + 0.5); }

void cross(const double a[3], const double b[3], double c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

bool inside_particle(const Oracle& o, const Oracle::Particle& P, int x, int y, int z) {
  const double d[3] = {min_image(x - P.r[0], o.nx), min_image(y - P.r[1], o.ny), min_image(z - P.r[2], o.nz)};
  return d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < P.R * P.R;
}

// loop over the lattice nodes of the box [r - R - m, r + R + m] (wrapped)
template <class Fn>
void for_box(const Oracle& o, const double r[3], double reach, Fn fn) {
  int lo[3], hi[3];
  const int n[3] = {o.nx, o.ny, o.nz};
  for (int a = 0; a < 3; ++a) {
    lo[a] = (int)std::floor(r[a] - reach);
    hi[a] = (int)std::ceil(r[a] + reach);
    if (hi[a] - lo[a] + 1 > n[a]) { lo[a] = 0; hi[a] = n[a] - 1; }   // never visit a node twice
  }
  for (int z = lo[2]; z <= hi[2]; ++z)
    for (int y = lo[1]; y <= hi[1]; ++y)
      for (int x = lo[0]; x <= hi[0]; ++x) fn(Oracle::wrap(x, o.nx), Oracle::wrap(y, o.ny), Oracle::wrap(z, o.nz));
}

// G32: mark the particle nodes (solid = 5, pid = p).  Walls keep their nodes.
void rasterize(Oracle& o) {
  for (size_t s = 0; s < o.S; ++s) {
    if (o.solid[s] == 5) o.solid[s] = 0;
    o.pid[s] = -1;
  }
  for (size_t p = 0; p < o.parts.size(); ++p)
    for_box(o, o.parts[p].r, o.parts[p].R + 1.0, [&](int x, int y, int z) {
      const size_t s = o.idx(x, y, z);
      if (o.solid[s] == 0 && inside_particle(o, o.parts[p], x, y, z)) { o.solid[s] = 5; o.pid[s] = (int)p; }
    });
}

// surface velocity of particle P at the point r_p + rel
void surface_velocity(const Oracle::Particle& P, const double rel[3], double ub[3]) {
  double wxr[3];
  cross(P.w, rel, wxr);
  for (int a = 0; a < 3; ++a) ub[a] = P.u[a] + wxr[a];
}

// G33 on one link: fluid node s = (x, y, z), direction j into a node of particle P (state P).
// Replaces fpost_j(s) by the reflected value and returns the momentum dP given to the particle.
void reflect_link(Oracle& o, const Oracle::Particle& P, int x, int y, int z, int j, double dP[3], double rel[3]) {
  const size_t s = o.idx(x, y, z);
  rel[0] = min_image(x - P.r[0], o.nx) + 0.5 * CX[j];
  rel[1] = min_image(y - P.r[1], o.ny) + 0.5 * CY[j];
  rel[2] = min_image(z - P.r[2], o.nz) + 0.5 * CZ[j];
  double ub[3];
  surface_velocity(P, rel, ub);
  const double cu = CX[j] * ub[0] + CY[j] * ub[1] + CZ[j] * ub[2];
  double tot = 0.0;
  for (int k = 0; k < (o.two ? 2 : 1); ++k) {
    const double rk = k == 0 ? o.rho_r[s] : o.rho_b[s];
    const double fp = o.fpost[k][s * Q + j];
    const double g = fp - 6.0 * W[j] * rk * cu;
    o.fpost[k][s * Q + j] = g;
    tot += fp + g;
  }
  dP[0] = tot * CX[j]; dP[1] = tot * CY[j]; dP[2] = tot * CZ[j];
}

// G33 for every link into a particle node, with the node map and the particle state of time t
void particle_links(Oracle& o) {
  for (size_t p = 0; p < o.parts.size(); ++p) {
    Oracle::Particle& P = o.parts[p];
    for (int a = 0; a < 3; ++a) P.F[a] = P.T[a] = 0.0;
    for_box(o, P.r, P.R + 2.0, [&](int x, int y, int z) {
      const size_t s = o.idx(x, y, z);
      if (o.solid[s]) return;
      for (int j = 1; j < Q; ++j) {
        const size_t n = o.nbr(x, y, z, CX[j], CY[j], CZ[j]);
        if (o.solid[n] != 5 || o.pid[n] != (int)p) continue;
        double dP[3], rel[3], t[3];
        reflect_link(o, P, x, y, z, j, dP, rel);
        cross(rel, dP, t);
        for (int a = 0; a < 3; ++a) { P.F[a] += dP[a]; P.T[a] += t[a]; }
      }
    });
  }
}

// G37
void interparticle(Oracle& o) {
  const size_t N = o.parts.size();
  for (size_t p = 0; p < N; ++p) for (int a = 0; a < 3; ++a) o.parts[p].Fpp[a] = 0.0;
  if (o.p_hc <= 0.0) return;
  const double mu = (o.tau_r - 0.5) / 3.0;   // rho_0 nu with rho_0 = 1
  for (size_t p = 0; p < N; ++p)
    for (size_t q = p + 1; q < N; ++q) {
      Oracle::Particle &A = o.parts[p], &Bq = o.parts[q];
      const double d[3] = {min_image(A.r[0] - Bq.r[0], o.nx), min_image(A.r[1] - Bq.r[1], o.ny), min_image(A.r[2] - Bq.r[2], o.nz)};
      const double dist = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
      double h = dist - A.R - Bq.R;
      if (h >= o.p_hc) continue;
      const double n[3] = {d[0] / dist, d[1] / dist, d[2] / dist};   // from q to p
      double f = o.p_K * std::pow(o.p_hc - h, 1.5);
      if (o.p_lub) {
        const double hh = h < 0.1 ? 0.1 : h;
        const double Reff = A.R * Bq.R / (A.R + Bq.R);
        const double un = (A.u[0] - Bq.u[0]) * n[0] + (A.u[1] - Bq.u[1]) * n[1] + (A.u[2] - Bq.u[2]) * n[2];
        f += -6.0 * M_PI * mu * Reff * Reff * (1.0 / hh - 1.0 / o.p_hc) * un;
      }
      for (int a = 0; a < 3; ++a) { A.Fpp[a] += f * n[a]; Bq.Fpp[a] -= f * n[a]; }
    }
}

// G35
void integrate(Oracle& o) {
  const int n[3] = {o.nx, o.ny, o.nz};
  for (auto& P : o.parts) {
    for (int a = 0; a < 3; ++a) {
      P.u[a] += (P.F[a] + P.Fpp[a] + P.Fext[a]) / P.mass;
      P.w[a] += (P.T[a] + P.Text[a]) / P.inertia;
      P.r[a] += P.u[a];
      P.r[a] -= n[a] * std::floor(P.r[a] / n[a]);
    }
    const double th = std::sqrt(P.w[0] * P.w[0] + P.w[1] * P.w[1] + P.w[2] * P.w[2]);
    if (th > 0.0) {
      const double sh = std::sin(0.5 * th) / th, ch = std::cos(0.5 * th);
      const double d[4] = {ch, sh * P.w[0], sh * P.w[1], sh * P.w[2]};
      const double* q = P.q;
      double r[4] = {d[0] * q[0] - d[1] * q[1] - d[2] * q[2] - d[3] * q[3],
                     d[0] * q[1] + d[1] * q[0] + d[2] * q[3] - d[3] * q[2],
                     d[0] * q[2] - d[1] * q[3] + d[2] * q[0] + d[3] * q[1],
                     d[0] * q[3] + d[1] * q[2] - d[2] * q[1] + d[3] * q[0]};
      const double nr = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + r[3] * r[3]);
      for (int a = 0; a < 4; ++a) P.q[a] = r[a] / nr;
    }
  }
}

// G36: node changes of particle p after its move from `old` to the current state
void remap_particle(Oracle& o, size_t p, const Oracle::Particle& old) {
  Oracle::Particle& P = o.parts[p];
  struct Node { int x, y, z; };
  std::vector<Node> covered, uncovered;
  for_box(o, P.r, P.R + 2.0, [&](int x, int y, int z) {
    const size_t s = o.idx(x, y, z);
    const bool was = o.solid[s] == 5 && o.pid[s] == (int)p;
    const bool now = inside_particle(o, P, x, y, z) && (was || o.solid[s] == 0);
    if (was && !now) uncovered.push_back({x, y, z});
    if (!was && now) covered.push_back({x, y, z});
  });
  const int nk = o.two ? 2 : 1;
  double dU[3] = {0, 0, 0}, dL[3] = {0, 0, 0};     // impulses: momentum and angular momentum
  auto is_new_cover = [&](size_t s) {
    for (const Node& c : covered) if (o.idx(c.x, c.y, c.z) == s) return true;
    return false;
  };
  auto give = [&](const double mom[3], const double rel[3], double sign) {
    double t[3];
    cross(rel, mom, t);
    for (int a = 0; a < 3; ++a) { dU[a] += sign * mom[a]; dL[a] += sign * t[a]; }
  };
  // nodes that leave the particle
  for (const Node& c : uncovered) {
    const size_t s = o.idx(c.x, c.y, c.z);
    double rk[2] = {0, 0};
    int cnt = 0;
    for (int j = 1; j < Q; ++j) {
      const size_t m = o.nbr(c.x, c.y, c.z, CX[j], CY[j], CZ[j]);
      if (o.solid[m] || is_new_cover(m)) continue;
      rk[0] += o.rho_r[m]; rk[1] += o.rho_b[m];
      ++cnt;
    }
    if (cnt) { rk[0] /= cnt; rk[1] /= cnt; }
    else { rk[0] = o.two ? 0.5 : 1.0; rk[1] = o.two ? 0.5 : 0.0; }
    const double rel[3] = {min_image(c.x - P.r[0], o.nx), min_image(c.y - P.r[1], o.ny), min_image(c.z - P.r[2], o.nz)};
    double ub[3];
    surface_velocity(P, rel, ub);
    for (int k = 0; k < nk; ++k)
      for (int i = 0; i < Q; ++i) o.fpost[k][s * Q + i] = feq(i, rk[k], ub[0], ub[1], ub[2]);
    const double rho = rk[0] + (o.two ? rk[1] : 0.0);
    const double mom[3] = {rho * ub[0], rho * ub[1], rho * ub[2]};
    give(mom, rel, -1.0);
    o.rho_r[s] = rk[0]; o.rho_b[s] = o.two ? rk[1] : 0.0;      // the new node's densities, for the link rule
    // the new node's own links into the particle (as it stands now) are reflected by G33
    for (int j = 1; j < Q; ++j) {
      const int mx = Oracle::wrap(c.x + CX[j], o.nx), my = Oracle::wrap(c.y + CY[j], o.ny), mz = Oracle::wrap(c.z + CZ[j], o.nz);
      if (!inside_particle(o, P, mx, my, mz)) continue;
      const size_t m = o.idx(mx, my, mz);
      if (o.solid[m] != 0 && !(o.solid[m] == 5 && o.pid[m] == (int)p)) continue;   // a wall's or another particle's node
      double dP[3], relb[3];
      reflect_link(o, P, c.x, c.y, c.z, j, dP, relb);
      give(dP, relb, +1.0);
    }
    // links of fluid neighbours into this node: the exchange of G33 is undone
    for (int j = 1; j < Q; ++j) {
      const int sx = Oracle::wrap(c.x - CX[j], o.nx), sy = Oracle::wrap(c.y - CY[j], o.ny), sz = Oracle::wrap(c.z - CZ[j], o.nz);
      const size_t t = o.idx(sx, sy, sz);
      if (o.solid[t] || is_new_cover(t)) continue;
      double relb[3] = {min_image(sx - old.r[0], o.nx) + 0.5 * CX[j], min_image(sy - old.r[1], o.ny) + 0.5 * CY[j],
                        min_image(sz - old.r[2], o.nz) + 0.5 * CZ[j]};
      double ubo[3];
      surface_velocity(old, relb, ubo);
      const double cu = CX[j] * ubo[0] + CY[j] * ubo[1] + CZ[j] * ubo[2];
      double tot = 0.0;
      for (int k = 0; k < nk; ++k) {
        const double rkk = k == 0 ? o.rho_r[t] : o.rho_b[t];
        const double g = o.fpost[k][t * Q + j];
        const double fp = g + 6.0 * W[j] * rkk * cu;
        o.fpost[k][t * Q + j] = fp;
        tot += fp + g;
      }
      const double dP[3] = {tot * CX[j], tot * CY[j], tot * CZ[j]};
      give(dP, relb, -1.0);
    }
  }
  // nodes that enter the particle
  for (const Node& c : covered) {
    const size_t s = o.idx(c.x, c.y, c.z);
    // What the node holds: fpost_i is the population that would be at the neighbour along c_i after
    // streaming, or, where that neighbour is solid, back at this node moving along -c_i (for a link
    // into the particle the stored value is already the reflected one, G33).
    double mom[3] = {0, 0, 0};
    for (int i = 0; i < Q; ++i) {
      const double sgn = o.solid[o.nbr(c.x, c.y, c.z, CX[i], CY[i], CZ[i])] ? -1.0 : 1.0;
      for (int k = 0; k < nk; ++k) {
        const double v = sgn * o.fpost[k][s * Q + i];
        mom[0] += v * CX[i]; mom[1] += v * CY[i]; mom[2] += v * CZ[i];
      }
    }
    const double rel[3] = {min_image(c.x - P.r[0], o.nx), min_image(c.y - P.r[1], o.ny), min_image(c.z - P.r[2], o.nz)};
    give(mom, rel, +1.0);
    for (int j = 1; j < Q; ++j) {
      const int sx = Oracle::wrap(c.x - CX[j], o.nx), sy = Oracle::wrap(c.y - CY[j], o.ny), sz = Oracle::wrap(c.z - CZ[j], o.nz);
      const size_t t = o.idx(sx, sy, sz);
      if (o.solid[t] || is_new_cover(t)) continue;
      double dP[3], relb[3];
      reflect_link(o, P, sx, sy, sz, j, dP, relb);
      give(dP, relb, +1.0);
    }
  }
  for (int a = 0; a < 3; ++a) { P.u[a] += dU[a] / P.mass; P.w[a] += dL[a] / P.inertia; }
  for (const Node& c : uncovered) { const size_t s = o.idx(c.x, c.y, c.z); o.solid[s] = 0; o.pid[s] = -1; }
  for (const Node& c : covered) { const size_t s = o.idx(c.x, c.y, c.z); o.solid[s] = 5; o.pid[s] = (int)p; }
}

// the particle part of a step, between collision and streaming
void particle_step(Oracle& o) {
  particle_links(o);
  if (!o.p_mobile) return;
  interparticle(o);
  std::vector<Oracle::Particle> old = o.parts;
  integrate(o);
  for (size_t p = 0; p < o.parts.size(); ++p) remap_particle(o, p, old[p]);
}

void one_step(Oracle& o) {
  moments(o);
  if (o.model == 1) {
#pragma omp parallel for schedule(static)
    for (int z = 0; z < o.nz; ++z)
      for (int y = 0; y < o.ny; ++y)
        for (int x = 0; x < o.nx; ++x)
          if (!o.solid[o.idx(x, y, z)]) collide_sc_at(o, x, y, z);
    stream(o);
    return;
  }
#pragma omp parallel for schedule(static)
  for (int z = 0; z < o.nz; ++z)
    for (int y = 0; y < o.ny; ++y)
      for (int x = 0; x < o.nx; ++x)
        if (!o.solid[o.idx(x, y, z)]) collide_at(o, x, y, z);
  if (!o.parts.empty()) particle_step(o);   // links (G33), Eq. 15 (G35), node changes (G36)
  stream(o);
}

void eval_forces(Oracle& o) {
  moments(o);
#pragma omp parallel for schedule(static)
  for (int z = 0; z < o.nz; ++z)
    for (int y = 0; y < o.ny; ++y)
      for (int x = 0; x < o.nx; ++x) {
        size_t s = o.idx(x, y, z);
        if (o.solid[s]) {
          o.Fx[s] = o.Fy[s] = o.Fz[s] = 0;
          o.Gx[s] = o.Gy[s] = o.Gz[s] = 0;
          o.hcontact[s] = 0;
          o.margin[s] = 1e300;
          continue;
        }
        if (o.model == 1) {
          double ar[3], ab[3];
          sc_accel_at(o, x, y, z, ar, ab);
          o.Fx[s] = o.rho_r[s] * ar[0] + o.rho_b[s] * ab[0];
          o.Fy[s] = o.rho_r[s] * ar[1] + o.rho_b[s] * ab[1];
          o.Fz[s] = o.rho_r[s] * ar[2] + o.rho_b[s] * ab[2];
          o.Gx[s] = o.Gy[s] = o.Gz[s] = 0;
          o.hcontact[s] = 0;
          o.margin[s] = 1e300;
          continue;
        }
        double a, b, c, d, e, f;
        force_at(o, x, y, z, a, b, c, d, e, f);
      }
}

}  // namespace

extern "C" {

enum { LBO_OK = 0, LBO_EINVAL = -1, LBO_ENOMEM = -2, LBO_ESTATE = -4 };

// params = {tau_r, tau_b, A, beta, A_nc} (order fixed by north_star)
int lbo_create(int nx, int ny, int nz, const double* params, void** out) {
  if (!out || !params || nx < 1 || ny < 1 || nz < 1) return LBO_EINVAL;
  if (!(params[0] > 0.5) || !(params[1] > 0.5)) return LBO_EINVAL;  // G17
  Oracle* o = new (std::nothrow) Oracle();
  if (!o) return LBO_ENOMEM;
  o->nx = nx; o->ny = ny; o->nz = nz;
  o->S = (size_t)nx * ny * nz;
  o->tau_r = params[0]; o->tau_b = params[1]; o->A = params[2]; o->beta = params[3]; o->A_nc = params[4];
  try {
    o->solid.assign(o->S, 0);
    for (auto* v : {&o->rho_r, &o->rho_b, &o->phi, &o->mx, &o->my, &o->mz, &o->Fx, &o->Fy, &o->Fz,
                    &o->Gx, &o->Gy, &o->Gz, &o->margin, &o->uex, &o->uey, &o->uez})
      v->assign(o->S, 0.0);
    o->hcontact.assign(o->S, 0);
    o->pid.assign(o->S, -1);
  } catch (...) {
    delete o;
    return LBO_ENOMEM;
  }
  *out = o;
  return LBO_OK;
}

void lbo_destroy(void* h) { delete static_cast<Oracle*>(h); }

int lbo_set_geometry(void* h, const uint8_t* mask) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o) return LBO_EINVAL;
  if (o->inited) return LBO_ESTATE;
  o->any_solid = false;
  for (size_t s = 0; s < o->S; ++s) {
    o->pid[s] = -1;
    o->solid[s] = mask ? (mask[s] > 4 ? 1 : mask[s]) : 0;   // 0 fluid, 1 wall at rest, 2 / 3 / 4 wall groups (three: the flow
                                                            // focuser has two kinds of inlet and an outlet; G31)
    o->any_solid |= o->solid[s] != 0;
  }
  return LBO_OK;
}

// velocity of the walls whose mask value is `group` (2, 3 or 4); walls with mask value 1 are at rest
int lbo_set_wall_velocity(void* h, int group, double ux, double uy, double uz) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || group < 2 || group > 4) return LBO_EINVAL;
  o->uw[group][0] = ux; o->uw[group][1] = uy; o->uw[group][2] = uz;
  return LBO_OK;
}

// What a wall group (2, 3 or 4) is (G31): 0 = moving wall (default; lbo_set_wall_velocity), 1 =
// velocity inlet (wall velocity = inflow velocity, prescribed densities rho_r, rho_b of the
// incoming fluid), 2 = pressure boundary with both densities prescribed (a reservoir), 3 = pressure
// outlet: rho_r + rho_b prescribes the total density, the composition is that of the outgoing
// fluid.  The wall velocity is not used by types 2 and 3.
int lbo_set_wall_type(void* h, int group, int type, double rho_r, double rho_b) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || group < 2 || group > 4 || type < 0 || type > 3) return LBO_EINVAL;
  if (type != 0 && (!(rho_r >= 0.0) || !(rho_b >= 0.0))) return LBO_EINVAL;
  o->wtype[group] = type;
  o->wrho[group][0] = rho_r; o->wrho[group][1] = rho_b;
  return LBO_OK;
}

int lbo_set_body_force(void* h, double gx, double gy, double gz) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o) return LBO_EINVAL;
  o->g[0] = gx; o->g[1] = gy; o->g[2] = gz;
  return LBO_OK;
}

int lbo_set_nc_cutoff(void* h, double phi_c) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o) return LBO_EINVAL;
  o->phi_c = phi_c;
  return LBO_OK;
}

// model 0 = colour gradient (A, beta, A_nc of lbo_create apply), 1 = Shan-Chen with exact-difference
// forcing, Eq. 5-10 of the paper (G_C applies; A, beta, A_nc are ignored; needs two components)
int lbo_set_model(void* h, int model, double G_C) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || (model != 0 && model != 1)) return LBO_EINVAL;
  if (o->inited) return LBO_ESTATE;
  o->model = model;
  o->G_C = G_C;
  return LBO_OK;
}

// 0 = Guo forcing (default), 1 = exact-difference forcing (Eq. 9)
int lbo_set_forcing(void* h, int mode) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || (mode != 0 && mode != 1)) return LBO_EINVAL;
  o->forcing = mode;
  return LBO_OK;
}

// 1 = colour-symmetric near-contact probe (G29); 0 = the probe toward decreasing phi only (default)
int lbo_set_nc_symmetric(void* h, int on) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || (on != 0 && on != 1)) return LBO_EINVAL;
  o->nc_sym = on;
  return LBO_OK;
}

// on = 1: solid nodes carry the prescribed value phi_wall in the colour-gradient stencil (G30);
// on = 0: a solid neighbour contributes the centre value (G8, default)
int lbo_set_wall_phi(void* h, int on, double phi_wall) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || (on != 0 && on != 1) || !(std::fabs(phi_wall) <= 1.0)) return LBO_EINVAL;
  o->wet = on;
  o->phi_wall = phi_wall;
  return LBO_OK;
}

int lbo_set_nc_mode(void* h, int mode) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || (mode != 0 && mode != 1)) return LBO_EINVAL;
  o->nc_mode = mode;
  return LBO_OK;
}

// S0. rho_b == NULL selects single-component mode. u is [3][z][y][x].
int lbo_init(void* h, const double* rho_r, const double* rho_b, const double* u) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || !rho_r || !u) return LBO_EINVAL;
  if (o->model == 1 && !rho_b) return LBO_EINVAL;   // the Shan-Chen model couples two components
  const size_t S = o->S;
  o->two = rho_b != nullptr;
  const int nk = o->two ? 2 : 1;
  try {
    for (int k = 0; k < nk; ++k) {
      o->f[k].assign(Q * S, 0.0);
      o->fpost[k].assign(Q * S, 0.0);
    }
  } catch (...) {
    return LBO_ENOMEM;
  }
  if (!o->parts.empty()) rasterize(*o);
  for (size_t s = 0; s < S; ++s) {
    if (o->solid[s]) continue;
    for (int i = 0; i < Q; ++i) {
      o->f[0][s * Q + i] = feq(i, rho_r[s], u[s], u[S + s], u[2 * S + s]);
      if (o->two) o->f[1][s * Q + i] = feq(i, rho_b[s], u[s], u[S + s], u[2 * S + s]);
    }
  }
  o->inited = true;
  return LBO_OK;
}

int lbo_step(void* h, int nsteps) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || nsteps < 0) return LBO_EINVAL;
  if (!o->inited) return LBO_ESTATE;
  for (int t = 0; t < nsteps; ++t) one_step(*o);
  return LBO_OK;
}

// rho_r, rho_b and the half-force-shifted velocity (G16); zeros on solid sites.
int lbo_get_macros(void* h, double* rho_r, double* rho_b, double* u) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o) return LBO_EINVAL;
  if (!o->inited) return LBO_ESTATE;
  eval_forces(*o);
  const size_t S = o->S;
  for (size_t s = 0; s < S; ++s) {
    double rho = o->rho_r[s] + o->rho_b[s];
    bool sol = o->solid[s];
    if (rho_r) rho_r[s] = sol ? 0.0 : o->rho_r[s];
    if (rho_b && o->two) rho_b[s] = sol ? 0.0 : o->rho_b[s];
    if (u) {
      u[s] = sol ? 0.0 : (o->mx[s] + 0.5 * o->Fx[s]) / rho;
      u[S + s] = sol ? 0.0 : (o->my[s] + 0.5 * o->Fy[s]) / rho;
      u[2 * S + s] = sol ? 0.0 : (o->mz[s] + 0.5 * o->Fz[s]) / rho;
    }
  }
  return LBO_OK;
}

// Debug accessors. Pre-collision populations f^k_i(x,t), layout [i][z][y][x].
int lbo_get_populations(void* h, int comp, double* f) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || !f || comp < 0 || comp > (o->two ? 1 : 0)) return LBO_EINVAL;
  if (!o->inited) return LBO_ESTATE;
  for (size_t s = 0; s < o->S; ++s)
    for (int i = 0; i < Q; ++i) f[i * o->S + s] = o->f[comp][s * Q + i];
  return LBO_OK;
}

int lbo_set_populations(void* h, int comp, const double* f) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || !f || comp < 0 || comp > (o->two ? 1 : 0)) return LBO_EINVAL;
  if (!o->inited) return LBO_ESTATE;
  for (size_t s = 0; s < o->S; ++s)
    for (int i = 0; i < Q; ++i) o->f[comp][s * Q + i] = f[i * o->S + s];
  return LBO_OK;
}

// Fields of the current state: phi, G[3][S], F[3][S] (total force), contact distance h
// (0 = none), and the smallest decision margin (G12). Any pointer may be NULL.
int lbo_get_fields(void* h, double* phi, double* G, double* F, int* hcontact, double* margin) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o) return LBO_EINVAL;
  if (!o->inited) return LBO_ESTATE;
  eval_forces(*o);
  const size_t S = o->S;
  for (size_t s = 0; s < S; ++s) {
    if (phi) phi[s] = o->phi[s];
    if (G) { G[s] = o->Gx[s]; G[S + s] = o->Gy[s]; G[2 * S + s] = o->Gz[s]; }
    if (F) { F[s] = o->Fx[s]; F[S + s] = o->Fy[s]; F[2 * S + s] = o->Fz[s]; }
    if (hcontact) hcontact[s] = o->hcontact[s];
    if (margin) margin[s] = o->margin[s];
  }
  return LBO_OK;
}

// ---- rigid particles.  state = n x 15 doubles: r[3], u[3], w[3], q[4], R, mass.
// Must precede lbo_init (the particle nodes hold no fluid).  Colour-gradient or one component.
int lbo_set_particles(void* h, int n, const double* state) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || n < 0 || (n > 0 && !state)) return LBO_EINVAL;
  if (o->inited) return LBO_ESTATE;
  if (o->model == 1) return LBO_EINVAL;
  o->parts.clear();
  for (int p = 0; p < n; ++p) {
    const double* v = state + 15 * p;
    Oracle::Particle P{};
    for (int a = 0; a < 3; ++a) { P.r[a] = v[a]; P.u[a] = v[3 + a]; P.w[a] = v[6 + a]; }
    for (int a = 0; a < 4; ++a) P.q[a] = v[9 + a];
    P.R = v[13]; P.mass = v[14];
    if (!(P.R > 0.0) || !(P.mass > 0.0)) return LBO_EINVAL;
    P.inertia = 0.4 * P.mass * P.R * P.R;
    o->parts.push_back(P);
  }
  return LBO_OK;
}

// state as in lbo_set_particles; force = n x 9 doubles: F[3], T[3] from the fluid links of the last
// step, F_pp[3] from the other particles.  Either may be NULL.
int lbo_get_particles(void* h, double* state, double* force) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o) return LBO_EINVAL;
  for (size_t p = 0; p < o->parts.size(); ++p) {
    const Oracle::Particle& P = o->parts[p];
    if (state) {
      double* v = state + 15 * p;
      for (int a = 0; a < 3; ++a) { v[a] = P.r[a]; v[3 + a] = P.u[a]; v[6 + a] = P.w[a]; }
      for (int a = 0; a < 4; ++a) v[9 + a] = P.q[a];
      v[13] = P.R; v[14] = P.mass;
    }
    if (force) for (int a = 0; a < 3; ++a) { force[9 * p + a] = P.F[a]; force[9 * p + 3 + a] = P.T[a]; force[9 * p + 6 + a] = P.Fpp[a]; }
  }
  return LBO_OK;
}

// mobile = 0 holds the particles in place (they still exchange momentum with the fluid);
// K, h_c, lubrication: the particle-particle force of G37 (h_c <= 0: none)
int lbo_set_particle_options(void* h, int mobile, double K, double h_c, int lubrication) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o) return LBO_EINVAL;
  o->p_mobile = mobile ? 1 : 0;
  o->p_K = K; o->p_hc = h_c; o->p_lub = lubrication ? 1 : 0;
  return LBO_OK;
}

int lbo_set_particle_force(void* h, int p, const double* F, const double* T) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o || p < 0 || p >= (int)o->parts.size()) return LBO_EINVAL;
  for (int a = 0; a < 3; ++a) { o->parts[p].Fext[a] = F ? F[a] : 0.0; o->parts[p].Text[a] = T ? T[a] : 0.0; }
  return LBO_OK;
}

// node map: 0 fluid, 1-4 walls, 5 particle; pid (may be NULL): particle index or -1
int lbo_get_node_map(void* h, uint8_t* solid, int* pid) {
  Oracle* o = static_cast<Oracle*>(h);
  if (!o) return LBO_EINVAL;
  for (size_t s = 0; s < o->S; ++s) {
    if (solid) solid[s] = o->solid[s];
    if (pid) pid[s] = o->pid[s];
  }
  return LBO_OK;
}

// Lattice constants, for pin P1: c[19][3], opp[19], w[19], B[19].
void lbo_constants(int* c, int* opp, double* w, double* b) {
  for (int i = 0; i < Q; ++i) {
    if (c) { c[3 * i] = CX[i]; c[3 * i + 1] = CY[i]; c[3 * i + 2] = CZ[i]; }
    if (opp) opp[i] = OPP[i];
    if (w) w[i] = W[i];
    if (b) b[i] = B[i];
  }
}

}  // extern "C"
