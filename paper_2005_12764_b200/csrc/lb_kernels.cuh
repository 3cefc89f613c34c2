// CUDA kernels of the colour-gradient D3Q19 hot path, written for sm_100a (B200).
//
// One LB step of a two-component run = k_fused + k_phase_fwd:
//   k_fused     K2  pull-stream + moments + grad phi from a TMA-staged shared-memory phi ring +
//                   near-contact probe (Eq. 11) + Guo force + BGK on the total
//                   (Eq. 1-2, 5-8) + perturbation + recolouring + store, and the
//                   moments of the NEXT state (Eq. 3) forwarded from registers
//   k_phase_fwd K1f phi of the next state from the forwarded moments + the brick-face terms
// Others:
//   k_phase     K1  full phase-field sweep: gather both components' populations, rho_r, rho_b, phi;
//                   runs after lb_init / lb_set_populations (phi is not forwarded yet)
//   k_single    K2s single-component BGK (Eq. 1-4), the pure-bandwidth baseline (config C2)
//   k_scatter   K0  place given pre-collision populations where the next gather finds them
//   k_gatherf       debug accessor: full pre-collision populations
//   k_macros    K3  rho_r, rho_b, u with the half-force shift
//
// Storage: SoA over the 19 directions, x fastest.  Two components: plane q holds
// one float2 {T_q, R_q} per site, T_q = f^r_q + f^b_q - w_q (the total as a deviation from the lattice
// weight, so that the hydrodynamic part keeps ~1e-9 absolute precision in fp32), R_q = f^r_q.
// Single component: plane q holds f_q - w_q.  The collision is carried out on the deviations
// directly (T^eq_q = w_q [drho + rho (3 cu + 4.5 cu^2 - 1.5 uu)]).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "lb_lattice.cuh"

namespace lb {

struct StepParams {
  const float* src;   // population buffer read by this step
  const float* ps[Q];   // base of every direction plane of src / dst: host-computed so that an access
  float* pd[Q];         // is one 64-bit add of a constant-bank operand and a 32-bit byte offset
  float* dst;         // buffer written (== src in AA modes)
  float* phi;         // padded phi array (written by K1 / K1f, read by K2 / K3)
  float* phi2;        // Shan-Chen model only: the padded array of rho_b (phi then holds rho_r)
  float* Md;          // forwarded moments of the next state (written by K2, read by K1f):
  float* Mt;          //   Md = sum (f^r - f^b), Mt = sum (f - w) over what arrives from inside the brick
  float* EX;          // the same sums for what crosses the x faces of the bricks: [z][y][tile][side]{D, Tm}
  Box box;
  int z0, z1;         // planes this launch covers: whole bricks, counted from box.zlo
  int zc;             // z planes per CTA
  int halo;           // ghost depth K1 must fill (1 without near contact, 4 with)
  float tau_r, tau_b, A, beta, A_nc, phi_c, gx, gy, gz;
  int two_tau, has_g;
  int edm;            // exact-difference forcing (Eq. 9) instead of Guo
  int nc_sym;         // colour-symmetric near-contact probe (G29)
  int wet;            // solid nodes carry phi_wall in the colour-gradient stencil (G30)
  float phi_wall;
  int has_moving;     // some walls move (mask groups 2, 3, 4): half-way bounce-back with the wall velocity (G28)
  float uw[3][3];     // velocities of groups 2, 3, 4
  int wtype[3];       // what these groups are (G31): 0 moving wall, 1 velocity inlet, 2 reservoir, 3 pressure outlet
  float wrho[3][2];   // prescribed rho_r, rho_b of an inlet / reservoir / outlet
  const PState* parts; // rigid particles (NEXT-4), or nullptr
  int sc;             // Shan-Chen model (Eq. 5-10 of the paper): the fields are rho_r, rho_b instead of phi
  float G_C;          // its coupling strength, positive = repulsive
};

constexpr int TX = 32, TY = 8;   // CTA tile in x-y; one warp per x row segment

// ----------------------------------------------------------------------------- addressing
// A population lives in plane `plane` (0..18, + 19 for the red set) at byte offset `off` inside
// the plane.  Offsets are 32-bit (a plane is < 4 GB: S < 2^30), plane bases are uniform across
// the warp, so one access costs one integer add instead of a 64-bit index computation.
struct Slot {
  int plane;
  uint32_t off;
};

struct Ctx {
  int idx;            // own site (elements)
  uint32_t ob;        // own site (bytes)
  // byte deltas to the wrapped neighbours, modulo 2^32: a wrap across the whole box exceeds
  // INT_MAX once S * 8 > 2^31 (656^3), so the arithmetic is unsigned, where wrap-around is defined
  uint32_t dxo[3];    // to x-1, x, x+1
  uint32_t dyo[3];    // to y-1, y, y+1
  uint32_t dzo[3];    // to z-1, z, z+1
};

// Byte delta from the own site to x - c_q.
template <int q>
__device__ __forceinline__ uint32_t delta_src(const Ctx& c) {
  return c.dxo[1 - cx(q)] + c.dyo[1 - cy(q)] + c.dzo[1 - cz(q)];
}

// Where f_q(x) of the current state is stored.  smask bit i set <=> x + c_i is solid.
template <int MODE, bool HAS_SOLID, int q>
__device__ __forceinline__ Slot read_slot(const Ctx& c, uint32_t smask) {
  if constexpr (MODE == MODE_AA_EVEN || q == 0) {
    return Slot{q, c.ob};
  } else {
    const uint32_t nb = c.ob + delta_src<q>(c);
    if constexpr (!HAS_SOLID) {
      return MODE == MODE_AB ? Slot{q, nb} : Slot{opp(q), nb};
    } else {
      const bool bounce = (smask >> opp(q)) & 1u;
      if constexpr (MODE == MODE_AB) return bounce ? Slot{opp(q), c.ob} : Slot{q, nb};
      else return bounce ? Slot{q, c.ob} : Slot{opp(q), nb};   // AA_ODD
    }
  }
}

// Where the post-collision value f*_q goes.
template <int MODE, bool HAS_SOLID, int q>
__device__ __forceinline__ Slot write_slot(const Ctx& c, uint32_t smask) {
  if constexpr (MODE == MODE_AB) {
    return Slot{q, c.ob};
  } else if constexpr (MODE == MODE_AA_EVEN) {
    return Slot{opp(q), c.ob};
  } else {
    return read_slot<MODE, HAS_SOLID, opp(q)>(c, smask);
  }
}

// Two-component buffers hold, per direction plane, one float2 {T_q, R_q} per site (T = total as a
// deviation, R = red), so a direction costs one 64-bit access.  Single-component buffers hold T_q.
template <class P>
__device__ __forceinline__ const float* src_ptr(const P& p, Slot s) {
  return reinterpret_cast<const float*>(reinterpret_cast<const char*>(p.ps[s.plane]) + s.off);
}
template <class P>
__device__ __forceinline__ float* dst_ptr(const P& p, Slot s) {
  return reinterpret_cast<float*>(reinterpret_cast<char*>(p.pd[s.plane]) + s.off);
}
template <int MODE>
__device__ __forceinline__ float2 ld_pair(const float* p) {
  if constexpr (MODE == MODE_AB) return __ldg(reinterpret_cast<const float2*>(p));   // read-only in A/B mode
  else return __ldcg(reinterpret_cast<const float2*>(p));   // in place: read through L2, not through a stale or thrashing L1
}

template <int MODE>
__device__ __forceinline__ float ld_pop(const float* p) {
  if constexpr (MODE == MODE_AB) return __ldg(p);   // source buffer is read-only in A/B mode
  else return *p;
}

// c_q . a without the multiplications by 0 and +-1 that IEEE arithmetic would not let the compiler drop
template <int q>
__device__ __forceinline__ float cdot(float ax, float ay, float az) {
  constexpr int X = cx(q), Y = cy(q), Z = cz(q);
  if constexpr (X != 0 && Y != 0) return (X > 0 ? ax : -ax) + (Y > 0 ? ay : -ay);
  else if constexpr (X != 0 && Z != 0) return (X > 0 ? ax : -ax) + (Z > 0 ? az : -az);
  else if constexpr (Y != 0 && Z != 0) return (Y > 0 ? ay : -ay) + (Z > 0 ? az : -az);
  else if constexpr (X != 0) return X > 0 ? ax : -ax;
  else if constexpr (Y != 0) return Y > 0 ? ay : -ay;
  else if constexpr (Z != 0) return Z > 0 ? az : -az;
  else return 0.0f;
}

// What a link q into a wall of group 2 + gi (gi = 0, 1, 2) sends back: the stored
// post-collision pair {ts = f* - w, rs = f^r*} is replaced by what the site reads along opp(q) in
// the next step.  Moving wall (G28): the reflected population loses 6 w_q rho^k (c_q . u_w), rho^k
// the site's own densities; velocity inlet (G31, type 1): the same with the prescribed densities.
// Reservoir / pressure outlet (G31, types 2 / 3; the flow focuser's open ends):
// anti-bounce-back, f^k <- -f^k* + 2 w_q rho^k_out [1 + 4.5 (c_q.u)^2 - 1.5 u.u] with u the
// velocity that entered f^eq; the outlet keeps the site's composition,
// rho^k_out = (rho_r + rho_b)_prescribed rho^k / rho.  In deviation form the total becomes
// -ts + 2 w_q [(rho_out - 1) + rho_out (4.5 (c.u)^2 - 1.5 u.u)].
// ONE: single component, whose density is the prescribed rho_r (the outlet's: rho_r + rho_b).
template <int q, bool ONE = false>
__device__ __forceinline__ void open_link(const StepParams& p, int gi, float rho, float rr, float inv_rho,
                                          float ux, float uy, float uz, float uu15, float& ts, float& rs) {
  constexpr float w = wq(q);
  const int wt = p.wtype[gi];
  const float pr = p.wrho[gi][0], pb = p.wrho[gi][1];
  if (wt >= 2) {
    const float cu = cdot<q>(ux, uy, uz);
    const float e1 = fmaf(4.5f * cu, cu, -uu15);
    const float ro = (ONE && wt == 2) ? pr : pr + pb;
    const float rro = wt == 3 ? ro * (rr * inv_rho) : pr;
    ts = fmaf(2.0f * w, fmaf(ro, e1, ro - 1.0f), -ts);
    rs = fmaf(2.0f * w * rro, 1.0f + e1, -rs);
  } else {
    const float cw = cdot<q>(p.uw[gi][0], p.uw[gi][1], p.uw[gi][2]);
    const float rt = wt == 1 ? (ONE ? pr : pr + pb) : rho, r1 = wt == 1 ? pr : rr;
    ts = fmaf(-6.0f * w * rt, cw, ts);
    rs = fmaf(-6.0f * w * r1, cw, rs);
  }
}

// ---- rigid particles (the paper's section 6; G32-G37) ----
// The hot kernels treat a particle's nodes as walls at rest; k_part_force then turns every stored
// value of a link into a particle into what comes back from the moving surface (G33).
// nearest periodic image of a difference of two positions inside the box (|d| < n): no division
__device__ __forceinline__ double min_image(double d, int n) {
  const double h = 0.5 * n;
  return d > h ? d - n : (d < -h ? d + n : d);
}

// Solid flags of the 18 neighbours from the bit-packed mask (bit i <=> x + c_i solid).
__device__ __forceinline__ uint32_t neighbour_mask(const Box& b, int x, int y, int z) {
  const int xs[3] = {wrap_m(x, b.nx), x, wrap_p(x, b.nx)};
  const int ys[3] = {wrap_m(y, b.ny), y, wrap_p(y, b.ny)};
  const int zs[3] = {wrap_m(z, b.nz), z, wrap_p(z, b.nz)};
  uint32_t m = 0;
  static_for<1, Q>([&](auto qc) {
    constexpr int q = decltype(qc)::value;
    if (solid_at(b, xs[1 + cx(q)], ys[1 + cy(q)], zs[1 + cz(q)])) m |= 1u << q;
  });
  return m;
}

// The same for the wall groups 2, 3, 4: bit i of g2 <=> x + c_i is a wall of group 2 or 4, of g3 <=>
// of group 3 or 4 (the two bit planes of Box::gmask).
__device__ __forceinline__ void neighbour_groups(const Box& b, int x, int y, int z, uint32_t& g2, uint32_t& g3) {
  const int xs[3] = {wrap_m(x, b.nx), x, wrap_p(x, b.nx)};
  const int ys[3] = {wrap_m(y, b.ny), y, wrap_p(y, b.ny)};
  const int zs[3] = {wrap_m(z, b.nz), z, wrap_p(z, b.nz)};
  g2 = g3 = 0;
  static_for<1, Q>([&](auto qc) {
    constexpr int q = decltype(qc)::value;
    const int g = wall_group_at(b, xs[1 + cx(q)], ys[1 + cy(q)], zs[1 + cz(q)]);
    if (g == 2 || g == 4) g2 |= 1u << q;
    if (g == 3 || g == 4) g3 |= 1u << q;
  });
}

// ESZ: bytes per site in a plane (8 for the {T, R} pairs of a two-component run, 4 for one component)
template <int ESZ>
__device__ __forceinline__ void make_ctx(Ctx& c, const Box& b, int x, int y, int z) {
  c.idx = x + b.nx * (y + b.ny * z);
  c.ob = (uint32_t)c.idx * (uint32_t)ESZ;
  constexpr uint32_t E = (uint32_t)ESZ;
  c.dxo[0] = x == 0 ? (uint32_t)(b.nx - 1) * E : 0u - E;
  c.dxo[1] = 0u;
  c.dxo[2] = x == b.nx - 1 ? 0u - (uint32_t)(b.nx - 1) * E : E;
  const uint32_t row = (uint32_t)b.nx * E;
  c.dyo[0] = y == 0 ? (uint32_t)(b.ny - 1) * row : 0u - row;
  c.dyo[1] = 0u;
  c.dyo[2] = y == b.ny - 1 ? 0u - (uint32_t)(b.ny - 1) * row : row;
  const uint32_t pl = (uint32_t)b.nx * (uint32_t)b.ny * E;
  c.dzo[0] = z == 0 ? (uint32_t)(b.nz - 1) * pl : 0u - pl;
  c.dzo[1] = 0u;
  c.dzo[2] = z == b.nz - 1 ? 0u - (uint32_t)(b.nz - 1) * pl : pl;
}

// s + e <- s + e + x with the rounding error of the addition kept in e (Knuth two-sum).
__device__ __forceinline__ void two_sum_acc(float& s, float& e, float x) {
  const float t = __fadd_rn(s, x);
  const float bp = __fsub_rn(t, s);
  e = __fadd_rn(e, __fadd_rn(__fsub_rn(s, __fsub_rn(t, bp)), __fsub_rn(x, bp)));
  s = t;
}

// phi of site (x, y, z) to its home in the padded array and to every periodic image that falls
// into the ghost layers (depth H).
__device__ __forceinline__ void store_field_with_images(float* field, const Box& b, int x, int y, int z, int H, float phi) {
  const int px = b.nx + 2 * HALO, py = b.ny + 2 * HALO;
  const bool zin = !b.zper || (z >= H && z < b.nz - H);      // a slab's z ghost planes come from its neighbours
  if (x >= H && x < b.nx - H && y >= H && y < b.ny - H && zin) {   // no image
    field[(size_t)(x + HALO) + (size_t)px * ((size_t)(y + HALO) + (size_t)py * (size_t)(z + HALO))] = phi;
    return;
  }
  const int sx[3] = {0, x < H ? b.nx : 0, x >= b.nx - H ? -b.nx : 0};
  const int sy[3] = {0, y < H ? b.ny : 0, y >= b.ny - H ? -b.ny : 0};
  const int sz[3] = {0, (b.zper && z < H) ? b.nz : 0, (b.zper && z >= b.nz - H) ? -b.nz : 0};
#pragma unroll
  for (int iz = 0; iz < 3; ++iz) {
    if (iz && !sz[iz]) continue;
#pragma unroll
    for (int iy = 0; iy < 3; ++iy) {
      if (iy && !sy[iy]) continue;
#pragma unroll
      for (int ix = 0; ix < 3; ++ix) {
        if (ix && !sx[ix]) continue;
        field[(size_t)(x + sx[ix] + HALO) + (size_t)px * ((size_t)(y + sy[iy] + HALO) + (size_t)py * (size_t)(z + sz[iz] + HALO))] = phi;
      }
    }
  }
}

// What the fused kernel needs of its neighbours at site (x, y, z), from d = rho_r - rho_b and rho:
// phi = d / rho for the colour-gradient model, the pair rho_r, rho_b for the Shan-Chen model.
// Solid sites carry the sentinel in the first field.
template <bool SC>
__device__ __forceinline__ void store_fields(const StepParams& p, int x, int y, int z, int H, bool solid, float d, float rho) {
  // the sentinel of a solid site also carries its wall group (1e30, 2e30, 3e30)
  const float sent = solid ? PHI_SOLID * (float)sentinel_code(p.box, x, y, z) : 0.f;
  if constexpr (!SC) {
    store_field_with_images(p.phi, p.box, x, y, z, H, solid ? sent : d / rho);
  } else {
    store_field_with_images(p.phi, p.box, x, y, z, H, solid ? sent : 0.5f * (rho + d));
    store_field_with_images(p.phi2, p.box, x, y, z, H, solid ? 0.f : 0.5f * (rho - d));
  }
}

// ----------------------------------------------------------------------------- K1 phase field
// One thread per site of a TX x TY tile, marching over zc planes.  152 B read, 4 B written.
template <int MODE, bool HAS_SOLID, bool SC>
__device__ __forceinline__ void phase_column(const StepParams& p, int x, int y, int zb, int ze) {
  const Box& b = p.box;
  const int H = p.halo;
  for (int z = zb; z < ze; ++z) {
    Ctx c;
    make_ctx<8>(c, b, x, y, z);
    float num = 0.f, rho = 1.f;
    bool self_solid = false;
    uint32_t smask = 0;
    if constexpr (HAS_SOLID) {
      self_solid = solid_at(b, x, y, z);
      if (!self_solid) smask = neighbour_mask(b, x, y, z);
    }
    if (!self_solid) {
      float t[Q], r[Q];
      static_for<0, Q>([&](auto qc) {
        constexpr int q = decltype(qc)::value;
        const Slot s = read_slot<MODE, HAS_SOLID, q>(c, smask);
        const float2 v = ld_pair<MODE>(src_ptr(p, s));
        t[q] = v.x;
        r[q] = v.y;
      });
      // Compensated (two-sum) accumulation: the direction of grad phi, which the perturbation and
      // the recolouring use, is ill-conditioned where |grad phi| is small, so phi is formed to
      // ~1e-8 instead of the ~1e-7 that a plain fp32 sum of 19 terms gives.
      float dr = 0.f, de = 0.f, rr = 0.f, re = 0.f;
      static_for<0, Q>([&](auto qc) {
        constexpr int q = decltype(qc)::value;
        two_sum_acc(dr, de, t[q]);
        two_sum_acc(rr, re, r[q]);
      });
      // rho_r - rho_b = 2 rho_r - rho = (2 rr - 1 - dr) + (2 re - de); rho = 1 + dr + de
      num = ((2.0f * rr - 1.0f) - dr) + (2.0f * re - de);
      rho = (1.0f + dr) + de;
    }
    store_fields<SC>(p, x, y, z, H, self_solid, num, rho);
  }
}

template <int MODE, bool HAS_SOLID, bool SC>
__global__ void __launch_bounds__(TX* TY) k_phase(const StepParams p) {
  const int x = blockIdx.x * TX + threadIdx.x;
  const int y = blockIdx.y * TY + threadIdx.y;
  if (x >= p.box.nx || y >= p.box.ny) return;
  const int zb = p.z0 + blockIdx.z * p.zc;
  phase_column<MODE, HAS_SOLID, SC>(p, x, y, zb, min(p.z1, zb + p.zc));
}

// ----------------------------------------------------------------------------- TMA / mbarrier
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
// 3-D tiled TMA load global -> shared, completion on an mbarrier (SASS: UTMALDG).
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}

template <int H>
struct Ring {
  // Box extent in x is TX + 2 HALO for every H and the box starts at padded x = x0: the TMA unit
  // faults (illegal instruction, measured on B200) when the innermost start
  // coordinate is not a multiple of 16 bytes, so the box cannot start at x0 + HALO - H for H = 1.
  static constexpr int BX = TX + 2 * HALO;
  static constexpr int BY = TY + 2 * H;
  static constexpr int PF = 2;                         // planes prefetched ahead
  static constexpr int NS = 2 * H + 1 + PF;            // ring slots
  static constexpr int SLOT = ((BX * BY * 4 + 127) / 128) * 32;   // floats per slot, 128-B multiple
  static constexpr uint32_t BYTES = BX * BY * 4;       // bytes one TMA box delivers
};

// ----------------------------------------------------------------------------- K2 fused
// Per thread: one site per plane, marching over zc planes; per CTA a TX x TY tile ("brick" =
// tile x z range of the CTA).  The phi planes z-H..z+H (+ 2 prefetched) of the tile with an H-wide
// halo live in a shared-memory ring filled by TMA from the padded phi array (ghost layers make
// every box in-bounds, so periodic wrap never reaches the TMA unit).  H = 1 without near
// contact, 4 with it.
//
// Moment forwarding.  The next step needs phi(t+1) = (rho_r - rho_b)/rho of the populations that
// will ARRIVE at each site, i.e. sums over the neighbours' post-collision values.  Instead of a
// second sweep over the 38 planes (k_phase), this kernel adds up, for every site of its brick,
// the contributions that come from inside the brick while the post-collision values are still in
// registers:  D(y) = sum_q (f^r*_q - f^b*_q)(y - c_q),  Tm(y) = sum_q (f*_q - w_q)(y - c_q).
// x: warp shuffles (a row of 32 sites is one warp); y: one shared-memory exchange per plane;
// z: carried in registers from one plane to the next (plane z-1 is complete once plane z is done).
// A population that would enter a solid site returns to its own site (bounce-back) and is added
// there.  What enters a brick through its faces is added by k_phase_fwd from the stored values.
template <int H, bool SC = false>
struct FusedSmem {
  static constexpr int NEX = 12;   // exchanged values: 6 (cy = +-1) x {D, Tm}
  static constexpr size_t RING1 = (size_t)Ring<H>::NS * Ring<H>::SLOT * sizeof(float);
  static constexpr size_t RING = (SC ? 2 : 1) * RING1;   // Shan-Chen: a second ring for rho_b
  static constexpr size_t YEX = (size_t)2 * NEX * TX * TY * sizeof(float);
  static constexpr size_t XEX = (size_t)2 * 2 * 4 * TY * sizeof(float);   // [buffer][side][(+1,-1) x {D, Tm}][row]
  static constexpr size_t BYTES = RING + YEX + XEX + Ring<H>::NS * sizeof(uint64_t);
};

// FMODE: bit 0 = a body force rho g acts, bit 1 = the force enters by the exact-difference source
// (Eq. 9) instead of the Guo term
// SC: the paper's section 3.1 as printed instead of the colour-gradient model: the two rings hold
// rho_r and rho_b, the Shan-Chen accelerations (Eq. 10; sign: DESIGN.md G27) replace
// grad phi, each component gets the exact-difference source of Eq. 9, and there is no perturbation,
// recolouring or near-contact force (HAS_NC = false; FMODE bit 0 only).
// WALLS: 0 = no solid sites, 1 = walls at rest, 2 = some walls move (G28; two CTAs per SM: the
// extra live values of the wall correction would spill at 80 registers)
template <int MODE, int WALLS, bool HAS_NC, int FMODE, bool SC = false>
__global__ void __launch_bounds__(TX* TY, ((MODE == MODE_AA_ODD && SC) || WALLS == 2) ? 2 : 3) k_fused(const StepParams p, const __grid_constant__ CUtensorMap tmap,
                                                     const __grid_constant__ CUtensorMap tmap2) {
  constexpr int H = HAS_NC ? H_MAX_NC : 1;
  constexpr bool HAS_SOLID = WALLS > 0, MOVING = WALLS == 2;
  constexpr bool HAS_G = (FMODE & 1) != 0, EDM = (FMODE & 2) != 0;
  static_assert(!SC || !HAS_NC, "the Shan-Chen model has no near-contact force");
  using R_ = Ring<H>;
  using SM_ = FusedSmem<H, SC>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* ring = reinterpret_cast<float*>(smem_raw);
  float* ring2 = reinterpret_cast<float*>(smem_raw + SM_::RING1);     // used only if SC
  float* yex = reinterpret_cast<float*>(smem_raw + SM_::RING);                 // [2][NEX][TY][TX]
  float* xex = reinterpret_cast<float*>(smem_raw + SM_::RING + SM_::YEX);     // [2][2][4][TY]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + SM_::RING + SM_::YEX + SM_::XEX);

  const Box& b = p.box;
  const int tid = threadIdx.y * TX + threadIdx.x;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int x = x0 + threadIdx.x, y = y0 + threadIdx.y;
  const bool active = x < b.nx && y < b.ny;
  const int zb = p.z0 + blockIdx.z * p.zc;
  const int ze = min(p.z1, zb + p.zc);
  const int npl = (ze - zb) + 2 * H;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < R_::NS; ++s) mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  auto issue = [&](int j) {
    const int s = j % R_::NS;
    mbar_expect_tx(&bars[s], (SC ? 2u : 1u) * R_::BYTES);
    tma_load_3d(&ring[s * R_::SLOT], &tmap, &bars[s], x0, y0 + HALO - H, zb - H + j + HALO);
    if constexpr (SC) tma_load_3d(&ring2[s * R_::SLOT], &tmap2, &bars[s], x0, y0 + HALO - H, zb - H + j + HALO);
  };
  if (tid == 0) {
    const int n0 = min(npl, R_::NS);
    for (int j = 0; j < n0; ++j) issue(j);
  }

  const float omega_same = 1.0f / p.tau_r;
  const float nu_r = (p.tau_r - 0.5f) * (1.0f / 3.0f), nu_b = (p.tau_b - 0.5f) * (1.0f / 3.0f);
  const int lx = threadIdx.x + HALO, ly = threadIdx.y + H;
  const size_t plane_sites = (size_t)b.nx * b.ny;
  const size_t col = (size_t)x + (size_t)b.nx * y;
  // carried between planes: pend = b0(z-1) + b+(z-2) (plane z-1 still misses b-(z)), bpc = b+(z-1)
  float pend_d = 0.f, pend_t = 0.f, bpc_d = 0.f, bpc_t = 0.f;
  // the same for what leaves the brick through its x faces (kept by the first and the last active
  // lane of each row): the sums land in p.EX, indexed by target row and plane, and k_phase_fwd adds
  // them to the first / last column of the neighbouring brick
  const int lastx = min(TX, b.nx - x0) - 1;
  const bool lL = threadIdx.x == 0, lR = (int)threadIdx.x == lastx;
  const int side = lR ? 1 : 0;
  float pe_d = 0.f, pe_t = 0.f, bpe_d = 0.f, bpe_t = 0.f;
  const int ntx = gridDim.x;

  for (int jz = 0; jz < ze - zb; ++jz) {
    const int z = zb + jz;
    if (jz == 0) {
#pragma unroll
      for (int j = 0; j <= 2 * H; ++j) mbar_wait(&bars[j % R_::NS], (j / R_::NS) & 1);
    } else {
      const int j = jz + 2 * H;
      mbar_wait(&bars[j % R_::NS], (j / R_::NS) & 1);
    }
    // plane dz of the ring
    auto plane = [&](int dz) -> const float* { return &ring[((jz + H + dz) % R_::NS) * R_::SLOT]; };
    const float* pl0 = plane(0);
    const float phi0 = pl0[ly * R_::BX + lx];
    const bool fluid = active && !(HAS_SOLID && phi0 > PHI_SOLID_TEST);
    // what this site sends along each direction: vd = f^r* - f^b*, vt = f* - w (zero if not fluid)
    float vd[Q], vt[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) { vd[q] = 0.f; vt[q] = 0.f; }
    if (fluid) {
      Ctx c;
      make_ctx<8>(c, b, x, y, z);
      // ---- grad phi (stencil of Eq. 10) and solid flags from the phi tile
      const float* plm = plane(-1);
      const float* plp = plane(+1);
      float Gx = 0.f, Gy = 0.f, Gz = 0.f;       // SC: sum_i w_i c_i rho_b(x + c_i)
      float Hx = 0.f, Hy = 0.f, Hz = 0.f;       // SC: sum_i w_i c_i rho_r(x + c_i)
      uint32_t smask = 0;
      if constexpr (!SC) {
        // a solid neighbour contributes the centre value (G8) or the prescribed wall value (G30)
        const float wallv = (HAS_SOLID && p.wet) ? p.phi_wall : phi0;
        static_for<1, Q>([&](auto qc) {
          constexpr int q = decltype(qc)::value;
          const float* pl = cz(q) == 0 ? pl0 : (cz(q) > 0 ? plp : plm);
          float v = pl[(ly + cy(q)) * R_::BX + lx + cx(q)];
          if constexpr (HAS_SOLID) {
            if (v > PHI_SOLID_TEST) { smask |= 1u << q; v = wallv; }
          }
          constexpr float k = 3.0f * wq(q);
          if constexpr (cx(q) != 0) Gx += (k * cx(q)) * v;
          if constexpr (cy(q) != 0) Gy += (k * cy(q)) * v;
          if constexpr (cz(q) != 0) Gz += (k * cz(q)) * v;
        });
      } else {
        const int ro = (int)(ring2 - ring);     // the rho_b tile sits at the same place in the second ring
        const float rb0 = pl0[ro + ly * R_::BX + lx];
        static_for<1, Q>([&](auto qc) {
          constexpr int q = decltype(qc)::value;
          const float* pl = cz(q) == 0 ? pl0 : (cz(q) > 0 ? plp : plm);
          const int o = (ly + cy(q)) * R_::BX + lx + cx(q);
          float vr = pl[o], vb = pl[ro + o];
          if constexpr (HAS_SOLID) {
            if (vr > PHI_SOLID_TEST) { smask |= 1u << q; vr = phi0; vb = rb0; }   // neutral wall
          }
          constexpr float k = wq(q);
          if constexpr (cx(q) != 0) { Gx += (k * cx(q)) * vb; Hx += (k * cx(q)) * vr; }
          if constexpr (cy(q) != 0) { Gy += (k * cy(q)) * vb; Hy += (k * cy(q)) * vr; }
          if constexpr (cz(q) != 0) { Gz += (k * cz(q)) * vb; Hz += (k * cz(q)) * vr; }
        });
      }
      // ---- gather.  Walls are rare: a warp none of whose sites has a solid neighbour takes the
      // addressing of the wall-free variant (no per-direction select between the two slots).
      bool near_wall = false;
      if constexpr (HAS_SOLID) near_wall = __any_sync(__activemask(), smask != 0u);
      float T[Q], R[Q];
      auto gather = [&](auto bounce) {
        static_for<0, Q>([&](auto qc) {
          constexpr int q = decltype(qc)::value;
          const Slot s = read_slot<MODE, decltype(bounce)::value, q>(c, smask);
          const float2 v = ld_pair<MODE>(src_ptr(p, s));
          T[q] = v.x;
          R[q] = v.y;
        });
      };
      if (HAS_SOLID && near_wall) gather(std::integral_constant<bool, HAS_SOLID>{});
      else gather(std::false_type{});
      // ---- moments (Eq. 3)
      float dr = 0.f, rr = 0.f, mx = 0.f, my = 0.f, mz = 0.f;
      static_for<0, Q>([&](auto qc) {
        constexpr int q = decltype(qc)::value;
        dr += T[q];
        rr += R[q];
        if constexpr (cx(q) != 0) mx += cx(q) * T[q];
        if constexpr (cy(q) != 0) my += cy(q) * T[q];
        if constexpr (cz(q) != 0) mz += cz(q) * T[q];
      });
      const float rho = 1.0f + dr;
      const float rb = rho - rr;
      const float inv_rho = 1.0f / rho;
      if constexpr (!SC) {
      const float Gn2 = Gx * Gx + Gy * Gy + Gz * Gz;
      const float Gn = sqrtf(Gn2);
      const bool aniso = Gn > EPS_G;
      const float invG = aniso ? 1.0f / Gn : 0.0f;
      const float Gne = aniso ? Gn : 0.0f;
      // ---- near-contact force (Eq. 11): F = A_h G / 2
      float Fx = 0.f, Fy = 0.f, Fz = 0.f;
      if constexpr (HAS_NC) {
        if (fabsf(phi0) < p.phi_c && aniso) {
          const float nx_ = -Gx * invG, ny_ = -Gy * invG, nz_ = -Gz * invG;
          // h: first k >= 2 along -G with phi(probe) >= phi(x); hp (symmetric probe, G29): first
          // k >= 2 along +G (the mirrored offsets) with phi(probe) <= phi(x)
          int h = 0, hp = 0;
          bool alive = true, alive2 = p.nc_sym != 0;
#pragma unroll
          for (int k = 1; k <= H_MAX_NC; ++k) {
            if (alive || alive2) {
              const int dx = (int)roundf(k * nx_), dy = (int)roundf(k * ny_), dz = (int)roundf(k * nz_);
              if (alive) {
                const float v = plane(dz)[(ly + dy) * R_::BX + lx + dx];
                if (HAS_SOLID && v > PHI_SOLID_TEST) alive = false;
                else if (k >= 2 && v >= phi0) { h = k; alive = false; }
              }
              if (alive2) {
                const float v = plane(-dz)[(ly - dy) * R_::BX + lx - dx];
                if (HAS_SOLID && v > PHI_SOLID_TEST) alive2 = false;
                else if (k >= 2 && v <= phi0) { hp = k; alive2 = false; }
              }
            }
          }
          auto A_h = [&](int hh) {
            return hh == 0 ? 0.f : (hh <= H_MIN_NC ? p.A_nc : p.A_nc * ((float)(H_MIN_NC * H_MIN_NC * H_MIN_NC) / (float)(hh * hh * hh)));
          };
          if (h > 0 || hp > 0) {
            const float Ah = A_h(h) - A_h(hp);
            Fx = 0.5f * Ah * Gx; Fy = 0.5f * Ah * Gy; Fz = 0.5f * Ah * Gz;
          }
        }
      }
      constexpr bool forced = HAS_NC || HAS_G;
      if constexpr (HAS_G) { Fx += rho * p.gx; Fy += rho * p.gy; Fz += rho * p.gz; }
      // ---- velocity with the half-force shift, relaxation rate (Eq. 7-8)
      // (exact difference: f^eq at the bare velocity m/rho, source f^eq(u + F/rho) - f^eq(u))
      constexpr float hs = EDM ? 0.0f : 0.5f;
      const float ux = (mx + hs * Fx) * inv_rho, uy = (my + hs * Fy) * inv_rho, uz = (mz + hs * Fz) * inv_rho;
      float omega = omega_same;
      if (p.two_tau) {
        const float inv_nu = (rr * inv_rho) / nu_r + (rb * inv_rho) / nu_b;
        omega = 1.0f / (3.0f / inv_nu + 0.5f);
      }
      const float uu15 = 1.5f * (ux * ux + uy * uy + uz * uz);
      const float uF = ux * Fx + uy * Fy + uz * Fz;
      const float fr_r = rr * inv_rho;                       // rho_r / rho
      const float kcol = p.beta * rr * rb * inv_rho * invG;   // recolouring amplitude / |G|
      const float om1 = 1.0f - omega;
      // Per-site constants of the three weight classes (rest, axis, diagonal), so that the loop
      // over directions is a handful of fused multiply-adds:
      //   omega f^eq_q - A B_q |G| = ob[c] + orw[c] cu (3 + 4.5 cu)
      //   A w_q (c.G)^2 / |G|      = (pa[c] cG) cG
      //   Guo source               = gw[c] (cF (1 + 3 cu) - u.F)   (-gw[c] u.F is folded into obf[c])
      //   red share                = fr_r (f*_q + w_q) + kc[c] cG
      const float eq0 = dr - rho * uu15;
      const float orw[3] = {omega * rho * wq(0), omega * rho * wq(1), omega * rho * wq(7)};
      const float ob[3] = {omega * wq(0) * eq0 - p.A * bq(0) * Gne, omega * wq(1) * eq0 - p.A * bq(1) * Gne,
                           omega * wq(7) * eq0 - p.A * bq(7) * Gne};
      const float pa[3] = {0.f, p.A * wq(1) * invG, p.A * wq(7) * invG};
      //   exact difference         = rw[c] ((cv - cu)(3 + 4.5 (cv + cu)) - 1.5 (v.v - u.u)),  v = u + F/rho
      const float fax = Fx * inv_rho, fay = Fy * inv_rho, faz = Fz * inv_rho;   // v - u
      const float vx = ux + fax, vy = uy + fay, vz = uz + faz;
      const float dvv15 = 1.5f * (vx * vx + vy * vy + vz * vz) - uu15;
      const float rw[3] = {rho * wq(0), rho * wq(1), rho * wq(7)};
      const float g3 = 3.0f * (1.0f - 0.5f * omega);
      const float gw[3] = {g3 * wq(0), g3 * wq(1), g3 * wq(7)};
      const float kc[3] = {0.f, kcol * wq(1), kcol * (wq(7) * inv_cnorm(7))};
      const float frw[3] = {fr_r * wq(0), fr_r * wq(1), fr_r * wq(7)};
      // ---- collide on the total (deviation form), perturb, recolour, store
      // Directions 1..18 first; the rest populations then take what is left of rho - 1 and of
      // rho_r (collision conserves both at every site), so that the per-site masses are conserved
      // to the rounding of one sum instead of carrying the relative error of rho_r/rho or of
      // w_q * drho (a systematic drift in uniform regions).
      float racc = 0.f, tacc = 0.f;
      // Guo forcing: opposite directions q, q+1 = opp(q) share (c.u)^2, (c.G)^2, (c.F)(c.u) and differ
      // in the sign of the odd terms, so a pair costs one even part s and one odd part a:
      //   f*_q, f*_opp = (1 - omega) T + s +- a,   red share = fr_r f* + frw +- kc cG
      const float orw45[3] = {0.f, 4.5f * orw[1], 4.5f * orw[2]};
      const float orw3[3] = {0.f, 3.0f * orw[1], 3.0f * orw[2]};
      const float gw3[3] = {0.f, 3.0f * gw[1], 3.0f * gw[2]};
      const float obf[3] = {0.f, (forced && !EDM) ? fmaf(-gw[1], uF, ob[1]) : ob[1], (forced && !EDM) ? fmaf(-gw[2], uF, ob[2]) : ob[2]};
      const float rw3[3] = {0.f, 3.0f * rw[1], 3.0f * rw[2]};
      auto collide = [&](auto bounce) {
      // what happens to every direction once its post-collision pair {ts, rs} is known
      auto finish = [&](auto qc, float ts, float rs) {
        constexpr int q = decltype(qc)::value;
        constexpr float w = wq(q);
        if constexpr (MOVING && q > 0) {
          // moving wall (G28) or open boundary (G31), see open_link; the wall group sits in the
          // neighbour's sentinel (1e30 x group).  The mass sums keep the uncorrected values:
          // a wall pushing on the fluid, an inlet or an outlet changes the mass.
          if ((smask >> q) & 1u) {
            const float sv = plane(cz(q))[(ly + cy(q)) * R_::BX + lx + cx(q)];
            if (sv > 1.5f * PHI_SOLID) open_link<q>(p, (int)(sv > 2.5f * PHI_SOLID) + (int)(sv > 3.5f * PHI_SOLID), rho, rr, inv_rho, ux, uy, uz, uu15, ts, rs);
          }
        }
        const Slot s = write_slot<MODE, decltype(bounce)::value, q>(c, smask);
        *reinterpret_cast<float2*>(dst_ptr(p, s)) = make_float2(ts, rs);
        // f^r* - f^b* = 2 f^r* - f* = (2 rs - w) - ts: the first difference is exact in the mixed
        // regions where phi matters, so the forwarded sum keeps ~1e-8 there
        vd[q] = (2.0f * rs - w) - ts;
        vt[q] = ts;
      };
      // (not in the in-place odd step with near contact or exact-difference forcing: there the pair form spills, and a spill
      // reload queued behind the shifted stores is expensive: C4 AA 15.2 -> 13.1 GLUPS)
      constexpr bool PAIRED = !(MODE == MODE_AA_ODD && (HAS_NC || EDM));
      if constexpr (PAIRED) {
        static_for<0, (Q - 1) / 2>([&](auto pc) {
          constexpr int q = 2 * decltype(pc)::value + 1;   // 1, 3, ..., 17; opp(q) = q + 1
          constexpr int k = q < 7 ? 1 : 2;
          const float cu = cdot<q>(ux, uy, uz);
          const float cG = cdot<q>(Gx, Gy, Gz);
          float s = fmaf(orw45[k], cu * cu, obf[k]);
          // (explicitly rounded product: a force-free run must give the same bits in the forced
          // instantiation, which the in-place modes use, and in the unforced one, where the
          // compiler would otherwise contract this product into the two sums below)
          float a = __fmul_rn(orw3[k], cu);
          if constexpr (forced && !EDM) {
            const float cF = cdot<q>(Fx, Fy, Fz);
            s = fmaf(gw3[k] * cF, cu, s);
            a = fmaf(gw[k], cF, a);
          }
          if constexpr (forced && EDM) {
            // exact difference, ca = c.(v - u) = c.F / rho:
            // S_q / (w rho) = [ca (4.5 ca + 9 cu) - 1.5 (v.v - u.u)] +- 3 ca
            const float ca = cdot<q>(fax, fay, faz);
            s = fmaf(rw[k], fmaf(ca, fmaf(4.5f, ca, 9.0f * cu), -dvv15), s);
            a = fmaf(rw3[k], ca, a);
          }
          s = fmaf(pa[k] * cG, cG, s);
          const float ts0 = __fadd_rn(fmaf(om1, T[q], s), a), ts1 = __fsub_rn(fmaf(om1, T[q + 1], s), a);
          const float rs0 = fmaf(fr_r, ts0, fmaf(kc[k], cG, frw[k])), rs1 = fmaf(fr_r, ts1, fmaf(-kc[k], cG, frw[k]));
          racc += rs0 + rs1;
          tacc += ts0 + ts1;
          finish(std::integral_constant<int, q>{}, ts0, rs0);
          finish(std::integral_constant<int, q + 1>{}, ts1, rs1);
        });
      } else if constexpr (!EDM && WALLS != 1) {
        // the same pairs with the constants of the direction loop only (no orw45, orw3, gw3, obf:
        // four live values fewer, two instructions more per pair), for the in-place odd step
        // (C5 AA 16.45 -> 16.58 GLUPS; not with walls at rest: one spilled value there, whose
        // reload behind the shifted stores took C4 AA from 15.3 to 12.6 GLUPS)
        static_for<0, (Q - 1) / 2>([&](auto pc) {
          constexpr int q = 2 * decltype(pc)::value + 1;
          constexpr int k = q < 7 ? 1 : 2;
          const float cu = cdot<q>(ux, uy, uz);
          const float cG = cdot<q>(Gx, Gy, Gz);
          const float cF = cdot<q>(Fx, Fy, Fz);
          const float cu3 = 3.0f * cu;
          float s = fmaf(orw[k], (1.5f * cu3) * cu, ob[k]);
          s = fmaf(gw[k], fmaf(cF, cu3, -uF), s);
          s = fmaf(pa[k] * cG, cG, s);
          const float a = fmaf(gw[k], cF, __fmul_rn(orw[k], cu3));
          const float ts0 = __fadd_rn(fmaf(om1, T[q], s), a), ts1 = __fsub_rn(fmaf(om1, T[q + 1], s), a);
          const float rs0 = fmaf(fr_r, ts0, fmaf(kc[k], cG, frw[k])), rs1 = fmaf(fr_r, ts1, fmaf(-kc[k], cG, frw[k]));
          racc += rs0 + rs1;
          tacc += ts0 + ts1;
          finish(std::integral_constant<int, q>{}, ts0, rs0);
          finish(std::integral_constant<int, q + 1>{}, ts1, rs1);
        });
      } else {
        static_for<1, Q>([&](auto qc) {
          constexpr int q = decltype(qc)::value;
          constexpr int k = q < 7 ? 1 : 2;
          const float cu = cdot<q>(ux, uy, uz);
          const float cG = cdot<q>(Gx, Gy, Gz);
          float ts = fmaf(om1, T[q], fmaf(orw[k], cu * fmaf(4.5f, cu, 3.0f), ob[k]));
          if constexpr (forced && !EDM) {
            const float cF = cdot<q>(Fx, Fy, Fz);
            ts = fmaf(gw[k], fmaf(cF, fmaf(3.0f, cu, 1.0f), -uF), ts);
          }
          if constexpr (forced && EDM) {
            const float cv = cdot<q>(vx, vy, vz);
            ts = fmaf(rw[k], fmaf(cv - cu, fmaf(4.5f, cv + cu, 3.0f), -dvv15), ts);
          }
          ts = fmaf(pa[k] * cG, cG, ts);
          const float rs = fmaf(fr_r, ts, fmaf(kc[k], cG, frw[k]));
          racc += rs;
          tacc += ts;
          finish(qc, ts, rs);
        });
      }
      finish(std::integral_constant<int, 0>{}, dr - tacc, rr - racc);
      };
      // only the in-place odd step writes to neighbouring sites, so only there the store slots
      // depend on the walls; everywhere else one copy of the loop serves both cases
      if (MODE == MODE_AA_ODD && HAS_SOLID && near_wall) collide(std::integral_constant<bool, HAS_SOLID>{});
      else collide(std::false_type{});
      } else {
        // ---- Shan-Chen model: Eq. 5-10 of the paper.  Accelerations
        // a^k = F^k / rho^k = -G_C sum_i w_i rho^kbar(x + c_i) c_i + g (never divides by rho^k),
        // common bare velocity u = m / rho, each component relaxes to f^eq(rho^k, u) and receives
        // S^k_q = f^eq_q(rho^k, u + a^k) - f^eq_q(rho^k, u)
        //       = w_q rho^k [(cv - cu)(3 + 4.5 (cv + cu)) - 1.5 (v.v - u.u)],  v = u + a^k.
        float arx = -p.G_C * Gx, ary = -p.G_C * Gy, arz = -p.G_C * Gz;
        float abx = -p.G_C * Hx, aby = -p.G_C * Hy, abz = -p.G_C * Hz;
        if constexpr (HAS_G) { arx += p.gx; ary += p.gy; arz += p.gz; abx += p.gx; aby += p.gy; abz += p.gz; }
        const float ux = mx * inv_rho, uy = my * inv_rho, uz = mz * inv_rho;
        float omega = omega_same;
        if (p.two_tau) {
          const float inv_nu = (rr * inv_rho) / nu_r + (rb * inv_rho) / nu_b;
          omega = 1.0f / (3.0f / inv_nu + 0.5f);
        }
        const float om1 = 1.0f - omega;
        const float uu15 = 1.5f * (ux * ux + uy * uy + uz * uz);
        const float vrx = ux + arx, vry = uy + ary, vrz = uz + arz;
        const float vbx = ux + abx, vby = uy + aby, vbz = uz + abz;
        const float dr15 = 1.5f * (vrx * vrx + vry * vry + vrz * vrz) - uu15;
        const float db15 = 1.5f * (vbx * vbx + vby * vby + vbz * vbz) - uu15;
        const float wr[3] = {wq(0) * rr, wq(1) * rr, wq(7) * rr};
        const float wb[3] = {wq(0) * rb, wq(1) * rb, wq(7) * rb};
        const float owd[3] = {omega * wq(0) * dr, omega * wq(1) * dr, omega * wq(7) * dr};
        const float owr[3] = {omega * wq(0) * rho, omega * wq(1) * rho, omega * wq(7) * rho};
        // Pair form (as in the colour-gradient branch): for opposite directions q, opp(q) = q + 1,
        // with cu = c.u and ca = c.a^k,
        //   f^eq_q / (w rho) - 1 = [4.5 cu^2 - 1.5 u.u] +- 3 cu
        //   S^k_q / (w rho^k)    = [ca (4.5 ca + 9 cu) - 1.5 (v.v - u.u)] +- 3 ca
        // so each pair costs one even part and one odd part per component.
        const float wr3[3] = {0.f, 3.0f * wr[1], 3.0f * wr[2]};
        const float wb3[3] = {0.f, 3.0f * wb[1], 3.0f * wb[2]};
        const float owr3[3] = {0.f, 3.0f * owr[1], 3.0f * owr[2]};
        float racc = 0.f, tacc = 0.f;
        auto collide = [&](auto bounce) {
        auto finish = [&](auto qc, float ts, float rs) {
          constexpr int q = decltype(qc)::value;
          constexpr float w = wq(q);
          if constexpr (MOVING && q > 0) {
            // moving wall (G28) or open boundary (G31), see open_link
            if ((smask >> q) & 1u) {
              const float sv = plane(cz(q))[(ly + cy(q)) * R_::BX + lx + cx(q)];
              if (sv > 1.5f * PHI_SOLID) open_link<q>(p, (int)(sv > 2.5f * PHI_SOLID) + (int)(sv > 3.5f * PHI_SOLID), rho, rr, inv_rho, ux, uy, uz, uu15, ts, rs);
            }
          }
          const Slot s = write_slot<MODE, decltype(bounce)::value, q>(c, smask);
          *reinterpret_cast<float2*>(dst_ptr(p, s)) = make_float2(ts, rs);
          vd[q] = (2.0f * rs - w) - ts;
          vt[q] = ts;
        };
        static_for<0, (Q - 1) / 2>([&](auto pc) {
          constexpr int q = 2 * decltype(pc)::value + 1;   // 1, 3, ..., 17; opp(q) = q + 1
          constexpr int k = q < 7 ? 1 : 2;
          const float cu = cdot<q>(ux, uy, uz);
          const float car = cdot<q>(arx, ary, arz), cab = cdot<q>(abx, aby, abz);
          const float cu9 = 9.0f * cu;
          const float ee = fmaf(4.5f * cu, cu, -uu15);                      // even part of f^eq / (w rho) - 1
          const float sre = fmaf(car, fmaf(4.5f, car, cu9), -dr15);          // even parts of S^k / (w rho^k)
          const float sbe = fmaf(cab, fmaf(4.5f, cab, cu9), -db15);
          // red: even and odd part (explicitly rounded products: no contraction into the sums, so
          // that every instantiation computes the same bits)
          const float re = __fmul_rn(wr[k], fmaf(omega, 1.0f + ee, sre));
          const float ro = __fmul_rn(wr3[k], fmaf(omega, cu, car));
          const float rs0 = __fadd_rn(fmaf(om1, R[q], re), ro), rs1 = __fsub_rn(fmaf(om1, R[q + 1], re), ro);
          // total
          const float te = fmaf(wb[k], sbe, fmaf(wr[k], sre, fmaf(owr[k], ee, owd[k])));
          const float to = fmaf(wb3[k], cab, fmaf(wr3[k], car, __fmul_rn(owr3[k], cu)));
          const float ts0 = __fadd_rn(fmaf(om1, T[q], te), to), ts1 = __fsub_rn(fmaf(om1, T[q + 1], te), to);
          racc += rs0 + rs1;
          tacc += ts0 + ts1;
          finish(std::integral_constant<int, q>{}, ts0, rs0);
          finish(std::integral_constant<int, q + 1>{}, ts1, rs1);
        });
        // the rest populations take what is left (mass is conserved)
        finish(std::integral_constant<int, 0>{}, dr - tacc, rr - racc);
        };
        if (MODE == MODE_AA_ODD && HAS_SOLID && near_wall) collide(std::integral_constant<bool, HAS_SOLID>{});
      else collide(std::false_type{});
      }
      if (HAS_SOLID && near_wall) {   // link bounce-back: what would enter a solid site comes back here
        float sd = 0.f, st = 0.f;
        static_for<1, Q>([&](auto qc) {
          constexpr int q = decltype(qc)::value;
          if ((smask >> q) & 1u) { sd += vd[q]; st += vt[q]; vd[q] = 0.f; vt[q] = 0.f; }
        });
        vd[0] += sd;
        vt[0] += st;
      }
    }
    // ---- forward the moments.  x: target lane L receives c_x = +1 values from lane L-1 and
    // c_x = -1 values from lane L+1; nothing crosses the ends of the warp row (brick faces).
    const unsigned full = 0xffffffffu;
    const bool l0 = threadIdx.x == 0, l31 = threadIdx.x == TX - 1;
    auto up = [&](float v) { const float t = __shfl_up_sync(full, v, 1); return l0 ? 0.f : t; };
    auto down = [&](float v) { const float t = __shfl_down_sync(full, v, 1); return l31 ? 0.f : t; };
    // a[cy][cz] after the x step (velocity order: include/lb.h)
    const float a00_d = vd[0] + up(vd[1]) + down(vd[2]),  a00_t = vt[0] + up(vt[1]) + down(vt[2]);
    const float ap0_d = vd[3] + up(vd[7]) + down(vd[10]), ap0_t = vt[3] + up(vt[7]) + down(vt[10]);
    const float am0_d = vd[4] + up(vd[9]) + down(vd[8]),  am0_t = vt[4] + up(vt[9]) + down(vt[8]);
    const float a0p_d = vd[5] + up(vd[11]) + down(vd[14]), a0p_t = vt[5] + up(vt[11]) + down(vt[14]);
    const float a0m_d = vd[6] + up(vd[13]) + down(vd[12]), a0m_t = vt[6] + up(vt[13]) + down(vt[12]);
    // what crosses the x faces: c_x = -1 values of lane 0 (left), c_x = +1 values of the last lane (right)
    const float e00_d = lL ? vd[2] : vd[1],   e00_t = lL ? vt[2] : vt[1];      // (0, 0)
    const float ep0_d = lL ? vd[10] : vd[7],  ep0_t = lL ? vt[10] : vt[7];     // (+1, 0)
    const float em0_d = lL ? vd[8] : vd[9],   em0_t = lL ? vt[8] : vt[9];      // (-1, 0)
    const float e0p_d = lL ? vd[14] : vd[11], e0p_t = lL ? vt[14] : vt[11];    // (0, +1)
    const float e0m_d = lL ? vd[12] : vd[13], e0m_t = lL ? vt[12] : vt[13];    // (0, -1)
    float* xe = xex + (size_t)((jz & 1) * 2 + side) * 4 * TY;
    if (lL || lR) {
      xe[0 * TY + threadIdx.y] = ep0_d; xe[1 * TY + threadIdx.y] = ep0_t;
      xe[2 * TY + threadIdx.y] = em0_d; xe[3 * TY + threadIdx.y] = em0_t;
    }
    // y: rows exchange their c_y = +-1 sums through shared memory (double-buffered by plane parity)
    float* ex = yex + (size_t)(jz & 1) * SM_::NEX * TX * TY;
    const int eo = threadIdx.y * TX + threadIdx.x;
    ex[0 * TX * TY + eo] = ap0_d;   ex[1 * TX * TY + eo] = ap0_t;      // (+1, 0)
    ex[2 * TX * TY + eo] = am0_d;   ex[3 * TX * TY + eo] = am0_t;      // (-1, 0)
    ex[4 * TX * TY + eo] = vd[15];  ex[5 * TX * TY + eo] = vt[15];     // (+1, +1)
    ex[6 * TX * TY + eo] = vd[18];  ex[7 * TX * TY + eo] = vt[18];     // (-1, +1)
    ex[8 * TX * TY + eo] = vd[17];  ex[9 * TX * TY + eo] = vt[17];     // (+1, -1)
    ex[10 * TX * TY + eo] = vd[16]; ex[11 * TX * TY + eo] = vt[16];    // (-1, -1)
    __syncthreads();   // exchange visible; also: every thread is done with ring plane j = jz
    if (tid == 0) {
      const int j = jz + R_::NS;
      if (j < npl) issue(j);
    }
    const bool has_below = threadIdx.y > 0, has_above = threadIdx.y < TY - 1;
    auto below = [&](int slot) { return has_below ? ex[slot * TX * TY + eo - TX] : 0.f; };   // c_y = +1 from row - 1
    auto above = [&](int slot) { return has_above ? ex[slot * TX * TY + eo + TX] : 0.f; };   // c_y = -1 from row + 1
    const float b0_d = a00_d + below(0) + above(2), b0_t = a00_t + below(1) + above(3);
    const float bp_d = a0p_d + below(4) + above(6), bp_t = a0p_t + below(5) + above(7);      // goes to plane z + 1
    const float bm_d = a0m_d + below(8) + above(10), bm_t = a0m_t + below(9) + above(11);    // goes to plane z - 1
    // z: plane z-1 is complete now
    if (jz > 0 && active) {
      const size_t s = col + plane_sites * (size_t)(z - 1);
      p.Md[s] = pend_d + bm_d;
      p.Mt[s] = pend_t + bm_t;
    }
    pend_d = b0_d + bpc_d; pend_t = b0_t + bpc_t;
    bpc_d = bp_d; bpc_t = bp_t;
    if ((lL || lR) && y < b.ny) {
      const float eb_d = e00_d + (has_below ? xe[0 * TY + threadIdx.y - 1] : 0.f) + (has_above ? xe[2 * TY + threadIdx.y + 1] : 0.f);
      const float eb_t = e00_t + (has_below ? xe[1 * TY + threadIdx.y - 1] : 0.f) + (has_above ? xe[3 * TY + threadIdx.y + 1] : 0.f);
      if (jz > 0) {
        float2* o = reinterpret_cast<float2*>(p.EX) + (((size_t)(z - 1) * b.ny + y) * ntx + blockIdx.x) * 2 + side;
        *o = make_float2(pe_d + e0m_d, pe_t + e0m_t);
      }
      pe_d = eb_d + bpe_d; pe_t = eb_t + bpe_t;
      bpe_d = e0p_d; bpe_t = e0p_t;
    }
  }
  if (active) {
    const size_t s = col + plane_sites * (size_t)(ze - 1);
    p.Md[s] = pend_d;
    p.Mt[s] = pend_t;
  }
  if ((lL || lR) && y < b.ny) {
    float2* o = reinterpret_cast<float2*>(p.EX) + (((size_t)(ze - 1) * b.ny + y) * ntx + blockIdx.x) * 2 + side;
    *o = make_float2(pe_d, pe_t);
  }
}

// ----------------------------------------------------------------------------- K1f phase field, forwarded
// phi(t+1) from the moments that k_fused forwarded plus what enters each brick through its faces:
// for a site on a face of its brick (tile-local x = 0 / TX-1, y = 0 / TY-1, z = first / last plane
// of the z chunk, or the last row / column / plane of the box) the directions whose source lies in
// another brick are gathered from the populations k_fused stored, with the read rule of the NEXT
// step (template MODE).  A solid source contributes nothing here: its link bounced back inside
// k_fused.  Interior sites read 8 bytes.  Writes phi with its periodic ghost images like k_phase.
template <int MODE, bool HAS_SOLID, bool SC>
__global__ void __launch_bounds__(TX* TY, 8) k_phase_fwd(const StepParams p) {
  // Four consecutive x sites per thread (128-bit loads and stores).  CTA = 32 quads x TY rows of
  // one plane (four k_fused tiles side by side), so that a warp is one row: the rows on a brick
  // face gather as whole warps and the others skip that code.  nx % 4 == 0: a quad is inside the
  // box or outside.
  const Box& b = p.box;
  const int x = (blockIdx.x * TX + threadIdx.x) * 4;
  const int y = blockIdx.y * TY + threadIdx.y;
  const int z = p.z0 + blockIdx.z;
  if (x >= b.nx || y >= b.ny) return;
  const int tile = x / TX;                            // k_fused tile (brick column) of this quad
  const int qx = threadIdx.x & (TX / 4 - 1);          // quad inside the tile row
  // z range of the k_fused brick this plane belongs to (bricks are counted from the first plane the handle updates)
  const int zb = b.zlo + ((z - b.zlo) / p.zc) * p.zc;
  const int ze = min(b.zhi, zb + p.zc);
  const int H = p.halo;
  const bool xm = qx == 0;                            // element 0 is the first column of its brick
  const bool xp = qx == TX / 4 - 1 || x + 4 == b.nx;  // element 3 is the last column of its brick
  const bool ym = threadIdx.y == 0, yp = threadIdx.y == TY - 1 || y == b.ny - 1;
  const bool zm = z == zb, zp = z == ze - 1;
  const int ntx = (b.nx + TX - 1) / TX;
  const size_t row = (size_t)b.nx * ((size_t)y + (size_t)b.ny * z);
  const size_t idx = row + x;
  const float4 d4 = __ldg(reinterpret_cast<const float4*>(p.Md + idx));
  const float4 t4 = __ldg(reinterpret_cast<const float4*>(p.Mt + idx));
  float d[4] = {d4.x, d4.y, d4.z, d4.w}, t[4] = {t4.x, t4.y, t4.z, t4.w};
  // what the neighbouring bricks sent through the x faces (rows and planes of this brick only)
  const float2* ex = reinterpret_cast<const float2*>(p.EX) + ((size_t)z * b.ny + y) * ntx * 2;
  if (xm) { const float2 v = __ldg(ex + (tile == 0 ? ntx - 1 : tile - 1) * 2 + 1); d[0] += v.x; t[0] += v.y; }
  if (xp) { const float2 v = __ldg(ex + (tile == ntx - 1 ? 0 : tile + 1) * 2 + 0); d[3] += v.x; t[3] += v.y; }
  bool solid[4] = {false, false, false, false};
  float sent[4] = {PHI_SOLID, PHI_SOLID, PHI_SOLID, PHI_SOLID};   // sentinel of a solid site: 1e30 x wall group
  // solid bits of the quad's own sites: x % 4 == 0, so the four bits sit in one mask word
  auto quad_bits = [&](int yy, int zz) -> uint32_t {
    return (b.mask[(size_t)(zz * b.ny + yy) * b.nxw + (x >> 5)] >> (x & 31)) & 0xfu;
  };
  if constexpr (HAS_SOLID) {
    const uint32_t m = quad_bits(y, z);
#pragma unroll
    for (int e = 0; e < 4; ++e) solid[e] = (m >> e) & 1u;
    if (b.gmask != nullptr && m != 0u) {     // moving walls somewhere in the box, and a solid site here
#pragma unroll
      for (int e = 0; e < 4; ++e) sent[e] = PHI_SOLID * (float)wall_group_at(b, x + e, y, z);
    }
  }
  if (ym || yp || zm || zp) {
    // sources in another row range or z chunk are gathered from the stored populations with the
    // read rule of the next step; x-only crossings came through EX; a solid source bounced back
    // inside k_fused
    static_for<1, Q>([&](auto qc) {
      constexpr int q = decltype(qc)::value;
      const bool crosses = (cy(q) > 0 && ym) || (cy(q) < 0 && yp) || (cz(q) > 0 && zm) || (cz(q) < 0 && zp);
      if (crosses) {
        constexpr bool own = MODE == MODE_AA_EVEN;          // AA-even reads its own site
        constexpr int plane = MODE == MODE_AA_ODD ? opp(q) : q;
        constexpr int sx = own ? 0 : cx(q);
        const int ys = own ? y : (cy(q) > 0 ? wrap_m(y, b.ny) : (cy(q) < 0 ? wrap_p(y, b.ny) : y));
        const int zs = own ? z : (cz(q) > 0 ? wrap_m(z, b.nz) : (cz(q) < 0 ? wrap_p(z, b.nz) : z));
        const size_t srow = (size_t)b.nx * ((size_t)ys + (size_t)b.ny * zs);
        float tq[4], rq[4];
        const float2* pl = reinterpret_cast<const float2*>(p.ps[plane]) + srow;   // {T, R} pairs of the source row
        if constexpr (sx == 0) {
          const float4 a = __ldg(reinterpret_cast<const float4*>(pl + x));
          const float4 r = __ldg(reinterpret_cast<const float4*>(pl + x + 2));
          tq[0] = a.x; rq[0] = a.y; tq[1] = a.z; rq[1] = a.w;
          tq[2] = r.x; rq[2] = r.y; tq[3] = r.z; rq[3] = r.w;
        } else {      // sources x - 1 .. x + 2 or x + 1 .. x + 4: the aligned quad plus one site beyond its end
          const float4 a = __ldg(reinterpret_cast<const float4*>(pl + x));
          const float4 r = __ldg(reinterpret_cast<const float4*>(pl + x + 2));
          const float2 ext = __ldg(pl + (sx > 0 ? (x == 0 ? b.nx - 1 : x - 1) : (x + 4 >= b.nx ? 0 : x + 4)));
          if constexpr (sx > 0) {
            tq[0] = ext.x; rq[0] = ext.y; tq[1] = a.x; rq[1] = a.y; tq[2] = a.z; rq[2] = a.w; tq[3] = r.x; rq[3] = r.y;
          } else {
            tq[0] = a.z; rq[0] = a.w; tq[1] = r.x; rq[1] = r.y; tq[2] = r.z; rq[2] = r.w; tq[3] = ext.x; rq[3] = ext.y;
          }
        }
        // is the site a population comes from (x + e - c_q) solid?  One mask word for the quad of
        // the source row, plus the one site beyond its end when c_x != 0
        uint32_t sm = 0;
        if constexpr (HAS_SOLID) {
          const int yq = cy(q) > 0 ? wrap_m(y, b.ny) : (cy(q) < 0 ? wrap_p(y, b.ny) : y);
          const int zq = cz(q) > 0 ? wrap_m(z, b.nz) : (cz(q) < 0 ? wrap_p(z, b.nz) : z);
          const uint32_t m = quad_bits(yq, zq);
          if constexpr (cx(q) == 0) sm = m;
          else if constexpr (cx(q) > 0) sm = (m << 1) | (solid_at(b, x == 0 ? b.nx - 1 : x - 1, yq, zq) ? 1u : 0u);
          else sm = (m >> 1) | (solid_at(b, x + 4 >= b.nx ? 0 : x + 4, yq, zq) ? 8u : 0u);
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const bool use = !((sm >> e) & 1u);
          if (use) {
            d[e] += (2.0f * rq[e] - wq(q)) - tq[e];
            t[e] += tq[e];
          }
        }
      }
    });
  }
  // phi of the quad goes to its home in the padded array and to every periodic image that falls into
  // the ghost layers (depth H).  Images are taken row by row: a row has at most one image along y and
  // one along z (two in a box thinner than 2 H), the same for a whole warp, and within a row only the
  // first and the last quad have images along x: one 128-bit store per row image plus the few x
  // images of those two quads.  (A warp spans 128 sites, so in a box of nx <= 256 EVERY warp holds
  // such a quad; sending whole warps through per-site image code, 27 candidates per site, was 40 % of
  // this kernel's instructions, and all of them in rows within H of a y or z face: C4.)
  float f0[4], f1[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    const float rho = 1.0f + t[e];
    if constexpr (!SC) {
      f0[e] = solid[e] ? sent[e] : d[e] / rho;
    } else {
      f0[e] = solid[e] ? sent[e] : 0.5f * (rho + d[e]);
      f1[e] = solid[e] ? 0.f : 0.5f * (rho - d[e]);
    }
  }
  const size_t px = b.nx + 2 * HALO, py = b.ny + 2 * HALO;
  const int sy[3] = {0, y < H ? b.ny : 0, y >= b.ny - H ? -b.ny : 0};
  const int sz[3] = {0, (b.zper && z < H) ? b.nz : 0, (b.zper && z >= b.nz - H) ? -b.nz : 0};    // (a slab's z ghost planes come from its neighbours)
#pragma unroll
  for (int iz = 0; iz < 3; ++iz) {
    if (iz && !sz[iz]) continue;
#pragma unroll
    for (int iy = 0; iy < 3; ++iy) {
      if (iy && !sy[iy]) continue;
      const size_t o = (size_t)(x + HALO) + px * ((size_t)(y + sy[iy] + HALO) + py * (size_t)(z + sz[iz] + HALO));
      *reinterpret_cast<float4*>(p.phi + o) = make_float4(f0[0], f0[1], f0[2], f0[3]);
      if constexpr (SC) *reinterpret_cast<float4*>(p.phi2 + o) = make_float4(f1[0], f1[1], f1[2], f1[3]);
      if (x < H) {                       // x = 0 (H <= 4 = the quad): sites 0 .. H-1 also stand behind nx - 1
#pragma unroll
        for (int e = 0; e < 4; ++e)
          if (e < H) {
            p.phi[o + b.nx + e] = f0[e];
            if constexpr (SC) p.phi2[o + b.nx + e] = f1[e];
          }
      }
      if (x + 4 > b.nx - H) {            // x = nx - 4: sites nx - H .. nx - 1 also stand before 0
#pragma unroll
        for (int e = 0; e < 4; ++e)
          if (e >= 4 - H) {
            p.phi[o - b.nx + e] = f0[e];
            if constexpr (SC) p.phi2[o - b.nx + e] = f1[e];
          }
      }
    }
  }
}

// ----------------------------------------------------------------------------- K2s single component
template <int MODE, bool HAS_SOLID>
__global__ void __launch_bounds__(TX* TY) k_single(const StepParams p) {
  const Box& b = p.box;
  const int x = blockIdx.x * TX + threadIdx.x;
  const int y = blockIdx.y * TY + threadIdx.y;
  if (x >= b.nx || y >= b.ny) return;
  const int zb = p.z0 + blockIdx.z * p.zc;
  const int ze = min(p.z1, zb + p.zc);
  const float omega = 1.0f / p.tau_r;
  const float om1 = 1.0f - omega, g0 = 1.0f - 0.5f * omega;
  for (int z = zb; z < ze; ++z) {
    uint32_t smask = 0, g2m = 0, g3m = 0;
    if constexpr (HAS_SOLID) {
      if (solid_at(b, x, y, z)) continue;
      smask = neighbour_mask(b, x, y, z);
      if (p.has_moving && smask) { neighbour_groups(b, x, y, z, g2m, g3m); g2m &= smask; g3m &= smask; }
    }
    Ctx c;
    make_ctx<4>(c, b, x, y, z);
    float T[Q];
    static_for<0, Q>([&](auto qc) {
      constexpr int q = decltype(qc)::value;
      T[q] = ld_pop<MODE>(src_ptr(p, read_slot<MODE, HAS_SOLID, q>(c, smask)));
    });
    float dr = 0.f, mx = 0.f, my = 0.f, mz = 0.f;
    static_for<0, Q>([&](auto qc) {
      constexpr int q = decltype(qc)::value;
      dr += T[q];
      if constexpr (cx(q) != 0) mx += cx(q) * T[q];
      if constexpr (cy(q) != 0) my += cy(q) * T[q];
      if constexpr (cz(q) != 0) mz += cz(q) * T[q];
    });
    const float rho = 1.0f + dr, inv_rho = 1.0f / rho;
    float Fx = 0.f, Fy = 0.f, Fz = 0.f;
    if (p.has_g) { Fx = rho * p.gx; Fy = rho * p.gy; Fz = rho * p.gz; }
    const float hs = p.edm ? 0.0f : 0.5f;
    const float ux = (mx + hs * Fx) * inv_rho, uy = (my + hs * Fy) * inv_rho, uz = (mz + hs * Fz) * inv_rho;
    const float uu15 = 1.5f * (ux * ux + uy * uy + uz * uz);
    const float uF = ux * Fx + uy * Fy + uz * Fz;
    const float vx = ux + Fx * inv_rho, vy = uy + Fy * inv_rho, vz = uz + Fz * inv_rho;
    const float dvv15 = 1.5f * (vx * vx + vy * vy + vz * vz) - uu15;
    float tacc = 0.f;   // the rest population takes what is left of rho - 1 (see k_fused)
    static_for<1, Q + 1>([&](auto qc) {
      constexpr int q = decltype(qc)::value % Q;   // 1, 2, ..., 18, 0
      constexpr float w = wq(q);
      const float cu = cdot<q>(ux, uy, uz);
      const float teq = w * (dr + rho * (3.0f * cu + 4.5f * cu * cu - uu15));
      float ts = om1 * T[q] + omega * teq;
      if (p.has_g) {
        if (p.edm) {      // exact difference (Eq. 9)
          const float cv = cdot<q>(vx, vy, vz);
          ts += (rho * w) * ((cv - cu) * (3.0f + 4.5f * (cv + cu)) - dvv15);
        } else {
          const float cF = cdot<q>(Fx, Fy, Fz);
          ts += g0 * w * (3.0f * (cF - uF) + 9.0f * cu * cF);
        }
      }
      if constexpr (q > 0) tacc += ts;
      else ts = dr - tacc;
      if constexpr (HAS_SOLID && q > 0) {      // moving wall (G28) or open boundary (G31), see open_link
        if ((g2m | g3m) >> q & 1u) {
          float rs = 0.f;                      // one component: rho_r is the density
          open_link<q, true>(p, (int)((g2m >> q) & 1u) + 2 * (int)((g3m >> q) & 1u) - 1, rho, rho, inv_rho, ux, uy, uz, uu15, ts, rs);
        }
      }
      *dst_ptr(p, write_slot<MODE, HAS_SOLID, q>(c, smask)) = ts;
    });
  }
}

// ----------------------------------------------------------------------------- cold kernels
// One thread per site of the planes [box.zlo, box.zhi) the handle owns.  The caller's arrays hold
// those planes only (a slab's ghost planes are internal): element e = s - s0 of a field, plane
// stride Sx = s1 - s0 between the 19 directions of a population array.  Addressing is that of the
// hot kernels (compile-time direction, Ctx byte deltas, one 64-bit access per {T, R} pair).
struct IoParams {
  float* buf;            // population buffer
  const float* ps[Q];    // its direction planes, as in StepParams
  float* pd[Q];
  Box box;
  long long s0, s1;      // allocated site indices the caller's arrays stand for: [zlo, zhi) x ny x nx
  long long c0, c1;      // elements [c0, c1) of those arrays that THIS launch treats (all: 0, s1 - s0)
  int comp;              // component of k_scatter / k_gatherf
  const float* in0;      // k_scatter: f[19][Sx] full populations (or nullptr: from rho,u)
  const float* rho_r;    // init fields
  const float* rho_b;
  const float* u;
  float* out0;           // k_gatherf / k_macros outputs
  float* out1;
  float* out2;
  const float* phi;      // padded phi (k_macros); rho_r in the Shan-Chen model
  const float* phi2;     // Shan-Chen model: padded rho_b
  int sc;                // Shan-Chen model
  float G_C;
  float tau_r, tau_b, A, beta, A_nc, phi_c, gx, gy, gz;
  int nc_sym, wet;       // as in StepParams
  float phi_wall;
};

struct IoSite {
  long long s, e, Sx;
  int x, y, z;
  bool inside, solid;
  uint32_t smask;
  Ctx c;
};

template <int ESZ, bool HAS_SOLID>
__device__ __forceinline__ IoSite io_site(const IoParams& p) {
  IoSite t;
  const Box& b = p.box;
  t.e = p.c0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;
  t.s = p.s0 + t.e;
  t.Sx = p.s1 - p.s0;
  t.inside = t.e < p.c1;
  t.solid = false;
  t.smask = 0;
  t.x = t.y = t.z = 0;
  if (t.inside) {
    t.x = (int)(t.s % b.nx); t.y = (int)((t.s / b.nx) % b.ny); t.z = (int)(t.s / ((long long)b.nx * b.ny));
    if constexpr (HAS_SOLID) {
      t.solid = solid_at(b, t.x, t.y, t.z);
      if (!t.solid) t.smask = neighbour_mask(b, t.x, t.y, t.z);
    }
    make_ctx<ESZ>(t.c, b, t.x, t.y, t.z);
  }
  return t;
}

// K0: write the pre-collision state where the next gather will look for it.
//   comp < 0 : equilibrium init from rho_r, rho_b, u (Eq. 2), both components
//   comp = 0 : red populations from in0; the T planes receive f^r - w (blue must follow)
//   comp = 1 : blue populations from in0 are ADDED to the T planes
template <int MODE, bool TWO, bool HAS_SOLID>
__global__ void __launch_bounds__(256) k_scatter(const IoParams p) {
  const IoSite t = io_site<TWO ? 8 : 4, HAS_SOLID>(p);
  if (!t.inside || t.solid) return;
  float rr = 0.f, rb = 0.f, ux = 0.f, uy = 0.f, uz = 0.f;
  if (p.comp < 0) {
    rr = __ldg(p.rho_r + t.e);
    rb = TWO ? __ldg(p.rho_b + t.e) : 0.f;
    ux = __ldg(p.u + t.e); uy = __ldg(p.u + t.Sx + t.e); uz = __ldg(p.u + 2 * t.Sx + t.e);
  }
  const float uu15 = 1.5f * (ux * ux + uy * uy + uz * uz);
  const float drho = (rr + rb) - 1.0f;
  static_for<0, Q>([&](auto qc) {
    constexpr int q = decltype(qc)::value;
    constexpr float w = wq(q);
    float* dst = const_cast<float*>(src_ptr(p, read_slot<MODE, HAS_SOLID, q>(t.c, t.smask)));
    if (p.comp < 0) {
      const float cu = cdot<q>(ux, uy, uz);
      const float e = 3.0f * cu + 4.5f * cu * cu - uu15;       // feq/(w rho) - 1
      const float tv = w * (drho + (rr + rb) * e);             // total as deviation
      if constexpr (TWO) *reinterpret_cast<float2*>(dst) = make_float2(tv, w * rr * (1.0f + e));
      else *dst = tv;
    } else {
      const float f = __ldg(p.in0 + (size_t)q * t.Sx + t.e);
      if (p.comp == 0) {
        if constexpr (TWO) *reinterpret_cast<float2*>(dst) = make_float2(f - w, f);
        else *dst = f - w;
      } else {
        *dst += f;
      }
    }
  });
}

// Debug accessor: full pre-collision populations of one component, [19][Sx].
template <int MODE, bool TWO, bool HAS_SOLID>
__global__ void __launch_bounds__(256) k_gatherf(const IoParams p) {
  const IoSite t = io_site<TWO ? 8 : 4, HAS_SOLID>(p);
  if (!t.inside) return;
  static_for<0, Q>([&](auto qc) {
    constexpr int q = decltype(qc)::value;
    float v = 0.f;
    if (!t.solid) {
      const float* src = src_ptr(p, read_slot<MODE, HAS_SOLID, q>(t.c, t.smask));
      if constexpr (TWO) {
        const float2 tr = __ldcg(reinterpret_cast<const float2*>(src));
        v = p.comp == 0 ? tr.y : (tr.x + wq(q)) - tr.y;
      } else {
        v = __ldcg(src) + wq(q);
      }
    }
    p.out0[(size_t)q * t.Sx + t.e] = v;
  });
}

// K3: rho_r, rho_b and u = (m + F/2)/rho (Eq. 3; half-force shift of Guo forcing).
// Needs the phi array of the current state (K1 must have run).  out0 = rho_r, out1 = rho_b,
// out2 = u[3][Sx]; any may be null.
template <int MODE, bool TWO, bool HAS_SOLID>
__global__ void __launch_bounds__(256) k_macros(const IoParams p) {
  const IoSite t = io_site<TWO ? 8 : 4, HAS_SOLID>(p);
  if (!t.inside) return;
  const Box& b = p.box;
  const int x = t.x, y = t.y, z = t.z;
  float rr = 0.f, rb = 0.f, ux = 0.f, uy = 0.f, uz = 0.f;
  if (!t.solid) {
    float dr = 0.f, mx = 0.f, my = 0.f, mz = 0.f;
    static_for<0, Q>([&](auto qc) {
      constexpr int q = decltype(qc)::value;
      const float* src = src_ptr(p, read_slot<MODE, HAS_SOLID, q>(t.c, t.smask));
      float tv;
      if constexpr (TWO) {
        const float2 tr = __ldcg(reinterpret_cast<const float2*>(src));
        tv = tr.x;
        rr += tr.y;
      } else {
        tv = __ldcg(src);
      }
      dr += tv;
      if constexpr (cx(q) != 0) mx += cx(q) * tv;
      if constexpr (cy(q) != 0) my += cy(q) * tv;
      if constexpr (cz(q) != 0) mz += cz(q) * tv;
    });
    const float rho = 1.0f + dr;
    if (!TWO) rr = rho;
    rb = TWO ? rho - rr : 0.f;
    float Fx = rho * p.gx, Fy = rho * p.gy, Fz = rho * p.gz;
    if (TWO && p.sc) {
      // Shan-Chen (Eq. 10; G27): F = rho_r a^r + rho_b a^b, g included
      const size_t o0 = phi_index(b, x, y, z);
      const long long px = b.nx + 2 * HALO, pxy = px * (b.ny + 2 * HALO);
      const float r0 = p.phi[o0], b0 = p.phi2[o0];
      float Sbx = 0.f, Sby = 0.f, Sbz = 0.f, Srx = 0.f, Sry = 0.f, Srz = 0.f;
      for (int q = 1; q < Q; ++q) {
        const long long d = c_cx[q] + px * c_cy[q] + pxy * c_cz[q];
        float vr = p.phi[o0 + d], vb = p.phi2[o0 + d];
        if (vr > PHI_SOLID_TEST) { vr = r0; vb = b0; }
        const float k = wq(q);
        Sbx += k * c_cx[q] * vb; Sby += k * c_cy[q] * vb; Sbz += k * c_cz[q] * vb;
        Srx += k * c_cx[q] * vr; Sry += k * c_cy[q] * vr; Srz += k * c_cz[q] * vr;
      }
      Fx += -p.G_C * (rr * Sbx + rb * Srx); Fy += -p.G_C * (rr * Sby + rb * Sry); Fz += -p.G_C * (rr * Sbz + rb * Srz);
    } else if (TWO && p.A_nc != 0.f) {
      const float* ph = p.phi + phi_index(b, x, y, z);
      const long long px = b.nx + 2 * HALO, pxy = px * (b.ny + 2 * HALO);
      const float phi0 = ph[0];
      float Gx = 0.f, Gy = 0.f, Gz = 0.f;
      for (int q = 1; q < Q; ++q) {
        float v = ph[c_cx[q] + px * c_cy[q] + pxy * c_cz[q]];
        if (v > PHI_SOLID_TEST) v = p.wet ? p.phi_wall : phi0;
        const float k = 3.0f * wq(q);
        Gx += k * c_cx[q] * v; Gy += k * c_cy[q] * v; Gz += k * c_cz[q] * v;
      }
      const float Gn = sqrtf(Gx * Gx + Gy * Gy + Gz * Gz);
      if (fabsf(phi0) < p.phi_c && Gn > EPS_G) {
        const float invG = 1.0f / Gn;
        const float nx_ = -Gx * invG, ny_ = -Gy * invG, nz_ = -Gz * invG;
        float Ah = 0.f;
        for (int sgn = 1; sgn >= (p.nc_sym ? -1 : 1); sgn -= 2) {     // +1: along -G; -1: the mirrored probe (G29)
          int h = 0;
          for (int k = 1; k <= H_MAX_NC; ++k) {
            const int dx = sgn * (int)roundf(k * nx_), dy = sgn * (int)roundf(k * ny_), dz = sgn * (int)roundf(k * nz_);
            const float v = ph[dx + px * dy + pxy * dz];
            if (v > PHI_SOLID_TEST) break;
            if (k >= 2 && (sgn > 0 ? v >= phi0 : v <= phi0)) { h = k; break; }
          }
          if (h > 0) Ah += sgn * (h <= H_MIN_NC ? p.A_nc : p.A_nc * ((float)(H_MIN_NC * H_MIN_NC * H_MIN_NC) / (float)(h * h * h)));
        }
        Fx += 0.5f * Ah * Gx; Fy += 0.5f * Ah * Gy; Fz += 0.5f * Ah * Gz;
      }
    }
    const float inv_rho = 1.0f / rho;
    ux = (mx + 0.5f * Fx) * inv_rho; uy = (my + 0.5f * Fy) * inv_rho; uz = (mz + 0.5f * Fz) * inv_rho;
  }
  if (p.out0) p.out0[t.e] = rr;
  if (p.out1 && TWO) p.out1[t.e] = rb;
  if (p.out2) { p.out2[t.e] = ux; p.out2[t.Sx + t.e] = uy; p.out2[2 * t.Sx + t.e] = uz; }
}

// State check (G23: "lb_step reports LB_ESTATE if the mass check it runs every 1000 steps
// is non-finite"; the paper names fault tolerance as an exascale issue): the component
// masses sum_x rho_k(x), rho_k = sum_q f^k_q (Eq. 3), over the handle's own fluid sites,
// gathered with the read rule of the current storage mode like every other kernel.
// out[0] += sum rho_r, out[1] += sum rho_b, out[2] += number of sites holding a non-finite value.
template <int MODE, bool TWO, bool HAS_SOLID>
__global__ void __launch_bounds__(256) k_check(const IoParams p, double* out) {
  const Box& b = p.box;
  double sr = 0.0, sb = 0.0, bad = 0.0;
  for (long long s = p.s0 + (long long)blockIdx.x * blockDim.x + threadIdx.x; s < p.s1; s += (long long)gridDim.x * blockDim.x) {
    const int x = (int)(s % b.nx), y = (int)((s / b.nx) % b.ny), z = (int)(s / ((long long)b.nx * b.ny));
    uint32_t smask = 0;
    if constexpr (HAS_SOLID) {
      if (solid_at(b, x, y, z)) continue;
      smask = neighbour_mask(b, x, y, z);
    }
    Ctx c;
    make_ctx<TWO ? 8 : 4>(c, b, x, y, z);
    float t = 0.f, r = 0.f;
    static_for<0, Q>([&](auto qc) {
      constexpr int q = decltype(qc)::value;
      const float* src = src_ptr(p, read_slot<MODE, HAS_SOLID, q>(c, smask));
      if constexpr (TWO) {
        const float2 v = __ldcg(reinterpret_cast<const float2*>(src));
        t += v.x; r += v.y;
      } else {
        t += __ldcg(src);
      }
    });
    if (!isfinite(t) || !isfinite(r)) { bad += 1.0; continue; }
    if constexpr (TWO) { sr += (double)r; sb += (double)(1.0f + t) - (double)r; }
    else sr += (double)(1.0f + t);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    sr += __shfl_down_sync(0xffffffffu, sr, o);
    sb += __shfl_down_sync(0xffffffffu, sb, o);
    bad += __shfl_down_sync(0xffffffffu, bad, o);
  }
  __shared__ double red[3][8];
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  if (lane == 0) { red[0][wp] = sr; red[1][wp] = sb; red[2][wp] = bad; }
  __syncthreads();
  if (threadIdx.x < 3) {
    double v = 0.0;
    for (int i = 0; i < 8; ++i) v += red[threadIdx.x][i];
    if (v != 0.0) atomicAdd(out + threadIdx.x, v);
  }
}

// phi without ghost layers or sentinels, for lb_get_phi (Shan-Chen: from the rho_r, rho_b arrays)
__global__ void k_unpad_phi(const float* phi, const float* phi2, float* out, Box b, long long s0, long long s1) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long s = s0 + e;
  if (s >= s1) return;
  const int x = (int)(s % b.nx), y = (int)((s / b.nx) % b.ny), z = (int)(s / ((long long)b.nx * b.ny));
  const float v = phi[phi_index(b, x, y, z)];
  if (v > PHI_SOLID_TEST) { out[e] = 0.f; return; }
  if (phi2) {
    const float w = phi2[phi_index(b, x, y, z)];
    out[e] = (v - w) / (v + w);
  } else {
    out[e] = v;
  }
}

// ----------------------------------------------------------------------------- rigid particles (NEXT-4)
// The paper's section 6: rigid spheres obeying Newton's equations (Eq. 15), solved
// "by a leapfrog approach, using quaternion algebra for the rotational component"; the coupling to the
// fluid is only cited there.  Readings G32-G37 (DESIGN.md section 2 states them in full).  Per
// time step, between the fused kernel (which applies the link rule G33 to what it stores) and the next
// step:  k_part_force (momentum the links handed over), k_part_pair (pair forces G37), k_part_integrate
// (leapfrog and quaternion G35), k_part_remap (nodes that entered or left a particle, G36).  A/B storage only: the
// kernels read the state of time t from the source buffer and work on the stored post-collision
// values of the destination buffer, each at its own site.  One CTA per particle; all sums in double
// precision and in a fixed order (the result does not depend on the scheduling).
struct PartParams {
  const float* ps[Q];    // source buffer (state of time t, pull layout)
  float* pd[Q];          // destination buffer: post-collision values of time t at their own sites
  Box box;               // mask and pid are those of time t until k_part_remap has changed them
  uint32_t* mask;        // writable view of box.mask; the particle index per site (-1: none)
  int* pid;
  PState* parts;
  int np;
  int mobile;            // 0: the particles are held in place
  double K, hc, mu;      // pair force (G37); mu = rho_0 nu
  int lub;
  int* overflow;         // set if a particle changed more nodes in one step than k_part_remap can list
  // a slab of a larger box (replicated data): every rank holds all particles and sums
  // what its own planes contribute; the sums over the ranks come back from the caller's all-reduce
  double* part_out;      // [np][6] this slab's share of the link sums (k_part_force) / of the impulses (k_part_remap); nullptr: undivided box
  const double* tot_in;  // [np][6] the sums over all slabs (k_part_pair: F, T; k_part_apply: dU, dL)
  const float* ghost_rho;   // [2 faces][2 components][ny * nx] densities of time t in the ghost planes (lb_slab_unpack_phi)
};

constexpr int PART_MAXCH = 384;   // changed nodes per particle and step that k_part_remap can hold

// Coordinates.  A particle lives in the whole periodic box, nx x ny x gnz, and its state is the same
// on every rank that holds a slab of that box ("replicated data").  The kernels
// below index SITES by the handle's allocated planes, z in [0, b.nz), of which [b.zlo, b.zhi) are its
// own; plane z stands at global z + b.zoff (mod gnz).  Distances to a particle are taken in global
// coordinates.  Undivided box: gnz = b.nz, zoff = 0, every plane its own.
__device__ __forceinline__ int global_z(const Box& b, int z) {
  const int g = z + b.zoff;
  return g < 0 ? g + b.gnz : (g >= b.gnz ? g - b.gnz : g);
}
__device__ __forceinline__ bool own_plane(const Box& b, int z) { return z >= b.zlo && z < b.zhi; }

struct PartBox { int lo[3], ext[3]; };    // in global coordinates
__device__ __forceinline__ PartBox part_box(const Box& b, const double r[3], double reach) {
  PartBox pb;
  const int n[3] = {b.nx, b.ny, b.gnz};
  for (int a = 0; a < 3; ++a) {
    int lo = (int)floor(r[a] - reach), hi = (int)ceil(r[a] + reach);
    if (hi - lo + 1 > n[a]) { lo = 0; hi = n[a] - 1; }      // never visit a node twice
    pb.lo[a] = lo; pb.ext[a] = hi - lo + 1;
  }
  return pb;
}
// The allocated plane that holds global plane zg, or -1.  A ring of ONE slab holds the planes next to its
// own faces twice (own plane and the ghost plane on the other side): img = 0 / 1 asks for the first /
// second copy.
__device__ __forceinline__ int local_z(const Box& b, int zg, int img = 0) {
  int z = zg - b.zoff;
  z = z < 0 ? z + b.gnz : (z >= b.gnz ? z - b.gnz : z);
  z += img * b.gnz;
  return z < b.nz ? z : -1;
}
// node i of the box: site coordinates (x, y, z); false if this handle does not hold (that copy of) its plane
__device__ __forceinline__ bool part_box_node(const Box& b, const PartBox& pb, int i, int& x, int& y, int& z, int img = 0) {
  const int lx = i % pb.ext[0], ly = (i / pb.ext[0]) % pb.ext[1], lz = i / (pb.ext[0] * pb.ext[1]);
  x = (pb.lo[0] + lx) % b.nx; if (x < 0) x += b.nx;
  y = (pb.lo[1] + ly) % b.ny; if (y < 0) y += b.ny;
  int zg = (pb.lo[2] + lz) % b.gnz; if (zg < 0) zg += b.gnz;
  z = local_z(b, zg, img);
  return z >= 0;
}
__device__ __forceinline__ bool inside_particle(const Box& b, const PState& P, int x, int y, int z) {
  const double dx = min_image(x - P.r[0], b.nx), dy = min_image(y - P.r[1], b.ny), dz = min_image(global_z(b, z) - P.r[2], b.gnz);
  return dx * dx + dy * dy + dz * dz < P.R * P.R;
}
__device__ __forceinline__ size_t site_of(const Box& b, int x, int y, int z) { return (size_t)x + (size_t)b.nx * ((size_t)y + (size_t)b.ny * z); }
// the neighbour of site (x, y, z) along c_q; false if this handle does not hold its plane (a slab's
// ghost planes have neighbours on one side only)
__device__ __forceinline__ bool nbr_of(const Box& b, int x, int y, int z, int q, int& xn, int& yn, int& zn) {
  xn = x + c_cx[q]; yn = y + c_cy[q]; zn = z + c_cz[q];
  xn = xn < 0 ? b.nx - 1 : (xn >= b.nx ? 0 : xn);
  yn = yn < 0 ? b.ny - 1 : (yn >= b.ny ? 0 : yn);
  if (b.zper) { zn = zn < 0 ? b.nz - 1 : (zn >= b.nz ? 0 : zn); return true; }
  return zn >= 0 && zn < b.nz;
}

// rho_r, rho_b (one component: rho, 0) of the fluid site (x, y, z) at time t (Eq. 3): its
// pre-collision populations gathered from the source buffer with the pull rule
template <bool TWO>
__device__ __forceinline__ void site_density(const PartParams& p, int x, int y, int z, float& rr, float& rb) {
  if (!own_plane(p.box, z)) {      // a slab's ghost plane: what the rank that owns it has sent (lb_slab_pack_phi)
    const size_t n = (size_t)p.box.nx * p.box.ny, o = (size_t)x + (size_t)p.box.nx * y;
    const float* g = p.ghost_rho + (z < p.box.zlo ? 0 : 2) * n;
    rr = g[o]; rb = g[n + o];
    return;
  }
  Ctx c;
  make_ctx<TWO ? 8 : 4>(c, p.box, x, y, z);
  const uint32_t smask = neighbour_mask(p.box, x, y, z);
  float t = 0.f, r = 0.f;
  static_for<0, Q>([&](auto qc) {
    constexpr int q = decltype(qc)::value;
    const float* src = src_ptr(p, read_slot<MODE_AB, true, q>(c, smask));
    if constexpr (TWO) { const float2 v = __ldcg(reinterpret_cast<const float2*>(src)); t += v.x; r += v.y; }
    else t += __ldcg(src);
  });
  if constexpr (TWO) { rr = r; rb = (1.0f + t) - r; }
  else { rr = 1.0f + t; rb = 0.f; }
}

// A slab with particles: rho_r, rho_b of its lowest and highest own plane (zero at solid sites), which
// travel with the phi halo and become the neighbours' ghost densities (site_density; G36 fills a node
// that leaves a particle at the mean densities of its fluid neighbours).  grid = (sites of a plane / 256, 2 faces).
template <bool TWO>
__global__ void __launch_bounds__(256) k_slab_rho(const PartParams p, float* out_lo, float* out_hi) {
  const Box& b = p.box;
  const int n = b.nx * b.ny, o = blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= n) return;
  const int x = o % b.nx, y = o / b.nx, z = blockIdx.y == 0 ? b.zlo : b.zhi - 1;
  float rr = 0.f, rb = 0.f;
  if (!solid_at(b, x, y, z)) site_density<TWO>(p, x, y, z, rr, rb);
  float* out = blockIdx.y == 0 ? out_lo : out_hi;
  out[o] = rr;
  out[n + o] = rb;
}

// stored post-collision pair of direction q at its own site (A/B layout)
template <bool TWO>
__device__ __forceinline__ float* own_slot(const PartParams& p, int q, size_t s) { return p.pd[q] + s * (TWO ? 2 : 1); }

// u_b . c_q at the midpoint of the link (x, y, z) -> + c_q, run-time q
__device__ __forceinline__ double link_cu_rt(const Box& b, const double r[3], const double u[3], const double w[3], int x, int y, int z, int q, double rel[3]) {
  rel[0] = min_image(x - r[0], b.nx) + 0.5 * c_cx[q];
  rel[1] = min_image(y - r[1], b.ny) + 0.5 * c_cy[q];
  rel[2] = min_image(global_z(b, z) - r[2], b.gnz) + 0.5 * c_cz[q];
  // in fp32 like k_fused (link_cu), so that undoing a link reproduces the stored value
  const float rx = (float)rel[0], ry = (float)rel[1], rz = (float)rel[2];
  const float wx = (float)w[0], wy = (float)w[1], wz = (float)w[2];
  const float ux = (float)u[0] + (wy * rz - wz * ry), uy = (float)u[1] + (wz * rx - wx * rz), uz = (float)u[2] + (wx * ry - wy * rx);
  return (double)((float)c_cx[q] * ux + (float)c_cy[q] * uy + (float)c_cz[q] * uz);
}

// sum of NV doubles per thread over the CTA in a fixed order; result in every thread of warp 0 lane 0 -> out
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* red /* [NV][8] shared */) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1)
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  if (lane == 0)
    for (int k = 0; k < NV; ++k) red[k * 8 + wp] = v[k];
  __syncthreads();
  if (threadIdx.x == 0)
    for (int k = 0; k < NV; ++k) {
      double a = 0.0;
      for (int i = 0; i < 8; ++i) a += red[k * 8 + i];
      v[k] = a;
    }
}

// A warp scans the rows row0, row0 + stride, ... of the bounding box pb of a sphere centred at r and
// queues the nodes with rin2 <= d^2 <= rout2 that pass keep(x, y, z); the costly part, process(site),
// then runs on 32 queued nodes at a time, all lanes busy.  Which lane treats which node is fixed by
// the scan order, so sums formed in process() do not depend on the scheduling.  queue: 64 ints of
// shared memory owned by this warp.
template <class Keep, class Process>
__device__ __forceinline__ void scan_shell(const Box& b, const PartBox& pb, const double r[3], float rin2, float rout2,
                                           int row0, int stride, int* queue, Keep keep, Process process) {
  const int lane = threadIdx.x & 31, nrows = pb.ext[1] * pb.ext[2];
  const float cxr = (float)r[0], cyr = (float)r[1], czr = (float)r[2];
  int qn = 0;
  for (int row = row0; row < nrows; row += stride) {
    const int ly = row % pb.ext[1], lz = row / pb.ext[1];
    int y = pb.lo[1] + ly, zg = pb.lo[2] + lz;
    y += y < 0 ? b.ny : (y >= b.ny ? -b.ny : 0);
    zg += zg < 0 ? b.gnz : (zg >= b.gnz ? -b.gnz : 0);
    float fy = (float)y - cyr, fz = (float)zg - czr;       // fp32 is enough for the prefilter
    fy += fy > 0.5f * b.ny ? -(float)b.ny : (fy < -0.5f * b.ny ? (float)b.ny : 0.f);
    fz += fz > 0.5f * b.gnz ? -(float)b.gnz : (fz < -0.5f * b.gnz ? (float)b.gnz : 0.f);
    const float ryz2 = fy * fy + fz * fz;
    if (ryz2 > rout2) continue;                            // a row in a corner of the box: it misses the shell
    for (int img = 0; img < 2; ++img) {                    // (the second copy of a plane: a ring of one slab only)
    const int z = local_z(b, zg, img);
    if (z < 0) continue;                                   // a plane of another slab
    for (int lx0 = 0; lx0 < pb.ext[0]; lx0 += 32) {
      const int lx = lx0 + lane;
      int x = pb.lo[0] + lx;
      x += x < 0 ? b.nx : (x >= b.nx ? -b.nx : 0);
      bool pass = lx < pb.ext[0];
      if (pass) {
        float fx = (float)x - cxr;
        fx += fx > 0.5f * b.nx ? -(float)b.nx : (fx < -0.5f * b.nx ? (float)b.nx : 0.f);
        const float d2 = fx * fx + ryz2;
        pass = d2 >= rin2 && d2 <= rout2 && keep(x, y, z);
      }
      const unsigned bal = __ballot_sync(0xffffffffu, pass);
      if (pass) queue[qn + __popc(bal & ((1u << lane) - 1u))] = (int)site_of(b, x, y, z);
      qn += __popc(bal);
      __syncwarp();
      if (qn >= 32) {
        process(queue[lane]);
        const int left = qn - 32;
        const int v = lane < left ? queue[32 + lane] : 0;
        __syncwarp();
        if (lane < left) queue[lane] = v;
        qn = left;
        __syncwarp();
      }
    }
    }
  }
  if (lane < qn) process(queue[lane]);
}

// the nodes of every particle at start-up (G32): solid bit and particle index
__global__ void __launch_bounds__(256) k_part_raster(const PartParams p) {
  const Box& b = p.box;
  const PState& P = p.parts[blockIdx.x];
  const PartBox pb = part_box(b, P.r, P.R + 1.0);
  const int nn = pb.ext[0] * pb.ext[1] * pb.ext[2];
  for (int i = threadIdx.x; i < 2 * nn; i += blockDim.x) {
    int x, y, z;
    if (!part_box_node(b, pb, i % nn, x, y, z, i / nn)) continue;       // (a slab marks its ghost planes too)
    if (solid_at(b, x, y, z) || !inside_particle(b, P, x, y, z)) continue;
    atomicOr(&p.mask[(size_t)(z * b.ny + y) * b.nxw + (x >> 5)], 1u << (x & 31));
    p.pid[site_of(b, x, y, z)] = blockIdx.x;
  }
}

// G33: the link rule at a moving surface and the momentum it hands over.  For a link j of the fluid
// site s into the particle the hot kernel stored f*_j at the site itself (bounce-back at a wall at
// rest: the site reads it back along -c_j); here it becomes g^k = f^k* - 6 w_j rho^k (c_j . u_b), rho^k
// the site's own densities of time t and u_b the surface velocity at the midpoint of the link, and
// the particle receives (f* + g) c_j, summed over the components.  Every link belongs to one
// particle, so no two threads touch the same value.
template <bool TWO>
__global__ void __launch_bounds__(256) k_part_force(const PartParams p) {
  __shared__ double red[6 * 8];
  __shared__ int queue[8][64];
  // the particle's state in shared memory: this kernel stores to global memory, so the compiler would
  // load r, u, w of a global PState again for every link (measured: a quarter of the kernel's stall samples)
  __shared__ PState P;
  const Box& b = p.box;
  {
    const double* src = reinterpret_cast<const double*>(&p.parts[blockIdx.x]);
    double* dst = reinterpret_cast<double*>(&P);
    for (int i = threadIdx.x; i < (int)(sizeof(PState) / sizeof(double)); i += blockDim.x) dst[i] = src[i];
  }
  __syncthreads();
  const PartBox pb = part_box(b, P.r, P.R + 2.0);
  double acc[6] = {0, 0, 0, 0, 0, 0};
  // everything a candidate site (a fluid node in the shell around the sphere) needs
  auto process = [&](int site) {
    const size_t s = (size_t)site;
    const int x = (int)(s % b.nx), y = (int)((s / b.nx) % b.ny), z = (int)(s / ((size_t)b.nx * b.ny));
    const uint32_t smask = neighbour_mask(b, x, y, z);      // 18 independent loads from the (small) bit mask
    if (smask == 0u) return;
    // which of the solid neighbours belong to this particle: the index loads are issued together
    uint32_t mine = 0u;
    static_for<1, Q>([&](auto qc) {
      constexpr int q = decltype(qc)::value;
      if ((smask >> q) & 1u) {
        int xn, yn, zn;
        nbr_of(b, x, y, z, q, xn, yn, zn);                 // (an own site: all its neighbours are held)
        if (p.pid[site_of(b, xn, yn, zn)] == (int)blockIdx.x) mine |= 1u << q;
      }
    });
    if (mine == 0u) return;
    float rr, rb;
    site_density<TWO>(p, x, y, z, rr, rb);
    for (int q = 1; q < Q; ++q) {
      if (!((mine >> q) & 1u)) continue;
      double rel[3];
      const double cu = link_cu_rt(b, P.r, P.u, P.w, x, y, z, q, rel);
      float* sl = own_slot<TWO>(p, q, s);
      const float k = -6.0f * wq(q) * (float)cu;
      const float ft = __ldcg(sl);                                       // f* - w (the T plane holds deviations)
      const float gt = fmaf(k, rr + rb, ft);
      sl[0] = gt;
      if constexpr (TWO) sl[1] = fmaf(k, rr, __ldcg(sl + 1));
      const double tot = ((double)ft + (double)wq(q)) + ((double)gt + (double)wq(q));
      const double d[3] = {tot * c_cx[q], tot * c_cy[q], tot * c_cz[q]};
      acc[0] += d[0]; acc[1] += d[1]; acc[2] += d[2];
      acc[3] += rel[1] * d[2] - rel[2] * d[1];
      acc[4] += rel[2] * d[0] - rel[0] * d[2];
      acc[5] += rel[0] * d[1] - rel[1] * d[0];
    }
  };
  // a fluid node with a link into the sphere lies in the shell R .. R + 1.75
  const float Rin = (float)P.R - 0.01f, Rout = (float)P.R + 1.75f;
  scan_shell(b, pb, P.r, Rin * Rin, Rout * Rout + 0.5f, threadIdx.x >> 5, 8, queue[threadIdx.x >> 5],
             [&](int x, int y, int z) { return own_plane(b, z) && !solid_at(b, x, y, z); }, process);
  block_sum<6>(acc, red);
  if (threadIdx.x == 0) {
    if (p.part_out)
      for (int a = 0; a < 6; ++a) p.part_out[(size_t)blockIdx.x * 6 + a] = acc[a];     // this slab's share
    else
      for (int a = 0; a < 3; ++a) { p.parts[blockIdx.x].F[a] = acc[a]; p.parts[blockIdx.x].T[a] = acc[3 + a]; }
  }
}

// G37: the force on particle i from all others.  One warp per particle, the lanes share the others;
// the lane sums are added in a fixed order.
__global__ void __launch_bounds__(256) k_part_pair(const PartParams p) {
  const Box& b = p.box;
  const int n[3] = {b.nx, b.ny, b.gnz};
  const int i = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (i >= p.np) return;
  PState& A = p.parts[i];
  if (p.tot_in && lane < 6) {      // a slab: the link sums over all slabs
    if (lane < 3) A.F[lane] = p.tot_in[(size_t)i * 6 + lane];
    else A.T[lane - 3] = p.tot_in[(size_t)i * 6 + lane];
  }
  double f[3] = {0, 0, 0};
  if (p.hc > 0.0)
    for (int j = lane; j < p.np; j += 32) {
      if (j == i) continue;
      const PState& B = p.parts[j];
      const double d[3] = {min_image(A.r[0] - B.r[0], n[0]), min_image(A.r[1] - B.r[1], n[1]), min_image(A.r[2] - B.r[2], n[2])};
      const double reach = A.R + B.R + p.hc;
      const double d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
      if (d2 >= reach * reach) continue;
      const double dist = sqrt(d2);
      const double h = dist - A.R - B.R;
      if (h >= p.hc) continue;
      const double e[3] = {d[0] / dist, d[1] / dist, d[2] / dist};     // from j to i
      double fm = p.K * pow(p.hc - h, 1.5);
      if (p.lub) {
        const double hh = h < 0.1 ? 0.1 : h, Reff = A.R * B.R / (A.R + B.R);
        const double un = (A.u[0] - B.u[0]) * e[0] + (A.u[1] - B.u[1]) * e[1] + (A.u[2] - B.u[2]) * e[2];
        fm += -6.0 * 3.14159265358979323846 * p.mu * Reff * Reff * (1.0 / hh - 1.0 / p.hc) * un;
      }
      for (int a = 0; a < 3; ++a) f[a] += fm * e[a];
    }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1)
#pragma unroll
    for (int a = 0; a < 3; ++a) f[a] += __shfl_down_sync(0xffffffffu, f[a], o);
  if (lane == 0)
    for (int a = 0; a < 3; ++a) A.Fpp[a] = f[a];
}

// G35: Eq. 15 by leapfrog with the quaternion update; one thread per particle
__global__ void __launch_bounds__(128) k_part_integrate(const PartParams p) {
  const Box& b = p.box;
  const int n[3] = {b.nx, b.ny, b.gnz};
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.np || !p.mobile) return;
  PState& P = p.parts[i];
  for (int a = 0; a < 3; ++a) {
    P.ro[a] = P.r[a]; P.uo[a] = P.u[a]; P.wo[a] = P.w[a];
    P.u[a] += (P.F[a] + P.Fpp[a] + P.Fext[a]) / P.mass;
    P.w[a] += (P.T[a] + P.Text[a]) / P.inertia;
    P.r[a] += P.u[a];
    P.r[a] -= n[a] * floor(P.r[a] / n[a]);
  }
  const double th = sqrt(P.w[0] * P.w[0] + P.w[1] * P.w[1] + P.w[2] * P.w[2]);
  if (th > 0.0) {
    const double sh = sin(0.5 * th) / th, ch = cos(0.5 * th);
    const double d[4] = {ch, sh * P.w[0], sh * P.w[1], sh * P.w[2]};
    const double q0 = P.q[0], q1 = P.q[1], q2 = P.q[2], q3 = P.q[3];
    double r[4] = {d[0] * q0 - d[1] * q1 - d[2] * q2 - d[3] * q3, d[0] * q1 + d[1] * q0 + d[2] * q3 - d[3] * q2,
                   d[0] * q2 - d[1] * q3 + d[2] * q0 + d[3] * q1, d[0] * q3 + d[1] * q2 - d[2] * q1 + d[3] * q0};
    const double nr = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + r[3] * r[3]);
    for (int a = 0; a < 4; ++a) P.q[a] = r[a] / nr;
  }
}

// G36: the nodes that entered or left particle blockIdx.x when it moved.  Phase 1 lists them (sorted
// by site, so that the sums below have a fixed order), phase 2 treats one node per thread, phase 3
// adds the impulses to the particle and rewrites the node map.
template <bool TWO>
__global__ void __launch_bounds__(256) k_part_remap(const PartParams p) {
  if (!p.mobile) return;
  __shared__ int raw[PART_MAXCH], list[PART_MAXCH];     // site index, bit 30 set = entered the particle
  __shared__ double imp[PART_MAXCH][6];
  __shared__ int nraw;
  const Box& b = p.box;
  const int me = blockIdx.x;
  PState& P = p.parts[me];
  if (threadIdx.x == 0) nraw = 0;
  __syncthreads();
  const PartBox pb = part_box(b, P.r, P.R + 2.0);
  const int nn = pb.ext[0] * pb.ext[1] * pb.ext[2];
  for (int i = threadIdx.x; i < 2 * nn; i += blockDim.x) {
    int x, y, z;
    if (!part_box_node(b, pb, i % nn, x, y, z, i / nn)) continue;       // (a slab lists the changes in its ghost planes too)
    const size_t s = site_of(b, x, y, z);
    const bool was = p.pid[s] == me;
    const bool now = inside_particle(b, P, x, y, z) && (was || !solid_at(b, x, y, z));
    if (was != now) {
      const int k = atomicAdd(&nraw, 1);
      if (k < PART_MAXCH) raw[k] = (int)s | (now ? (1 << 30) : 0);
    }
  }
  __syncthreads();
  const int nch = min(nraw, PART_MAXCH);
  if (nraw > PART_MAXCH && threadIdx.x == 0) atomicExch(p.overflow, 1);
  for (int i = threadIdx.x; i < nch; i += blockDim.x) {       // rank sort by (site, kind)
    const int v = raw[i] & ~(1 << 30);
    int rank = 0;
    for (int j = 0; j < nch; ++j) rank += (raw[j] & ~(1 << 30)) < v;
    list[rank] = raw[i];
  }
  __syncthreads();
  auto newly_covered = [&](size_t s) {
    for (int j = 0; j < nch; ++j) if (list[j] == ((int)s | (1 << 30))) return true;
    return false;
  };
  // One WARP per changed node, lane q = direction q (lanes 19..31 idle): the work of a node is 18
  // neighbours, each a chain of dependent loads (mask, densities, stored values), and one thread per
  // node ran them one after the other (70 us per step at 241 colloids).  The lanes' shares of the
  // impulse are added by a shuffle tree: a fixed order.
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int i = wid; i < nch; i += 8) {
    const bool entered = (list[i] >> 30) & 1;
    const size_t s = (size_t)(list[i] & ~(1 << 30));
    const int x = (int)(s % b.nx), y = (int)((s / b.nx) % b.ny), z = (int)(s / ((size_t)b.nx * b.ny));
    const int q = lane;
    const bool dir = q >= 1 && q < Q;                  // this lane stands for a link direction
    double dU[3] = {0, 0, 0}, dL[3] = {0, 0, 0};
    auto give = [&](const double m[3], const double rel[3], double sg) {
      dU[0] += sg * m[0]; dU[1] += sg * m[1]; dU[2] += sg * m[2];
      dL[0] += sg * (rel[1] * m[2] - rel[2] * m[1]);
      dL[1] += sg * (rel[2] * m[0] - rel[0] * m[2]);
      dL[2] += sg * (rel[0] * m[1] - rel[1] * m[0]);
    };
    // G33 with the particle's NEW state on the link (xs, ys, zs) -> + c_qq; the particle receives the sum
    auto reflect = [&](int xs, int ys, int zs, int qq, float rr, float rb) {
      double rel[3];
      const double cu = link_cu_rt(b, P.r, P.u, P.w, xs, ys, zs, qq, rel);
      float* sl = own_slot<TWO>(p, qq, site_of(b, xs, ys, zs));
      const float k = -6.0f * wq(qq) * (float)cu;
      const float fpt = sl[0] + wq(qq);                  // f* (total)
      const float gt = fmaf(k, rr + rb, fpt);
      sl[0] = gt - wq(qq);
      if constexpr (TWO) sl[1] = fmaf(k, rr, sl[1]);
      const double tot = (double)fpt + (double)gt;
      const double d[3] = {tot * c_cx[qq], tot * c_cy[qq], tot * c_cz[qq]};
      give(d, rel, +1.0);
    };
    const double rel0[3] = {min_image(x - P.r[0], b.nx), min_image(y - P.r[1], b.ny), min_image(global_z(b, z) - P.r[2], b.gnz)};
    // A slab treats what belongs to its own planes: the node itself if it owns it, and of every changed
    // node (its ghost planes included) the links of its own fluid sites into that node.
    const bool own_s = own_plane(b, z);
    // the neighbour along c_q and the one against it (xs + c_q = this node)
    int xn = 0, yn = 0, zn = 0, xs = 0, ys = 0, zs = 0;
    const bool has_n = dir && nbr_of(b, x, y, z, q, xn, yn, zn);
    const bool has_s = dir && nbr_of(b, x, y, z, opp(dir ? q : 1), xs, ys, zs) && own_plane(b, zs);
    if (!entered) {
      if (own_s) {
        // the node leaves the particle: equilibrium (Eq. 2) at the mean densities of its fluid neighbours
        // and the surface velocity; its momentum comes out of the particle's
        float a = 0.f, c2 = 0.f;
        int one = 0;
        if (has_n && !solid_at(b, xn, yn, zn) && !newly_covered(site_of(b, xn, yn, zn))) {
          site_density<TWO>(p, xn, yn, zn, a, c2);
          one = 1;
        }
        // sums over the directions in the order 1, 2, ..., 18 (what one thread did): lane 0 adds them up
        float sr = 0.f, sb = 0.f;
        int cnt = 0;
        for (int k = 1; k < Q; ++k) {
          sr += __shfl_sync(0xffffffffu, a, k);
          sb += __shfl_sync(0xffffffffu, c2, k);
          cnt += __shfl_sync(0xffffffffu, one, k);
        }
        float rr = TWO ? 0.5f : 1.0f, rb = TWO ? 0.5f : 0.0f;
        if (cnt) { rr = sr / (float)cnt; rb = sb / (float)cnt; }
        const double wxr[3] = {P.w[1] * rel0[2] - P.w[2] * rel0[1], P.w[2] * rel0[0] - P.w[0] * rel0[2], P.w[0] * rel0[1] - P.w[1] * rel0[0]};
        const float ux = (float)(P.u[0] + wxr[0]), uy = (float)(P.u[1] + wxr[1]), uz = (float)(P.u[2] + wxr[2]);
        const float uu15 = 1.5f * (ux * ux + uy * uy + uz * uz), rho = rr + rb;
        if (q < Q) {
          const float cu = c_cx[q] * ux + c_cy[q] * uy + c_cz[q] * uz;
          const float e = 3.0f * cu + 4.5f * cu * cu - uu15;
          float* sl = own_slot<TWO>(p, q, s);
          sl[0] = wq(q) * ((rho - 1.0f) + rho * e);
          if constexpr (TWO) sl[1] = wq(q) * rr * (1.0f + e);
        }
        if (lane == 0) {
          const double mom[3] = {(double)rho * ux, (double)rho * uy, (double)rho * uz};
          give(mom, rel0, -1.0);
        }
        // its own links into the particle as it stands now (the lane that wrote slot q reflects it)
        if (has_n && inside_particle(b, P, xn, yn, zn)) {
          const int pn = p.pid[site_of(b, xn, yn, zn)];
          if (!(solid_at(b, xn, yn, zn) && pn != me)) reflect(x, y, z, q, rr, rb);    // (not a wall's or another particle's node)
        }
      }
      // links of fluid neighbours into this node: undone
      if (has_s) {
        const size_t t = site_of(b, xs, ys, zs);
        if (!solid_at(b, xs, ys, zs) && !newly_covered(t)) {
          float a, c2;
          site_density<TWO>(p, xs, ys, zs, a, c2);
          double rel[3];
          const double cu = link_cu_rt(b, P.ro, P.uo, P.wo, xs, ys, zs, q, rel);
          float* sl = own_slot<TWO>(p, q, t);
          const float k = 6.0f * wq(q) * (float)cu;
          const float gt = sl[0] + wq(q);
          const float fpt = fmaf(k, a + c2, gt);
          sl[0] = fpt - wq(q);
          if constexpr (TWO) sl[1] = fmaf(k, a, sl[1]);
          const double tot = (double)fpt + (double)gt;
          const double d[3] = {tot * c_cx[q], tot * c_cy[q], tot * c_cz[q]};
          give(d, rel, -1.0);
        }
      }
    } else {
      // the node enters the particle: what it holds goes to the particle.  A stored value stands for a
      // population that after streaming moves along c_q, or, where the neighbour is solid, along -c_q.
      if (own_s && q < Q) {
        const double sg = (dir && has_n && solid_at(b, xn, yn, zn)) ? -1.0 : 1.0;
        const double v = sg * ((double)own_slot<TWO>(p, q, s)[0] + (double)wq(q));
        const double mom[3] = {v * c_cx[q], v * c_cy[q], v * c_cz[q]};
        give(mom, rel0, +1.0);
      }
      // links of fluid neighbours into this node: reflected
      if (has_s && !solid_at(b, xs, ys, zs) && !newly_covered(site_of(b, xs, ys, zs))) {
        float a, c2;
        site_density<TWO>(p, xs, ys, zs, a, c2);
        reflect(xs, ys, zs, q, a, c2);
      }
    }
    // the lanes' shares, added by a tree of fixed shape
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        dU[a] += __shfl_down_sync(0xffffffffu, dU[a], o);
        dL[a] += __shfl_down_sync(0xffffffffu, dL[a], o);
      }
    if (lane == 0)
      for (int a = 0; a < 3; ++a) { imp[i][a] = dU[a]; imp[i][3 + a] = dL[a]; }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double t[6] = {0, 0, 0, 0, 0, 0};
    for (int i = 0; i < nch; ++i)
      for (int a = 0; a < 6; ++a) t[a] += imp[i][a];
    if (p.part_out)
      for (int a = 0; a < 6; ++a) p.part_out[(size_t)me * 6 + a] = t[a];      // this slab's share: k_part_apply adds the total
    else
      for (int a = 0; a < 3; ++a) { P.u[a] += t[a] / P.mass; P.w[a] += t[3 + a] / P.inertia; }
  }
  for (int i = threadIdx.x; i < nch; i += blockDim.x) {       // the node map of time t + 1
    const bool entered = (list[i] >> 30) & 1;
    const size_t s = (size_t)(list[i] & ~(1 << 30));
    const int x = (int)(s % b.nx), y = (int)((s / b.nx) % b.ny), z = (int)(s / ((size_t)b.nx * b.ny));
    uint32_t* wd = &p.mask[(size_t)(z * b.ny + y) * b.nxw + (x >> 5)];
    if (entered) { atomicOr(wd, 1u << (x & 31)); p.pid[s] = me; }
    else { atomicAnd(wd, ~(1u << (x & 31))); p.pid[s] = -1; }
  }
}

// A slab: the impulses of the node changes, summed over all slabs by the caller, go to the particles
// (what the last lines of k_part_remap do in an undivided box).  One thread per particle.
__global__ void __launch_bounds__(128) k_part_apply(const PartParams p) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.np || !p.mobile) return;
  PState& P = p.parts[i];
  for (int a = 0; a < 3; ++a) {
    P.u[a] += p.tot_in[(size_t)i * 6 + a] / P.mass;
    P.w[a] += p.tot_in[(size_t)i * 6 + 3 + a] / P.inertia;
  }
}

// The phase field around the particles.  k_phase_fwd has written phi(t + 1) from the moments k_fused
// forwarded, i.e. for walls at rest and the node map of time t.  Near a particle both have changed
// since: k_part_force rewrote the values that come back from the surface, and a node that entered
// or left the particle (k_part_remap) changes what its neighbours will read.  So phi is formed
// again, from the stored populations with the node map of time t + 1, in the shell of nodes around
// every particle's surface, R - dr <= d <= R + sqrt(2) + dr from the new centre, dr = the distance the
// centre moved in this step: a fluid node with a link into the particle lies within R + sqrt(2) of the
// old centre, a changed node within R of the old or the new one and its neighbours sqrt(2) further;
// nodes deeper inside than R - dr were and are the particle's and keep their sentinel.  Shells of two particles may overlap: both write the same
// values.  A/B storage (the particles' only one).
// grid = (particles, slices of the box's rows): the gathers are latency-bound, so the rows of a
// box are spread over several CTAs.
__global__ void __launch_bounds__(256) k_part_phi(const StepParams p) {
  __shared__ int queue[8][64];
  const Box& b = p.box;
  const PState& P = p.parts[blockIdx.x];
  // how far the centre moved in this step
  const double mx = min_image(P.r[0] - P.ro[0], b.nx), my = min_image(P.r[1] - P.ro[1], b.ny), mz = min_image(P.r[2] - P.ro[2], b.gnz);
  const float dr = (float)sqrt(mx * mx + my * my + mz * mz) + 0.05f;
  const float Rin = (float)P.R > dr ? (float)P.R - dr : 0.f, Rout = (float)P.R + 1.4143f + dr;
  const PartBox pb = part_box(b, P.r, (double)Rout + 0.5);
  scan_shell(b, pb, P.r, Rin * Rin, Rout * Rout + 0.5f, blockIdx.y * 8 + (threadIdx.x >> 5), 8 * gridDim.y, queue[threadIdx.x >> 5],
             [&](int, int, int z) { return own_plane(b, z); },
             [&](int site) {
               const int x = site % b.nx, y = (site / b.nx) % b.ny, z = site / (b.nx * b.ny);
               phase_column<MODE_AB, true, false>(p, x, y, z, z + 1);
             });
}

// ----------------------------------------------------------------------------- slab halo
// z-slab decomposition ("the domain is equally distributed (according to a either 1D, or 2D or 3D
// domain decomposition)"; streaming reaches first neighbours only): what
// crosses a z face per step is the 5 populations per component with c_z = +1 (upwards) or -1
// (downwards).  One (direction, plane) block is contiguous in the SoA layout; the message of a face
// is the 5 blocks behind each other.  The same kernel packs (blocks -> message) and unpacks (message
// -> blocks of the ghost plane, or of the own boundary plane after an in-place odd step); which
// blocks is the host's choice (lb_api.cu, slab_blocks).  grid = (ceil(n4 / 256), 5, 2 faces).
struct HaloCopy {
  const float4* src[2][5];
  float4* dst[2][5];
  long long n4;          // float4 elements per block
};
__global__ void __launch_bounds__(256) k_halo_copy(const HaloCopy p) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.n4) return;
  const int k = blockIdx.y, f = blockIdx.z;
  p.dst[f][k][i] = __ldcg(p.src[f][k] + i);
}

// Unpacking after an in-place ODD step with walls.  That step pushed f*_q into slot (q, x + c_q); what
// it pushed across a z face sits in the sender's ghost plane and belongs to the receiver's boundary
// plane.  But a receiver site y whose source y - c_q is SOLID keeps the value it wrote itself (the
// bounced-back population went to slot (q, y) at its own site), so the message may only overwrite
// the slots whose source site, in the receiver's ghost plane zsrc[f], is fluid.
struct HaloMerge {
  const float* src[2][5];
  float* dst[2][5];
  int dirs[2][5];
  int zsrc[2];
  Box box;
};
template <int ESZ>       // bytes per site: 8 = {T, R} pair, 4 = one component
__global__ void __launch_bounds__(256) k_halo_merge(const HaloMerge p) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const Box& b = p.box;
  if (i >= (long long)b.nx * b.ny) return;
  const int k = blockIdx.y, f = blockIdx.z, q = p.dirs[f][k];
  const int x = (int)(i % b.nx), y = (int)(i / b.nx);
  int xs = x - c_cx[q], ys = y - c_cy[q];
  xs = xs < 0 ? b.nx - 1 : (xs >= b.nx ? 0 : xs);
  ys = ys < 0 ? b.ny - 1 : (ys >= b.ny ? 0 : ys);
  if (solid_at(b, xs, ys, p.zsrc[f])) return;
  if constexpr (ESZ == 8) reinterpret_cast<float2*>(p.dst[f][k])[i] = __ldcg(reinterpret_cast<const float2*>(p.src[f][k]) + i);
  else p.dst[f][k][i] = __ldcg(p.src[f][k] + i);
}

// bytes [S] (0 fluid, 1 wall at rest, 2 / 3 / 4 wall groups) -> bit-packed words: solid, and
// (if groups != nullptr) two bit planes behind each other that hold group - 1 in binary
__global__ void k_pack_mask(const uint8_t* bytes, uint32_t* words, uint32_t* groups, Box b) {
  const long long wi = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long nw = (long long)b.nxw * b.ny * b.nz;
  if (wi >= nw) return;
  const long long row = wi / b.nxw;
  const int xw = (int)(wi % b.nxw);
  uint32_t m = 0, g2 = 0, g3 = 0;
  for (int i = 0; i < 32; ++i) {
    const int x = xw * 32 + i;
    if (x < b.nx) {
      const uint8_t v = bytes[row * b.nx + x];
      if (v) m |= 1u << i;
      if (v == 2 || v == 4) g2 |= 1u << i;
      if (v == 3 || v == 4) g3 |= 1u << i;
    }
  }
  words[wi] = m;
  if (groups) { groups[wi] = g2; groups[nw + wi] = g3; }
}

// does the byte mask hold a moving wall group?  out[0] |= 1
__global__ void k_any_moving(const uint8_t* bytes, long long S, int* out) {
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < S && bytes[s] >= 2 && bytes[s] <= 4) atomicOr(out, 1);
}

}  // namespace lb
