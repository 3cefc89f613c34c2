// CUDA kernels of the colour-gradient D3Q19 hot path, written for sm_100a (B200).
//
//   k_phase   K1  gather both components' populations, rho_r, rho_b, phi (Eq. 3),
//                 write phi (+ periodic ghost images, + sentinel at solid sites)
//   k_fused   K2  pull-stream + moments + grad phi from a TMA-staged shared-memory phi ring +
//                 near-contact probe (Eq. 11) + Guo force + BGK on the total
//                 (Eq. 1-2, 5-8) + perturbation + recolouring + store
//   k_single  K2s single-component BGK (Eq. 1-4), the pure-bandwidth baseline (config C2)
//   k_scatter K0  place given pre-collision populations where the next gather finds them
//   k_gatherf     debug accessor: full pre-collision populations
//   k_macros  K3  rho_r, rho_b, u with the half-force shift
//
// Storage: SoA planes, x fastest.  Two components: planes 0..18 hold
// T_q = f^r_q + f^b_q - w_q (the total as a deviation from the lattice weights, so that the
// hydrodynamic part keeps ~1e-9 absolute precision in fp32), planes 19..37 hold R_q = f^r_q.
// Single component: planes 0..18 hold f_q - w_q.  The collision is carried out on the
// deviations directly (T^eq_q = w_q [drho + rho (3 cu + 4.5 cu^2 - 1.5 uu)]).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "lb_lattice.cuh"

namespace lb {

struct StepParams {
  const float* src;   // population buffer read by this step
  float* dst;         // buffer written (== src in AA modes)
  float* phi;         // padded phi array (written by K1, read by K2/K3)
  Box box;
  int zc;             // z planes per CTA
  int halo;           // ghost depth K1 must fill (1 without near contact, 4 with)
  float tau_r, tau_b, A, beta, A_nc, phi_c, gx, gy, gz;
  int two_tau, has_g;
};

constexpr int TX = 32, TY = 8;   // CTA tile in x-y; one warp per x row segment

// ----------------------------------------------------------------------------- addressing
struct Ctx {
  int idx;            // own site
  int dxo[3];         // index deltas to x-1, x, x+1 (wrapped)
  int dyo[3];         // to y-1, y, y+1
  int dzo[3];         // to z-1, z, z+1
  long long S;
};

// Index delta from the own site to x - c_q.
template <int q>
__device__ __forceinline__ int delta_src(const Ctx& c) {
  return c.dxo[1 - cx(q)] + c.dyo[1 - cy(q)] + c.dzo[1 - cz(q)];
}

// Flattened (plane * S + site) location that holds f_q(x) of the current state.
// smask bit i set <=> x + c_i is solid.
template <int MODE, bool HAS_SOLID, int q>
__device__ __forceinline__ size_t read_slot(const Ctx& c, uint32_t smask) {
  if constexpr (MODE == MODE_AA_EVEN || q == 0) {
    return (size_t)q * c.S + c.idx;
  } else {
    const bool bounce = HAS_SOLID && ((smask >> opp(q)) & 1u);
    if constexpr (MODE == MODE_AB) {
      return bounce ? (size_t)opp(q) * c.S + c.idx : (size_t)q * c.S + (c.idx + delta_src<q>(c));
    } else {  // AA_ODD
      return bounce ? (size_t)q * c.S + c.idx : (size_t)opp(q) * c.S + (c.idx + delta_src<q>(c));
    }
  }
}

// Where the post-collision value f*_q goes.
template <int MODE, bool HAS_SOLID, int q>
__device__ __forceinline__ size_t write_slot(const Ctx& c, uint32_t smask) {
  if constexpr (MODE == MODE_AB) {
    return (size_t)q * c.S + c.idx;
  } else if constexpr (MODE == MODE_AA_EVEN) {
    return (size_t)opp(q) * c.S + c.idx;
  } else {
    return read_slot<MODE, HAS_SOLID, opp(q)>(c, smask);
  }
}

template <int MODE>
__device__ __forceinline__ float ld_pop(const float* p) {
  if constexpr (MODE == MODE_AB) return __ldg(p);   // source buffer is read-only in A/B mode
  else return *p;
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

__device__ __forceinline__ void make_ctx(Ctx& c, const Box& b, int x, int y, int z) {
  c.S = b.S;
  c.idx = x + b.nx * (y + b.ny * z);
  c.dxo[0] = (x == 0 ? b.nx - 1 : -1);
  c.dxo[1] = 0;
  c.dxo[2] = (x == b.nx - 1 ? -(b.nx - 1) : 1);
  c.dyo[0] = (y == 0 ? b.ny - 1 : -1) * b.nx;
  c.dyo[1] = 0;
  c.dyo[2] = (y == b.ny - 1 ? -(b.ny - 1) : 1) * b.nx;
  const int pl = b.nx * b.ny;
  c.dzo[0] = (z == 0 ? b.nz - 1 : -1) * pl;
  c.dzo[1] = 0;
  c.dzo[2] = (z == b.nz - 1 ? -(b.nz - 1) : 1) * pl;
}

// s + e <- s + e + x with the rounding error of the addition kept in e (Knuth two-sum).
__device__ __forceinline__ void two_sum_acc(float& s, float& e, float x) {
  const float t = __fadd_rn(s, x);
  const float bp = __fsub_rn(t, s);
  e = __fadd_rn(e, __fadd_rn(__fsub_rn(s, __fsub_rn(t, bp)), __fsub_rn(x, bp)));
  s = t;
}

// ----------------------------------------------------------------------------- K1 phase field
// One thread per site of a TX x TY tile, marching over zc planes.  152 B read, 4 B written.
template <int MODE, bool HAS_SOLID>
__device__ __forceinline__ void phase_column(const StepParams& p, int x, int y, int zb, int ze) {
  const Box& b = p.box;
  const int H = p.halo;
  const int px = b.nx + 2 * HALO, py = b.ny + 2 * HALO;
  for (int z = zb; z < ze; ++z) {
    Ctx c;
    make_ctx(c, b, x, y, z);
    float phi;
    bool self_solid = false;
    uint32_t smask = 0;
    if constexpr (HAS_SOLID) {
      self_solid = solid_at(b, x, y, z);
      if (!self_solid) smask = neighbour_mask(b, x, y, z);
    }
    if (self_solid) {
      phi = PHI_SOLID;
    } else {
      float t[Q], r[Q];
      static_for<0, Q>([&](auto qc) {
        constexpr int q = decltype(qc)::value;
        const size_t s = read_slot<MODE, HAS_SOLID, q>(c, smask);
        t[q] = ld_pop<MODE>(p.src + s);
        r[q] = ld_pop<MODE>(p.src + (size_t)Q * c.S + s);
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
      const float num = ((2.0f * rr - 1.0f) - dr) + (2.0f * re - de);
      const float rho = (1.0f + dr) + de;
      phi = num / rho;
    }
    // home location plus the periodic images that fall into the ghost layers
    const int sx[3] = {0, x < H ? b.nx : 0, x >= b.nx - H ? -b.nx : 0};
    const int sy[3] = {0, y < H ? b.ny : 0, y >= b.ny - H ? -b.ny : 0};
    const int sz[3] = {0, z < H ? b.nz : 0, z >= b.nz - H ? -b.nz : 0};
#pragma unroll
    for (int iz = 0; iz < 3; ++iz) {
      if (iz && !sz[iz]) continue;
#pragma unroll
      for (int iy = 0; iy < 3; ++iy) {
        if (iy && !sy[iy]) continue;
#pragma unroll
        for (int ix = 0; ix < 3; ++ix) {
          if (ix && !sx[ix]) continue;
          p.phi[(size_t)(x + sx[ix] + HALO) + (size_t)px * ((size_t)(y + sy[iy] + HALO) + (size_t)py * (size_t)(z + sz[iz] + HALO))] = phi;
        }
      }
    }
  }
}

template <int MODE, bool HAS_SOLID>
__global__ void __launch_bounds__(TX* TY) k_phase(const StepParams p) {
  const int x = blockIdx.x * TX + threadIdx.x;
  const int y = blockIdx.y * TY + threadIdx.y;
  if (x >= p.box.nx || y >= p.box.ny) return;
  const int zb = blockIdx.z * p.zc;
  phase_column<MODE, HAS_SOLID>(p, x, y, zb, min(p.box.nz, zb + p.zc));
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
// Per thread: one site per plane, marching over zc planes; per CTA a TX x TY tile.  The phi
// planes z-H..z+H (+2 prefetched) of the tile with an H-wide halo live in a shared-memory ring
// filled by TMA from the padded phi array (ghost layers make every box in-bounds, so periodic
// wrap never reaches the TMA unit).  H = 1 without near contact, 4 with it.
// One TX x TY tile starting at (x0, y0), planes [zb, ze).  `ring`/`bars` are the CTA's phi ring and
// its mbarriers (initialised once per CTA); `jbase` counts the planes this CTA has pushed through the
// ring so far, so that slot numbers and mbarrier phase parities carry over from one call to the next.
template <int MODE, bool HAS_SOLID, bool HAS_NC>
__device__ __forceinline__ void fused_column(const StepParams& p, const CUtensorMap& tmap, float* ring, uint64_t* bars,
                                             int x0, int y0, int ylim, int zb, int ze, uint32_t& jbase) {
  constexpr int H = HAS_NC ? H_MAX_NC : 1;
  using R_ = Ring<H>;
  const Box& b = p.box;
  const int tid = threadIdx.y * TX + threadIdx.x;
  const int x = x0 + threadIdx.x, y = y0 + threadIdx.y;
  const bool active = x < b.nx && y < ylim;
  const int npl = (ze - zb) + 2 * H;
  const uint32_t jb = jbase;
  jbase += npl;

  auto issue = [&](int j) {
    const int s = (jb + j) % R_::NS;
    mbar_expect_tx(&bars[s], R_::BYTES);
    tma_load_3d(&ring[s * R_::SLOT], &tmap, &bars[s], x0, y0 + HALO - H, zb - H + j + HALO);
  };
  auto wait = [&](int j) { mbar_wait(&bars[(jb + j) % R_::NS], ((jb + j) / R_::NS) & 1); };
  if (tid == 0) {
    const int n0 = min(npl, R_::NS - 1);
    for (int j = 0; j < n0; ++j) issue(j);
  }

  const float omega_same = 1.0f / p.tau_r;
  const float nu_r = (p.tau_r - 0.5f) * (1.0f / 3.0f), nu_b = (p.tau_b - 0.5f) * (1.0f / 3.0f);
  const int lx = threadIdx.x + HALO, ly = threadIdx.y + H;

  for (int jz = 0; jz < ze - zb; ++jz) {
    const int z = zb + jz;
    if (tid == 0) {
      const int j = jz + R_::NS - 1;
      if (j < npl) issue(j);
    }
    if (jz == 0) {
#pragma unroll
      for (int j = 0; j <= 2 * H; ++j) wait(j);
    } else {
      wait(jz + 2 * H);
    }
    // plane dz of the ring
    auto plane = [&](int dz) -> const float* { return &ring[((jb + jz + H + dz) % R_::NS) * R_::SLOT]; };
    const float* pl0 = plane(0);
    const float phi0 = pl0[ly * R_::BX + lx];
    const bool fluid = active && !(HAS_SOLID && phi0 > PHI_SOLID_TEST);
    if (fluid) {
      Ctx c;
      make_ctx(c, b, x, y, z);
      // ---- grad phi (stencil of Eq. 10) and solid flags from the phi tile
      const float* plm = plane(-1);
      const float* plp = plane(+1);
      float Gx = 0.f, Gy = 0.f, Gz = 0.f;
      uint32_t smask = 0;
      static_for<1, Q>([&](auto qc) {
        constexpr int q = decltype(qc)::value;
        const float* pl = cz(q) == 0 ? pl0 : (cz(q) > 0 ? plp : plm);
        float v = pl[(ly + cy(q)) * R_::BX + lx + cx(q)];
        if constexpr (HAS_SOLID) {
          if (v > PHI_SOLID_TEST) { smask |= 1u << q; v = phi0; }
        }
        constexpr float k = 3.0f * wq(q);
        if constexpr (cx(q) != 0) Gx += (k * cx(q)) * v;
        if constexpr (cy(q) != 0) Gy += (k * cy(q)) * v;
        if constexpr (cz(q) != 0) Gz += (k * cz(q)) * v;
      });
      // ---- gather
      float T[Q], R[Q];
      static_for<0, Q>([&](auto qc) {
        constexpr int q = decltype(qc)::value;
        const size_t s = read_slot<MODE, HAS_SOLID, q>(c, smask);
        T[q] = ld_pop<MODE>(p.src + s);
        R[q] = ld_pop<MODE>(p.src + (size_t)Q * c.S + s);
      });
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
          int h = 0;
          bool alive = true;
#pragma unroll
          for (int k = 1; k <= H_MAX_NC; ++k) {
            if (alive) {
              const int dx = (int)roundf(k * nx_), dy = (int)roundf(k * ny_), dz = (int)roundf(k * nz_);
              const float v = plane(dz)[(ly + dy) * R_::BX + lx + dx];
              if (HAS_SOLID && v > PHI_SOLID_TEST) alive = false;
              else if (k >= 2 && v >= phi0) { h = k; alive = false; }
            }
          }
          if (h > 0) {
            const float Ah = h <= H_MIN_NC ? p.A_nc : p.A_nc * ((float)(H_MIN_NC * H_MIN_NC * H_MIN_NC) / (float)(h * h * h));
            Fx = 0.5f * Ah * Gx; Fy = 0.5f * Ah * Gy; Fz = 0.5f * Ah * Gz;
          }
        }
      }
      const bool forced = HAS_NC || p.has_g;
      if (p.has_g) { Fx += rho * p.gx; Fy += rho * p.gy; Fz += rho * p.gz; }
      // ---- velocity with the half-force shift, relaxation rate (Eq. 7-8)
      const float ux = (mx + 0.5f * Fx) * inv_rho, uy = (my + 0.5f * Fy) * inv_rho, uz = (mz + 0.5f * Fz) * inv_rho;
      float omega = omega_same;
      if (p.two_tau) {
        const float inv_nu = (rr * inv_rho) / nu_r + (rb * inv_rho) / nu_b;
        omega = 1.0f / (3.0f / inv_nu + 0.5f);
      }
      const float uu15 = 1.5f * (ux * ux + uy * uy + uz * uz);
      const float uF = ux * Fx + uy * Fy + uz * Fz;
      const float g0 = 1.0f - 0.5f * omega;
      const float fr_r = rr * inv_rho;                       // rho_r / rho
      const float kcol = p.beta * rr * rb * inv_rho * invG;   // recolouring amplitude / |G|
      const float om1 = 1.0f - omega;
      // ---- collide on the total (deviation form), perturb, recolour, store
      float* dT = p.dst;
      float* dR = p.dst + (size_t)Q * c.S;
      // Directions 1..18 first; the rest populations then take what is left of rho - 1 and of
      // rho_r (collision conserves both at every site), so that the per-site masses are conserved
      // to the rounding of one sum instead of carrying the relative error of rho_r/rho or of
      // w_q * drho (a systematic drift in uniform regions).
      float racc = 0.f, tacc = 0.f;
      static_for<1, Q + 1>([&](auto qc) {
        constexpr int q = decltype(qc)::value % Q;   // 1, 2, ..., 18, 0
        constexpr float w = wq(q);
        const float cu = cx(q) * ux + cy(q) * uy + cz(q) * uz;
        const float cG = cx(q) * Gx + cy(q) * Gy + cz(q) * Gz;
        const float teq = w * (dr + rho * (3.0f * cu + 4.5f * cu * cu - uu15));
        float ts = om1 * T[q] + omega * teq;
        if (forced) {
          const float cF = cx(q) * Fx + cy(q) * Fy + cz(q) * Fz;
          ts += g0 * w * (3.0f * (cF - uF) + 9.0f * cu * cF);
        }
        ts += p.A * (w * cG * cG * invG - bq(q) * Gne);
        float rs;
        if constexpr (q > 0) {
          rs = fr_r * (ts + w) + kcol * (w * inv_cnorm(q)) * cG;
          racc += rs;
          tacc += ts;
        } else {
          ts = dr - tacc;
          rs = rr - racc;
        }
        const size_t s = write_slot<MODE, HAS_SOLID, q>(c, smask);
        dT[s] = ts;
        dR[s] = rs;
      });
    }
    __syncthreads();   // everyone is done with plane jz before its slot is refilled
  }
}

template <int H>
__device__ __forceinline__ void ring_init(uint64_t* bars) {
  if (threadIdx.y * TX + threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < Ring<H>::NS; ++s) mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
}

template <int MODE, bool HAS_SOLID, bool HAS_NC>
__global__ void __launch_bounds__(TX* TY) k_fused(const StepParams p, const __grid_constant__ CUtensorMap tmap) {
  constexpr int H = HAS_NC ? H_MAX_NC : 1;
  __shared__ __align__(128) float ring[Ring<H>::NS * Ring<H>::SLOT];
  __shared__ __align__(8) uint64_t bars[Ring<H>::NS];
  ring_init<H>(bars);
  uint32_t jbase = 0;
  const int zb = blockIdx.z * p.zc;
  fused_column<MODE, HAS_SOLID, HAS_NC>(p, tmap, ring, bars, blockIdx.x * TX, blockIdx.y * TY, p.box.ny, zb, min(p.box.nz, zb + p.zc), jbase);
}

// ----------------------------------------------------------------------------- K12 pipelined step
// One launch per LB step doing the work of K1 and K2 in an order that lets K2's gather hit in L2.
// The box is cut into pencils (y strips of YS rows, full x extent, all z) that are processed one
// after another; inside a pencil the work is cut into items of one TX x TY tile x ZS planes and
// ordered z-slab by z-slab: the phase-field items P(k) of slab k run LEAD slabs ahead of the fused
// items F(s).  P(k) pulls the 38 planes of slab k from HBM; F(k) gathers the same lines a few
// hundred items later, while they are still in the 126 MB L2, so HBM sees each population once.
// Persistent CTAs draw items from a global ticket counter in schedule order.  F(s) needs phi on
// planes [s ZS - H, (s+1) ZS + H) of its tile and halo, i.e. completed P items with SMALLER ticket
// numbers only; P items never wait.  The CTA holding the smallest unfinished ticket can therefore
// always proceed: no deadlock, whether or not all CTAs are co-resident.  Completion is published
// per (pencil, slab) with a release (fence + atomic add) and observed by one polling thread with an
// acquire followed by fence.proxy.async, because the consumer of phi is the TMA unit.
struct Sched {
  int ZS, nzs, HS, LEAD;     // planes per slab, slabs, halo in slabs, lead of P over F in slabs
  int H;                     // phi halo (1 or 4)
  int ntx;                   // tiles along x
  int NP, YS;                // pencils, rows per pencil (multiple of TY; the last pencil takes the rest)
  // pencil classes: 0 = first, 1 = middle, 2 = last (a single pencil is class 0 with no halo)
  int hb[3], prow[3], frow[3];   // backward halo rows, P rows (interior + halos), F rows
  int nPt[3], nFt[3];            // P tiles and F tiles per slab
  long long tk[3];               // tickets per pencil of this class
  long long total;               // tickets per step
  int* ticket;                   // global ticket counter (zeroed before the launch)
  int* pdone;                    // [NP][nzs] completed P items (zeroed before the launch)
  int prefetch;                  // hint the next P item's lines into L2 while the current item runs
};

struct Item {
  int type;      // 0 = P, 1 = F, -1 = none
  int pencil, cls, slab, tx, ty;
};

__device__ __forceinline__ Item decode_ticket(const Sched& sc, long long t) {
  Item it;
  it.type = -1;
  if (t >= sc.total) return it;
  int pencil = 0, cls = 0;
  if (t >= sc.tk[0]) {
    t -= sc.tk[0];
    const long long nmid = sc.NP - 2;
    if (nmid > 0 && t < nmid * sc.tk[1]) {
      pencil = 1 + (int)(t / sc.tk[1]);
      t -= (long long)(pencil - 1) * sc.tk[1];
      cls = 1;
    } else {
      if (nmid > 0) t -= nmid * sc.tk[1];
      pencil = sc.NP - 1;
      cls = 2;
    }
  }
  it.pencil = pencil;
  it.cls = cls;
  const int nP = sc.nPt[cls], nF = sc.nFt[cls];
  int u = (int)t, tile;
  const int A = sc.LEAD * nP;
  if (u < A) {
    it.type = 0; it.slab = u / nP; tile = u - it.slab * nP;
  } else {
    u -= A;
    const int pair = nP + nF, npairs = sc.nzs - sc.LEAD;
    if (u < npairs * pair) {
      const int i = u / pair, r = u - i * pair;
      if (r < nF) { it.type = 1; it.slab = i; tile = r; }
      else { it.type = 0; it.slab = sc.LEAD + i; tile = r - nF; }
    } else {
      u -= npairs * pair;
      const int i = u / nF;
      it.type = 1; it.slab = npairs + i; tile = u - i * nF;
    }
  }
  if (it.type == 0) {   // P slabs start HS slabs below the top so that F(0) finds its lower halo
    it.slab = it.slab + sc.nzs - sc.HS;
    if (it.slab >= sc.nzs) it.slab -= sc.nzs;
  }
  it.ty = tile / sc.ntx;
  it.tx = tile - it.ty * sc.ntx;
  return it;
}

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ int ld_relaxed(const int* p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// Block until every P item that F(pencil, slab) depends on has been published (one thread calls).
// All counters are read with independent relaxed loads (their latencies overlap), then one fence
// gives the acquire; fence.proxy.async orders the phi data before the TMA reads that follow.
__device__ __forceinline__ void wait_phi_ready(const Sched& sc, const Box& b, int pencil, int slab) {
  const int zb = slab * sc.ZS, ze = min(b.nz, zb + sc.ZS);
  // own pencil, the pencil behind (its interior holds our backward halo rows) and, for the last
  // pencil, pencil 0 (our forward halo rows wrap onto it)
  int who[3] = {pencil, pencil, pencil};
  if (sc.NP > 1) {
    if (pencil > 0) who[1] = pencil - 1;
    if (pencil == sc.NP - 1) who[2] = 0;
  }
  int need[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) need[i] = sc.nPt[who[i] == 0 ? 0 : (who[i] == sc.NP - 1 ? 2 : 1)];
  bool ok;
  do {
    ok = true;
    for (int pl = zb - sc.H; pl < ze + sc.H; ++pl) {
      int w = pl;
      while (w < 0) w += b.nz;
      while (w >= b.nz) w -= b.nz;
      const int k = w / sc.ZS;
#pragma unroll
      for (int i = 0; i < 3; ++i) ok &= ld_relaxed(sc.pdone + (size_t)who[i] * sc.nzs + k) >= need[i];
    }
    if (!ok) __nanosleep(100);
  } while (!ok);
  __threadfence();
  asm volatile("fence.proxy.async;" ::: "memory");
}

// Hint the lines that P item `it` will gather into L2 (one line per component, direction, row, plane).
template <int MODE>
__device__ __forceinline__ void prefetch_p_item(const StepParams& p, const Sched& sc, const Item& it, int tid) {
  const Box& b = p.box;
  const int zb = it.slab * sc.ZS, ze = min(b.nz, zb + sc.ZS);
  const int rows = min(TY, sc.prow[it.cls] - it.ty * TY);
  const int x0 = it.tx * TX;
  const int n = 2 * Q * rows * (ze - zb);
  for (int i = tid; i < n; i += TX * TY) {
    const int pq = i % (2 * Q);
    const int rz = i / (2 * Q);
    const int r = rz % rows, z = zb + rz / rows;
    const int q = pq % Q;
    int y = it.pencil * sc.YS - sc.hb[it.cls] + it.ty * TY + r;
    int dx = 0, dy = 0, dz = 0, plane = q;
    if (MODE != MODE_AA_EVEN) { dx = c_cx[q]; dy = c_cy[q]; dz = c_cz[q]; }
    if (MODE == MODE_AA_ODD) plane = opp(q);
    y -= dy;
    while (y < 0) y += b.ny;
    while (y >= b.ny) y -= b.ny;
    int zz = z - dz;
    if (zz < 0) zz += b.nz;
    if (zz >= b.nz) zz -= b.nz;
    int xx = x0 + (dx < 0 ? TX - 1 : 0);          // the line that holds all but one element of the row
    if (xx >= b.nx) xx = b.nx - 1;
    const float* a = p.src + (size_t)(plane + (pq >= Q ? Q : 0)) * b.S + ((size_t)xx + (size_t)b.nx * ((size_t)y + (size_t)b.ny * zz));
    asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
  }
}

template <int MODE, bool HAS_SOLID, bool HAS_NC>
__global__ void __launch_bounds__(TX* TY, 3) k_step(const StepParams p, const __grid_constant__ CUtensorMap tmap, const Sched sc) {
  constexpr int H = HAS_NC ? H_MAX_NC : 1;
  __shared__ __align__(128) float ring[Ring<H>::NS * Ring<H>::SLOT];
  __shared__ __align__(8) uint64_t bars[Ring<H>::NS];
  __shared__ int tq[4];          // ticket queue: current, next (prefetched into L2), two in flight
  const int tid = threadIdx.y * TX + threadIdx.x;
  const Box& b = p.box;
  if (tid < 3) tq[tid] = atomicAdd(sc.ticket, 1);
  ring_init<H>(bars);          // ends with __syncthreads: the queue is visible
  uint32_t jbase = 0;
  for (int i = 0;; ++i) {
    const Item it = decode_ticket(sc, tq[i & 3]);
    if (it.type < 0) break;
    const Item nx = decode_ticket(sc, tq[(i + 1) & 3]);
    if (tid == 0) tq[(i + 3) & 3] = atomicAdd(sc.ticket, 1);
    if (sc.prefetch && nx.type == 0) prefetch_p_item<MODE>(p, sc, nx, tid);
    const int y0p = (it.pencil * sc.YS);                           // first interior row of the pencil
    const int zb = it.slab * sc.ZS, ze = min(b.nz, zb + sc.ZS);
    if (it.type == 0) {
      const int r = it.ty * TY + threadIdx.y;                        // row inside the pencil's P range
      const int x = it.tx * TX + threadIdx.x;
      if (r < sc.prow[it.cls] && x < b.nx) {
        int y = y0p - sc.hb[it.cls] + r;
        if (y < 0) y += b.ny;
        if (y >= b.ny) y -= b.ny;
        phase_column<MODE, HAS_SOLID>(p, x, y, zb, ze);
      }
      __syncthreads();
      if (tid == 0) {
        __threadfence();
        atomicAdd(sc.pdone + (size_t)it.pencil * sc.nzs + it.slab, 1);
      }
    } else {
      if (tid == 0) wait_phi_ready(sc, b, it.pencil, it.slab);
      fused_column<MODE, HAS_SOLID, HAS_NC>(p, tmap, ring, bars, it.tx * TX, y0p + it.ty * TY,
                                            min(b.ny, y0p + sc.frow[it.cls]), zb, ze, jbase);
      // fused_column ends with __syncthreads
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
  const int zb = blockIdx.z * p.zc;
  const int ze = min(b.nz, zb + p.zc);
  const float omega = 1.0f / p.tau_r;
  const float om1 = 1.0f - omega, g0 = 1.0f - 0.5f * omega;
  for (int z = zb; z < ze; ++z) {
    uint32_t smask = 0;
    if constexpr (HAS_SOLID) {
      if (solid_at(b, x, y, z)) continue;
      smask = neighbour_mask(b, x, y, z);
    }
    Ctx c;
    make_ctx(c, b, x, y, z);
    float T[Q];
    static_for<0, Q>([&](auto qc) {
      constexpr int q = decltype(qc)::value;
      T[q] = ld_pop<MODE>(p.src + read_slot<MODE, HAS_SOLID, q>(c, smask));
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
    const float ux = (mx + 0.5f * Fx) * inv_rho, uy = (my + 0.5f * Fy) * inv_rho, uz = (mz + 0.5f * Fz) * inv_rho;
    const float uu15 = 1.5f * (ux * ux + uy * uy + uz * uz);
    const float uF = ux * Fx + uy * Fy + uz * Fz;
    float tacc = 0.f;   // the rest population takes what is left of rho - 1 (see k_fused)
    static_for<1, Q + 1>([&](auto qc) {
      constexpr int q = decltype(qc)::value % Q;   // 1, 2, ..., 18, 0
      constexpr float w = wq(q);
      const float cu = cx(q) * ux + cy(q) * uy + cz(q) * uz;
      const float teq = w * (dr + rho * (3.0f * cu + 4.5f * cu * cu - uu15));
      float ts = om1 * T[q] + omega * teq;
      if (p.has_g) {
        const float cF = cx(q) * Fx + cy(q) * Fy + cz(q) * Fz;
        ts += g0 * w * (3.0f * (cF - uF) + 9.0f * cu * cF);
      }
      if constexpr (q > 0) tacc += ts;
      else ts = dr - tacc;
      p.dst[write_slot<MODE, HAS_SOLID, q>(c, smask)] = ts;
    });
  }
}

// ----------------------------------------------------------------------------- cold kernels
struct IoParams {
  float* buf;            // population buffer
  Box box;
  int two;               // two components?
  int comp;              // component of k_scatter / k_gatherf
  const float* in0;      // k_scatter: f[19][S] full populations (or nullptr: from rho,u)
  const float* rho_r;    // init fields
  const float* rho_b;
  const float* u;
  float* out0;           // k_gatherf / k_macros outputs
  float* out1;
  float* out2;
  const float* phi;      // padded phi (k_macros)
  float tau_r, tau_b, A, beta, A_nc, phi_c, gx, gy, gz;
};

template <int MODE>
__device__ __forceinline__ size_t read_slot_rt(const Box& b, int q, int x, int y, int z) {
  // run-time-q version of read_slot for the cold kernels
  const int cxs[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
  const int cys[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
  const int czs[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
  const size_t own = (size_t)x + (size_t)b.nx * ((size_t)y + (size_t)b.ny * z);
  if (MODE == MODE_AA_EVEN || q == 0) return (size_t)q * b.S + own;
  int xs = x - cxs[q], ys = y - cys[q], zs = z - czs[q];
  xs = xs < 0 ? b.nx - 1 : (xs >= b.nx ? 0 : xs);
  ys = ys < 0 ? b.ny - 1 : (ys >= b.ny ? 0 : ys);
  zs = zs < 0 ? b.nz - 1 : (zs >= b.nz ? 0 : zs);
  const bool bounce = b.mask && solid_at(b, xs, ys, zs);
  const size_t nb = (size_t)xs + (size_t)b.nx * ((size_t)ys + (size_t)b.ny * zs);
  const int o = opp(q);
  if (MODE == MODE_AB) return bounce ? (size_t)o * b.S + own : (size_t)q * b.S + nb;
  return bounce ? (size_t)q * b.S + own : (size_t)o * b.S + nb;
}

// K0: write the pre-collision state where the next gather will look for it.
//   comp < 0 : equilibrium init from rho_r, rho_b, u (Eq. 2), both components
//   comp = 0 : red populations from in0; the T planes receive f^r - w (blue must follow)
//   comp = 1 : blue populations from in0 are ADDED to the T planes
template <int MODE>
__global__ void k_scatter(const IoParams p) {
  const Box& b = p.box;
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= b.S) return;
  const int x = (int)(s % b.nx), y = (int)((s / b.nx) % b.ny), z = (int)(s / ((long long)b.nx * b.ny));
  if (b.mask && solid_at(b, x, y, z)) return;
  float rr = 0.f, rb = 0.f, ux = 0.f, uy = 0.f, uz = 0.f;
  if (p.comp < 0) {
    rr = p.rho_r[s];
    rb = p.two ? p.rho_b[s] : 0.f;
    ux = p.u[s]; uy = p.u[b.S + s]; uz = p.u[2 * b.S + s];
  }
  const float uu15 = 1.5f * (ux * ux + uy * uy + uz * uz);
  const int cxs[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
  const int cys[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
  const int czs[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
  for (int q = 0; q < Q; ++q) {
    const size_t slot = read_slot_rt<MODE>(b, q, x, y, z);
    const float w = wq(q);
    if (p.comp < 0) {
      const float cu = cxs[q] * ux + cys[q] * uy + czs[q] * uz;
      const float e = 3.0f * cu + 4.5f * cu * cu - uu15;       // feq/(w rho) - 1
      const float drho = (rr + rb) - 1.0f;
      p.buf[slot] = w * (drho + (rr + rb) * e);                 // total as deviation
      if (p.two) p.buf[(size_t)Q * b.S + slot] = w * rr * (1.0f + e);
    } else if (p.comp == 0) {
      const float f = p.in0[(size_t)q * b.S + s];
      p.buf[slot] = f - w;
      if (p.two) p.buf[(size_t)Q * b.S + slot] = f;
    } else {
      p.buf[slot] += p.in0[(size_t)q * b.S + s];
    }
  }
}

// Debug accessor: full pre-collision populations of one component, [19][S].
template <int MODE>
__global__ void k_gatherf(const IoParams p) {
  const Box& b = p.box;
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= b.S) return;
  const int x = (int)(s % b.nx), y = (int)((s / b.nx) % b.ny), z = (int)(s / ((long long)b.nx * b.ny));
  const bool sol = b.mask && solid_at(b, x, y, z);
  for (int q = 0; q < Q; ++q) {
    float v = 0.f;
    if (!sol) {
      const size_t slot = read_slot_rt<MODE>(b, q, x, y, z);
      const float t = p.buf[slot] + wq(q);
      if (!p.two) v = t;
      else {
        const float r = p.buf[(size_t)Q * b.S + slot];
        v = p.comp == 0 ? r : t - r;
      }
    }
    p.out0[(size_t)q * b.S + s] = v;
  }
}

// K3: rho_r, rho_b and u = (m + F/2)/rho (Eq. 3; half-force shift of Guo forcing).
// Needs the phi array of the current state (K1 must have run).  out0 = rho_r, out1 = rho_b,
// out2 = u[3][S]; any may be null.
template <int MODE>
__global__ void k_macros(const IoParams p) {
  const Box& b = p.box;
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= b.S) return;
  const int x = (int)(s % b.nx), y = (int)((s / b.nx) % b.ny), z = (int)(s / ((long long)b.nx * b.ny));
  float rr = 0.f, rb = 0.f, ux = 0.f, uy = 0.f, uz = 0.f;
  if (!(b.mask && solid_at(b, x, y, z))) {
    const int cxs[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
    const int cys[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
    const int czs[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
    float dr = 0.f, mx = 0.f, my = 0.f, mz = 0.f;
    for (int q = 0; q < Q; ++q) {
      const size_t slot = read_slot_rt<MODE>(b, q, x, y, z);
      const float t = p.buf[slot];
      dr += t;
      mx += cxs[q] * t; my += cys[q] * t; mz += czs[q] * t;
      if (p.two) rr += p.buf[(size_t)Q * b.S + slot];
    }
    const float rho = 1.0f + dr;
    if (!p.two) rr = rho;
    rb = p.two ? rho - rr : 0.f;
    float Fx = rho * p.gx, Fy = rho * p.gy, Fz = rho * p.gz;
    if (p.two && p.A_nc != 0.f) {
      const float* ph = p.phi + phi_index(b, x, y, z);
      const long long px = b.nx + 2 * HALO, pxy = px * (b.ny + 2 * HALO);
      const float phi0 = ph[0];
      float Gx = 0.f, Gy = 0.f, Gz = 0.f;
      for (int q = 1; q < Q; ++q) {
        float v = ph[cxs[q] + px * cys[q] + pxy * czs[q]];
        if (v > PHI_SOLID_TEST) v = phi0;
        const float k = 3.0f * wq(q);
        Gx += k * cxs[q] * v; Gy += k * cys[q] * v; Gz += k * czs[q] * v;
      }
      const float Gn = sqrtf(Gx * Gx + Gy * Gy + Gz * Gz);
      if (fabsf(phi0) < p.phi_c && Gn > EPS_G) {
        const float invG = 1.0f / Gn;
        const float nx_ = -Gx * invG, ny_ = -Gy * invG, nz_ = -Gz * invG;
        int h = 0;
        for (int k = 1; k <= H_MAX_NC; ++k) {
          const int dx = (int)roundf(k * nx_), dy = (int)roundf(k * ny_), dz = (int)roundf(k * nz_);
          const float v = ph[dx + px * dy + pxy * dz];
          if (v > PHI_SOLID_TEST) break;
          if (k >= 2 && v >= phi0) { h = k; break; }
        }
        if (h > 0) {
          const float Ah = h <= H_MIN_NC ? p.A_nc : p.A_nc * ((float)(H_MIN_NC * H_MIN_NC * H_MIN_NC) / (float)(h * h * h));
          Fx += 0.5f * Ah * Gx; Fy += 0.5f * Ah * Gy; Fz += 0.5f * Ah * Gz;
        }
      }
    }
    const float inv_rho = 1.0f / rho;
    ux = (mx + 0.5f * Fx) * inv_rho; uy = (my + 0.5f * Fy) * inv_rho; uz = (mz + 0.5f * Fz) * inv_rho;
  }
  if (p.out0) p.out0[s] = rr;
  if (p.out1 && p.two) p.out1[s] = rb;
  if (p.out2) { p.out2[s] = ux; p.out2[b.S + s] = uy; p.out2[2 * b.S + s] = uz; }
}

// phi without ghost layers or sentinels, for lb_get_phi
__global__ void k_unpad_phi(const float* phi, float* out, Box b) {
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= b.S) return;
  const int x = (int)(s % b.nx), y = (int)((s / b.nx) % b.ny), z = (int)(s / ((long long)b.nx * b.ny));
  const float v = phi[phi_index(b, x, y, z)];
  out[s] = v > PHI_SOLID_TEST ? 0.f : v;
}

// bytes [S] -> bit-packed words
__global__ void k_pack_mask(const uint8_t* bytes, uint32_t* words, Box b) {
  const long long wi = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long nw = (long long)b.nxw * b.ny * b.nz;
  if (wi >= nw) return;
  const long long row = wi / b.nxw;
  const int xw = (int)(wi % b.nxw);
  uint32_t m = 0;
  for (int i = 0; i < 32; ++i) {
    const int x = xw * 32 + i;
    if (x < b.nx && bytes[row * b.nx + x]) m |= 1u << i;
  }
  words[wi] = m;
}

}  // namespace lb
