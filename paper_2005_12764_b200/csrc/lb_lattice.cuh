// D3Q19 lattice constants and small device helpers for the CUDA path (sm_100a).
// Velocity order: include/lb.h.  The paper numbers i = 1..19 and fixes no order;
// weights "normalized to unity" are the standard D3Q19 values.
// This header is part of the product; the oracle (oracle/) has its own, separate tables.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace lb {

constexpr int Q = 19;
constexpr int HALO = 4;        // ghost layers of the phi array on every side (>= H_MAX)
constexpr int H_MIN_NC = 3;    // "h_min = 3-4 lattice units"
constexpr int H_MAX_NC = 4;    // outer cut-off of the contact probe (G10)
constexpr float EPS_G = 1e-12f;        // guard on |grad phi| (G7)
constexpr float PHI_SOLID = 1.0e30f;   // sentinel stored in the phi array at solid sites
constexpr float PHI_SOLID_TEST = 1.0e29f;

__host__ __device__ constexpr int cx(int q) {
  constexpr int t[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
  return t[q];
}
__host__ __device__ constexpr int cy(int q) {
  constexpr int t[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
  return t[q];
}
__host__ __device__ constexpr int cz(int q) {
  constexpr int t[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
  return t[q];
}
__host__ __device__ constexpr int opp(int q) { return q == 0 ? 0 : ((q & 1) ? q + 1 : q - 1); }
__host__ __device__ constexpr float wq(int q) {
  return q == 0 ? 1.0f / 3.0f : (q < 7 ? 1.0f / 18.0f : 1.0f / 36.0f);
}
// B_i of the colour-gradient perturbation: sum B_i = 1/3, sum B_i c_ia c_ib = delta_ab/3.
__host__ __device__ constexpr float bq(int q) {
  return q == 0 ? -1.0f / 3.0f : (q < 7 ? 1.0f / 18.0f : 1.0f / 36.0f);
}
// 1/|c_q| for q >= 1
__host__ __device__ constexpr float inv_cnorm(int q) {
  return q == 0 ? 0.0f : (q < 7 ? 1.0f : 0.70710678118654752440f);
}

// run-time-indexed copies of the velocity set (constant memory)
__constant__ int c_cx[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
__constant__ int c_cy[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
__constant__ int c_cz[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};

// Compile-time loop: f(std::integral_constant<int, i>) for i in [B, E).
template <int B, int E, class F>
__device__ __forceinline__ void static_for(F&& f) {
  if constexpr (B < E) {
    f(std::integral_constant<int, B>{});
    static_for<B + 1, E>(f);
  }
}

// How the populations of the state at time t are found in memory.
//   AB       pull from the previous step's post-collision buffer: f_q(x) = F_q(x - c_q), or
//            F_opp(q)(x) when x - c_q is solid; results go to the other buffer at (q, x).
//   AA_EVEN  single buffer, natural layout: f_q(x) = slot(q, x); results go to slot(opp q, x).
//   AA_ODD   single buffer after an even step: f_q(x) = slot(opp q, x - c_q), or slot(q, x) when
//            x - c_q is solid; f*_q goes to the slot that f_opp(q) was read from.
enum Mode { MODE_AB = 0, MODE_AA_EVEN = 1, MODE_AA_ODD = 2 };

struct Box {
  int nx, ny, nz;        // allocated extents (a z slab holds one ghost plane below and one above its own planes)
  int zlo, zhi;          // planes this handle updates: [zlo, zhi) = [0, nz), or [1, nz - 1) for a z slab
  int zper;              // z is periodic inside this box (0 for a slab: its z neighbours are other handles)
  int gnz, zoff;         // z extent of the whole (periodic) box and global z of the allocated plane 0: nz, 0 unless a slab
  int nxw;               // 32-bit mask words per x row
  long long S;           // sites (allocated)
  const uint32_t* mask;  // bit-packed solid mask (bit x&31 of word row*nxw + x>>5), or nullptr
  const uint32_t* gmask; // wall groups: two more bit planes of the same shape behind each other (group - 1 in binary), or nullptr
};

// State of one rigid spherical particle (the paper's section 6, Eq. 15).  Double
// precision: a position of a few hundred lattice units advanced by ~1e-3 per step loses its
// increments in fp32.  The first 15 values are lb_particle of include/lb.h.
struct PState {
  double r[3], u[3], w[3], q[4];   // centre, velocity, angular velocity, orientation quaternion (w, x, y, z)
  double R, mass;
  double inertia;                  // 2/5 m R^2
  double F[3], T[3];               // force and torque from the fluid links of the last step (G33)
  double Fpp[3];                   // from the other particles (G37)
  double Fext[3], Text[3];
  double ro[3], uo[3], wo[3];      // r, u, w before the last move (the node changes undo links made with them, G36)
};

__device__ __forceinline__ bool solid_at(const Box& b, int x, int y, int z) {
  return (b.mask[(size_t)(z * b.ny + y) * b.nxw + (x >> 5)] >> (x & 31)) & 1u;
}

// Wall group of a solid site: 1 = at rest, 2 / 3 / 4 = moving or open, StepParams::uw, wtype, wrho.
__device__ __forceinline__ int wall_group_at(const Box& b, int x, int y, int z) {
  if (!b.gmask) return 1;
  const size_t w = (size_t)(z * b.ny + y) * b.nxw + (x >> 5);
  const size_t nw = (size_t)b.nxw * b.ny * b.nz;
  const uint32_t g2 = (b.gmask[w] >> (x & 31)) & 1u, g3 = (b.gmask[nw + w] >> (x & 31)) & 1u;
  return 1 + (int)g2 + 2 * (int)g3;
}

// what the phi sentinel of a solid site encodes: the wall group (a particle's node counts as a wall at rest)
__device__ __forceinline__ int sentinel_code(const Box& b, int x, int y, int z) { return wall_group_at(b, x, y, z); }

__device__ __forceinline__ int wrap_m(int a, int n) { return a == 0 ? n - 1 : a - 1; }
__device__ __forceinline__ int wrap_p(int a, int n) { return a == n - 1 ? 0 : a + 1; }

// index of site (x,y,z) in the padded phi array
__device__ __forceinline__ size_t phi_index(const Box& b, int x, int y, int z) {
  return (size_t)(x + HALO) + (size_t)(b.nx + 2 * HALO) * ((size_t)(y + HALO) + (size_t)(b.ny + 2 * HALO) * (size_t)(z + HALO));
}

}  // namespace lb
