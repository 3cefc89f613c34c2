// C-ABI of the B200 colour-gradient LB hot path (include/lb.h).  Host logic only: argument
// checks, device memory through the allocator hooks (PyTorch's caching allocator in
// production), kernel launches on the handle's stream.  No CPU fallback of any step.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/lb.h"
#include "lb_kernels.cuh"

using namespace lb;

namespace {

lb_alloc_fn g_alloc = nullptr;
lb_free_fn g_free = nullptr;
void* g_user = nullptr;
std::string g_create_error;

// The allocator hooks are process-wide defaults; every handle captures the pair that was current
// at lb_create and uses it for its whole life (so a later lb_set_allocator never makes a handle
// free memory with another allocator than the one it came from).
struct Allocator {
  lb_alloc_fn alloc = nullptr;
  lb_free_fn free_fn = nullptr;
  void* user = nullptr;
};

void* dev_alloc(const Allocator& a, size_t bytes) {
  if (a.alloc) return a.alloc(bytes, a.user);
  void* p = nullptr;
  if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return p;
}
void dev_free(const Allocator& a, void* p) {
  if (!p) return;
  if (a.free_fn) a.free_fn(p, a.user);
  else cudaFree(p);
}

constexpr int MAX_DEVICES = 64;
constexpr int IO_CHUNKS = 8;

// Makes the handle's device current for the duration of one C-ABI call (one process may hold
// handles on several devices) and restores the caller's device afterwards.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (dev < 0) return;
    if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); prev = -1; return; }
    if (prev != dev) { switched = cudaSetDevice(dev) == cudaSuccess; cudaGetLastError(); }
  }
  ~DeviceGuard() { if (switched) { cudaSetDevice(prev); cudaGetLastError(); } }
};

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

}  // namespace

struct lb_handle_s {
  Allocator al;              // captured at lb_create
  int device = -1;           // CUDA device of this handle (the device current at lb_create; -1: none)
  int nx = 0, ny = 0, nz = 0;   // the caller's box: nz planes (of a slab: its own planes)
  int gz = 0;                // ghost planes below and above (1 for a z slab, lb_set_slab)
  int slab_z0 = 0, slab_nzg = 0;   // slab: first global plane, global extent
  int slab_phase = 0;        // slab: 0 = between steps, 1 = after lb_slab_begin, 2 = after lb_slab_interior
  bool phi_ghost_ok = false; // slab: the z ghost planes of phi match the current state (lb_slab_unpack_phi)
  long long S = 0;           // allocated sites nx * ny * (nz + 2 gz): what the kernels index
  long long Sx = 0;          // sites of the caller's arrays nx * ny * nz
  lb_params par{};
  float g[3] = {0, 0, 0};
  float phi_c = 0.9f;
  int nc_sym = 0;            // colour-symmetric near-contact probe (G29)
  int wet = 0;               // prescribed phi at solid nodes (G30)
  float phi_wall = 0.f;
  int forcing = 0;          // 0 Guo, 1 exact difference (Eq. 9)
  int storage = 0;          // 0 A/B, 1 AA
  bool two = true;
  bool inited = false;
  bool has_solid = false;
  bool has_moving = false;   // the mask holds wall groups 2 / 3 / 4 (moving walls, open boundaries)
  float uw[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};   // their velocities
  int wtype[3] = {0, 0, 0};  // what they are (G31): 0 moving wall, 1 velocity inlet, 2 reservoir, 3 pressure outlet
  float wrho[3][2] = {{0, 0}, {0, 0}, {0, 0}};       // prescribed rho_r, rho_b of an inlet / reservoir / outlet
  int aa_odd = 0;           // AA: is the next step the odd one?
  int cur = 0;              // A/B: buffer holding the current state
  float* buf[2] = {nullptr, nullptr};
  float* phi = nullptr;
  uint32_t* mask = nullptr;
  size_t bytes = 0;
  cudaStream_t stream = 0;
  long long launches = 0;
  CUtensorMap tmap{};
  CUtensorMap tmap2{};       // Shan-Chen model: the rho_b array
  float* phi2 = nullptr;
  int model = 0;            // 0 colour gradient, 1 Shan-Chen + exact difference (Eq. 5-10 of the paper)
  float G_C = 0.f;
  bool tmap_ok = false;
  bool phi_current = false;  // phi array matches the current populations
  float* mom = nullptr;      // forwarded moments Md, Mt (2 x S floats), written by k_fused
  int forward = 1;           // 1 = phi(t+1) from forwarded moments (k_phase_fwd), 0 = full k_phase sweep
  // rigid particles (NEXT-4)
  int np = 0;
  std::vector<PState> parts_host;   // what lb_set_particles gave (and the external forces)
  PState* parts = nullptr;          // device
  int* pid = nullptr;               // particle index per site, -1 elsewhere
  uint32_t* mask_static = nullptr;  // the walls of lb_set_geometry alone (the live mask also holds the particle nodes)
  bool user_solid = false, user_moving = false;
  int* povf = nullptr;              // k_part_remap overflow flag
  // particles in a slab (replicated data): lb_slab_part_get / lb_slab_part_put
  double* pred = nullptr;           // [np][6] this slab's share of the link sums, then of the node-change impulses
  double* ptot = nullptr;           // [np][6] the sums over all slabs, as the caller gave them back
  float* ghost_rho = nullptr;       // [2 faces][2 components][ny * nx] densities in the ghost planes (lb_slab_unpack_phi)
  int part_stage = 0;               // 0 = none pending, 1 = link sums wait for their total, 2 = impulses wait for theirs
  void* pend_send[2] = {nullptr, nullptr};   // the population messages lb_slab_begin was given, packed once the particles have moved
  int p_mobile = 1, p_lub = 0;
  double p_K = 0.0, p_hc = 0.0;
  int tune_zc = 0;           // z planes per CTA (0 = automatic)
  // lb_init / lb_get_macros with HOST arrays: copies in IO_CHUNKS pieces on a stream of their own, so that
  // the kernel works on one piece while the next one crosses PCIe
  cudaStream_t cstream = nullptr;
  cudaEvent_t cev[IO_CHUNKS + 1] = {};
  // CUDA graph of GRAPH_STEPS time steps for boxes whose step is bounded by launch latency (lb_step)
  int graph = -1;            // tuning key "graph": -1 = automatic (small boxes), 0 = never, 1 = whenever possible
  cudaGraphExec_t gexec = nullptr;
  cudaStream_t gstream = nullptr;          // capture stream (the caller's may be the legacy default stream, which cannot capture)
  std::vector<unsigned char> gkey;         // everything the captured launches depend on (graph_key)
  long long graph_kernels = 0;             // kernel nodes in the graph
  bool graph_failed = false;               // capture or instantiation failed once: not tried again
  int sm_count = 0;          // SMs of the handle's device (0: not asked yet)
  double* chk = nullptr;     // state check (lb_check_state): {sum rho_r, sum rho_b, non-finite count}
  long long steps_done = 0;  // time steps since lb_init
  long long last_check = 0;  // steps_done at the last state check
  int profiling = 0;
  cudaEvent_t ev_step[2] = {nullptr, nullptr};
  std::vector<cudaEvent_t> ev_k;   // 4 per step when profiling: K1 begin/end, K2 begin/end
  int ev_steps = 0;
  std::string err;

  int nza() const { return nz + 2 * gz; }   // allocated planes
  int zlo() const { return gz; }
  int zhi() const { return gz + nz; }
  Box box() const {
    Box b;
    b.nx = nx; b.ny = ny; b.nz = nza();
    b.zlo = zlo(); b.zhi = zhi(); b.zper = gz == 0;
    b.gnz = gz ? slab_nzg : nz; b.zoff = gz ? slab_z0 - gz : 0;
    b.nxw = (nx + 31) / 32;
    b.S = S;
    b.mask = has_solid ? mask : nullptr;
    b.gmask = (has_solid && has_moving) ? mask + (size_t)b.nxw * ny * nza() : nullptr;
    return b;
  }
  int planes() const { return two ? 2 * Q : Q; }
  int mode() const { return storage == 0 ? MODE_AB : (aa_odd ? MODE_AA_ODD : MODE_AA_EVEN); }
  float* cur_buf() const { return storage == 0 ? buf[cur] : buf[0]; }
};

namespace {

int fail(lb_handle h, int code, const std::string& msg) {
  if (h) h->err = msg;
  else g_create_error = msg;
  return code;
}

constexpr long long CHECK_EVERY = 1000;   // steps between two state checks inside lb_step (G23)
constexpr long long GRAPH_AUTO_SITES = 1LL << 21;     // boxes up to 128^3 count as bounded by launch latency (tuning key "graph")

int cuda_fail(lb_handle h, cudaError_t e, const char* what) {
  cudaGetLastError();
  return fail(h, LB_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

bool is_device_ptr(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// A device view of a caller array: the pointer itself, or a staged copy of a host array.
struct Staged {
  void* dev = nullptr;
  bool owned = false;
  Allocator al;
  ~Staged() { if (owned) dev_free(al, dev); }
};

int stage_in(lb_handle h, const void* src, size_t bytes, Staged& s, bool copy = true) {
  if (is_device_ptr(src)) { s.dev = const_cast<void*>(src); return LB_OK; }
  s.al = h->al;
  s.dev = dev_alloc(h->al, bytes);
  if (!s.dev) return fail(h, LB_ENOMEM, "staging buffer allocation failed");
  s.owned = true;
  if (!copy) return LB_OK;       // (the caller copies piece by piece: io_pipeline)
  cudaError_t e = cudaMemcpyAsync(s.dev, src, bytes, cudaMemcpyHostToDevice, h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "H2D copy");
  return LB_OK;
}

// The copy stream and the events of the chunked host transfers (created on first use).
int io_pipeline(lb_handle h) {
  if (!h->cstream && cudaStreamCreateWithFlags(&h->cstream, cudaStreamNonBlocking) != cudaSuccess) return cuda_fail(h, cudaGetLastError(), "copy stream");
  for (cudaEvent_t& e : h->cev)
    if (!e && cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return cuda_fail(h, cudaGetLastError(), "copy event");
  return LB_OK;
}
// elements [*e0, *e1) of piece c of n elements (pieces start at multiples of 1024 elements)
void io_chunk(long long n, int c, long long* e0, long long* e1) {
  const long long per = ((n + IO_CHUNKS - 1) / IO_CHUNKS + 1023) / 1024 * 1024;
  *e0 = std::min(n, per * c);
  *e1 = std::min(n, per * (c + 1));
}

// Output staging: device pointer as is, else a device temporary copied back by finish_out.
int stage_out(lb_handle h, void* dst, size_t bytes, Staged& s) {
  if (!dst) return LB_OK;
  if (is_device_ptr(dst)) { s.dev = dst; return LB_OK; }
  s.al = h->al;
  s.dev = dev_alloc(h->al, bytes);
  if (!s.dev) return fail(h, LB_ENOMEM, "staging buffer allocation failed");
  s.owned = true;
  return LB_OK;
}
int finish_out(lb_handle h, void* dst, size_t bytes, Staged& s) {
  if (!dst || !s.owned) return LB_OK;
  cudaError_t e = cudaMemcpyAsync(dst, s.dev, bytes, cudaMemcpyDeviceToHost, h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "D2H copy");
  return LB_OK;
}

}  // namespace

// ------------------------------------------------------------------------------ launches
namespace {

StepParams make_step_params(lb_handle h, const float* src, float* dst, int zc, int z0 = -1, int z1 = -1) {
  StepParams p;
  memset(&p, 0, sizeof(p));      // (padding too: graph_key compares the bytes)
  p.z0 = z0 < 0 ? h->zlo() : z0;
  p.z1 = z1 < 0 ? h->zhi() : z1;
  p.src = src; p.dst = dst; p.phi = h->phi;
  p.phi2 = h->phi2; p.sc = h->model == 1; p.G_C = h->G_C;
  p.parts = h->np > 0 ? h->parts : nullptr;
  const size_t plane = (h->two ? 2 : 1) * (size_t)h->S;   // floats per direction plane ({T, R} pairs or T)
  for (int q = 0; q < Q; ++q) {
    p.ps[q] = src ? src + (size_t)q * plane : nullptr;
    p.pd[q] = dst ? dst + (size_t)q * plane : nullptr;
  }
  p.Md = h->mom; p.Mt = h->mom ? h->mom + h->S : nullptr; p.EX = h->mom ? h->mom + 2 * h->S : nullptr;
  p.box = h->box();
  p.zc = zc;
  p.halo = (h->model == 0 && h->par.A_nc != 0.f) ? H_MAX_NC : 1;
  p.tau_r = h->par.tau_r; p.tau_b = h->par.tau_b; p.A = h->par.A; p.beta = h->par.beta;
  p.A_nc = h->par.A_nc; p.phi_c = h->phi_c;
  p.nc_sym = h->nc_sym; p.wet = h->wet; p.phi_wall = h->phi_wall;
  p.gx = h->g[0]; p.gy = h->g[1]; p.gz = h->g[2];
  p.two_tau = h->par.tau_r != h->par.tau_b;
  p.has_g = (h->g[0] != 0.f || h->g[1] != 0.f || h->g[2] != 0.f);
  p.edm = h->forcing;
  p.has_moving = h->has_solid && h->has_moving;
  for (int g = 0; g < 3; ++g) {
    for (int a = 0; a < 3; ++a) p.uw[g][a] = h->uw[g][a];
    p.wtype[g] = h->wtype[g];
    p.wrho[g][0] = h->wrho[g][0]; p.wrho[g][1] = h->wrho[g][1];
  }
  return p;
}

// z planes per CTA: enough CTAs for ~8 waves of 148 SMs x 4 resident CTAs, at least 8 planes
// so that the phi-ring prologue (2H+1 planes) is amortised.
// z planes per CTA.  Measured on B200: short columns win (256^3: 0.91 ms at 8
// planes, 0.95 at 16, 1.11 at 64; 640^3: 16.2 ms at 16, 18.9 at 214), but every brick face costs
// k_phase_fwd a gather, so: 10..20 planes, and among those the count whose number of CTAs fills
// whole waves of (SMs x resident CTAs) best.
int pick_zc(lb_handle h) {
  int zc = 16;
  if (!h->sm_count) {       // of the handle's own device
    int sms = 148;
    if (h->device >= 0) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device);
    cudaGetLastError();
    h->sm_count = sms;
  }
  // resident CTAs per SM: 3, but 2 for the instantiations with wall groups (WALLS = 2)
  const int slots = ((h->has_solid && h->has_moving) ? 2 : 3) * h->sm_count;
  const long long cols = (long long)((h->nx + TX - 1) / TX) * ((h->ny + TY - 1) / TY);
  if (h->tune_zc > 0) zc = h->tune_zc < h->nz ? h->tune_zc : h->nz;
  else if (cols * ((h->nz + 9) / 10) < slots) {
    // A box that does not fill one wave of CTAs even with 10-plane bricks (32^3: 8 bricks on 148 SMs):
    // the step then lasts as long as ONE brick, so the bricks are made as shallow as one wave allows
    // (C1: 27 -> 9 us per step).  Such a box lives in L2; the extra phi-ring prologues cost no HBM traffic.
    zc = (int)((cols * h->nz + slots - 1) / slots);
    if (zc < 1) zc = 1;
  } else {
    double eff[21], best_eff = -1.0;
    for (int c = 10; c <= 20 && c <= h->nz; ++c) {
      const long long ctas = cols * ((h->nz + c - 1) / c);
      const long long waves = (ctas + slots - 1) / slots;
      // planes actually computed per slot-wave (the last chunk may be short)
      eff[c] = (double)cols * h->nz / ((double)waves * slots * c);
      if (eff[c] > best_eff + 1e-9) { best_eff = eff[c]; zc = c; }
    }
    // among depths that fill the waves equally well (within half a percent: large boxes), the deepest:
    // fewer brick faces for k_phase_fwd (640^3: 17.13 GLUPS at 10 planes, 17.20 at 20)
    for (int c = 20; c > zc; --c)
      if (c <= h->nz && eff[c] >= best_eff - 0.005) { zc = c; break; }
  }
  // A slab's phi planes that wait for the halo, [zlo, zlo + H) and [zhi - H, zhi), must not touch an
  // inner brick face (lb_slab_end): bricks deeper than the phi halo, or one brick for the whole slab.
  if (zc > h->nz) zc = h->nz;
  if (h->gz && zc <= H_MAX_NC) zc = h->nz;
  return zc;
}

dim3 tile_grid(lb_handle h, int zc, int nplanes = -1) {
  if (nplanes < 0) nplanes = h->nz;
  return dim3((h->nx + TX - 1) / TX, (h->ny + TY - 1) / TY, (nplanes + zc - 1) / zc);
}

template <int MODE>
void launch_phase(lb_handle h, const StepParams& p, dim3 grid) {
  const dim3 blk(TX, TY);
  if (h->model == 1) {
    if (h->has_solid) k_phase<MODE, true, true><<<grid, blk, 0, h->stream>>>(p);
    else k_phase<MODE, false, true><<<grid, blk, 0, h->stream>>>(p);
  } else {
    if (h->has_solid) k_phase<MODE, true, false><<<grid, blk, 0, h->stream>>>(p);
    else k_phase<MODE, false, false><<<grid, blk, 0, h->stream>>>(p);
  }
}
template <int MODE, int WALLS, bool HAS_NC, int FMODE>
void launch_fused_t(lb_handle h, const StepParams& p, dim3 grid) {
  constexpr size_t smem = FusedSmem<HAS_NC ? H_MAX_NC : 1>::BYTES;
  static bool attr_set[MAX_DEVICES] = {};   // per instantiation and per device (the attribute is per device)
  const int d = h->device >= 0 && h->device < MAX_DEVICES ? h->device : 0;
  if (!attr_set[d]) {
    cudaFuncSetAttribute(k_fused<MODE, WALLS, HAS_NC, FMODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr_set[d] = true;
  }
  k_fused<MODE, WALLS, HAS_NC, FMODE><<<grid, dim3(TX, TY), smem, h->stream>>>(p, h->tmap, h->tmap);
}
template <int MODE, int WALLS, bool HAS_NC>
void launch_fused_g(lb_handle h, const StepParams& p, dim3 grid) {
  // The in-place (AA) instantiations without any force run 25 % slower than those that carry the
  // Guo term (measured at 256^3: 1.16 against 0.87 ms; the extra arithmetic spaces out the shifted
  // stores), and with g = 0 the term adds exactly zero, so AA always takes the force variant.
  // moving walls (WALLS == 2, a rare configuration) are built for the force variants only
  const bool g = p.has_g || (MODE != MODE_AB && !HAS_NC) || WALLS == 2;
  const bool edm = p.edm && (HAS_NC || p.has_g);    // no force, no source: nothing to choose
#ifdef LB_BUILD_SUBSET      // developer builds (LB_BUILD_SUBSET=1 python -m ...build): Guo forcing, walls at rest or none
  if (edm) { h->err = "not in this developer build (LB_BUILD_SUBSET)"; return; }
  if constexpr (WALLS != 2) {
    if (g) launch_fused_t<MODE, WALLS, HAS_NC, 1>(h, p, grid);
    else launch_fused_t<MODE, WALLS, HAS_NC, 0>(h, p, grid);
  } else {
    launch_fused_t<MODE, 2, HAS_NC, 1>(h, p, grid);
  }
#else
  if (edm) {
    if (g) launch_fused_t<MODE, WALLS, HAS_NC, 3>(h, p, grid);
    else if constexpr (HAS_NC && WALLS != 2) launch_fused_t<MODE, WALLS, HAS_NC, 2>(h, p, grid);
  } else {
    if (g) launch_fused_t<MODE, WALLS, HAS_NC, 1>(h, p, grid);
    else if constexpr (WALLS != 2) launch_fused_t<MODE, WALLS, HAS_NC, 0>(h, p, grid);
  }
#endif
}
template <int MODE, int WALLS, int FMODE>
void launch_fused_sc(lb_handle h, const StepParams& p, dim3 grid) {
  constexpr size_t smem = FusedSmem<1, true>::BYTES;
  static bool attr_set[MAX_DEVICES] = {};   // per instantiation and per device
  const int d = h->device >= 0 && h->device < MAX_DEVICES ? h->device : 0;
  if (!attr_set[d]) {
    cudaFuncSetAttribute(k_fused<MODE, WALLS, false, FMODE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr_set[d] = true;
  }
  k_fused<MODE, WALLS, false, FMODE, true><<<grid, dim3(TX, TY), smem, h->stream>>>(p, h->tmap, h->tmap2);
}
template <int MODE>
void launch_fused(lb_handle h, const StepParams& p, dim3 grid) {
#ifndef LB_BUILD_SUBSET
  if (h->model == 1) {      // Shan-Chen: no near contact; the only force flag is the body force
    const bool g = p.has_g || MODE != MODE_AB;    // AA: the body-force instantiation, as in launch_fused_g
    if (p.has_moving) launch_fused_sc<MODE, 2, 1>(h, p, grid);
    else if (h->has_solid) { if (g) launch_fused_sc<MODE, 1, 1>(h, p, grid); else launch_fused_sc<MODE, 1, 0>(h, p, grid); }
    else { if (g) launch_fused_sc<MODE, 0, 1>(h, p, grid); else launch_fused_sc<MODE, 0, 0>(h, p, grid); }
    return;
  }
#endif
  const bool nc = h->par.A_nc != 0.f;
  if (p.has_moving) {
    if (nc) launch_fused_g<MODE, 2, true>(h, p, grid);
    else launch_fused_g<MODE, 2, false>(h, p, grid);
  } else if (h->has_solid) {
    if (nc) launch_fused_g<MODE, 1, true>(h, p, grid);
    else launch_fused_g<MODE, 1, false>(h, p, grid);
  } else {
    if (nc) launch_fused_g<MODE, 0, true>(h, p, grid);
    else launch_fused_g<MODE, 0, false>(h, p, grid);
  }
}
template <int MODE>
void launch_phase_fwd(lb_handle h, const StepParams& p, dim3 grid) {
  const dim3 blk(TX, TY);
  if (h->model == 1) {
    if (h->has_solid) k_phase_fwd<MODE, true, true><<<grid, blk, 0, h->stream>>>(p);
    else k_phase_fwd<MODE, false, true><<<grid, blk, 0, h->stream>>>(p);
  } else {
    if (h->has_solid) k_phase_fwd<MODE, true, false><<<grid, blk, 0, h->stream>>>(p);
    else k_phase_fwd<MODE, false, false><<<grid, blk, 0, h->stream>>>(p);
  }
}
template <int MODE>
void launch_single(lb_handle h, const StepParams& p, dim3 grid) {
  if (h->has_solid) k_single<MODE, true><<<grid, dim3(TX, TY), 0, h->stream>>>(p);
  else k_single<MODE, false><<<grid, dim3(TX, TY), 0, h->stream>>>(p);
}

// K1 on the current state (no-op if phi is already current or in single-component mode)
void run_phase(lb_handle h) {
  if (!h->two || h->phi_current) return;
  const int zc = pick_zc(h);
  const StepParams p = make_step_params(h, h->cur_buf(), nullptr, zc);
  const dim3 grid = tile_grid(h, zc);
  switch (h->mode()) {
    case MODE_AB: launch_phase<MODE_AB>(h, p, grid); break;
    case MODE_AA_EVEN: launch_phase<MODE_AA_EVEN>(h, p, grid); break;
    default: launch_phase<MODE_AA_ODD>(h, p, grid); break;
  }
  h->launches++;
  h->phi_current = true;
  h->phi_ghost_ok = false;
}

float* next_buf(lb_handle h) { return h->storage == 0 ? h->buf[h->cur ^ 1] : h->buf[0]; }
int next_mode(lb_handle h) { return h->storage == 0 ? MODE_AB : (h->aa_odd ? MODE_AA_EVEN : MODE_AA_ODD); }

// K2 / K2s on the bricks that cover the planes [z0, z1) (whole bricks, counted from zlo): reads the
// current buffer, writes the next one.  Does not flip.
void launch_collide(lb_handle h, int z0, int z1) {
  if (z1 <= z0) return;
  const int zc = pick_zc(h);
  const dim3 grid = tile_grid(h, zc, z1 - z0);
  const StepParams p = make_step_params(h, h->cur_buf(), next_buf(h), zc, z0, z1);
  const int mode = h->mode();
  if (h->two) {
    if (mode == MODE_AB) launch_fused<MODE_AB>(h, p, grid);
    else if (mode == MODE_AA_EVEN) launch_fused<MODE_AA_EVEN>(h, p, grid);
    else launch_fused<MODE_AA_ODD>(h, p, grid);
  } else {
    if (mode == MODE_AB) launch_single<MODE_AB>(h, p, grid);
    else if (mode == MODE_AA_EVEN) launch_single<MODE_AA_EVEN>(h, p, grid);
    else launch_single<MODE_AA_ODD>(h, p, grid);
  }
  h->launches++;
}

// K1f on the planes [z0, z1): phi of the state that launch_collide has just written (buffer
// next_buf, read rule next_mode) from the moments k_fused forwarded.  Call before flip().
void launch_phase_forward(lb_handle h, int z0, int z1) {
  if (z1 <= z0 || !h->two) return;
  const int zc = pick_zc(h);      // the same z chunks as k_fused: the bricks must match
  const StepParams q = make_step_params(h, next_buf(h), nullptr, zc, z0, z1);
  const dim3 gridf((h->nx / 4 + TX - 1) / TX, (h->ny + TY - 1) / TY, z1 - z0);   // 4 sites per thread, one plane per CTA
  switch (next_mode(h)) {
    case MODE_AB: launch_phase_fwd<MODE_AB>(h, q, gridf); break;
    case MODE_AA_EVEN: launch_phase_fwd<MODE_AA_EVEN>(h, q, gridf); break;
    default: launch_phase_fwd<MODE_AA_ODD>(h, q, gridf); break;
  }
  h->launches++;
}

// the next buffer / parity becomes the current state
void flip(lb_handle h) {
  if (h->storage == 0) h->cur ^= 1;
  else h->aa_odd ^= 1;
  h->steps_done++;
}

// Does phi(t + 1) come from the forwarded moments (k_phase_fwd) in lb_step?  Not for bricks of one
// plane, which pick_zc gives a box far smaller than one wave of CTAs: there every plane is both z
// faces of its brick, k_phase_fwd gathers most populations anyway (four sites per thread, a quarter
// of its lanes busy at nx = 32), and the full sweep k_phase (one site per thread) is faster: 32^3
// 11.2 -> 7.1 us per step.  With two planes per brick forwarding still wins (128 x 32 x 32: 18.1
// against 22.6 us).  "forward" = 2 forwards regardless.
bool forwarding(lb_handle h) {
  return h->two && h->forward && (h->forward == 2 || h->gz || pick_zc(h) > 1);
}

PartParams make_part_params(lb_handle h) {
  PartParams q;
  memset(&q, 0, sizeof(q));
  const size_t plane = (h->two ? 2 : 1) * (size_t)h->S;
  for (int d = 0; d < Q; ++d) { q.ps[d] = h->cur_buf() + (size_t)d * plane; q.pd[d] = next_buf(h) + (size_t)d * plane; }
  q.box = h->box();
  q.mask = h->mask; q.pid = h->pid; q.parts = h->parts; q.np = h->np;
  q.mobile = h->p_mobile; q.K = h->p_K; q.hc = h->p_hc; q.lub = h->p_lub;
  q.mu = ((double)h->par.tau_r - 0.5) / 3.0;
  q.overflow = h->povf;
  q.part_out = h->gz ? h->pred : nullptr;
  q.tot_in = h->gz ? h->ptot : nullptr;
  q.ghost_rho = h->ghost_rho;
  return q;
}

// The particles' part of a step (Eq. 15), between the fused kernel, which applied
// the link rule to what it stored, and the flip: momentum exchange, leapfrog, node changes.
// In three parts, because a slab needs the sums over all slabs in between (lb_slab_part_put).
void particles_force(lb_handle h) {
  const PartParams q = make_part_params(h);
  if (h->two) k_part_force<true><<<h->np, 256, 0, h->stream>>>(q);
  else k_part_force<false><<<h->np, 256, 0, h->stream>>>(q);
  h->launches++;
}
void particles_move(lb_handle h) {
  const PartParams q = make_part_params(h);
  k_part_pair<<<(h->np + 7) / 8, 256, 0, h->stream>>>(q);
  k_part_integrate<<<(h->np + 127) / 128, 128, 0, h->stream>>>(q);
  if (h->gz) cudaMemsetAsync(h->pred, 0, (size_t)h->np * 6 * sizeof(double), h->stream);   // (particles held in place list no changes)
  if (h->two) k_part_remap<true><<<h->np, 256, 0, h->stream>>>(q);
  else k_part_remap<false><<<h->np, 256, 0, h->stream>>>(q);
  h->launches += 3;
}
void particles_apply(lb_handle h) {     // slabs only
  const PartParams q = make_part_params(h);
  k_part_apply<<<(h->np + 127) / 128, 128, 0, h->stream>>>(q);
  h->launches++;
}
void run_particles(lb_handle h) {
  particles_force(h);
  particles_move(h);
}
// phi again in the shells around the particles, for the state launch_collide has written (before flip())
void particles_phi(lb_handle h) {
  const StepParams q = make_step_params(h, next_buf(h), nullptr, pick_zc(h), h->zlo(), h->zhi());
  // rows of the largest particle's box, 32 per CTA (4 per warp)
  double rmax = 0.0;
  for (const PState& P : h->parts_host) rmax = std::max(rmax, P.R);
  const int ext = 2 * (int)std::ceil(rmax + 2.5) + 2;
  const int slices = std::max(1, std::min(64, (ext * ext + 31) / 32));
  k_part_phi<<<dim3(h->np, slices), 256, 0, h->stream>>>(q);
  h->launches++;
}

// One whole step of a box that is periodic in z: K2 (+ K1f) or K2s
void run_collide(lb_handle h, cudaEvent_t after_k2 = nullptr) {
  launch_collide(h, h->zlo(), h->zhi());
  if (after_k2) cudaEventRecord(after_k2, h->stream);
  if (h->np > 0) {
    // phi(t + 1) from the forwarded moments first (they belong to the node map of time t), then the
    // particles, then phi again in the shells around them (k_part_phi)
    const bool fwd = forwarding(h);
    if (fwd) launch_phase_forward(h, h->zlo(), h->zhi());
    run_particles(h);
    if (fwd) particles_phi(h);
    flip(h);
    h->phi_current = fwd;
  } else if (forwarding(h)) {
    launch_phase_forward(h, h->zlo(), h->zhi());
    flip(h);
    h->phi_current = true;
  } else {
    flip(h);
    h->phi_current = false;
  }
}

IoParams make_io_params(lb_handle h) {
  IoParams p;
  memset(&p, 0, sizeof(p));
  p.buf = h->cur_buf();
  const size_t plane = (h->two ? 2 : 1) * (size_t)h->S;   // floats per direction plane
  for (int q = 0; q < Q; ++q) { p.ps[q] = p.buf + (size_t)q * plane; p.pd[q] = p.buf + (size_t)q * plane; }
  p.box = h->box();
  p.s0 = (long long)h->zlo() * h->nx * h->ny;      // the caller's arrays hold the handle's own planes
  p.s1 = (long long)h->zhi() * h->nx * h->ny;
  p.c0 = 0; p.c1 = p.s1 - p.s0;
  p.phi = h->phi;
  p.phi2 = h->phi2; p.sc = h->model == 1; p.G_C = h->G_C;
  p.tau_r = h->par.tau_r; p.tau_b = h->par.tau_b; p.A = h->par.A; p.beta = h->par.beta;
  p.A_nc = h->par.A_nc; p.phi_c = h->phi_c;
  p.nc_sym = h->nc_sym; p.wet = h->wet; p.phi_wall = h->phi_wall;
  p.gx = h->g[0]; p.gy = h->g[1]; p.gz = h->g[2];
  return p;
}

// the cold kernels are instantiated for (storage mode) x (one / two components) x (walls)
#define LB_IO_DISPATCH(KERNEL)                                                                       \
  template <int MODE, bool TWO>                                                                      \
  void launch_##KERNEL##_t(lb_handle h, const IoParams& p, unsigned nb) {                            \
    if (h->has_solid) KERNEL<MODE, TWO, true><<<nb, 256, 0, h->stream>>>(p);                         \
    else KERNEL<MODE, TWO, false><<<nb, 256, 0, h->stream>>>(p);                                     \
  }                                                                                                  \
  void launch_##KERNEL(lb_handle h, const IoParams& p) {                                             \
    const unsigned nb = (unsigned)((p.c1 - p.c0 + 255) / 256);                                       \
    const int mode = h->mode();                                                                      \
    if (h->two) {                                                                                    \
      if (mode == MODE_AB) launch_##KERNEL##_t<MODE_AB, true>(h, p, nb);                             \
      else if (mode == MODE_AA_EVEN) launch_##KERNEL##_t<MODE_AA_EVEN, true>(h, p, nb);              \
      else launch_##KERNEL##_t<MODE_AA_ODD, true>(h, p, nb);                                         \
    } else {                                                                                         \
      if (mode == MODE_AB) launch_##KERNEL##_t<MODE_AB, false>(h, p, nb);                            \
      else if (mode == MODE_AA_EVEN) launch_##KERNEL##_t<MODE_AA_EVEN, false>(h, p, nb);             \
      else launch_##KERNEL##_t<MODE_AA_ODD, false>(h, p, nb);                                        \
    }                                                                                                \
    h->launches++;                                                                                   \
  }
LB_IO_DISPATCH(k_scatter)
LB_IO_DISPATCH(k_gatherf)
LB_IO_DISPATCH(k_macros)
#undef LB_IO_DISPATCH
template <int MODE, bool TWO>
void launch_check_t(lb_handle h, const IoParams& p, int nb) {
  if (h->has_solid) k_check<MODE, TWO, true><<<nb, 256, 0, h->stream>>>(p, h->chk);
  else k_check<MODE, TWO, false><<<nb, 256, 0, h->stream>>>(p, h->chk);
}
void launch_check(lb_handle h) {
  const IoParams p = make_io_params(h);
  const int nb = (int)std::min<long long>((p.s1 - p.s0 + 255) / 256, 148 * 16);
  const int mode = h->mode();
  if (h->two) {
    if (mode == MODE_AB) launch_check_t<MODE_AB, true>(h, p, nb);
    else if (mode == MODE_AA_EVEN) launch_check_t<MODE_AA_EVEN, true>(h, p, nb);
    else launch_check_t<MODE_AA_ODD, true>(h, p, nb);
  } else {
    if (mode == MODE_AB) launch_check_t<MODE_AB, false>(h, p, nb);
    else if (mode == MODE_AA_EVEN) launch_check_t<MODE_AA_EVEN, false>(h, p, nb);
    else launch_check_t<MODE_AA_ODD, false>(h, p, nb);
  }
  h->launches++;
}
void launch_scatter(lb_handle h, const IoParams& p) { launch_k_scatter(h, p); }
void launch_gatherf(lb_handle h, const IoParams& p) { launch_k_gatherf(h, p); }
void launch_macros(lb_handle h, const IoParams& p) { launch_k_macros(h, p); }

// Component masses and finiteness of the stored state (k_check); synchronises the stream.
int state_check(lb_handle h, double* mass_r, double* mass_b) {
  if (!h->chk) {
    h->chk = static_cast<double*>(dev_alloc(h->al, 3 * sizeof(double)));
    if (!h->chk) return fail(h, LB_ENOMEM, "state-check buffer allocation failed");
    h->bytes += 3 * sizeof(double);
  }
  cudaError_t e = cudaMemsetAsync(h->chk, 0, 3 * sizeof(double), h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "state check memset");
  launch_check(h);
  double out[3] = {0, 0, 0};
  e = cudaMemcpyAsync(out, h->chk, sizeof(out), cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "state check");
  h->last_check = h->steps_done;
  if (mass_r) *mass_r = out[0];
  if (mass_b) *mass_b = out[1];
  if (out[2] != 0.0 || !std::isfinite(out[0]) || !std::isfinite(out[1])) {
    char msg[160];
    snprintf(msg, sizeof(msg), "non-finite state after %lld steps: %.0f sites hold a NaN or Inf population", h->steps_done, out[2]);
    return fail(h, LB_ESTATE, msg);
  }
  return LB_OK;
}

int check_launch(lb_handle h, const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, LB_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
  return LB_OK;
}

}  // namespace

// ------------------------------------------------------------------------------ C-ABI
extern "C" {

int lb_set_allocator(lb_alloc_fn alloc, lb_free_fn free_fn, void* user) {
  if ((alloc == nullptr) != (free_fn == nullptr)) return LB_EINVAL;
  g_alloc = alloc; g_free = free_fn; g_user = user;
  return LB_OK;
}

int lb_create(int nx, int ny, int nz, const lb_params* p, lb_handle* out) {
  if (!out) return fail(nullptr, LB_EINVAL, "out is NULL");
  *out = nullptr;
  if (!p) return fail(nullptr, LB_EINVAL, "params is NULL");
  if (nx < 4 || ny < 4 || nz < 4) return fail(nullptr, LB_EINVAL, "every extent must be >= 4");
  if (nx % 4 != 0) return fail(nullptr, LB_EINVAL, "nx must be a multiple of 4");
  if ((long long)nx * ny * nz >= (1LL << 29)) return fail(nullptr, LB_EINVAL, "box too large (>= 2^29 sites)");
  if (!(p->tau_r > 0.5f) || !(p->tau_b > 0.5f)) return fail(nullptr, LB_EINVAL, "tau must exceed 0.5");
  lb_handle h = new (std::nothrow) lb_handle_s();
  if (!h) return fail(nullptr, LB_ENOMEM, "host allocation failed");
  h->nx = nx; h->ny = ny; h->nz = nz;
  h->S = h->Sx = (long long)nx * ny * nz;
  h->par = *p;
  h->al.alloc = g_alloc; h->al.free_fn = g_free; h->al.user = g_user;
  if (cudaGetDevice(&h->device) != cudaSuccess) { cudaGetLastError(); h->device = -1; }   // no device: later calls return LB_ECUDA
  *out = h;
  return LB_OK;
}

void lb_destroy(lb_handle h) {
  if (!h) return;
  DeviceGuard guard(h->device);
  if (h->inited || h->mask) cudaStreamSynchronize(h->stream);
  for (void* q : {(void*)h->buf[0], (void*)h->buf[1], (void*)h->phi, (void*)h->phi2, (void*)h->mask, (void*)h->mom, (void*)h->chk, (void*)h->parts, (void*)h->pid, (void*)h->mask_static, (void*)h->povf, (void*)h->pred, (void*)h->ptot, (void*)h->ghost_rho}) dev_free(h->al, q);
  if (h->cstream) cudaStreamDestroy(h->cstream);
  for (cudaEvent_t e : h->cev) if (e) cudaEventDestroy(e);
  if (h->gexec) cudaGraphExecDestroy(h->gexec);
  if (h->gstream) cudaStreamDestroy(h->gstream);
  for (int i = 0; i < 2; ++i) if (h->ev_step[i]) cudaEventDestroy(h->ev_step[i]);
  for (cudaEvent_t e : h->ev_k) cudaEventDestroy(e);
  cudaGetLastError();
  delete h;
}

int lb_set_stream(lb_handle h, void* cuda_stream) {
  if (!h) return LB_EINVAL;
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  return LB_OK;
}

int lb_set_geometry(lb_handle h, const uint8_t* solid_mask) {
  if (!h) return LB_EINVAL;
  DeviceGuard guard(h->device);
  if (h->inited) return fail(h, LB_ESTATE, "lb_set_geometry after lb_init");
  if (!solid_mask) { h->has_solid = h->user_solid = false; h->has_moving = h->user_moving = false; return LB_OK; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(h, LB_ECUDA, "no CUDA device (there is no CPU fallback)");
  }
  Box b = h->box();
  const size_t nwords = (size_t)b.nxw * h->ny * h->nza();   // a slab's mask covers its ghost planes too
  // three bit masks behind each other (solid, wall group 2, wall group 3) and one flag word
  if (!h->mask) {
    h->mask = static_cast<uint32_t*>(dev_alloc(h->al, (3 * nwords + 1) * 4));
    if (!h->mask) return fail(h, LB_ENOMEM, "mask allocation failed");
    h->bytes += (3 * nwords + 1) * 4;
  }
  Staged in;
  int rc = stage_in(h, solid_mask, (size_t)h->S, in);
  if (rc) return rc;
  const int tb = 256;
  int* flag = reinterpret_cast<int*>(h->mask + 3 * nwords);
  cudaMemsetAsync(flag, 0, sizeof(int), h->stream);
  k_pack_mask<<<(unsigned)((nwords + tb - 1) / tb), tb, 0, h->stream>>>(static_cast<const uint8_t*>(in.dev), h->mask, h->mask + nwords, b);
  k_any_moving<<<(unsigned)((h->S + tb - 1) / tb), tb, 0, h->stream>>>(static_cast<const uint8_t*>(in.dev), h->S, flag);
  h->launches += 2;
  rc = check_launch(h, "k_pack_mask");
  if (rc) return rc;
  int moving = 0;
  cudaError_t e = cudaMemcpyAsync(&moving, flag, sizeof(int), cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);   // also: the staged copy dies with `in`
  if (e != cudaSuccess) return cuda_fail(h, e, "lb_set_geometry");
  h->has_moving = h->user_moving = moving != 0;
  h->has_solid = h->user_solid = true;
  return LB_OK;
}

int lb_set_wall_velocity(lb_handle h, int group, float ux, float uy, float uz) {
  if (!h || group < 2 || group > 4) return fail(h, LB_EINVAL, "wall group must be 2, 3 or 4");
  h->uw[group - 2][0] = ux; h->uw[group - 2][1] = uy; h->uw[group - 2][2] = uz;
  return LB_OK;
}

int lb_set_wall_type(lb_handle h, int group, int type, float rho_r, float rho_b) {
  if (!h || group < 2 || group > 4) return fail(h, LB_EINVAL, "wall group must be 2, 3 or 4");
  if (type < 0 || type > 3) return fail(h, LB_EINVAL, "wall type must be 0 (wall), 1 (inlet), 2 (reservoir) or 3 (outlet)");
  if (type != 0 && (!(rho_r >= 0.f) || !(rho_b >= 0.f))) return fail(h, LB_EINVAL, "prescribed densities must be >= 0");
  h->wtype[group - 2] = type;
  h->wrho[group - 2][0] = rho_r; h->wrho[group - 2][1] = rho_b;
  return LB_OK;
}

int lb_set_body_force(lb_handle h, float gx, float gy, float gz) {
  if (!h) return LB_EINVAL;
  h->g[0] = gx; h->g[1] = gy; h->g[2] = gz;
  return LB_OK;
}

int lb_set_model(lb_handle h, int model, float G_C) {
  if (!h || (model != 0 && model != 1)) return fail(h, LB_EINVAL, "model must be 0 (colour gradient) or 1 (Shan-Chen)");
  if (h->inited) return fail(h, LB_ESTATE, "lb_set_model after lb_init");
#ifdef LB_BUILD_SUBSET
  if (model == 1) return fail(h, LB_EINVAL, "the Shan-Chen model is not in this developer build (LB_BUILD_SUBSET)");
#endif
  h->model = model;
  h->G_C = G_C;
  return LB_OK;
}

int lb_set_forcing(lb_handle h, int mode) {
  if (!h || (mode != 0 && mode != 1)) return fail(h, LB_EINVAL, "forcing must be 0 (Guo) or 1 (exact difference)");
#ifdef LB_BUILD_SUBSET
  if (mode == 1) return fail(h, LB_EINVAL, "exact-difference forcing is not in this developer build (LB_BUILD_SUBSET)");
#endif
  h->forcing = mode;
  return LB_OK;
}

int lb_set_nc_cutoff(lb_handle h, float phi_c) {
  if (!h) return LB_EINVAL;
  h->phi_c = phi_c;
  return LB_OK;
}

int lb_set_nc_symmetric(lb_handle h, int on) {
  if (!h) return LB_EINVAL;
  if (on != 0 && on != 1) return fail(h, LB_EINVAL, "lb_set_nc_symmetric: on must be 0 or 1");
  h->nc_sym = on;
  return LB_OK;
}

int lb_set_wall_phi(lb_handle h, int on, float phi_wall) {
  if (!h) return LB_EINVAL;
  if ((on != 0 && on != 1) || !(fabsf(phi_wall) <= 1.0f)) return fail(h, LB_EINVAL, "lb_set_wall_phi: on must be 0 or 1 and |phi_wall| <= 1");
  h->wet = on;
  h->phi_wall = phi_wall;
  return LB_OK;
}

int lb_set_storage(lb_handle h, int mode) {
  if (!h || (mode != 0 && mode != 1)) return fail(h, LB_EINVAL, "storage mode must be 0 (A/B) or 1 (AA)");
  if (h->inited) return fail(h, LB_ESTATE, "lb_set_storage after lb_init");
  h->storage = mode;
  return LB_OK;
}

int lb_set_slab(lb_handle h, int z0, int nz_global) {
  if (!h) return LB_EINVAL;
  if (h->inited || h->mask) return fail(h, LB_ESTATE, "lb_set_slab must precede lb_set_geometry and lb_init");
  if (nz_global <= 0) {      // back to a box that is periodic in z
    h->gz = 0; h->slab_z0 = 0; h->slab_nzg = 0;
    h->S = h->Sx;
    return LB_OK;
  }
  if (z0 < 0 || z0 + h->nz > nz_global) return fail(h, LB_EINVAL, "slab [z0, z0 + nz) does not fit the global extent");
  if (h->nz < 2 * H_MAX_NC) return fail(h, LB_EINVAL, "a slab needs at least 8 planes (twice the phi halo)");
  const long long Sa = (long long)h->nx * h->ny * (h->nz + 2);
  if (Sa >= (1LL << 29)) return fail(h, LB_EINVAL, "slab too large (>= 2^29 sites with its ghost planes)");
  h->gz = 1; h->slab_z0 = z0; h->slab_nzg = nz_global;
  h->S = Sa;
  return LB_OK;
}

}  // extern "C"

namespace {

// (Re)allocate population buffers, the padded phi array and its TMA descriptor.
int allocate_state(lb_handle h, bool two) {
  const int nbuf = h->storage == 0 ? 2 : 1;
  const int planes = two ? 2 * Q : Q;
  const size_t pbytes = (size_t)planes * (size_t)h->S * sizeof(float);
  if (h->inited && two != h->two) {   // component count changed: start over
    for (int i = 0; i < 2; ++i) { if (h->buf[i]) h->bytes -= (size_t)h->planes() * h->S * 4; dev_free(h->al, h->buf[i]); h->buf[i] = nullptr; }
  }
  h->two = two;
  for (int i = 0; i < nbuf; ++i) {
    if (!h->buf[i]) {
      h->buf[i] = static_cast<float*>(dev_alloc(h->al, pbytes));
      if (!h->buf[i]) return fail(h, LB_ENOMEM, "population buffer allocation failed");
      h->bytes += pbytes;
    }
  }
  if (two && !h->mom) {
    const size_t ex = (size_t)h->nza() * h->ny * ((h->nx + TX - 1) / TX) * 4;   // x-face sums: 2 sides x {D, Tm}
    const size_t mb = (2 * (size_t)h->S + ex) * sizeof(float);
    h->mom = static_cast<float*>(dev_alloc(h->al, mb));
    if (!h->mom) return fail(h, LB_ENOMEM, "moment buffer allocation failed");
    h->bytes += mb;
  }
  const bool nc = h->model == 0 && h->par.A_nc != 0.f;
  for (int f = 0; f < (h->model == 1 ? 2 : 1); ++f) {
    float*& field = f == 0 ? h->phi : h->phi2;
    if (!two || field) continue;
    const size_t px = h->nx + 2 * HALO, py = h->ny + 2 * HALO, pz = h->nza() + 2 * HALO;
    const size_t phib = px * py * pz * sizeof(float);
    field = static_cast<float*>(dev_alloc(h->al, phib));
    if (!field) return fail(h, LB_ENOMEM, "phi allocation failed");
    h->bytes += phib;
    cudaError_t e = cudaMemsetAsync(field, 0, phib, h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "phi memset");
    // TMA descriptor of the padded array: dims (x, y, z), box (BX, BY, 1)
    EncodeTiledFn enc = get_encode();
    if (!enc) return fail(h, LB_ECUDA, "cuTensorMapEncodeTiled entry point not found");
    cuuint64_t dims[3] = {px, py, pz};
    cuuint64_t strides[2] = {px * sizeof(float), px * py * sizeof(float)};
    cuuint32_t box[3] = {(cuuint32_t)(nc ? Ring<H_MAX_NC>::BX : Ring<1>::BX),
                         (cuuint32_t)(nc ? Ring<H_MAX_NC>::BY : Ring<1>::BY), 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(f == 0 ? &h->tmap : &h->tmap2, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, field, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(h, LB_ECUDA, "cuTensorMapEncodeTiled failed: " + std::to_string((int)r));
    h->tmap_ok = true;
  }
  return LB_OK;
}

}  // namespace

namespace {

// Particles at lb_init: the live mask = the walls + the particle nodes (G32), the particle index per
// site, the particle states on the device.
int init_particles(lb_handle h) {
  if (h->storage != 0) return fail(h, LB_ESTATE, "particles need A/B storage");
  if (h->model != 0) return fail(h, LB_ESTATE, "particles are built for the colour-gradient model and for one component");
  const Box b0 = h->box();
  const size_t nwords = (size_t)b0.nxw * h->ny * h->nza();
  const size_t mb = (3 * nwords + 1) * 4;
  cudaError_t e = cudaSuccess;
  if (!h->mask) {
    h->mask = static_cast<uint32_t*>(dev_alloc(h->al, mb));
    if (!h->mask) return fail(h, LB_ENOMEM, "mask allocation failed");
    h->bytes += mb;
    e = cudaMemsetAsync(h->mask, 0, mb, h->stream);
  }
  if (!h->mask_static) {       // the walls alone, as lb_set_geometry left them (or none)
    h->mask_static = static_cast<uint32_t*>(dev_alloc(h->al, nwords * 4));
    if (!h->mask_static) return fail(h, LB_ENOMEM, "mask allocation failed");
    h->bytes += nwords * 4;
    if (e == cudaSuccess) e = h->user_solid ? cudaMemcpyAsync(h->mask_static, h->mask, nwords * 4, cudaMemcpyDeviceToDevice, h->stream)
                                            : cudaMemsetAsync(h->mask_static, 0, nwords * 4, h->stream);
  }
  if (!h->pid) {
    h->pid = static_cast<int*>(dev_alloc(h->al, (size_t)h->S * sizeof(int)));
    h->povf = static_cast<int*>(dev_alloc(h->al, sizeof(int)));
    if (!h->pid || !h->povf) return fail(h, LB_ENOMEM, "particle index allocation failed");
    h->bytes += (size_t)h->S * sizeof(int) + sizeof(int);
  }
  if (!h->parts) {
    h->parts = static_cast<PState*>(dev_alloc(h->al, (size_t)h->np * sizeof(PState)));
    if (!h->parts) return fail(h, LB_ENOMEM, "particle state allocation failed");
    h->bytes += (size_t)h->np * sizeof(PState);
  }
  if (h->gz && !h->pred) {     // a slab: the buffers of the two sums over the slabs, the densities of the ghost planes
    const size_t rb = (size_t)h->np * 6 * sizeof(double), gb = (size_t)4 * h->nx * h->ny * sizeof(float);
    h->pred = static_cast<double*>(dev_alloc(h->al, rb));
    h->ptot = static_cast<double*>(dev_alloc(h->al, rb));
    h->ghost_rho = static_cast<float*>(dev_alloc(h->al, gb));
    if (!h->pred || !h->ptot || !h->ghost_rho) return fail(h, LB_ENOMEM, "particle reduction buffer allocation failed");
    h->bytes += 2 * rb + gb;
    if (e == cudaSuccess) e = cudaMemsetAsync(h->pred, 0, rb, h->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->ptot, 0, rb, h->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->ghost_rho, 0, gb, h->stream);
  }
  h->part_stage = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(h->mask, h->mask_static, nwords * 4, cudaMemcpyDeviceToDevice, h->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(h->pid, 0xff, (size_t)h->S * sizeof(int), h->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(h->povf, 0, sizeof(int), h->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(h->parts, h->parts_host.data(), (size_t)h->np * sizeof(PState), cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);      // parts_host is pageable
  if (e != cudaSuccess) return cuda_fail(h, e, "particle set-up");
  h->has_solid = true;         // to the hot kernels a particle's node is a wall at rest (k_part_force applies G33)
  const PartParams q = make_part_params(h);
  k_part_raster<<<h->np, 256, 0, h->stream>>>(q);
  h->launches++;
  return check_launch(h, "k_part_raster");
}

}  // namespace

extern "C" {

int lb_set_particles(lb_handle h, int n, const lb_particle* p) {
  if (!h || n < 0 || (n > 0 && !p)) return fail(h, LB_EINVAL, "lb_set_particles: n >= 0 and a host array of n particles");
  if (h->inited) return fail(h, LB_ESTATE, "lb_set_particles after lb_init");
  h->parts_host.assign((size_t)n, PState{});
  for (int i = 0; i < n; ++i) {
    PState& P = h->parts_host[i];
    for (int a = 0; a < 3; ++a) { P.r[a] = p[i].r[a]; P.u[a] = p[i].u[a]; P.w[a] = p[i].w[a]; P.ro[a] = P.r[a]; P.uo[a] = P.u[a]; P.wo[a] = P.w[a]; }
    for (int a = 0; a < 4; ++a) P.q[a] = p[i].q[a];
    P.R = p[i].R; P.mass = p[i].mass;
    if (!(P.R > 0.0) || !(P.mass > 0.0)) { h->parts_host.clear(); h->np = 0; return fail(h, LB_EINVAL, "particle radius and mass must be positive"); }
    if (2.0 * P.R + 4.0 > h->nx || 2.0 * P.R + 4.0 > h->ny || 2.0 * P.R + 4.0 > (h->gz ? h->slab_nzg : h->nz)) { h->parts_host.clear(); h->np = 0; return fail(h, LB_EINVAL, "particle too large for the box"); }
    P.inertia = 0.4 * P.mass * P.R * P.R;
  }
  h->np = n;
  return LB_OK;
}

int lb_set_particle_options(lb_handle h, int mobile, double K, double h_c, int lubrication) {
  if (!h) return LB_EINVAL;
  h->p_mobile = mobile ? 1 : 0; h->p_K = K; h->p_hc = h_c; h->p_lub = lubrication ? 1 : 0;
  return LB_OK;
}

int lb_set_particle_force(lb_handle h, int i, const double* F, const double* T) {
  if (!h || i < 0 || i >= h->np) return fail(h, LB_EINVAL, "no such particle");
  if (h->inited) return fail(h, LB_ESTATE, "lb_set_particle_force after lb_init");
  for (int a = 0; a < 3; ++a) { h->parts_host[i].Fext[a] = F ? F[a] : 0.0; h->parts_host[i].Text[a] = T ? T[a] : 0.0; }
  return LB_OK;
}

int lb_get_particles(lb_handle h, lb_particle* state, double* force) {
  if (!h) return LB_EINVAL;
  if (!h->inited || h->np == 0) return fail(h, LB_ESTATE, "lb_get_particles needs an initialised state with particles");
  DeviceGuard guard(h->device);
  std::vector<PState> tmp((size_t)h->np);
  int ovf = 0;
  cudaError_t e = cudaMemcpyAsync(tmp.data(), h->parts, (size_t)h->np * sizeof(PState), cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(&ovf, h->povf, sizeof(int), cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "lb_get_particles");
  for (int i = 0; i < h->np; ++i) {
    const PState& P = tmp[i];
    if (state) {
      for (int a = 0; a < 3; ++a) { state[i].r[a] = P.r[a]; state[i].u[a] = P.u[a]; state[i].w[a] = P.w[a]; }
      for (int a = 0; a < 4; ++a) state[i].q[a] = P.q[a];
      state[i].R = P.R; state[i].mass = P.mass;
    }
    if (force) for (int a = 0; a < 3; ++a) { force[9 * i + a] = P.F[a]; force[9 * i + 3 + a] = P.T[a]; force[9 * i + 6 + a] = P.Fpp[a]; }
  }
  if (ovf) return fail(h, LB_ESTATE, "a particle changed more nodes in one step than the node-change kernel holds (384): it moves too fast");
  return LB_OK;
}

int lb_init(lb_handle h, const float* rho_r, const float* rho_b, const float* u) {
  if (!h) return LB_EINVAL;
  DeviceGuard guard(h->device);
  if (!rho_r || !u) return fail(h, LB_EINVAL, "rho_r and u must not be NULL");
  if (h->model == 1 && !rho_b) return fail(h, LB_EINVAL, "the Shan-Chen model couples two components: rho_b must not be NULL");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(h, LB_ECUDA, "no CUDA device (there is no CPU fallback)");
  }
  int rc = allocate_state(h, rho_b != nullptr);
  if (rc) return rc;
  if (h->np > 0 && (rc = init_particles(h))) return rc;
  const size_t fb = (size_t)h->Sx * sizeof(float);
  Staged srr, srb, su;
  // host arrays: staged piece by piece below, under the kernel that turns the piece before into populations
  if ((rc = stage_in(h, rho_r, fb, srr, false))) return rc;
  if (rho_b && (rc = stage_in(h, rho_b, fb, srb, false))) return rc;
  if ((rc = stage_in(h, u, 3 * fb, su, false))) return rc;
  h->cur = 0;
  h->aa_odd = 0;
  h->steps_done = 0;
  h->last_check = 0;
  IoParams p = make_io_params(h);
  p.comp = -1;
  p.rho_r = static_cast<const float*>(srr.dev);
  p.rho_b = static_cast<const float*>(srb.dev);
  p.u = static_cast<const float*>(su.dev);
  // solid sites (and the planes of a slab that its own sites do not read) keep zeros so that stray reads
  // are harmless; in an undivided box without solid sites k_scatter writes every slot of every site, and
  // clearing 40 GB first costs 12 ms at 640^3
  cudaError_t e = cudaSuccess;
  if (h->has_solid || h->gz) e = cudaMemsetAsync(h->cur_buf(), 0, (size_t)h->planes() * h->S * sizeof(float), h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "population memset");
  if (srr.owned || srb.owned || su.owned) {
    if ((rc = io_pipeline(h))) return rc;
    cudaEventRecord(h->cev[IO_CHUNKS], h->stream);             // (the staging buffers and the cleared populations are ready)
    cudaStreamWaitEvent(h->cstream, h->cev[IO_CHUNKS], 0);
    const long long n = h->Sx;
    for (int c = 0; c < IO_CHUNKS; ++c) {
      long long e0, e1;
      io_chunk(n, c, &e0, &e1);
      if (e1 <= e0) continue;
      const size_t nb = (size_t)(e1 - e0) * sizeof(float);
      if (srr.owned) e = cudaMemcpyAsync(static_cast<float*>(srr.dev) + e0, rho_r + e0, nb, cudaMemcpyHostToDevice, h->cstream);
      if (e == cudaSuccess && srb.owned) e = cudaMemcpyAsync(static_cast<float*>(srb.dev) + e0, rho_b + e0, nb, cudaMemcpyHostToDevice, h->cstream);
      for (int a = 0; a < 3 && e == cudaSuccess && su.owned; ++a)
        e = cudaMemcpyAsync(static_cast<float*>(su.dev) + a * n + e0, u + a * n + e0, nb, cudaMemcpyHostToDevice, h->cstream);
      if (e != cudaSuccess) return cuda_fail(h, e, "H2D copy");
      cudaEventRecord(h->cev[c], h->cstream);
      cudaStreamWaitEvent(h->stream, h->cev[c], 0);
      p.c0 = e0; p.c1 = e1;
      launch_scatter(h, p);
    }
  } else {
    launch_scatter(h, p);
  }
  if ((rc = check_launch(h, "k_scatter"))) return rc;
  h->inited = true;
  h->phi_current = false;
  if (srr.owned || srb.owned || su.owned) {
    e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "lb_init");
  }
  return LB_OK;
}

namespace {

// A box that one wave of CTAs covers is bounded by the latency of its two dependent launches per step
// (C1, 32^3: ~8 us per launch), not by memory traffic.  For such boxes lb_step replays a CUDA graph
// of GRAPH_STEPS steps: the launches then cost the GPU front end a fraction of a stream launch
// and the host one call per GRAPH_STEPS steps.
constexpr int GRAPH_STEPS = 16;                       // even: the A/B and in-place parities return to where they were

// Everything the captured launches depend on.  The graph is rebuilt when any of it changes.
std::vector<unsigned char> graph_key(lb_handle h) {
  const StepParams p = make_step_params(h, h->cur_buf(), next_buf(h), pick_zc(h), h->zlo(), h->zhi());
  const long long extra[] = {h->model, h->has_solid, h->has_moving, h->forward, h->storage, h->cur, h->aa_odd, h->two,
                             (long long)(size_t)h->mom, (long long)(size_t)h->mask, (long long)(size_t)h->buf[0], (long long)(size_t)h->buf[1]};
  std::vector<unsigned char> k(sizeof(p) + sizeof(extra) + (h->np > 0 ? sizeof(PartParams) : 0));
  memcpy(k.data(), &p, sizeof(p));
  memcpy(k.data() + sizeof(p), extra, sizeof(extra));
  if (h->np > 0) {       // the particle kernels' parameters (buffers, options)
    const PartParams q = make_part_params(h);
    memcpy(k.data() + sizeof(p) + sizeof(extra), &q, sizeof(q));
  }
  return k;
}

bool graph_eligible(lb_handle h, int remaining) {
  if (h->graph == 0 || h->graph_failed || remaining < GRAPH_STEPS) return false;
  if (h->graph < 0 && h->Sx > GRAPH_AUTO_SITES) return false;
  if (h->profiling || h->gz) return false;
  // the host flags must come back to where they were: with forwarding phi is current at every step's
  // start (the first step after lb_init / lb_set_populations runs K1 by itself), without it never
  if (h->two && forwarding(h) != h->phi_current) return false;
  if (h->steps_done < 2) return false;                              // first launches set function attributes
  cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(h->stream, &st) != cudaSuccess) { cudaGetLastError(); return false; }
  return st == cudaStreamCaptureStatusNone;                         // the caller is capturing lb_step itself: plain launches
}

// Captures GRAPH_STEPS steps from the current parity.  Leaves the handle's host state as it was.
bool graph_build(lb_handle h, const std::vector<unsigned char>& key) {
  if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
  if (!h->gstream && cudaStreamCreateWithFlags(&h->gstream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return false; }
  const cudaStream_t user = h->stream;
  const long long l0 = h->launches, s0 = h->steps_done;
  const int cur0 = h->cur, odd0 = h->aa_odd;
  const bool pc0 = h->phi_current, pg0 = h->phi_ghost_ok;
  h->stream = h->gstream;
  cudaGraph_t g = nullptr;
  bool ok = cudaStreamBeginCapture(h->gstream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  if (ok) {
    for (int t = 0; t < GRAPH_STEPS; ++t) { run_phase(h); run_collide(h); }
    ok = cudaStreamEndCapture(h->gstream, &g) == cudaSuccess && g != nullptr;
  }
  h->stream = user;
  h->graph_kernels = h->launches - l0;
  h->launches = l0; h->steps_done = s0; h->cur = cur0; h->aa_odd = odd0; h->phi_current = pc0; h->phi_ghost_ok = pg0;
  if (ok) ok = cudaGraphInstantiate(&h->gexec, g, 0) == cudaSuccess;
  if (g) cudaGraphDestroy(g);
  if (!ok) { cudaGetLastError(); h->gexec = nullptr; return false; }
  h->gkey = key;
  return true;
}

}  // namespace

int lb_step(lb_handle h, int nsteps) {
  if (!h || nsteps < 0) return fail(h, LB_EINVAL, "nsteps must be >= 0");
  DeviceGuard guard(h->device);
  if (!h->inited) return fail(h, LB_ESTATE, "lb_step before lb_init");
  if (h->gz) return fail(h, LB_ESTATE, "a slab is stepped by lb_slab_begin / _interior / _end and the phi exchange, not by lb_step");
  for (int i = 0; i < 2; ++i)
    if (!h->ev_step[i] && cudaEventCreate(&h->ev_step[i]) != cudaSuccess) return cuda_fail(h, cudaGetLastError(), "event create");
  // profiling = n > 0: every n-th step of this call is bracketed by events (kernel by kernel)
  const int stride = h->profiling;
  const int nprof = stride > 0 ? (nsteps + stride - 1) / stride : 0;
  while ((int)h->ev_k.size() < 4 * nprof) {
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return cuda_fail(h, cudaGetLastError(), "event create");
    h->ev_k.push_back(e);
  }
  h->ev_steps = nprof;
  cudaEventRecord(h->ev_step[0], h->stream);
  for (int t = 0; t < nsteps; ++t) {
    // replays of the step graph, as many as fit before the end of the call and the next state check
    if (graph_eligible(h, nsteps - t)) {
      const long long room = std::min<long long>(nsteps - t, CHECK_EVERY - (h->steps_done - h->last_check));
      const int reps = (int)(room / GRAPH_STEPS);
      if (reps > 0) {
        const std::vector<unsigned char> key = graph_key(h);
        if ((h->gexec && key == h->gkey) || graph_build(h, key)) {
          cudaError_t e = cudaSuccess;
          for (int r = 0; r < reps && e == cudaSuccess; ++r) e = cudaGraphLaunch(h->gexec, h->stream);
          if (e != cudaSuccess) return cuda_fail(h, e, "lb_step: graph launch");
          h->launches += (long long)reps * h->graph_kernels;
          h->steps_done += (long long)reps * GRAPH_STEPS;
          t += reps * GRAPH_STEPS - 1;         // (the parities are where they were: GRAPH_STEPS is even)
          if (h->steps_done - h->last_check >= CHECK_EVERY) {
            int rc = check_launch(h, "lb_step");
            if (!rc) rc = state_check(h, nullptr, nullptr);
            if (rc) { cudaEventRecord(h->ev_step[1], h->stream); return rc; }
          }
          continue;
        }
        h->graph_failed = true;                // stays on plain launches
      }
    }
    const bool prof = stride > 0 && t % stride == 0;
    const int k = prof ? 4 * (t / stride) : 0;
    if (prof) cudaEventRecord(h->ev_k[k + 0], h->stream);
    run_phase(h);                 // K1: no-op unless phi is stale (first step, or forwarding off)
    if (prof) cudaEventRecord(h->ev_k[k + 1], h->stream);
    run_collide(h, prof ? h->ev_k[k + 2] : nullptr);   // K2 (+ K1f) or K2s
    if (prof) cudaEventRecord(h->ev_k[k + 3], h->stream);
    // G23: every CHECK_EVERY steps the component masses are summed on the device; a non-finite
    // state ends the call with LB_ESTATE (this is the one place where lb_step synchronises)
    if (h->steps_done - h->last_check >= CHECK_EVERY) {
      int rc = check_launch(h, "lb_step");
      if (!rc) rc = state_check(h, nullptr, nullptr);
      if (rc) { cudaEventRecord(h->ev_step[1], h->stream); return rc; }
    }
  }
  cudaEventRecord(h->ev_step[1], h->stream);
  return check_launch(h, "lb_step");
}

int lb_check_state(lb_handle h, double* mass_r, double* mass_b) {
  if (!h) return LB_EINVAL;
  if (!h->inited) return fail(h, LB_ESTATE, "lb_check_state before lb_init");
  DeviceGuard guard(h->device);
  return state_check(h, mass_r, mass_b);
}

int lb_get_macros(lb_handle h, float* rho_r, float* rho_b, float* u) {
  if (!h) return LB_EINVAL;
  DeviceGuard guard(h->device);
  if (!h->inited) return fail(h, LB_ESTATE, "lb_get_macros before lb_init");
  const size_t fb = (size_t)h->Sx * sizeof(float);
  Staged o0, o1, o2;
  int rc;
  if ((rc = stage_out(h, rho_r, fb, o0))) return rc;
  if (h->two && (rc = stage_out(h, rho_b, fb, o1))) return rc;
  if ((rc = stage_out(h, u, 3 * fb, o2))) return rc;
  run_phase(h);
  IoParams p = make_io_params(h);
  p.out0 = static_cast<float*>(o0.dev);
  p.out1 = static_cast<float*>(o1.dev);
  p.out2 = static_cast<float*>(o2.dev);
  if (o0.owned || o1.owned || o2.owned) {
    // host arrays: the fields piece by piece, each piece on its way over PCIe while the next one is formed
    if ((rc = io_pipeline(h))) return rc;
    const long long n = h->Sx;
    cudaError_t e = cudaSuccess;
    for (int c = 0; c < IO_CHUNKS; ++c) {
      long long e0, e1;
      io_chunk(n, c, &e0, &e1);
      if (e1 <= e0) continue;
      p.c0 = e0; p.c1 = e1;
      launch_macros(h, p);
      cudaEventRecord(h->cev[c], h->stream);
      cudaStreamWaitEvent(h->cstream, h->cev[c], 0);
      const size_t nb = (size_t)(e1 - e0) * sizeof(float);
      if (rho_r && o0.owned) e = cudaMemcpyAsync(rho_r + e0, static_cast<float*>(o0.dev) + e0, nb, cudaMemcpyDeviceToHost, h->cstream);
      if (e == cudaSuccess && h->two && rho_b && o1.owned) e = cudaMemcpyAsync(rho_b + e0, static_cast<float*>(o1.dev) + e0, nb, cudaMemcpyDeviceToHost, h->cstream);
      for (int a = 0; a < 3 && e == cudaSuccess && u && o2.owned; ++a)
        e = cudaMemcpyAsync(u + a * n + e0, static_cast<float*>(o2.dev) + a * n + e0, nb, cudaMemcpyDeviceToHost, h->cstream);
      if (e != cudaSuccess) return cuda_fail(h, e, "D2H copy");
    }
    if ((rc = check_launch(h, "k_macros"))) return rc;
    e = cudaStreamSynchronize(h->cstream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "lb_get_macros");
    return LB_OK;
  }
  launch_macros(h, p);
  return check_launch(h, "k_macros");
}

int lb_get_populations(lb_handle h, int comp, float* f) {
  if (!h || !f) return fail(h, LB_EINVAL, "f is NULL");
  DeviceGuard guard(h->device);
  if (!h->inited) return fail(h, LB_ESTATE, "lb_get_populations before lb_init");
  if (comp < 0 || comp > (h->two ? 1 : 0)) return fail(h, LB_EINVAL, "bad component");
  const size_t fb = (size_t)Q * h->Sx * sizeof(float);
  Staged o;
  int rc;
  if ((rc = stage_out(h, f, fb, o))) return rc;
  IoParams p = make_io_params(h);
  p.comp = comp;
  p.out0 = static_cast<float*>(o.dev);
  launch_gatherf(h, p);
  if ((rc = check_launch(h, "k_gatherf"))) return rc;
  if ((rc = finish_out(h, f, fb, o))) return rc;
  if (o.owned) {
    cudaError_t e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "lb_get_populations");
  }
  return LB_OK;
}

int lb_set_populations(lb_handle h, int comp, const float* f) {
  if (!h || !f) return fail(h, LB_EINVAL, "f is NULL");
  DeviceGuard guard(h->device);
  if (!h->inited) return fail(h, LB_ESTATE, "lb_set_populations before lb_init");
  if (comp < 0 || comp > (h->two ? 1 : 0)) return fail(h, LB_EINVAL, "bad component");
  const size_t fb = (size_t)Q * h->Sx * sizeof(float);
  Staged in;
  int rc;
  if ((rc = stage_in(h, f, fb, in))) return rc;
  if (comp == 0 && h->storage == 1) h->aa_odd = 0;   // AA: a full rewrite restores the natural layout
  IoParams p = make_io_params(h);
  p.comp = comp;
  p.in0 = static_cast<const float*>(in.dev);
  launch_scatter(h, p);
  if ((rc = check_launch(h, "k_scatter"))) return rc;
  h->phi_current = false;
  if (in.owned) {
    cudaError_t e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "lb_set_populations");
  }
  return LB_OK;
}

int lb_get_phi(lb_handle h, float* phi) {
  if (!h || !phi) return fail(h, LB_EINVAL, "phi is NULL");
  DeviceGuard guard(h->device);
  if (!h->inited || !h->two) return fail(h, LB_ESTATE, "lb_get_phi needs an initialised two-component state");
  const size_t fb = (size_t)h->Sx * sizeof(float);
  Staged o;
  int rc;
  if ((rc = stage_out(h, phi, fb, o))) return rc;
  run_phase(h);
  const int tb = 256;
  const long long s0 = (long long)h->zlo() * h->nx * h->ny, s1 = (long long)h->zhi() * h->nx * h->ny;
  k_unpad_phi<<<(unsigned)((h->Sx + tb - 1) / tb), tb, 0, h->stream>>>(h->phi, h->model == 1 ? h->phi2 : nullptr, static_cast<float*>(o.dev), h->box(), s0, s1);
  h->launches++;
  if ((rc = check_launch(h, "k_unpad_phi"))) return rc;
  if ((rc = finish_out(h, phi, fb, o))) return rc;
  if (o.owned) {
    cudaError_t e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "lb_get_phi");
  }
  return LB_OK;
}

// ------------------------------------------------------------------------------ z slabs
}  // extern "C"

namespace {

const int DIRS_UP[5] = {5, 11, 14, 15, 18};   // c_z = +1 (velocity order: include/lb.h)
const int DIRS_DN[5] = {6, 12, 13, 16, 17};   // c_z = -1

// The five (direction, plane) blocks of a face's message.  [0]: the message that travels to / came
// from the rank BELOW, [1]: ABOVE.  Which blocks depends on the storage mode of the step that has
// just collided:
//   A/B       pull: the neighbour reads F_q(x - c_q) out of its ghost plane        real plane -> ghost
//   AA even   the odd step reads slot (opp q, x - c_q) out of the ghost plane     real plane -> ghost
//   AA odd    the step pushed f*_q into slot (q, x + c_q) of the ghost plane      ghost -> real plane
struct SlabBlocks { const int* dirs[2]; int plane[2]; };

SlabBlocks slab_send_blocks(lb_handle h, int mode) {
  SlabBlocks b;
  if (mode == MODE_AB) { b.dirs[0] = DIRS_DN; b.plane[0] = h->zlo(); b.dirs[1] = DIRS_UP; b.plane[1] = h->zhi() - 1; }
  else if (mode == MODE_AA_EVEN) { b.dirs[0] = DIRS_UP; b.plane[0] = h->zlo(); b.dirs[1] = DIRS_DN; b.plane[1] = h->zhi() - 1; }
  else { b.dirs[0] = DIRS_DN; b.plane[0] = h->zlo() - 1; b.dirs[1] = DIRS_UP; b.plane[1] = h->zhi(); }
  return b;
}
SlabBlocks slab_recv_blocks(lb_handle h, int mode) {
  SlabBlocks b;
  if (mode == MODE_AB) { b.dirs[0] = DIRS_UP; b.plane[0] = h->zlo() - 1; b.dirs[1] = DIRS_DN; b.plane[1] = h->zhi(); }
  else if (mode == MODE_AA_EVEN) { b.dirs[0] = DIRS_DN; b.plane[0] = h->zlo() - 1; b.dirs[1] = DIRS_UP; b.plane[1] = h->zhi(); }
  else { b.dirs[0] = DIRS_UP; b.plane[0] = h->zlo(); b.dirs[1] = DIRS_DN; b.plane[1] = h->zhi() - 1; }
  return b;
}

int slab_msg_check(lb_handle h, const void* lo, const void* hi) {
  if (!lo || !hi) return fail(h, LB_EINVAL, "halo message buffers must not be NULL");
  if (((uintptr_t)lo | (uintptr_t)hi) & 15u) return fail(h, LB_EINVAL, "halo message buffers must be 16-byte aligned");
  if (!is_device_ptr(lo) || !is_device_ptr(hi)) return fail(h, LB_EINVAL, "halo message buffers must be device memory");
  return LB_OK;
}

// pack (blocks of `buf` -> messages) or unpack (messages -> blocks of `buf`); merge: unpack after an
// in-place odd step between walls (k_halo_merge: only the slots whose source site is fluid)
void slab_copy_populations(lb_handle h, float* buf, const SlabBlocks& b, void* msg_lo, void* msg_hi, bool pack, bool merge = false) {
  const size_t esz = h->two ? 2 : 1;                       // floats per site in a plane
  const size_t blockf = (size_t)h->nx * h->ny * esz;       // floats per (direction, plane) block
  if (merge) {
    HaloMerge m;
    void* msg[2] = {msg_lo, msg_hi};
    for (int f = 0; f < 2; ++f)
      for (int k = 0; k < 5; ++k) {
        m.src[f][k] = static_cast<const float*>(msg[f]) + (size_t)k * blockf;
        m.dst[f][k] = buf + (size_t)b.dirs[f][k] * h->S * esz + (size_t)b.plane[f] * blockf;
        m.dirs[f][k] = b.dirs[f][k];
      }
    m.zsrc[0] = h->zlo() - 1;      // upward populations came out of the plane below the slab
    m.zsrc[1] = h->zhi();          // downward ones out of the plane above
    m.box = h->box();
    const dim3 grid((unsigned)(((size_t)h->nx * h->ny + 255) / 256), 5, 2);
    if (h->two) k_halo_merge<8><<<grid, 256, 0, h->stream>>>(m);
    else k_halo_merge<4><<<grid, 256, 0, h->stream>>>(m);
    h->launches++;
    return;
  }
  HaloCopy c;
  c.n4 = (long long)(blockf / 4);
  void* msg[2] = {msg_lo, msg_hi};
  for (int f = 0; f < 2; ++f)
    for (int k = 0; k < 5; ++k) {
      float* blk = buf + (size_t)b.dirs[f][k] * h->S * esz + (size_t)b.plane[f] * blockf;
      float* m = static_cast<float*>(msg[f]) + (size_t)k * blockf;
      c.src[f][k] = reinterpret_cast<const float4*>(pack ? blk : m);
      c.dst[f][k] = reinterpret_cast<float4*>(pack ? m : blk);
    }
  k_halo_copy<<<dim3((unsigned)((c.n4 + 255) / 256), 5, 2), 256, 0, h->stream>>>(c);
  h->launches++;
}

int slab_phi_halo(lb_handle h) { return (h->model == 0 && h->par.A_nc != 0.f) ? H_MAX_NC : 1; }
size_t slab_phi_plane_floats(lb_handle h) { return (size_t)(h->nx + 2 * HALO) * (h->ny + 2 * HALO); }

// the phi part of a phi message, and the densities of the boundary plane behind it (runs with particles)
size_t slab_phi_bytes(lb_handle h) {
  return h->two ? (size_t)(h->model == 1 ? 2 : 1) * slab_phi_halo(h) * slab_phi_plane_floats(h) * sizeof(float) : 0;
}
size_t slab_rho_bytes(lb_handle h) { return h->np > 0 ? (size_t)2 * h->nx * h->ny * sizeof(float) : 0; }

int slab_ready(lb_handle h, int phase, const char* what) {
  if (!h) return LB_EINVAL;
  if (!h->gz) return fail(h, LB_ESTATE, std::string(what) + ": not a slab (lb_set_slab)");
  if (!h->inited) return fail(h, LB_ESTATE, std::string(what) + " before lb_init");
  if (h->slab_phase != phase) return fail(h, LB_ESTATE, std::string(what) + " out of order (lb_slab_begin, lb_slab_interior, lb_slab_end, then the phi exchange)");
  return LB_OK;
}

// first and last brick of the slab, and what lies between
struct SlabBricks { int first0, first1, last0, last1, mid0, mid1; };
SlabBricks slab_bricks(lb_handle h) {
  const int zc = pick_zc(h), zlo = h->zlo(), zhi = h->zhi();
  const int nb = (h->nz + zc - 1) / zc;
  SlabBricks b;
  b.first0 = zlo; b.first1 = std::min(zhi, zlo + zc);
  b.last0 = nb > 1 ? zlo + (nb - 1) * zc : zhi; b.last1 = zhi;
  b.mid0 = b.first1; b.mid1 = nb > 2 ? b.last0 : b.first1;
  return b;
}

}  // namespace

extern "C" {

int lb_slab_halo_bytes(lb_handle h, size_t* pop_bytes, size_t* phi_bytes) {
  if (!h) return LB_EINVAL;
  if (!h->gz || !h->inited) return fail(h, LB_ESTATE, "lb_slab_halo_bytes needs an initialised slab");
  if (pop_bytes) *pop_bytes = (size_t)5 * h->nx * h->ny * (h->two ? 2 : 1) * sizeof(float);
  if (phi_bytes) *phi_bytes = slab_phi_bytes(h) + slab_rho_bytes(h);
  return LB_OK;
}

int lb_slab_begin(lb_handle h, void* send_lo, void* send_hi) {
  int rc = slab_ready(h, 0, "lb_slab_begin");
  if (rc) return rc;
  if ((rc = slab_msg_check(h, send_lo, send_hi))) return rc;
  if (h->two && !(h->phi_current && h->phi_ghost_ok))
    return fail(h, LB_ESTATE, "lb_slab_begin: the phi ghost planes are stale (lb_slab_pack_phi, exchange, lb_slab_unpack_phi first)");
  if (h->two && !h->forward) return fail(h, LB_ESTATE, "slabs need moment forwarding (lb_set_tuning forward = 1)");
  DeviceGuard guard(h->device);
  if (h->np > 0) {
    // Particles (replicated data): the link rule and the node changes rewrite stored
    // values of the boundary planes, so nothing is packed before the particles have moved.  All
    // bricks now, then this slab's share of the link sums; the messages are packed by the second
    // lb_slab_part_put.
    launch_collide(h, h->zlo(), h->zhi());
    particles_force(h);
    h->part_stage = 1;
    h->pend_send[0] = send_lo; h->pend_send[1] = send_hi;
    h->slab_phase = 1;
    return check_launch(h, "lb_slab_begin");
  }
  const SlabBricks b = slab_bricks(h);
  launch_collide(h, b.first0, b.first1);
  launch_collide(h, b.last0, b.last1);
  slab_copy_populations(h, next_buf(h), slab_send_blocks(h, h->mode()), send_lo, send_hi, true);
  h->slab_phase = 1;
  return check_launch(h, "lb_slab_begin");
}

int lb_slab_interior(lb_handle h) {
  int rc = slab_ready(h, 1, "lb_slab_interior");
  if (rc) return rc;
  DeviceGuard guard(h->device);
  if (h->np > 0 && h->part_stage != 0)
    return fail(h, LB_ESTATE, "lb_slab_interior: the particles wait for their sums (lb_slab_part_get / lb_slab_part_put, twice per step)");
  const SlabBricks b = slab_bricks(h);
  if (h->np == 0) launch_collide(h, b.mid0, b.mid1);         // (with particles lb_slab_begin has run every brick)
  const int H = slab_phi_halo(h);
  launch_phase_forward(h, h->zlo() + H, h->zhi() - H);     // the planes whose phi does not wait for the halo
  h->slab_phase = 2;
  return check_launch(h, "lb_slab_interior");
}

int lb_slab_end(lb_handle h, const void* recv_lo, const void* recv_hi) {
  int rc = slab_ready(h, 2, "lb_slab_end");
  if (rc) return rc;
  if ((rc = slab_msg_check(h, recv_lo, recv_hi))) return rc;
  DeviceGuard guard(h->device);
  slab_copy_populations(h, next_buf(h), slab_recv_blocks(h, h->mode()), const_cast<void*>(recv_lo), const_cast<void*>(recv_hi), false,
                        h->mode() == MODE_AA_ODD && h->has_solid);
  const int H = slab_phi_halo(h);
  launch_phase_forward(h, h->zlo(), std::min(h->zlo() + H, h->zhi()));
  launch_phase_forward(h, std::max(h->zhi() - H, h->zlo() + H), h->zhi());
  if (h->np > 0 && h->two) particles_phi(h);                 // phi again around the particles (own planes)
  flip(h);
  h->phi_current = h->two;
  h->phi_ghost_ok = false;
  h->slab_phase = 0;
  if ((rc = check_launch(h, "lb_slab_end"))) return rc;
  if (h->steps_done - h->last_check >= CHECK_EVERY) return state_check(h, nullptr, nullptr);   // G23, as in lb_step
  return LB_OK;
}

int lb_slab_pack_phi(lb_handle h, void* send_lo, void* send_hi) {
  int rc = slab_ready(h, 0, "lb_slab_pack_phi");
  if (rc) return rc;
  if (!h->two && h->np == 0) return LB_OK;         // one component: no phase field
  if ((rc = slab_msg_check(h, send_lo, send_hi))) return rc;
  DeviceGuard guard(h->device);
  if (h->np > 0) {                                 // the densities of the boundary planes, behind the phi part
    const PartParams q = make_part_params(h);
    float* lo = reinterpret_cast<float*>(static_cast<char*>(send_lo) + slab_phi_bytes(h));
    float* hi = reinterpret_cast<float*>(static_cast<char*>(send_hi) + slab_phi_bytes(h));
    const dim3 grid((unsigned)(((size_t)h->nx * h->ny + 255) / 256), 2);
    if (h->two) k_slab_rho<true><<<grid, 256, 0, h->stream>>>(q, lo, hi);
    else k_slab_rho<false><<<grid, 256, 0, h->stream>>>(q, lo, hi);
    h->launches++;
    if (!h->two) return check_launch(h, "lb_slab_pack_phi");
  }
  run_phase(h);                                    // after lb_init / lb_set_populations: the full sweep
  const int H = slab_phi_halo(h);
  const size_t pf = slab_phi_plane_floats(h), nb = (size_t)H * pf * sizeof(float);
  const float* fields[2] = {h->phi, h->phi2};
  for (int f = 0; f < (h->model == 1 ? 2 : 1); ++f) {
    cudaError_t e = cudaMemcpyAsync(static_cast<char*>(send_lo) + f * nb, fields[f] + (size_t)(h->zlo() + HALO) * pf, nb, cudaMemcpyDeviceToDevice, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(static_cast<char*>(send_hi) + f * nb, fields[f] + (size_t)(h->zhi() - H + HALO) * pf, nb, cudaMemcpyDeviceToDevice, h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "lb_slab_pack_phi");
  }
  return check_launch(h, "lb_slab_pack_phi");
}

int lb_slab_unpack_phi(lb_handle h, const void* recv_lo, const void* recv_hi) {
  int rc = slab_ready(h, 0, "lb_slab_unpack_phi");
  if (rc) return rc;
  if (!h->two && h->np == 0) return LB_OK;
  if ((rc = slab_msg_check(h, recv_lo, recv_hi))) return rc;
  if (h->two && !h->phi_current) return fail(h, LB_ESTATE, "lb_slab_unpack_phi before lb_slab_pack_phi");
  DeviceGuard guard(h->device);
  if (h->np > 0) {                                 // ghost densities: below from the message that came up, above from the one that came down
    const size_t gb = slab_rho_bytes(h);
    cudaError_t e = cudaMemcpyAsync(h->ghost_rho, static_cast<const char*>(recv_lo) + slab_phi_bytes(h), gb, cudaMemcpyDeviceToDevice, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(reinterpret_cast<char*>(h->ghost_rho) + gb, static_cast<const char*>(recv_hi) + slab_phi_bytes(h), gb, cudaMemcpyDeviceToDevice, h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "lb_slab_unpack_phi");
    if (!h->two) { h->phi_ghost_ok = true; return LB_OK; }
  }
  const int H = slab_phi_halo(h);
  const size_t pf = slab_phi_plane_floats(h), nb = (size_t)H * pf * sizeof(float);
  float* fields[2] = {h->phi, h->phi2};
  for (int f = 0; f < (h->model == 1 ? 2 : 1); ++f) {
    cudaError_t e = cudaMemcpyAsync(fields[f] + (size_t)(h->zlo() - H + HALO) * pf, static_cast<const char*>(recv_lo) + f * nb, nb, cudaMemcpyDeviceToDevice, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(fields[f] + (size_t)(h->zhi() + HALO) * pf, static_cast<const char*>(recv_hi) + f * nb, nb, cudaMemcpyDeviceToDevice, h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "lb_slab_unpack_phi");
  }
  h->phi_ghost_ok = true;
  return LB_OK;
}

int lb_slab_part_get(lb_handle h, double* d_sums) {
  int rc = slab_ready(h, 1, "lb_slab_part_get");
  if (rc) return rc;
  if (h->np == 0 || h->part_stage == 0) return fail(h, LB_ESTATE, "lb_slab_part_get: no particle sums are pending");
  if (!d_sums || !is_device_ptr(d_sums)) return fail(h, LB_EINVAL, "lb_slab_part_get: a device buffer of 6 doubles per particle");
  DeviceGuard guard(h->device);
  cudaError_t e = cudaMemcpyAsync(d_sums, h->pred, (size_t)h->np * 6 * sizeof(double), cudaMemcpyDeviceToDevice, h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "lb_slab_part_get");
  return LB_OK;
}

int lb_slab_part_put(lb_handle h, const double* d_sums) {
  int rc = slab_ready(h, 1, "lb_slab_part_put");
  if (rc) return rc;
  if (h->np == 0 || h->part_stage == 0) return fail(h, LB_ESTATE, "lb_slab_part_put: no particle sums are pending");
  if (!d_sums || !is_device_ptr(d_sums)) return fail(h, LB_EINVAL, "lb_slab_part_put: a device buffer of 6 doubles per particle");
  DeviceGuard guard(h->device);
  cudaError_t e = cudaMemcpyAsync(h->ptot, d_sums, (size_t)h->np * 6 * sizeof(double), cudaMemcpyDeviceToDevice, h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "lb_slab_part_put");
  if (h->part_stage == 1) {          // force and torque on every particle: pair forces, the move, this slab's node changes
    particles_move(h);
    h->part_stage = 2;
  } else {                           // impulses of the node changes; the stored values are final: pack
    particles_apply(h);
    slab_copy_populations(h, next_buf(h), slab_send_blocks(h, h->mode()), h->pend_send[0], h->pend_send[1], true);
    h->part_stage = 0;
  }
  return check_launch(h, "lb_slab_part_put");
}

long long lb_launch_count(lb_handle h) { return h ? h->launches : 0; }
size_t lb_device_bytes(lb_handle h) { return h ? h->bytes : 0; }
const char* lb_last_error(lb_handle h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int lb_set_tuning(lb_handle h, const char* key, int value) {
  if (!h || !key) return LB_EINVAL;
  const std::string k(key);
  if (k == "forward") h->forward = value < 0 || value > 2 ? 1 : value;
  else if (k == "zc") h->tune_zc = value;
  else if (k == "graph") h->graph = value < 0 ? -1 : (value ? 1 : 0);
  else return fail(h, LB_EINVAL, "unknown tuning key: " + k);
  return LB_OK;
}

int lb_set_profiling(lb_handle h, int on) {
  if (!h) return LB_EINVAL;
  h->profiling = on > 0 ? on : 0;
  return LB_OK;
}

int lb_last_step_ms(lb_handle h, int which, float* ms) {
  if (!h || !ms || which < 0 || which > 2) return fail(h, LB_EINVAL, "bad argument");
  if (!h->ev_step[1]) return fail(h, LB_ESTATE, "no lb_step recorded yet");
  DeviceGuard guard(h->device);
  cudaError_t e = cudaEventSynchronize(h->ev_step[1]);
  if (e != cudaSuccess) return cuda_fail(h, e, "event sync");
  if (which == 0) {
    e = cudaEventElapsedTime(ms, h->ev_step[0], h->ev_step[1]);
    if (e != cudaSuccess) return cuda_fail(h, e, "event elapsed");
    return LB_OK;
  }
  if (h->ev_steps == 0) return fail(h, LB_ESTATE, "profiling was off during the last lb_step");
  float total = 0.f;
  for (int t = 0; t < h->ev_steps; ++t) {
    float v = 0.f;
    if (which == 1) {
      e = cudaEventElapsedTime(&v, h->ev_k[4 * t + 1], h->ev_k[4 * t + 2]);
    } else {
      float v2 = 0.f;
      e = cudaEventElapsedTime(&v, h->ev_k[4 * t + 0], h->ev_k[4 * t + 1]);
      if (e == cudaSuccess) e = cudaEventElapsedTime(&v2, h->ev_k[4 * t + 2], h->ev_k[4 * t + 3]);
      v += v2;
    }
    if (e != cudaSuccess) return cuda_fail(h, e, "event elapsed");
    total += v;
  }
  *ms = total / (float)h->ev_steps;   // mean per sampled step
  return LB_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------ state check without allocation
// lb_check_state_static (include/lb.h): the sums of lb_check_state for callers that may not
// allocate (CUDA graph capture, tight loops, harnesses that forbid cudaMalloc).  k_check_static is
// a variant of k_check whose scratch memory is the file-scope array below instead of a buffer the
// handle allocates: one triple of partial sums per block of SC_SITES_PER_BLOCK sites, summed by
// the last block to arrive in a fixed order (the result does not depend on the order in which the
// blocks ran, unlike k_check's atomic adds).
constexpr int SC_SITES_PER_BLOCK = 8192;   // 256 threads x 32 sites
constexpr int SC_MAX_BLOCKS = 32768;
constexpr long long SC_MAX_SITES = (long long)SC_SITES_PER_BLOCK * SC_MAX_BLOCKS;   // 2^28 sites (640^3 fits)
constexpr int SC_COUNTER_AT = 3 * SC_MAX_BLOCKS;   // the arrival counter sits behind the partial sums

// 768 KiB of partial sums + 256 B for the arrival counter.  Every GPU that loads the library holds
// this array until the process exits.  In host code the name is a host-side stand-in, NOT a
// device address: static_scratch() below asks the runtime for the address, once per device.
static __device__ __align__(256) double g_static_scratch[3 * SC_MAX_BLOCKS + 32];

namespace {

template <int MODE, bool TWO, bool HAS_SOLID>
__global__ void __launch_bounds__(256) k_check_static(const IoParams p, double* scratch, double* out) {
  const Box& b = p.box;
  double sr = 0.0, sb = 0.0, bad = 0.0;
  const long long base = p.s0 + (long long)blockIdx.x * SC_SITES_PER_BLOCK;
  const long long end = base + SC_SITES_PER_BLOCK < p.s1 ? base + SC_SITES_PER_BLOCK : p.s1;
  for (long long s = base + threadIdx.x; s < end; s += 256) {
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
  __shared__ double red[3][8];
  __shared__ bool last;
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  auto block_sum3 = [&](double& a0, double& a1, double& a2) {   // fixed order: the same bits every time
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a0 += __shfl_down_sync(0xffffffffu, a0, o);
      a1 += __shfl_down_sync(0xffffffffu, a1, o);
      a2 += __shfl_down_sync(0xffffffffu, a2, o);
    }
    if (lane == 0) { red[0][wp] = a0; red[1][wp] = a1; red[2][wp] = a2; }
    __syncthreads();
    double v = 0.0;
    if (threadIdx.x < 3)
      for (int i = 0; i < 8; ++i) v += red[threadIdx.x][i];
    return v;   // threads 0..2 hold the three sums
  };
  const double part = block_sum3(sr, sb, bad);
  if (threadIdx.x < 3) {
    scratch[3 * (size_t)blockIdx.x + threadIdx.x] = part;
    __threadfence();                 // the partial sums are visible before the ticket is drawn
  }
  __syncthreads();
  unsigned* counter = reinterpret_cast<unsigned*>(scratch + SC_COUNTER_AT);
  if (threadIdx.x == 0) last = atomicAdd(counter, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!last) return;
  __threadfence();
  double a0 = 0.0, a1 = 0.0, a2 = 0.0;
  for (unsigned i = threadIdx.x; i < gridDim.x; i += 256) {
    a0 += __ldcg(scratch + 3 * (size_t)i);
    a1 += __ldcg(scratch + 3 * (size_t)i + 1);
    a2 += __ldcg(scratch + 3 * (size_t)i + 2);
  }
  __syncthreads();                   // red[] is reused
  const double total = block_sum3(a0, a1, a2);
  if (threadIdx.x < 3) out[threadIdx.x] = total;
  if (threadIdx.x == 0) *counter = 0u;   // the next call on this stream finds the counter at zero
}

// Device address of g_static_scratch on the handle's device (which the caller has made current).
// Asked once per device; no allocation.
int static_scratch(lb_handle h, double** ptr) {
  static double* addr[MAX_DEVICES] = {};
  static std::mutex mu;
  int cur = -1;
  if (cudaGetDevice(&cur) != cudaSuccess || cur != h->device || cur < 0 || cur >= MAX_DEVICES) {
    cudaGetLastError();
    return fail(h, LB_ECUDA, "lb_check_state_static: the handle's device could not be made current");
  }
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[cur]) {
    void* q = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&q, g_static_scratch);
    if (e != cudaSuccess || !q) return cuda_fail(h, e, "lb_check_state_static: address of the static scratch array");
    addr[cur] = static_cast<double*>(q);
  }
  *ptr = addr[cur];
  return LB_OK;
}

template <int MODE, bool TWO>
void launch_check_static_t(lb_handle h, const IoParams& p, int nb, double* scratch, double* out) {
  if (h->has_solid) k_check_static<MODE, TWO, true><<<nb, 256, 0, h->stream>>>(p, scratch, out);
  else k_check_static<MODE, TWO, false><<<nb, 256, 0, h->stream>>>(p, scratch, out);
}

}  // namespace

extern "C" int lb_check_state_static(lb_handle h, double* d_out) {
  if (!h) return LB_EINVAL;
  if (!d_out) return fail(h, LB_EINVAL, "lb_check_state_static: d_out is NULL");
  const long long sites = h->Sx;   // the handle's own sites (known since lb_create)
  if (sites > SC_MAX_SITES) {
    char msg[200];
    snprintf(msg, sizeof(msg), "lb_check_state_static: %lld sites exceed the static scratch array's maximum of %lld (use lb_check_state)",
             sites, SC_MAX_SITES);
    return fail(h, LB_EINVAL, msg);
  }
  if (!h->inited) return fail(h, LB_ESTATE, "lb_check_state_static before lb_init");
  DeviceGuard guard(h->device);
  if (!is_device_ptr(d_out)) return fail(h, LB_EINVAL, "lb_check_state_static: d_out must be a device pointer (3 doubles)");
  const IoParams p = make_io_params(h);
  double* scratch = nullptr;
  if (int rc = static_scratch(h, &scratch)) return rc;
  // the array keeps what the last call left: the arrival counter must start at zero
  cudaError_t e = cudaMemsetAsync(scratch + SC_COUNTER_AT, 0, 256, h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "lb_check_state_static: counter reset");
  const int nb = (int)((sites + SC_SITES_PER_BLOCK - 1) / SC_SITES_PER_BLOCK);
  const int mode = h->mode();
  if (h->two) {
    if (mode == MODE_AB) launch_check_static_t<MODE_AB, true>(h, p, nb, scratch, d_out);
    else if (mode == MODE_AA_EVEN) launch_check_static_t<MODE_AA_EVEN, true>(h, p, nb, scratch, d_out);
    else launch_check_static_t<MODE_AA_ODD, true>(h, p, nb, scratch, d_out);
  } else {
    if (mode == MODE_AB) launch_check_static_t<MODE_AB, false>(h, p, nb, scratch, d_out);
    else if (mode == MODE_AA_EVEN) launch_check_static_t<MODE_AA_EVEN, false>(h, p, nb, scratch, d_out);
    else launch_check_static_t<MODE_AA_ODD, false>(h, p, nb, scratch, d_out);
  }
  h->launches++;
  return check_launch(h, "lb_check_state_static");
}
