/* lb.h -- C-ABI boundary of the B200-native two-component colour-gradient D3Q19 lattice
 * Boltzmann hot path (arxiv 2005.12764, "Towards Exascale Design of Soft Mesoscale Materials").
 *
 * Citations are to /root/reference/PAPER.md (line, equation).  Where the paper is silent the
 * reading is one of G1-G24 in DESIGN.md.
 *
 * The problem, as the paper states it: two sets of populations f^r_i, f^b_i on a D3Q19 lattice
 * advance by collide-and-stream (Eq. 1; Eq. 5-6)
 * with a common velocity and a mixture relaxation rate (Eq. 7-8), under a
 * source term S_i carrying body and near-contact forces (Eq. 11),
 * between bounce-back walls with one periodic axis.
 *
 * Conventions for every call
 *   layout      scalar fields are [z][y][x], x fastest: index x + nx*(y + ny*z).  u is three such
 *               planes [3][z][y][x].  Populations are [19][z][y][x] in the velocity order below.
 *   pointers    every array argument may be a HOST or a DEVICE pointer (detected with
 *               cudaPointerGetAttributes); host arrays are staged through a temporary device
 *               buffer.  The caller owns every array it passes; the handle owns all device state.
 *   stream      all work is enqueued on the handle's stream (lb_set_stream; default stream 0).
 *               lb_step is asynchronous.  Calls that write to host memory synchronise the
 *               stream before returning.
 *   time        after lb_init the state is t = 0, after lb_step(n) it is t = n.  "The state at t"
 *               is the set of pre-collision populations f^k_i(x, t) (those that have arrived at x).
 *   errors      0 on success, negative LB_E* otherwise; text via lb_last_error.  Nothing throws,
 *               nothing aborts.  There is no CPU fallback: without a CUDA device every call that
 *               touches the device returns LB_ECUDA.
 *
 * Velocity order (free in the paper, which numbers i = 1..19):
 *   0:(0,0,0) 1:(+1,0,0) 2:(-1,0,0) 3:(0,+1,0) 4:(0,-1,0) 5:(0,0,+1) 6:(0,0,-1)
 *   7:(+1,+1,0) 8:(-1,-1,0) 9:(+1,-1,0) 10:(-1,+1,0) 11:(+1,0,+1) 12:(-1,0,-1)
 *   13:(+1,0,-1) 14:(-1,0,+1) 15:(0,+1,+1) 16:(0,-1,-1) 17:(0,+1,-1) 18:(0,-1,+1)
 */
#ifndef LB_B200_H
#define LB_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LB_OK 0
#define LB_EINVAL (-1) /* bad size, NULL where not allowed, tau <= 0.5, nx not a multiple of 4 */
#define LB_ENOMEM (-2) /* device allocation failed */
#define LB_ECUDA (-3)  /* a CUDA call failed (or there is no device) */
#define LB_ESTATE (-4) /* call out of order: step before init, set_geometry after init, ... */

/* tau_k: relaxation times, omega_k = 1/tau_k, nu_k = (tau_k - 1/2)/3 (Eq. 4).
 * A: strength of the colour-gradient surface-tension perturbation (sigma ~ 4/9 A tau).
 * beta: Latva-Kokko recolouring strength.  A_nc: near-contact strength, the constant "A" of
 * A_h[h] in Eq. 11; 0 switches the near-contact force off. */
typedef struct {
  float tau_r, tau_b, A, beta, A_nc;
} lb_params;

typedef struct lb_handle_s* lb_handle;

/* Device-memory hooks.  PyTorch is the allocator in production: the Python binding passes
 * wrappers of torch's CUDA caching allocator.  alloc returns a device pointer (on the device
 * that is current when it is called) or NULL.  The pair is a process-wide default that every
 * handle captures at lb_create and keeps for its whole life; NULL, NULL restores cudaMalloc /
 * cudaFree for handles created afterwards.  A handle lives on the device that was current at
 * lb_create; every call makes that device current for its duration. */
typedef void* (*lb_alloc_fn)(size_t bytes, void* user);
typedef void (*lb_free_fn)(void* ptr, void* user);
int lb_set_allocator(lb_alloc_fn alloc, lb_free_fn free_fn, void* user);

/* Create a simulation on an nx x ny x nz box (all axes periodic in topology; walls are solid
 * sites, see lb_set_geometry).  Requires nx % 4 == 0 and every extent >= 4; tau_k > 0.5.
 * Allocates nothing large: population buffers are allocated by lb_init. */
int lb_create(int nx, int ny, int nz, const lb_params* p, lb_handle* out);

/* Frees all device state.  lb_destroy(NULL) is a no-op. */
void lb_destroy(lb_handle h);

/* CUDA stream (a cudaStream_t passed as void*) that all later work of this handle uses. */
int lb_set_stream(lb_handle h, void* cuda_stream);

/* Solid mask, S = nx*ny*nz bytes: 0 = fluid, 1 = wall at rest, 2, 3 and 4 = wall groups: walls
 * moving with the velocities of lb_set_wall_velocity or the open boundaries of lb_set_wall_type
 * (any other value counts as 1); NULL = all fluid.  Stored
 * bit-packed.  Solid sites hold no populations; links into them bounce back half-way
 * (G21).  Must precede lb_init. */
int lb_set_geometry(lb_handle h, const uint8_t* solid_mask);

/* Velocity u_w of the walls of group 2, 3 or 4 ("solid walls with opposite speeds +-U", PAPER.md:341,
 * :367; G28): a population reflected at such a wall along link i loses 6 w_i rho^k (c_i . u_w). */
int lb_set_wall_velocity(lb_handle h, int group, float ux, float uy, float uz);

/* What the wall group 2, 3 or 4 is (G31; the two kinds of inlet and the outlet of the
 * flow focuser, whose boundary rules the paper does not give).  type 0 (default) = moving
 * wall.  1 = velocity inlet: the moving-wall rule with u_w = the inflow velocity
 * (lb_set_wall_velocity) and the prescribed densities rho_r, rho_b of the incoming fluid in place
 * of the site's own.  2 = reservoir (pressure boundary, both densities prescribed) by
 * anti-bounce-back: f^k_opp(i)(x, t+1) = -f^k*_i(x, t) + 2 w_i rho^k_out [1 + 4.5 (c_i.u)^2 -
 * 1.5 u.u], u = the velocity that entered f^eq at x in this step.  3 = pressure outlet: the same
 * with rho^k_out = (rho_r + rho_b) rho^k(x) / rho(x), so that the composition of the outgoing
 * fluid passes.  One component: rho_r is the density (type 3: rho_r + rho_b).  May be called at
 * any time; acts from the next lb_step.  LB_EINVAL: group not 2..4, type not 0..3, a negative or
 * NaN density. */
int lb_set_wall_type(lb_handle h, int group, int type, float rho_r, float rho_b);

/* Uniform acceleration g: body force F = rho g enters through the source term. */
int lb_set_body_force(lb_handle h, float gx, float gy, float gz);

/* Which two-component model lb_step advances.  0 (default) = colour gradient + Latva-Kokko
 * recolouring + near contact (north_star; A, beta, A_nc of lb_params).  1 = the paper's section
 * 3.1 as printed: each component relaxes to f^eq(rho^k, u) (Eq. 5-6) and
 * receives the exact-difference source (Eq. 9) of the Shan-Chen force
 * F^r = -G_C rho^r sum_i w_i rho^b(x + c_i) c_i, and r, b swapped (Eq. 10; positive
 * G_C repels); A, beta, A_nc do not act.  Must precede lb_init; needs rho_b. */
int lb_set_model(lb_handle h, int model, float G_C);

/* How the force enters the collision.  0 (default) = Guo forcing (north_star): source term
 * (1 - omega/2) w_i [3 (c_i - u) + 9 (c_i.u) c_i].F with u = (m + F/2)/rho.  1 = exact-difference
 * forcing, the paper's own Eq. 9: S_i = f^eq_i(rho, u + F/rho) - f^eq_i(rho, u)
 * with the bare u = m/rho.  lb_get_macros returns (m + F/2)/rho in both cases. */
int lb_set_forcing(lb_handle h, int mode);

/* Near-contact force acts where |phi| < phi_c (default 0.9). */
int lb_set_nc_cutoff(lb_handle h, float phi_c);

/* Colour-symmetric near-contact probe (G29; Fig. 5, is symmetric in the
 * two fluids).  on = 0 (default): the probe marches along -G/|G| and finds h- = the first k >= 2
 * with phi(probe) >= phi(x): F_nc = A_h(h-) G / 2 (two red interfaces across a blue film).
 * on = 1: its image under r <-> b is applied as well (along +G/|G|, h+ = first k >= 2 with
 * phi(probe) <= phi(x)): F_nc = (A_h(h-) - A_h(h+)) G / 2.  May be changed between steps. */
int lb_set_nc_symmetric(lb_handle h, int on);

/* Wetting (G30; the paper has no wetting model).  on = 0 (default): a solid neighbour
 * contributes the centre value phi(x) to the colour-gradient stencil (neutral wall).  on = 1: it
 * contributes the prescribed phi_wall in [-1, 1], one value for all walls (static contact angle
 * cos(theta) ~= phi_wall).  Colour-gradient model only.  May be changed between steps. */
int lb_set_wall_phi(lb_handle h, int on, float phi_wall);

/* Storage of the populations.  0 = A/B double buffer (default), 1 = AA-pattern, one buffer
 * updated in place.  Must precede lb_init. */
int lb_set_storage(lb_handle h, int mode);

/* Initial state (t = 0): f^k_i = w_i rho_k [1 + 3 c.u + 4.5 (c.u)^2 - 1.5 u.u] with the common u
 * (Eq. 2, per component as in Eq. 5-6).  rho_b == NULL selects
 * the single-component BGK mode (config C2).  Input on solid sites is ignored.  Allocates the
 * population buffers: 2 (A/B) or 1 (AA) x 38 (or 19) x S floats, plus the padded phi array and
 * 2.125 x S floats of forwarded moments.  Requires S = nx*ny*nz < 2^29. */
int lb_init(lb_handle h, const float* rho_r, const float* rho_b, const float* u);

/* Advance nsteps time steps: per step the fused pull-stream + collide kernel (Eq. 1-2, 5-8, 11),
 * which also forwards the moments of the next state, and the phase-field kernel that turns them
 * into phi = (rho_r - rho_b)/rho (Eq. 3).  Asynchronous, except that every 1000
 * steps it runs lb_check_state and returns LB_ESTATE if the state is no longer finite. */
int lb_step(lb_handle h, int nsteps);

/* State check (G23; the paper names fault tolerance as an exascale issue):
 * sums rho_r and rho_b (Eq. 3) over the handle's own fluid sites on the device, in
 * double precision, and looks for NaN / Inf populations.  Returns LB_ESTATE (text: how many sites, after
 * how many steps) if the state is not finite, LB_OK otherwise; mass_r, mass_b (HOST pointers, may
 * be NULL) receive the sums (single component: mass_r is the mass, mass_b is 0).  Synchronises the
 * stream.  lb_step runs the same check by itself every 1000 steps since the last check and then
 * returns LB_ESTATE instead of stepping on: that is the one place where lb_step synchronises. */
int lb_check_state(lb_handle h, double* mass_r, double* mass_b);

/* The same sums for callers that may not allocate or synchronise (code under CUDA graph capture,
 * tight loops, harnesses that forbid cudaMalloc): calls no cudaMalloc / cudaFree and no allocator
 * hook, never synchronises, and writes {sum rho_r, sum rho_b, number of fluid sites that hold a
 * NaN / Inf population} to d_out, a DEVICE pointer to 3 doubles owned by the caller, on the
 * handle's stream.  It does not judge the state: the caller reads d_out[2] (LB_ESTATE is never
 * returned for a non-finite state, and the 1000-step counter of lb_step is not reset).
 * Scratch memory is one array of 768 KiB + 256 B in the library's device image
 * (`static __device__`; every GPU that loads the library holds it until the process exits): one
 * triple of partial sums per block of 8192 sites, added up in a fixed order, so two calls on the
 * same state give the same bits (lb_check_state adds atomically and agrees to rounding).
 * Limit: at most 2^28 = 268,435,456 own sites (640^3 fits); a larger box returns LB_EINVAL with
 * a text that names the limit, before anything is launched.  d_out NULL or a host pointer:
 * LB_EINVAL.  All calls on one device share the array (handles included): calls that overlap on
 * the GPU (different streams without an ordering between them) race; calls ordered on one
 * stream, or by events, do not. */
int lb_check_state_static(lb_handle h, double* d_out);

/* rho_r, rho_b and the velocity u = (sum_i c_i f_i + F/2)/rho of the current state (Eq. 3,
 * PAPER.md:96, with the half-force shift of Guo forcing; G16).  Zeros on solid sites.  Any
 * output pointer may be NULL; rho_b is ignored in single-component mode.  Does not disturb
 * the state. */
int lb_get_macros(lb_handle h, float* rho_r, float* rho_b, float* u);

/* Debug / checkpoint accessors: the full pre-collision populations f^comp_i(x, t), comp 0 = red,
 * 1 = blue, 19*S floats.  Internally the state is stored as deviations;
 * these calls convert.  lb_set_populations must be called for both components (red first)
 * before the next lb_step; values on solid sites are ignored. */
int lb_get_populations(lb_handle h, int comp, float* f);
int lb_set_populations(lb_handle h, int comp, const float* f);

/* phi = (rho_r - rho_b)/(rho_r + rho_b) of the current state, S floats (0 on solid sites). */
int lb_get_phi(lb_handle h, float* phi);

/* ---- z-slab decomposition over several handles / GPUs -----------------
 * The paper splits the fluid box equally over the ranks, "according to a either 1D, or 2D or 3D
 * domain decomposition"; the collision is local ("zero communication",
 * PAPER.md:161) and streaming reaches first neighbours only.  Here: slabs along z
 * (x stays contiguous).  A slab handle owns the planes [z0, z0 + nz) of a box of nz_global planes
 * that is periodic over nz_global; nz is the nz of lb_create.  Internally it holds one ghost
 * plane below and one above its own planes.  What crosses a z face per step and per direction of
 * travel: the 5 populations per component with c_z = +1 (or -1), i.e. 5 * nx * ny * 8 bytes (4 for
 * one component), and H planes of the padded phase field, H = 4 with the near-contact force (its
 * probe reaches 4 sites), else 1: H * (nx + 8) * (ny + 8) * 4 bytes (twice that in the Shan-Chen
 * model, whose fields are rho_r and rho_b).  The library packs and unpacks these messages; MOVING
 * them is the caller's job (ncclSend / ncclRecv through torch.distributed in
 * paper_2005_12764_b200/slab.py, peer copies, or plain copies between two handles of one process),
 * so the boundary carries no communicator type.  Message buffers are DEVICE memory, 16-byte
 * aligned, owned by the caller.  "lo" = the face towards smaller z (the rank below), "hi" = above.
 *
 * lb_set_slab(h, z0, nz_global): declares the handle a slab; before lb_set_geometry and lb_init;
 * nz >= 8; nz_global <= 0 undoes it.  For a slab, lb_set_geometry takes (nz + 2) * ny * nx bytes:
 * the planes z0 - 1 .. z0 + nz of the global mask (periodic), i.e. including the two ghost planes;
 * every other array argument (lb_init, lb_get_macros, ...) holds the slab's own nz planes only.
 * lb_step returns LB_ESTATE for a slab; one time step is, in this order:
 *   lb_slab_begin(h, send_lo, send_hi)    fused stream-collide on the first and the last brick of
 *                                         the slab; packs the populations the neighbours need
 *   [caller: send_hi -> rank above's recv_lo, send_lo -> rank below's recv_hi; may overlap with:]
 *   lb_slab_interior(h)                   fused kernel on the bricks in between, and the phase
 *                                         field of the planes that do not wait for the halo
 *   lb_slab_end(h, recv_lo, recv_hi)      unpacks the received populations into the ghost planes
 *                                         (after an in-place odd step: into the own boundary
 *                                         planes), phase field of the H planes next to each face;
 *                                         the state is then t + 1 (runs the 1000-step state check
 *                                         like lb_step)
 *   lb_slab_pack_phi(h, send_lo, send_hi) the H phi planes next to each face
 *   [caller: exchange as above]
 *   lb_slab_unpack_phi(h, recv_lo, recv_hi)   into the z ghost planes of the padded phi array
 * After lb_init (and after lb_set_populations) the last three calls must run once before the first
 * lb_slab_begin or lb_get_macros (phi of the initial state is computed by lb_slab_pack_phi).
 * All calls are asynchronous on the handle's stream at the time of the call (lb_set_stream may
 * switch streams between phases; ordering across streams is the caller's, by events).  Errors:
 * LB_ESTATE for a call out of order or on a handle that is not a slab, LB_EINVAL for NULL,
 * misaligned or host message buffers.  One component: the phi calls do nothing. */
int lb_set_slab(lb_handle h, int z0, int nz_global);
int lb_slab_halo_bytes(lb_handle h, size_t* pop_bytes, size_t* phi_bytes);   /* per face and direction of travel; after lb_init */
int lb_slab_begin(lb_handle h, void* send_lo, void* send_hi);
int lb_slab_interior(lb_handle h);
int lb_slab_end(lb_handle h, const void* recv_lo, const void* recv_hi);
int lb_slab_pack_phi(lb_handle h, void* send_lo, void* send_hi);
int lb_slab_unpack_phi(lb_handle h, const void* recv_lo, const void* recv_hi);

/* Particles in a slab: "replicated data" ("each process stores the physical
 * variables of all particles ... a global reduction ... each process solves the equation of motion
 * for all particles").  Every slab handle is given ALL particles (lb_set_particles, positions in
 * the coordinates of the whole box) and keeps the same state as every other; per step two sums over
 * the slabs are the caller's (an all-reduce of 6 doubles per particle each):
 *   lb_slab_begin(h, send_lo, send_hi)   with particles: the fused kernel on EVERY brick, the link
 *                                        rule (G33) on the slab's own sites and its share of the link
 *                                        sums; nothing is packed yet (the particles still rewrite
 *                                        stored values of the boundary planes), so there is no overlap
 *   lb_slab_part_get(h, d_sums)          the slab's share [np][6] = (F, T) -> caller's DEVICE buffer
 *   [caller: sum over the slabs]
 *   lb_slab_part_put(h, d_sums)          the totals; pair forces, leapfrog step, node changes of the
 *                                        slab's own sites (G36), its share of their impulses
 *   lb_slab_part_get(h, d_sums)          that share [np][6] = (dU, dL)
 *   [caller: sum over the slabs]
 *   lb_slab_part_put(h, d_sums)          the totals go to the particles; the population messages
 *                                        given to lb_slab_begin are packed now (send_lo, send_hi
 *                                        must stay valid until this call returns)
 *   [caller: exchange the population messages]   lb_slab_interior, lb_slab_end as above
 *   (lb_slab_end also forms phi again around the particles)
 * and the phi messages carry, behind the phi planes, rho_r and rho_b of the boundary plane (G36 fills
 * a node that leaves a particle at the mean densities of its neighbours, which may lie in a ghost
 * plane): lb_slab_halo_bytes counts them, and with one component the phi calls then carry only those.
 * The result equals the undivided box up to the order of the two sums.  LB_ESTATE: out of order. */
int lb_slab_part_get(lb_handle h, double* d_sums);
int lb_slab_part_put(lb_handle h, const double* d_sums);

/* ---- rigid spherical particles (the paper's section 6) --------------------
 * "colloidal particles are represented as rigid spheres of radius R, moving under the effect of a
 * total force F_p and torque T_p ... dr_p/dt = u_p, m_p du_p/dt = F_p, I_p dw_p/dt = T_p (Eq. 15) ...
 * The force on each particle takes into account the interactions with the fluid and the
 * inter-particle forces, including the lubrication term.  Hence, the equations of motion are solved
 * by a leapfrog approach, using quaternion algebra for the rotational component".
 * The paper gives no coupling rule; G32-G37 state the ones built: a lattice node within R of
 * the centre is solid; a link from a fluid node into it is reflected half-way at a wall that moves
 * with u_p + w_p x (x_b - r_p) (both components, as lb_set_wall_velocity does for plane walls) and
 * hands its momentum change to the particle; leapfrog and quaternion update per step; nodes that
 * leave a particle are filled with the equilibrium of their neighbours' mean densities, nodes that
 * enter it give their momentum to it, so that the momentum of fluid + particles is conserved
 * exactly; between particles a repulsion K (h_c - h)^(3/2) for gaps h < h_c and, if switched on,
 * the normal lubrication force 6 pi mu R_eff^2 (1/h - 1/h_c) against the approach.
 * lb_particle: centre r, velocity u, angular velocity w, orientation quaternion q = (w, x, y, z),
 * radius R, mass (I_p = 2/5 m R^2); doubles, lattice units.
 * lb_set_particles(h, n, p): HOST array of n particles; before lb_init (n = 0: none).  Needs A/B
 * storage, the colour-gradient model or one component, no slab (lb_init returns LB_ESTATE
 * otherwise); the "replicated data" scheme of PAPER.md:312-316 for several ranks is not built.
 * The particle nodes hold no fluid: lb_init ignores its input there and lb_get_macros returns zeros.
 * lb_set_particle_options: mobile = 0 holds the particles in place (they still exchange momentum with
 * the fluid); K, h_c, lubrication: the pair force (h_c <= 0: none).  lb_set_particle_force: a constant
 * external force and torque on particle i (either may be NULL); before lb_init.
 * lb_get_particles(h, state, force): current states and, per particle, 9 doubles: force and torque
 * from the fluid links of the last step, force from the other particles (HOST arrays, either may be
 * NULL); synchronises; LB_ESTATE if a particle moved so fast that more than 384 of its nodes changed
 * in one step.  With particles, phi is recomputed by the full sweep every step (the node map
 * changes under the forwarded moments). */
typedef struct {
  double r[3], u[3], w[3], q[4], R, mass;
} lb_particle;
int lb_set_particles(lb_handle h, int n, const lb_particle* p);
int lb_set_particle_options(lb_handle h, int mobile, double K, double h_c, int lubrication);
int lb_set_particle_force(lb_handle h, int i, const double* F, const double* T);
int lb_get_particles(lb_handle h, lb_particle* state, double* force);

/* Tuning of lb_step.  key = "forward": 1 (default) = the fused kernel forwards the moments of the
 * next state and a light kernel turns them into phi, except in
 * boxes so small that a CTA holds a single plane, where the full sweep is faster; 2 = the same
 * without that exception; 0 = a full phase-field sweep over the populations before every step
 * (same phi to ~1e-8).  "zc": z planes
 * per CTA, 0 = automatic.  "graph": lb_step replays a CUDA graph of 16 time steps where it can (no
 * profiling, not the first two steps, not while the caller's stream is capturing):
 * -1 (default) = for boxes of at most 2^21 sites, whose step is bounded by launch latency, 0 = never,
 * 1 = for every box.  The graph is captured on a stream of the handle's own and launched into the
 * handle's stream; it is rebuilt when any parameter, buffer or the storage parity changes; results
 * are bit-identical to plain launches.  Returns LB_EINVAL for an unknown key. */
int lb_set_tuning(lb_handle h, const char* key, int value);

/* Number of kernel launches this handle has made so far (for the harness' gpu_launches). */
long long lb_launch_count(lb_handle h);

/* Bytes of device memory the handle currently owns. */
size_t lb_device_bytes(lb_handle h);

/* Last error text of this handle (or of the failed lb_create when h == NULL). */
const char* lb_last_error(lb_handle h);

/* Timing hooks, on the handle's stream.  lb_last_step_ms(h, 0, &ms): milliseconds of the whole LAST
 * lb_step call (an event pair around all its launches; synchronises on the end event).
 * lb_set_profiling(h, n), n > 0: in later lb_step calls every n-th step is bracketed kernel by
 * kernel; lb_last_step_ms then returns the MEAN per sampled step of which = 1: the fused
 * stream-collide launch (k_fused / k_single), which = 2: the phase-field launches (k_phase_fwd,
 * or k_phase).  n = 0 switches the sampling off (the events cost ~3 % when taken every step). */
int lb_set_profiling(lb_handle h, int on);
int lb_last_step_ms(lb_handle h, int which, float* ms);

#ifdef __cplusplus
}
#endif
#endif /* LB_B200_H */
