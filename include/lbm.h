/*
 * lbm.h -- C ABI of the B200-native particle-resolved thermal lattice Boltzmann hot path.
 *
 * Method: Xu & Li, "Particle-resolved thermal lattice Boltzmann simulation using OpenACC on
 * multi-GPUs" (arXiv 2308.16597).  Citations below are PAPER.md:<line> (the paper text) and
 * SURVEY.md section 8 (the scope contract: rows a1..a6, boundary (b), readings (c)).
 *
 * One handle = one simulation on one GPU.  All lattice state lives in ONE caller-supplied
 * device workspace (PyTorch allocates it; the library never calls cudaMalloc inside lbm_step).
 * Every array argument below is a HOST pointer unless it says "device".  Output buffers are
 * caller-owned and caller-sized.  No exception crosses the boundary: every function that can
 * fail returns an int (0 = LBM_OK, negative = error) and lbm_last_error() gives the text.
 *
 * Lattice conventions (SURVEY.md 8(c) "Lattice"; the paper does not print its numbering):
 *   nodes (i,j), 0<=i<nx, 0<=j<ny, host arrays dense with x fastest: idx = j*nx + i
 *   e0=(0,0) e1=(1,0) e2=(0,1) e3=(-1,0) e4=(0,-1) e5=(1,1) e6=(-1,1) e7=(-1,-1) e8=(1,-1)
 *   D2Q5 (temperature) uses e0..e4.  Cavity walls lie half a spacing outside the outermost
 *   nodes.  +y is up; gravity pulls particles along -y; hot fluid rises (Eq. 1b).
 *   Everything is in lattice units, fp64.
 */
#ifndef LBM_B200_H
#define LBM_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LBM_OK            0
#define LBM_E_ARG        (-1)  /* bad argument (NULL, non-positive size, overlap on insert ...)  */
#define LBM_E_STATE      (-2)  /* call not legal in the handle's current state                   */
#define LBM_E_CAPACITY   (-3)  /* a fixed-capacity array (particles, links, cells, newborn) full */
#define LBM_E_CUDA       (-4)  /* a CUDA runtime call failed; lbm_last_error() has the string    */
#define LBM_E_NONFINITE  (-5)  /* a particle state became NaN/Inf                                */

typedef struct lbm lbm_t;

/* Problem statement of the paper: closed cavity, Boussinesq fluid (Eqs. 1-6),
 * circular particles with repulsion (Eq. 15). */
typedef struct {
  double nu, kappa;            /* kinematic viscosity, thermal diffusivity (kappa = nu/Pr)        */
  double rho0, T0;             /* reference density, reference temperature (Eq. 1b)              */
  double g;                    /* gravity magnitude; acts along -y on particles (Eq. 15's C too)  */
  double gbeta;                /* g*beta_T: fluid buoyancy acceleration = +gbeta*(T-T0) along +y  */
  double body_ax, body_ay;     /* extra uniform body acceleration (Poiseuille check); default 0    */
  int    periodic_x;           /* 0 = closed cavity (all configs); 1 = x-periodic (closed-form checks) */
  int    wall_T_type[4];       /* W,E,S,N: 0 adiabatic, 1 Dirichlet                              */
  double wall_T[4];            /* W,E,S,N wall temperature (Dirichlet only)                      */
  double rep_s, rep_eps;       /* Eq. (15): threshold distance s, stiffness eps_w                */
  int    rep_power;            /* Eq. (15) exponent: 2 = paper, 1 = linear (BASELINE configs)     */
  int    max_particles;        /* capacity of the particle arrays                                */
  int    max_links_per_particle; /* capacity of one particle's segment of the fixed index array
                                    (paper: 12N-12)                                */
} lbm_params;

/* Fills *p with: nu=0.02 kappa=0.02/0.7 rho0=1 T0=0 g=0 gbeta=0 body=0 periodic_x=0
 * walls adiabatic, rep_s=2 rep_eps=1e-3 rep_power=1 max_particles=0 max_links_per_particle=0. */
void lbm_params_default(lbm_params* p);

/* Bytes of device workspace lbm_create needs for this lattice and these capacities
 * (two copies of the 9+5 populations, flag and owner maps, particle/link/cell arrays).
 * Returns 0 on bad arguments. */
size_t lbm_workspace_bytes(int nx, int ny, const lbm_params* p);

/* Creates a simulation.  dev_workspace: DEVICE pointer, >= lbm_workspace_bytes(), 256-byte
 * aligned, owned by the caller and kept alive until lbm_destroy.  cuda_stream: a cudaStream_t
 * (as void*; NULL = default stream) on which every kernel and copy of this handle is issued.
 * Initial state (SURVEY 8(c) "Initial state"): f = f_eq(rho0, 0), g = g_eq(T0, 0), no particles.
 * Errors: LBM_E_ARG (sizes, nu/kappa out of range: need nu>0, 0<kappa<0.144, nx,ny>=4),
 * LBM_E_CAPACITY (workspace too small), LBM_E_CUDA. */
int lbm_create(int nx, int ny, const lbm_params* p, void* dev_workspace, size_t bytes,
               void* cuda_stream, lbm_t** out);

/* T_host: nx*ny doubles.  Sets g = g_eq(T, u=0) on every node (Eq. 17's equilibrium with u=0).
 * Only before the first lbm_step (LBM_E_STATE afterwards). */
int lbm_set_temperature(lbm_t* h, const double* T_host);

/* Adds n circular particles (position, diameter, density, surface temperature).
 * x,y: centres; diam: diameters; rho_ratio: rho_p/rho_f; T_w: surface temperature (Eq. 11, 17).
 * ux,uy,omega: initial velocity (each may be NULL = at rest).  fixed: may be NULL; 1 = immobile
 * (skips Eqs. 7-8; the momentum-exchange force is still computed).
 * Errors: LBM_E_STATE after the first lbm_step (the paper never inserts particles mid-run);
 * LBM_E_CAPACITY beyond max_particles or if 12N-12 exceeds max_links_per_particle;
 * LBM_E_ARG if a disc is not strictly inside the cavity walls, overlaps another particle,
 * or (periodic_x=1) its search zone would cross the periodic seam. */
int lbm_add_particles(lbm_t* h, int n, const double* x, const double* y, const double* diam,
                      const double* rho_ratio, const double* T_w,
                      const double* ux, const double* uy, const double* omega,
                      const unsigned char* fixed);

/* Adds n ELLIPTICAL particles (PAPER.md:206-224 and Appendix A): full axes major x minor, the
 * major-labelled axis at angle theta (radians) to the x axis; everything else as in
 * lbm_add_particles, with which it may be mixed.  Equal axes give a circle through the circle
 * formulas.  Readings: the orientation is carried as a unit
 * vector advanced by a Cayley rotation (no cos / sin after set-up); the repulsion gap of a pair is
 * taken along the line of centres through the support functions, and the overlap test on insert
 * uses the same (conservative) gap; mass rho_p pi a b, inertia M (a^2 + b^2) / 4.
 * max_links_per_particle must admit 12N-12 with N = floor(largest full axis) + 4. */
int lbm_add_ellipses(lbm_t* h, int n, const double* x, const double* y, const double* major,
                     const double* minor, const double* theta, const double* rho_ratio,
                     const double* T_w, const double* ux, const double* uy, const double* omega,
                     const unsigned char* fixed);

/* Advances nsteps time steps (each = rows a1..a6 of SURVEY 8(a); order PAPER.md:347-353):
 * bounce-back (Eqs. 9-12) + momentum exchange (Eqs. 13-14) on the links of x_p(t) -> { particle
 * update (Eqs. 7, 8, 15) -> flag update -> refill (Eqs. 16-17, into a stash) -> link build for
 * x_p(t+1) } concurrently with { fused pull-stream-collide (Eqs. 5, 6) } -> refill commit.
 * Asynchronous kernels on the handle's stream, then ONE stream synchronisation at the end of the
 * call to read the device status word.  Errors: LBM_E_NONFINITE (a particle state is NaN/Inf,
 * checked once per call), LBM_E_CAPACITY (a link segment, cell or the newborn list overflowed;
 * the state is then undefined), LBM_E_CUDA. */
int lbm_step(lbm_t* h, int nsteps);

/* Optional set-up call: does everything a following lbm_step(h, nsteps) would do before its first
 * time step -- collides the initial state, builds the first links, plans the band and
 * captures, instantiates and uploads the CUDA graphs that call will replay -- without advancing
 * time, so that a short timed lbm_step (tens of steps) does not pay for graph instantiation (about
 * a millisecond per graph; like building an FFT plan before the loop).  The graphs are keyed by
 * the state's phase and the band plan, both unchanged by this call.  After it the set-up calls
 * (lbm_set_temperature, lbm_add_particles) return LBM_E_STATE, as after lbm_step. */
int lbm_prepare(lbm_t* h, int nsteps);

/* Environment variables read by lbm_create / lbm_add_particles (defaults in brackets):
 *   LBM_GRAPH [1], LBM_BAND [1] (0 / 1 / 2), LBM_BAND_STEPS [3] (2 / 3), LBM_STEPS_PER_PASS [3] (1 / 2 / 3), LBM_TMA [2] (0 / 1 / 2), LBM_PDL [1] (programmatic dependent launch along
 *   the kernels of a stream), LBM_CHAIN_CTAS_PER_SM [chosen from the sizes],
 *   LBM_DEBUG_SYNC [0] (debugging: synchronise after every direct launch, abort naming the first
 *   kernel that fails). */

/* on = 1 (default): the particle update chain of a step (integrator, flag update, refill, link
 * build for the next step) runs on the library's own high-priority stream concurrently with the
 * lattice kernel on the handle's stream, as a few persistent CTAs per SM (chosen from the lattice
 * and particle sizes; the environment variable LBM_CHAIN_CTAS_PER_SM, read by lbm_add_particles,
 * overrides it, 0 = one CTA per particle); forked and joined with events inside every step, so
 * the handle's stream still orders everything for the caller.  on = 0: one stream, strictly
 * sequential, one CTA per particle (same results bit for bit on every fluid node; used for
 * per-kernel timing and by the tests). */
int lbm_set_overlap(lbm_t* h, int on);

/* on = 1 (default; the environment variable LBM_GRAPH=0 turns the default off): lbm_step replays
 * whole periods of the step schedule as CUDA graphs -- 8 time steps per graph launch while that
 * many remain, then 2, an odd last step launched directly -- instead of issuing every kernel,
 * event record and stream wait from the host (the single-GPU analogue of the paper's async(n)
 * work queues).  The graph is captured on streams the library owns (the fork /
 * join onto the particle-chain stream becomes graph edges) and launched into the handle's stream,
 * so the caller's ordering is unchanged; the kernels, their arguments and their order are those of
 * on = 0, hence the same results bit for bit.  Event profiling (lbm_profile_enable) always uses
 * direct launches. */
int lbm_set_graph(lbm_t* h, int on);

/* Particle-free lattices (no particle added): time steps per pass over the populations.
 * on = 0: one (the fused one-step kernel, 224 B of HBM traffic per lattice update);
 * on = 1 or 2: two (shared-memory tile of 30 x 14 nodes with a one-node halo, about 137 B requested
 *   and 111 B of DRAM traffic per update);
 * on = 3 (default; the environment variable LBM_STEPS_PER_PASS = 1 / 2 / 3 sets the default): three
 *   (tile of 28 x 12 nodes with a two-node halo, the intermediate levels written back in place in
 *   shared memory; about 105 B requested per update), the last one or two steps of a call through
 *   the two-step and one-step kernels.
 * The arithmetic per node and step is the same in all three, so results are identical bit for bit. */
int lbm_set_two_step(lbm_t* h, int on);

/* Time steps per pass in a band (lbm_set_band): 3 (default; the environment variable
 * LBM_BAND_STEPS = 2 / 3 sets the default): periods of six steps, the band kernel
 * k_stream_collide_3step<BAND> advances the band's rows three steps per pass and hands its row next
 * to the seam, at the two intermediate times, to the rows outside through the spare row; 2: periods
 * of four steps with k_stream_collide_2step.  Identical results bit for bit.
 * Errors: LBM_E_ARG unless steps is 2 or 3. */
int lbm_set_band_steps(lbm_t* h, int steps);

/* Which kernel takes the three-steps-per-pass passes of a particle-free lattice.
 * on = 2 (default on closed cavities of at least 2^20 nodes; the environment variable LBM_TMA =
 *   0 / 1 / 2 sets the default): the persistent TMA-fed kernel k_stream_collide_3step_tma -- one CTA
 *   per SM walks the tiles, each tile's input image (tile + three-node halo, all 14 populations)
 *   arrives by two cp.async.bulk.tensor box copies into a three-deep shared-memory ring with an
 *   mbarrier per stage, two groups of 512 threads collide alternate tiles in place while the next
 *   ones load; inside a group each warp owns a tile row and hands over to its two neighbour rows
 *   through per-row mbarriers instead of group-wide barriers.
 *   Closed cavities only (periodic_x = 0), not for slab handles; needs cuTensorMapEncodeTiled.
 * on = 1: the same kernel with group-wide named barriers between the levels.
 * on = 0: k_stream_collide_3step (one CTA per tile, plain loads).
 * Same arithmetic per node and step: identical results bit for bit.
 * Errors: LBM_E_STATE if on != 0 and the handle has no tensor maps. */
int lbm_set_tma(lbm_t* h, int on);

/* on = 1 (default; the environment variable LBM_BAND = 0 / 1 / 2 sets the default): lattices WITH
 * particles also use a multi-step kernel, on the particle-free rows [0, Q) below the lowest
 * particle (DESIGN.md sections 6a, 6b), in lbm_step calls of at least 16 steps (such
 * a call plans the band once on entry to size its grids: one more synchronisation).  In periods of
 * six time steps (four with lbm_set_band_steps(h, 2)) a device kernel picks Q from the particle
 * positions and speeds (far enough below the lowest particle that no link or refill stencil reaches
 * the band within the period; fewer than 28 free rows: no band); the band is advanced t -> t+3 ->
 * t+6 by the three-step kernel (t -> t+2 -> t+4 by the two-step kernel) while the rows above it
 * take ordinary steps, reading the band's top row at the intermediate times from a spare row.  The
 * arithmetic per node and step is unchanged: results are identical bit for bit to on = 0.
 * on = 1 uses a band only if it holds at least 2^18 nodes (below that its extra launches cost more
 * than the traffic it saves); on = 2 uses every band of at least 28 rows (the tests).
 * A settled bed leaves the rows under the lid free instead: the plan at the start of a call picks
 * the larger of the two bands (rows [0, Q) under the lowest particle, rows [Q, ny) above the
 * highest) and the call keeps that orientation.
 * lbm_get_band: *rows = Q of the last plan (0: none; > 0: the band is [0, Q); < 0: [-Q, ny)). */
int lbm_set_band(lbm_t* h, int on);
int lbm_get_band(lbm_t* h, int* rows);

/* ---- y-slabs: domain decomposition along y (PAPER.md:287-291 ghost layers,
 * 303-321 domain lists, 347-355 schedule).  BASELINE.json's north_star keeps the measured path on
 * one GPU; this is the library side of the next step, testable on one device.
 *
 * A slab handle stores and updates the rows [j0, j1) of a cavity ny_global rows high (its OWN rows)
 * plus `halo` ghost rows on every side that is not a cavity wall.  Every slab holds EVERY particle
 * (lbm_add_particles with the same arrays on each; coordinates are global) and advances all of
 * them identically; which slab does what for a particle follows from positions alone (the paper's
 * domain lists): each slab rasterises, builds links and runs the bounce-back for whatever part of
 * a particle lies in its stored rows (that parks the values its own rows pull); the slab whose own
 * rows hold the particle's centre sees all of its links -- the halo must be at least d/2 + 8 rows,
 * checked by lbm_add_particles -- and its force sum, in the single domain's order, is the
 * particle's force.  Results on own rows and all particle states are bit-identical to one
 * lbm_create domain (tests/test_gpu_slabs.py).
 *
 * One time step, for all slabs:
 *   lbm_slab_forces(h)      bounce-back + momentum exchange; the slab's share of F, T_z (zeros for
 *                           particles it does not own) is left in lbm_slab_force_buffer
 *   -- force combine: element-wise sum of the slabs' buffers (3 * n doubles: Fx[n], Fy[n], Tz[n]),
 *      written back to every slab's buffer.  One process: lbm_slab_combine_forces; ranks: an
 *      all-reduce (the sum is exact: one non-zero term per entry)
 *   lbm_slab_advance(h)     particle update from the combined forces, flags, refill, links, lattice
 *                           kernel on the own rows
 *   -- halo exchange: lbm_slab_pack(h, side, buf) / lbm_slab_unpack(h, side, buf) with
 *      lbm_slab_halo_doubles values per face (14 populations x halo rows), or, in one process,
 *      lbm_slab_exchange_halos (direct copies, peer copies between devices)
 * lbm_slab_check reads the device status word (one synchronisation; same errors as lbm_step).
 * lbm_step refuses slab handles.  lbm_set_temperature takes the STORED rows (own + ghost:
 * global rows [j0 - halo, j1 + halo) clipped to the cavity), lbm_get_fields returns the OWN rows.
 * Errors: LBM_E_ARG (halo < 4, a slab lower than its halo, ranges that do not adjoin), LBM_E_STATE. */
size_t lbm_slab_workspace_bytes(int nx, int ny_global, int j0, int j1, int halo, const lbm_params* p);
int lbm_create_slab(int nx, int ny_global, int j0, int j1, int halo, const lbm_params* p,
                    void* dev_workspace, size_t bytes, void* cuda_stream, lbm_t** out);
int lbm_slab_forces(lbm_t* h);
int lbm_slab_force_buffer(lbm_t* h, double** dev_buf, int* count);   /* DEVICE pointer, 3 * n doubles */
int lbm_slab_advance(lbm_t* h);
int lbm_slab_check(lbm_t* h);
int lbm_slab_halo_doubles(const lbm_t* h, long long* doubles);
int lbm_slab_pack(lbm_t* h, int side, double* dev_buf);           /* side 0: lowest own rows, 1: highest */
int lbm_slab_unpack(lbm_t* h, int side, const double* dev_buf);   /* side 0: ghost rows below, 1: above */
int lbm_slab_exchange_halos(lbm_t** slabs, int n);                /* ascending row ranges, one process */
/* Fused halo exchange for slabs of one process (ascending row ranges): after lbm_slab_link_peers
 * the lattice kernel and the refill commit of lbm_slab_advance also write the rows next to a cut
 * straight into the neighbour slab's ghost rows (peer memory: the same GPU, or another GPU of the
 * node with peer access over NVLink) -- the exchange becomes the epilogue of the kernel that
 * produces the data.  lbm_slab_fence (instead of lbm_slab_exchange_halos) then ends a step: all
 * slabs' streams are synchronised, so every push has landed before the next step reads it.
 * Every slab must be advanced once per step.  Same bits as the copy-based exchange. */
int lbm_slab_link_peers(lbm_t** slabs, int n);
int lbm_slab_fence(lbm_t** slabs, int n);
int lbm_slab_combine_forces(lbm_t** slabs, int n);                /* same (peer access between devices) */

/* Readout.  Any pointer may be NULL = not wanted.
 * rho, ux, uy, T: nx*ny doubles each; on fluid nodes rho = sum f, T = sum g,
 *   u = (sum e f + F/2)/rho; on solid nodes rho0, rigid-body velocity, T_w.
 * f: 9*nx*ny, g: 5*nx*ny doubles, population-major (f[k*nx*ny + j*nx + i]): the POST-collision
 *   populations f+(x,t), g+(x,t) (right-hand sides of Eqs. 5, 6 before streaming) -- the quantity
 *   Eqs. 9-13 consume and the state the fused kernel keeps resident.  Values on solid nodes are
 *   unspecified (parity is taken on fluid nodes).
 * flag: nx*ny bytes, 0 fluid, 1 solid. */
int lbm_get_fields(lbm_t* h, double* rho, double* ux, double* uy, double* T,
                   double* f, double* g, unsigned char* flag);

/* The macroscopic read-out for callers that cannot allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc) and want the workspace left untouched:
 * the same kernel as lbm_get_fields, but its dense outputs are staged in a file-scope
 * `static __device__` array of the library instead of the dead copy of the populations, then
 * copied to the caller's HOST buffers (each nx*ny doubles; any may be NULL).  Calls no cudaMalloc,
 * cudaFree or allocating library routine.
 * Limit: nx*ny <= LBM_STATIC_MAX_NODES (2^20 nodes: 4 fields x 8 MiB = 32 MiB of device memory,
 * held by every GPU that loads the library until the process exits); larger lattices (and slab
 * handles) are rejected with LBM_E_CAPACITY resp. LBM_E_STATE and a text in lbm_last_error.
 * Every call on a device shares that array, which keeps the last call's contents (every node of
 * the requested outputs is rewritten, so nothing stale is ever returned); calls that overlap on
 * the GPU -- two handles on different streams -- race on it: serialise them.
 * Results are bit-identical to lbm_get_fields(h, rho, ux, uy, T, NULL, NULL, NULL). */
#define LBM_STATIC_MAX_NODES (1 << 20)
int lbm_get_macroscopic_static(lbm_t* h, double* rho, double* ux, double* uy, double* T);

/* Particle state (r, U, theta, Omega_z; F, T_z of the last completed step).
 * *n receives the particle count; arrays (each may be NULL) need that many entries. */
int lbm_get_particles(lbm_t* h, int* n, double* x, double* y, double* theta,
                      double* ux, double* uy, double* omega, double* Fx, double* Fy, double* Tz);

/* Runs the link builder (row a2) on the CURRENT particle positions and returns
 * the compacted fluid-particle links: fluid node (i,j), lattice direction alpha in 1..8 with
 * (i,j)+e_alpha inside particle pid, and q.  In: *n = capacity of the arrays
 * (arrays may be NULL if *n = 0).  Out: *n = number of links.  LBM_E_CAPACITY if too small
 * (then *n = required).  Order: by particle, then the builder's scan order (callers sort). */
int lbm_get_links(lbm_t* h, long long* n, int* pid, int* i, int* j, int* alpha, double* q);

/* Per-kernel device timing with CUDA events on the handle's stream (used by bench.py for the
 * roofline line).  on=1 starts recording around every kernel launch of lbm_step (events are
 * pre-created; at most LBM_PROFILE_MAX_SAMPLES launches per kernel are sampled, the rest run
 * untimed); on=0 stops.  lbm_profile_get: kernel ids 0..lbm_profile_kernels()-1; returns the
 * summed duration in ms over the sampled launches and their number. */
#define LBM_PROFILE_MAX_SAMPLES 512
int lbm_profile_enable(lbm_t* h, int on);
int lbm_profile_kernels(void);
const char* lbm_profile_kernel_name(int kernel_id);
int lbm_profile_get(lbm_t* h, int kernel_id, double* total_ms, long long* launches);

/* Number of CUDA kernels this handle has launched since lbm_create (set-up, step and read-out
 * kernels; memsets and copies are not counted).  bench.py reports the difference across its
 * timed region as "gpu_launches".  Returns -1 for a NULL handle. */
long long lbm_kernel_launches(const lbm_t* h);

/* Frees the handle (not the workspace).  NULL is a no-op. */
int lbm_destroy(lbm_t* h);

/* Text of the last error on this handle; with h = NULL, of the last failed lbm_create. */
const char* lbm_last_error(const lbm_t* h);

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
