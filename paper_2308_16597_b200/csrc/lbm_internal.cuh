// lbm_internal.cuh -- shared declarations of the CUDA path (product).  Not part of the C ABI.
//
// HBM layout: structure of arrays, fp64, node (i,j) at x = j*px + i,
//   px = nx rounded up to 16 doubles, ps = px*ny rounded up to 32 doubles.
//   populations: the D2Q5 directions k = 0..4 carry a flow AND a temperature population that
//   stream along the same e_k, so they are stored as pairs: pair plane k (k = 0..4) at
//   base + 2*k*ps holds (f_k(x), g_k(x)) at doubles 2x, 2x+1 (one 16-byte access per node and
//   direction for the lattice kernel, the bounce-back kernel and the parked slot); the diagonal
//   flow populations f5..f8 are plain planes at base + (k+5)*ps + x.  14*ps doubles per copy;
//   two copies A (read) and B (written), swapped per step.
//   flag : 1 byte/node, 0 fluid, 1 solid, 2 newborn (solid at t, fluid at t+1; only between the
//          flag update and the refill kernel of one step)
//   owner: int32/node, id of the lowest-numbered particle covering the node, OWNER_NONE = fluid
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lbm.h"

#define OWNER_NONE 0x7f7f7f7f   // = cudaMemset(0x7f): larger than any particle id
#define CELL_CAP 32          // particle centres per repulsion-grid cell
#define MIN_CELL 16.0        // smallest repulsion-grid cell edge (workspace is sized for it)
#define NEWBORN_PER_PARTICLE 32
#define LBM_MAX_GRAPHS 8
#define LBM_TMA_MIN_NODES (1LL << 20)   // three-step passes go through the persistent TMA-fed kernel from this size up

// status bits written by kernels, read once per lbm_step call
#define ST_NONFINITE 1
#define ST_LINK_OVERFLOW 2
#define ST_CELL_OVERFLOW 4
#define ST_NEWBORN_OVERFLOW 8
#define ST_BAND_REACHED 16

enum {
  K_STREAM_COLLIDE = 0, K_BUILD_LINKS, K_BOUNCE_BACK, K_MOVE, K_COVER, K_REFILL,
  K_INIT, K_REFILL_COMMIT, K_STREAM_COLLIDE_2STEP, K_BAND_PLAN, K_STREAM_COLLIDE_3STEP,
  K_STREAM_COLLIDE_3STEP_TMA, K_COUNT
};

// link_dir byte: bits 0-3 = alpha (1..8), bits 4-5 = number of fluid nodes behind x_f along
// -e_alpha (0, 1 or 2: which rung of the interpolation ladder of DESIGN.md reading 6 applies).
// The link builder fills it from the flag map of the step the links belong to, so that the
// bounce-back kernel needs no dependent flag loads.
#define LINK_DIR_MASK 0x0f
#define LINK_BEHIND_SHIFT 4

// double index of f_k / g_k of node x inside one copy of the populations
__host__ __device__ __forceinline__ long long f_at(int k, long long x, long long ps) {
  return k <= 4 ? 2 * k * ps + 2 * x : (k + 5) * ps + x;
}
__host__ __device__ __forceinline__ long long g_at(int k, long long x, long long ps) {
  return 2 * k * ps + 2 * x + 1;
}

// constants every kernel needs; passed by value (lands in the constant bank)
struct LbmConst {
  int nx, ny, px;          // lattice size (rows this handle stores), row pitch (doubles)
  // y-slabs: the handle stores the global rows [yoff, yoff + ny)
  // of a cavity NY rows high.  Particle coordinates, link nodes and every row index the particle
  // kernels compute with are GLOBAL; only memory indices are local.  Single domain: 0, ny.
  int yoff, NY;
  long long ps;            // plane stride (doubles)
  int periodic_x;
  // D2Q9 MRT (DESIGN.md readings): relaxation rates and the (1 - s/2) forcing factors
  double s_e, s_eps, s_q, s_nu;
  // D2Q5 MRT
  double q_k, q_e, q_nu, aT, wT0, wT;   // wT0 = (1-aT)/5, wT = (4+aT)/20
  double rho0, T0, gbeta, ax, ay, g;
  int wall_type[4];        // W,E,S,N
  double wall_T[4];
  double rep_s, rep_eps;
  int rep_power;
};

// y-slabs: where the rows next to a cut also go -- the ghost rows of the neighbour slab's copy of
// the state being written (peer memory of the same process).  lo: my local rows
// [lo_start, lo_end) = the lowest `halo` own rows land in the lower neighbour at its local row
// (j + lo_shift); hi: the highest own rows [hi_start, hi_end) in the upper neighbour.
struct HaloPush {
  double* lo;
  long long lo_ps;
  int lo_shift, lo_start, lo_end;
  double* hi;
  long long hi_ps;
  int hi_shift, hi_start, hi_end;
};

struct ParticleArrays {      // SoA in the workspace, each max_particles long
  double *x[2], *y[2], *theta[2], *ux[2], *uy[2], *omega[2];   // double-buffered state
  double *r, *rho_ratio, *Tw;   // r: radius of a circle, largest semi-axis of an ellipse
  // elliptical particles: semi-axes a, b
  // (a == b: a circle, which takes the circle formulas bit for bit) and the orientation as a unit
  // vector (cs, sn), double-buffered with the state and advanced without any cos / sin
  double *a, *b, *cs[2], *sn[2];
  double *Fx, *Fy, *Tz;      // hydrodynamic force / torque of the last step (Eqs. 13, 14)
  unsigned char* fixed;
  unsigned char* ovl;        // sticky: the disc may share nodes with another particle's (k_cover)
};

struct LinkArrays {          // the paper's fixed index array: segment p = [p*cap, (p+1)*cap)
  int* node;                 // fluid node x_f, packed i | j << 16 (nx, ny <= 46000 < 2^16)
  unsigned char* dir;        // alpha in 1..8
  double* q;
  int* count;                // links of particle p
  int cap;
};

struct lbm {
  int nx, ny, px;            // ny: rows stored by this handle
  // y-slab (lbm_create_slab): global rows [yoff, yoff + ny) of a cavity NY rows high are stored,
  // the own rows [own0, own1) (global) are updated, `halo` ghost rows on each interior side.
  // row0, row1: the own rows as LOCAL indices.  A single domain: 0, ny, 0, ny, halo 0.
  int is_slab, yoff, NY, own0, own1, halo, row0, row1;
  lbm *peer_lo, *peer_hi;    // neighbour slabs in the same process (lbm_slab_link_peers): the halo push targets
  long long ps;
  lbm_params P;
  LbmConst C;
  cudaStream_t stream;       // the caller's stream: bounce-back, lattice kernel, refill, set-up, read-out
  cudaStream_t chain;        // the serial chain: bounce-back, particle update, flags, links, refill commit
  cudaStream_t side;         // refill (beside the link builder)
  cudaStream_t chain_own;    // the stream we created (NULL if creation failed)
  cudaStream_t side_own;     // refill runs here, beside the link builder
  cudaEvent_t ev_in, ev_out, ev_bb, ev_sc, ev_cov, ev_ref;
  int overlap;               // 1: chain runs on `chain_own` concurrently with the lattice kernel
  int chain_ctas;            // CTAs per chain kernel while it runs under the lattice kernel (0 = one per item)
  int sm_count;
  int two_step;              // particle-free lattice: advance two steps per pass (lbm_set_two_step)
  int links_ready;           // the index array holds the links of the current particle positions
  double *A, *B;             // 14 planes each
  unsigned char* flag;
  int* owner;
  ParticleArrays pa;
  LinkArrays la;
  int cur;                   // which particle state buffer is current
  int np;                    // particles added
  int n_ell;                 // of which ellipses (a != b): selects the kernel instantiations
  double d_max;              // largest diameter (sizes the repulsion grid)
  int* cell_count[2];        // repulsion grid, double-buffered by the particle buffer index
  int* cell_items[2];
  int ncx, ncy;
  double cell;               // cell edge
  int max_cells;
  int* newborn_node;
  int* newborn_pid;
  int* newborn_count;        // two counters, [step parity = cur at the start of the step]
  double* stash;             // 14 refilled populations per newborn-list entry
  int newborn_cap;
  int* status_dev;
  int* status_host;          // pinned: [0] status word, [1] band height of the last banded period
  // two-step band: band[0] = Q, rows
  // [0, Q) are advanced two steps per pass; band[1] = 0 (what the plain schedule's kernels read)
  int* band;
  double* force_buf;         // y-slabs: 3 * max_particles doubles (Fx, Fy, Tz), the slab's share of the force combine
  int band_hint;             // rows certainly inside the band as the host last saw it (part of the graph key)
  int band_l1_rows;          // CTA rows of the one-step kernel in banded steps (the rows outside that, + a margin)
  int band_orient;           // 0: the call-start plan chooses; +1 band under the suspension, -1 above it
  int band_live;             // the step being enqueued belongs to a banded period (k_cover checks the margin)
  int band_cap;              // most rows the band may have in this call (sizes the band kernel's grid)
  int band_on;               // lbm_set_band / LBM_BAND: use the banded schedule where it applies
  int band_steps;            // lbm_set_band_steps / LBM_BAND_STEPS: 2 or 3 time steps per pass in a band under the suspension
  int want3;                 // this call may use periods of six steps (band under the suspension, band_steps == 3)
  int band3;                 // the unit being enqueued is such a period: the band advances three steps per pass
  cudaEvent_t ev_p2;         // the band kernel's part of a step has been issued (the particle chain follows it)
  cudaEvent_t ev_plan;       // the band plan of a period has been issued (the caller's stream follows it)
  int primed;                // 0: A holds pre-collision f(x,0); 1: A holds post-collision f+(x,t)
  long long steps_done;
  long long launches;        // kernels launched (lbm_kernel_launches)
  int device;                // the device the handle was created on (every entry point selects it)
  int two_step_ok;           // the two-step kernel's attributes could be set
  // k_stream_collide_3step_tma: tensor maps of the two copies ([2*copy] pair planes, [2*copy+1]
  // diagonal planes; opaque CUtensorMap bytes), the copies' base pointers, and whether they exist
  unsigned long long tmaps[4][16];
  const double* tma_base[2];
  int tma_ok;
  int use_tma;               // lbm_set_tma / LBM_TMA: three-step passes go through the TMA-fed kernel
  // CUDA graphs: a period of the schedule -- an even number of steps,
  // after which A/B and the particle buffer index are back where they started -- is captured once
  // per (phase, length, schedule) and replayed; the fork/join onto the chain stream is part of
  // the capture.  The single-GPU analogue of the paper's async(n) queues.
  int use_graph;
  int use_pdl;               // programmatic dependent launch along the chain (LBM_PDL=0 turns it off)
  cudaStream_t cap_stream;   // capture happens here (the caller's stream may be the legacy stream)
  void* cap_nodes;           // during capture: std::vector<cudaGraphNode_t>* of the chain's kernel nodes
  int chain_priority;        // priority of the chain stream, given to those nodes
  struct StepGraph {
    cudaGraphExec_t exec;
    const double* A;         // phase the graph was captured in
    int cur, steps, overlap, chain_ctas, banded, band_hint, band_cap, band_orient;
    long long launches;      // kernels per replay
  } graphs[LBM_MAX_GRAPHS];
  int n_graphs;
  // profiling
  int prof_on;
  cudaEvent_t* ev0[K_COUNT];
  cudaEvent_t* ev1[K_COUNT];
  int ev_n[K_COUNT];
  char err[512];
};

// global row j of the cavity: is it stored by this handle, and where
__host__ __device__ __forceinline__ bool row_here(const LbmConst& c, int j) {
  return j >= c.yoff && j < c.yoff + c.ny;
}
__host__ __device__ __forceinline__ long long node_index(const LbmConst& c, int i, int j) {
  return (long long)(j - c.yoff) * c.px + i;
}

// ---- programmatic dependent launch (PDL).  Every kernel of the step's serial chain starts with
// pdl_wait(): launched with the programmatic-serialisation attribute it may begin while its
// predecessor in the stream still runs, and this is where it waits for that kernel to have
// completed and flushed; launched normally the instruction returns at once.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }

#ifdef __CUDACC__
#include <utility>
// <<<grid, block, smem, st>>> with the PDL attribute on request
template <typename... KArgs, typename... Args>
inline void launch_k(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                     bool pdl, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}
#endif

// ---- kernel launchers (each in its own translation unit) ----
// stream_collide.cu
void launch_stream_collide(lbm* h, int band, const double* low);   // on h->stream, h->A -> h->B
void launch_stream_collide_slab(lbm* h, const HaloPush& hp);       // on h->stream; own rows, with the halo push
void launch_stream_collide_2step(lbm* h);  // on h->stream; particle-free lattices only
void launch_stream_collide_3step(lbm* h);  // on h->stream; particle-free lattices only
int stream_collide_tma_setup(lbm* h);      // tensor maps for the TMA-fed three-step kernel (0 = ok, sets h->tma_ok)
void launch_stream_collide_3step_tma(lbm* h);  // on h->stream; particle-free closed cavities, needs h->tma_ok
void launch_stream_collide_band(lbm* h, const double* src_band, const double* src_top, double* dst_band,
                                int nparts, int part);   // on h->stream; rows [0, *h->band)
void launch_stream_collide_band3(lbm* h, double* src, double* dst, int nparts, int part);   // on h->stream; rows [0, *h->band), three steps per pass
int stream_collide_configure();            // kernel attributes (0 = ok)
void launch_init_collide(lbm* h, double* dst);   // dst = h->A (in place) or scratch
void launch_set_temperature(lbm* h, const double* T_dev_dense);
void launch_set_equilibrium(lbm* h);
void launch_export(lbm* h, double* f_dense, double* g_dense);    // dense f[9][n], g[5][n], device
void launch_macroscopic(lbm* h, double* rho, double* ux, double* uy, double* T);  // dense nx*ny, device
int launch_macroscopic_static(lbm* h, double** fields4);   // into the library's static scratch array; 0 / -1 too large / -2
// particles.cu (compiled with -fmad=false)
// `pdl`: launch with the programmatic-serialisation attribute (the kernel then waits for its
// predecessor in `st` itself, see pdl_wait)
void launch_build_links(lbm* h, int which_buffer, cudaStream_t st, bool pdl);
void launch_move(lbm* h, cudaStream_t st, bool pdl);   // integrator + uncover, buffer cur -> cur ^ 1
int particles_configure(lbm* h);           // per-handle kernel attributes (0 = ok)
void launch_cover(lbm* h, int which_buffer, cudaStream_t st, bool pdl);   // (band margin check: 4 rows, 5 with h->band3)
void launch_band_plan(lbm* h, cudaStream_t st);
void launch_slab_forces_out(lbm* h);   // owned particles' F, T_z -> h->force_buf (zeros for the others)
void launch_slab_forces_in(lbm* h);    // h->force_buf (combined over the slabs) -> F, T_z
void launch_add_buffer(double* dst, const double* src, int n, cudaStream_t st);   // h->band[0] from the positions of buffer h->cur
// bounce_back.cu
void launch_bounce_back(lbm* h, cudaStream_t st, bool pdl);
void launch_refill(lbm* h, cudaStream_t st); // reads A, writes the stash; called before cur is flipped
void launch_refill_commit(lbm* h, int step_parity, cudaStream_t st, bool pdl, const HaloPush* hp = nullptr);  // stash -> B (and the neighbours' ghost rows), newborn flags cleared
