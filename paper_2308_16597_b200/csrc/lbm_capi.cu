// lbm_capi.cu -- the C ABI of include/lbm.h: workspace carving, host-side validation, the per-step
// launch sequence (SURVEY.md 3 / 7 "legal fused ordering"), read-out copies and event profiling.
// No torch types, no exceptions across the boundary, no cudaMalloc of lattice state: everything
// lives in the caller's workspace (only the pinned status word and the events are ours).
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <utility>
#include <vector>

#include "lbm_internal.cuh"

namespace {

char g_create_error[512] = "";

const char* const kKernelNames[K_COUNT] = {
    "stream_collide", "build_links", "bounce_back_force", "integrate_uncover",
    "flags_cover", "refill", "init_collide", "refill_commit", "stream_collide_2step", "band_plan",
    "stream_collide_3step", "stream_collide_3step_tma"};

int fail(lbm* h, int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(h ? h->err : g_create_error, 512, fmt, ap);
  va_end(ap);
  return code;
}

#define CUDA_OK(h, call)                                                              \
  do {                                                                                \
    cudaError_t e_ = (call);                                                          \
    if (e_ != cudaSuccess)                                                            \
      return fail(h, LBM_E_CUDA, "%s: %s", #call, cudaGetErrorString(e_));            \
  } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

constexpr long long LBM_BAND_MIN_NODES = 1LL << 18;
constexpr int LBM_BAND_MIN_STEPS = 16;   // shortest lbm_step call that uses the two-step band
constexpr int LBM_GRAPH_STEPS = 8;   // time steps per graph launch (an even number: one or more periods)

// Every entry point runs on the device the handle was created on, whatever device is current in
// the calling thread, and leaves the caller's choice as it found it.
struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(const lbm* h) {
    if (h && cudaGetDevice(&prev) == cudaSuccess && prev != h->device) cudaSetDevice(h->device);
    else prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Lays the arrays out in the workspace.  With base == nullptr only the size is computed.
struct Carver {
  char* base;
  size_t off = 0;
  explicit Carver(void* b) : base((char*)b) {}
  template <typename T>
  T* take(size_t count) {
    off = align_up(off, 256);
    T* p = base ? (T*)(base + off) : nullptr;
    off += sizeof(T) * count;
    return p;
  }
};

struct Layout {
  int px;
  long long ps;
  int max_cells, mcx, mcy;
  int newborn_cap;
};

// ny: rows stored; NY: height of the whole cavity (the repulsion grid covers all of it)
Layout layout_of(int nx, int ny, int NY, const lbm_params* p) {
  Layout L;
  L.px = (int)align_up((size_t)nx, 16);
  L.ps = (long long)align_up((size_t)L.px * (ny + 1), 32);   // one spare row (the band seam's)
  L.mcx = (int)std::ceil(nx / MIN_CELL) + 1;
  L.mcy = (int)std::ceil(NY / MIN_CELL) + 1;
  L.max_cells = p->max_particles > 0 ? L.mcx * L.mcy : 0;
  L.newborn_cap = p->max_particles * NEWBORN_PER_PARTICLE;
  return L;
}

size_t carve(lbm* h, void* base, int nx, int ny, int NY, const lbm_params* p) {
  const Layout L = layout_of(nx, ny, NY, p);
  Carver c(base);
  const size_t np = (size_t)p->max_particles;
  double* A = c.take<double>(14 * (size_t)L.ps);
  double* B = c.take<double>(14 * (size_t)L.ps);
  unsigned char* flag = c.take<unsigned char>((size_t)L.px * ny);
  int* owner = c.take<int>((size_t)L.px * ny);
  ParticleArrays pa;
  for (int b = 0; b < 2; ++b) {
    pa.x[b] = c.take<double>(np);
    pa.y[b] = c.take<double>(np);
    pa.theta[b] = c.take<double>(np);
    pa.ux[b] = c.take<double>(np);
    pa.uy[b] = c.take<double>(np);
    pa.omega[b] = c.take<double>(np);
  }
  for (int b = 0; b < 2; ++b) {
    pa.cs[b] = c.take<double>(np);
    pa.sn[b] = c.take<double>(np);
  }
  pa.a = c.take<double>(np);
  pa.b = c.take<double>(np);
  pa.r = c.take<double>(np);
  pa.rho_ratio = c.take<double>(np);
  pa.Tw = c.take<double>(np);
  pa.Fx = c.take<double>(np);
  pa.Fy = c.take<double>(np);
  pa.Tz = c.take<double>(np);
  pa.fixed = c.take<unsigned char>(np);
  pa.ovl = c.take<unsigned char>(np);
  LinkArrays la;
  const size_t nl = np * (size_t)p->max_links_per_particle;
  la.node = c.take<int>(nl);
  la.dir = c.take<unsigned char>(nl);
  la.q = c.take<double>(nl);
  la.count = c.take<int>(np);
  la.cap = p->max_links_per_particle;
  int* cell_count[2];
  int* cell_items[2];
  for (int b = 0; b < 2; ++b) {
    cell_count[b] = c.take<int>((size_t)L.max_cells);
    cell_items[b] = c.take<int>((size_t)L.max_cells * CELL_CAP);
  }
  int* nb_node = c.take<int>((size_t)L.newborn_cap);
  int* nb_pid = c.take<int>((size_t)L.newborn_cap);
  int* nb_count = c.take<int>(2);
  double* stash = c.take<double>((size_t)L.newborn_cap * 14);
  int* status = c.take<int>(1);
  int* band = c.take<int>(2);
  double* fbuf = c.take<double>(3 * np);
  if (h) {
    h->force_buf = fbuf;
    h->band = band;
    h->px = L.px;
    h->ps = L.ps;
    h->A = A;
    h->B = B;
    h->flag = flag;
    h->owner = owner;
    h->pa = pa;
    h->la = la;
    for (int b = 0; b < 2; ++b) {
      h->cell_count[b] = cell_count[b];
      h->cell_items[b] = cell_items[b];
    }
    h->max_cells = L.max_cells;
    h->newborn_node = nb_node;
    h->newborn_pid = nb_pid;
    h->newborn_count = nb_count;
    h->stash = stash;
    h->newborn_cap = L.newborn_cap;
    h->status_dev = status;
  }
  return align_up(c.off, 256);
}

bool params_ok(int nx, int ny, const lbm_params* p) {
  return p && nx >= 4 && ny >= 4 && nx <= 46000 && ny <= 46000 && p->nu > 0.0 && p->kappa > 0.0 &&
         p->kappa < 0.144 && p->rho0 > 0.0 && p->max_particles >= 0 &&
         p->max_links_per_particle >= 0 && p->max_links_per_particle <= 12000 && p->rep_s > 0.0 && p->rep_eps > 0.0 &&
         p->rep_power >= 1 && std::isfinite(p->nu) && std::isfinite(p->kappa);
}

void fill_const(lbm* h) {
  LbmConst& c = h->C;
  const lbm_params& p = h->P;
  c.nx = h->nx;
  c.ny = h->ny;
  c.yoff = h->yoff;
  c.NY = h->NY;
  c.px = h->px;
  c.ps = h->ps;
  c.periodic_x = p.periodic_x ? 1 : 0;
  // DESIGN.md readings: s_nu = 1/tau, tau = 3 nu + 1/2, s_e = s_eps = s_nu, s_q = 8(2-s_nu)/(8-s_nu)
  const double tau = 3.0 * p.nu + 0.5;
  c.s_nu = 1.0 / tau;
  c.s_e = c.s_nu;
  c.s_eps = c.s_nu;
  c.s_q = 8.0 * (2.0 - c.s_nu) / (8.0 - c.s_nu);
  const double r3 = std::sqrt(3.0);
  c.q_k = 3.0 - r3;
  c.q_e = 4.0 * r3 - 6.0;
  c.q_nu = 4.0 * r3 - 6.0;
  c.aT = 20.0 * r3 * p.kappa - 4.0;
  c.wT0 = (1.0 - c.aT) / 5.0;
  c.wT = (4.0 + c.aT) / 20.0;
  c.rho0 = p.rho0;
  c.T0 = p.T0;
  c.gbeta = p.gbeta;
  c.ax = p.body_ax;
  c.ay = p.body_ay;
  c.g = p.g;
  for (int k = 0; k < 4; ++k) {
    c.wall_type[k] = p.wall_T_type[k];
    c.wall_T[k] = p.wall_T[k];
  }
  c.rep_s = p.rep_s;
  c.rep_eps = p.rep_eps;
  c.rep_power = p.rep_power;
}

// ---- profiling helpers ----
struct Timed {
  lbm* h;
  int k;
  cudaStream_t st;
  bool on;
  Timed(lbm* h_, int k_, cudaStream_t st_) : h(h_), k(k_), st(st_), on(false) {
    if (h->prof_on && h->ev_n[k] < LBM_PROFILE_MAX_SAMPLES) {
      on = true;
      cudaEventRecord(h->ev0[k][h->ev_n[k]], st);
    }
  }
  ~Timed() {
    // debugging aid (LBM_DEBUG_SYNC=1, with LBM_GRAPH=0): synchronise after every launch and name
    // the first kernel that fails, instead of a sticky error at the end of the call
    static const int dbg = getenv("LBM_DEBUG_SYNC") ? atoi(getenv("LBM_DEBUG_SYNC")) : 0;
    if (dbg) {
      cudaError_t e = cudaDeviceSynchronize();
      if (e != cudaSuccess) {
        fprintf(stderr, "[lbm debug] %s failed at step %lld: %s\n", kKernelNames[k], h->steps_done, cudaGetErrorString(e));
        fflush(stderr);
        abort();
      }
    }
    if (on) {
      cudaEventRecord(h->ev1[k][h->ev_n[k]], st);
      h->ev_n[k]++;
    }
  }
};

int check_status(lbm* h) {
  CUDA_OK(h, cudaMemcpyAsync(h->status_host, h->status_dev, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CUDA_OK(h, cudaMemcpyAsync(h->status_host + 1, h->band, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CUDA_OK(h, cudaStreamSynchronize(h->stream));
  CUDA_OK(h, cudaGetLastError());
  const int st = *h->status_host;
  if (st & ST_NONFINITE) return fail(h, LBM_E_NONFINITE, "a particle state became NaN/Inf");
  if (st & ST_LINK_OVERFLOW) return fail(h, LBM_E_CAPACITY, "a particle has more links than max_links_per_particle");
  if (st & ST_CELL_OVERFLOW) return fail(h, LBM_E_CAPACITY, "more than %d particle centres in one repulsion cell", CELL_CAP);
  if (st & ST_NEWBORN_OVERFLOW) return fail(h, LBM_E_CAPACITY, "newborn-node list overflow");
  if (st & ST_BAND_REACHED) return fail(h, LBM_E_STATE, "a particle came within 4 rows of the two-step band (lbm_set_band(h, 0) runs without it)");
  return LBM_OK;
}

// CTAs of a particle-chain kernel while it runs under the lattice kernel (DESIGN.md "Step
// schedule").  Measured on B200: the lattice kernel keeps its speed when other work holds up to
// two of its nine 128-thread CTA slots per SM and loses 7 % at three; a 64-thread chain CTA under a
// saturated memory system needs about 45 us per d = 20 particle for its three zone kernels (75 us
// at d = 40).  Pick the fewest CTAs per SM (at least 2) with which the chain still ends within
// 50 % of the time the lattice kernel needs for the WHOLE lattice (224 B per node at 6 TB/s) --
// with a two-step band below the suspension the kernel covers about two thirds of it.
// Configs 3 and 4: 5 and 6 per SM, the paper's d = 40 workload: 9.  LBM_CHAIN_CTAS_PER_SM
// overrides (0 = one CTA per particle).
void size_chain(lbm* h) {
  if (const char* e = getenv("LBM_CHAIN_CTAS_PER_SM")) {
    h->chain_ctas = atoi(e) * h->sm_count;
    return;
  }
  if (h->np == 0) { h->chain_ctas = 0; return; }
  const double sc_us = (double)h->nx * h->ny * 224.0 / 6.0e6;
  const double tau_us = 45.0 * std::max(1.0, std::pow(h->d_max / 20.0, 0.75));
  double per_sm = std::ceil(h->np * tau_us / (h->sm_count * 0.5 * sc_us));
  per_sm = std::min(std::max(per_sm, 2.0), 24.0);
  h->chain_ctas = (int)per_sm * h->sm_count;
}

void prime(lbm* h) {
  if (h->primed) return;
  Timed t(h, K_INIT, h->stream);
  launch_init_collide(h, h->A);
  h->primed = 1;
}

// links of the current positions (the first step's; afterwards every step builds the next one's)
void ensure_links(lbm* h) {
  if (h->links_ready || h->np == 0) return;
  launch_build_links(h, h->cur, h->stream, false);
  h->links_ready = 1;
}

} // namespace

extern "C" {

void lbm_params_default(lbm_params* p) {
  if (!p) return;
  std::memset(p, 0, sizeof(*p));
  p->nu = 0.02;
  p->kappa = 0.02 / 0.7;
  p->rho0 = 1.0;
  p->rep_s = 2.0;
  p->rep_eps = 1e-3;
  p->rep_power = 1;
}

size_t lbm_workspace_bytes(int nx, int ny, const lbm_params* p) {
  if (!params_ok(nx, ny, p)) return 0;
  return carve(nullptr, nullptr, nx, ny, ny, p);
}

// Shared by lbm_create (a whole cavity: yoff = 0, NY = ny, no halo) and lbm_create_slab (global
// rows [yoff, yoff + ny) of a cavity NY rows high, of which [own0, own1) are the slab's own).
static int create_impl(int is_slab, int nx, int ny, int yoff, int NY, int own0, int own1, int halo, const lbm_params* p,
                       void* dev_workspace, size_t bytes, void* cuda_stream, lbm_t** out) {
  if (!out) return fail(nullptr, LBM_E_ARG, "lbm_create: out is NULL");
  *out = nullptr;
  if (!params_ok(nx, ny, p) || NY > 46000) return fail(nullptr, LBM_E_ARG, "lbm_create: bad size or parameter");
  if (!dev_workspace || ((uintptr_t)dev_workspace & 255))
    return fail(nullptr, LBM_E_ARG, "lbm_create: workspace NULL or not 256-byte aligned");
  const size_t need = carve(nullptr, nullptr, nx, ny, NY, p);
  if (bytes < need) return fail(nullptr, LBM_E_CAPACITY, "lbm_create: workspace %zu < %zu bytes", bytes, need);
  if ((long long)layout_of(nx, ny, NY, p).px * ny >= 0x7fffffffLL)
    return fail(nullptr, LBM_E_ARG, "lbm_create: lattice too large for 32-bit node indices");
  lbm* h = new (std::nothrow) lbm;
  if (!h) return fail(nullptr, LBM_E_ARG, "lbm_create: out of host memory");
  std::memset(h, 0, sizeof(*h));
  h->nx = nx;
  h->ny = ny;
  h->P = *p;
  h->stream = (cudaStream_t)cuda_stream;
  h->is_slab = is_slab;
  h->yoff = yoff;
  h->NY = NY;
  h->own0 = own0;
  h->own1 = own1;
  h->halo = halo;
  h->row0 = own0 - yoff;
  h->row1 = own1 - yoff;
  carve(h, dev_workspace, nx, ny, NY, p);
  fill_const(h);
  cudaGetDevice(&h->device);
  h->two_step_ok = stream_collide_configure() == 0 ? 1 : 0;
  h->two_step = h->two_step_ok ? 2 : 0;   // 0: one step per pass, 1: two, 2: three (then two, then one)
  if (h->two_step_ok) {
    const char* e3 = getenv("LBM_STEPS_PER_PASS");
    if (e3) h->two_step = atoi(e3) >= 3 ? 2 : (atoi(e3) == 2 ? 1 : 0);
  }
  h->band_steps = 3;
  if (const char* eb = getenv("LBM_BAND_STEPS")) h->band_steps = atoi(eb) >= 3 ? 3 : 2;
  // three steps per pass through the persistent TMA-fed kernel where it can run (closed cavity,
  // tensor maps encodable); LBM_TMA=0 keeps the plain three-step kernel
  h->use_tma = 0;
  if (h->two_step_ok && stream_collide_tma_setup(h) == 0) {
    const char* et = getenv("LBM_TMA");
    // default: from 2^20 nodes up, with the row-wise hand-over (2).  Measured per pass against the
    // plain three-step kernel (CUDA events, 402 steps): 1024^2 64.0 / 68.1 us, 2048^2 217 / 236 us,
    // 4096^2 855 / 903 us; with group barriers (1): 66.7 / 229 / 886 us
    h->use_tma = et ? std::min(std::max(atoi(et), 0), 2) : ((long long)nx * ny >= LBM_TMA_MIN_NODES ? 2 : 0);
  }
  if (particles_configure(h) != 0) {
    delete h;
    return fail(nullptr, LBM_E_CUDA, "lbm_create: max_links_per_particle needs more shared memory than the device has");
  }
  cudaError_t e = cudaMallocHost((void**)&h->status_host, 2 * sizeof(int));
  if (e != cudaSuccess) {
    fail(nullptr, LBM_E_CUDA, "cudaMallocHost: %s", cudaGetErrorString(e));
    delete h;
    return LBM_E_CUDA;
  }
  // streams of the step schedule: the serial chain of small kernels
  // (bounce-back, particle update, flags, links, refill commit) on a stream of the highest
  // priority, so that its latency-bound kernels get SM slots as CTAs of the lattice kernel retire;
  // the refill on a third stream beside the link builder; the lattice kernel on the caller's stream
  h->chain = h->stream;
  h->side = h->stream;
  {
    int lo = 0, hi = 0;
    cudaDeviceGetStreamPriorityRange(&lo, &hi);
    h->chain_priority = hi;
    bool ok = cudaStreamCreateWithPriority(&h->chain_own, cudaStreamNonBlocking, hi) == cudaSuccess &&
              cudaStreamCreateWithPriority(&h->side_own, cudaStreamNonBlocking, hi) == cudaSuccess;
    cudaEvent_t* evs[7] = {&h->ev_in, &h->ev_out, &h->ev_bb, &h->ev_sc, &h->ev_cov, &h->ev_ref, &h->ev_plan};
    for (cudaEvent_t* e : evs) ok = ok && cudaEventCreateWithFlags(e, cudaEventDisableTiming) == cudaSuccess;
    if (ok) {
      h->overlap = 1;
      h->chain = h->chain_own;
      h->side = h->side_own;
    } else {
      cudaGetLastError();
      h->chain_own = nullptr;
    }
  }
  if (cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) == cudaSuccess) {
    const char* e = getenv("LBM_GRAPH");
    h->use_graph = (e && atoi(e) == 0) ? 0 : 1;
    const char* e2 = getenv("LBM_PDL");
    h->use_pdl = (e2 && atoi(e2) == 0) ? 0 : 1;
  } else {
    cudaGetLastError();
    h->cap_stream = nullptr;
  }
  {
    const int dev = h->device;
    cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (h->sm_count <= 0) h->sm_count = 148;
    h->chain_ctas = 0;   // set by add_particles (size_chain)
  }
  // initial state: fluid everywhere, f = f_eq(rho0, 0), g = g_eq(T0, 0)
  const size_t nn = (size_t)h->px * ny;
  cudaMemsetAsync(h->flag, 0, nn, h->stream);
  cudaMemsetAsync(h->owner, 0x7f, nn * sizeof(int), h->stream);   // OWNER_NONE = 0x7f7f7f7f
  cudaMemsetAsync(h->status_dev, 0, sizeof(int), h->stream);
  cudaMemsetAsync(h->band, 0, 2 * sizeof(int), h->stream);
  cudaMemsetAsync(h->newborn_count, 0, 2 * sizeof(int), h->stream);
  h->status_host[1] = 0;
  {
    const char* eb = getenv("LBM_BAND");
    h->band_on = eb ? std::min(std::max(atoi(eb), 0), 2) : 1;   // 0 off, 1 where it pays, 2 every band
    if (cudaEventCreateWithFlags(&h->ev_p2, cudaEventDisableTiming) != cudaSuccess) {
      cudaGetLastError();
      h->band_on = 0;
      h->ev_p2 = nullptr;
    }
  }
  for (int b = 0; b < 2; ++b)
    if (h->max_cells) cudaMemsetAsync(h->cell_count[b], 0, sizeof(int) * (size_t)h->max_cells, h->stream);
  cudaMemsetAsync(h->B, 0, sizeof(double) * 14 * (size_t)h->ps, h->stream);
  launch_set_equilibrium(h);
  e = cudaStreamSynchronize(h->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) {
    fail(nullptr, LBM_E_CUDA, "lbm_create: %s", cudaGetErrorString(e));
    cudaFreeHost(h->status_host);
    delete h;
    return LBM_E_CUDA;
  }
  if (h->is_slab) {
    // a slab is stepped in two halves by its caller (lbm_slab_forces / lbm_slab_advance), on one
    // stream, with direct launches; no band (its plan would need every slab's agreement)
    h->overlap = 0;
    h->chain = h->side = h->stream;
    h->use_graph = 0;
    h->band_on = 0;
  }
  *out = h;
  return LBM_OK;
}

int lbm_create(int nx, int ny, const lbm_params* p, void* dev_workspace, size_t bytes,
               void* cuda_stream, lbm_t** out) {
  return create_impl(0, nx, ny, 0, ny, 0, ny, 0, p, dev_workspace, bytes, cuda_stream, out);
}

// ---- y-slabs (PAPER.md:287-291 ghost layers, 303-321 domain lists) ----
// rows stored by the slab that owns [j0, j1): `halo` ghost rows on each side that is not a cavity wall
static void slab_extent(int ny_global, int j0, int j1, int halo, int* yoff, int* rows) {
  const int lo = j0 == 0 ? 0 : j0 - halo, hi = j1 == ny_global ? ny_global : j1 + halo;
  *yoff = lo;
  *rows = hi - lo;
}

static bool slab_ok(int nx, int ny_global, int j0, int j1, int halo) {
  if (nx < 4 || ny_global < 4 || j0 < 0 || j1 > ny_global || j1 <= j0 || halo < 4) return false;
  if (j0 != 0 && j0 - halo < 0) return false;                 // the slab below must be at least `halo` high
  if (j1 != ny_global && j1 + halo > ny_global) return false;
  return j1 - j0 >= halo;
}

size_t lbm_slab_workspace_bytes(int nx, int ny_global, int j0, int j1, int halo, const lbm_params* p) {
  if (!slab_ok(nx, ny_global, j0, j1, halo)) return 0;
  int yoff, rows;
  slab_extent(ny_global, j0, j1, halo, &yoff, &rows);
  if (!params_ok(nx, rows, p)) return 0;
  return carve(nullptr, nullptr, nx, rows, ny_global, p);
}

int lbm_create_slab(int nx, int ny_global, int j0, int j1, int halo, const lbm_params* p,
                    void* dev_workspace, size_t bytes, void* cuda_stream, lbm_t** out) {
  if (!slab_ok(nx, ny_global, j0, j1, halo))
    return fail(nullptr, LBM_E_ARG, "lbm_create_slab: bad row range or halo (need halo >= 4 and every slab at least halo rows high)");
  int yoff, rows;
  slab_extent(ny_global, j0, j1, halo, &yoff, &rows);
  return create_impl(1, nx, rows, yoff, ny_global, j0, j1, halo, p, dev_workspace, bytes, cuda_stream, out);
}

int lbm_set_temperature(lbm_t* h, const double* T_host) {
  if (!h || !T_host) return h ? fail(h, LBM_E_ARG, "set_temperature: NULL") : LBM_E_ARG;
  if (h->primed) return fail(h, LBM_E_STATE, "set_temperature after the first step");
  DeviceGuard dg(h);
  // B is scratch until the first step writes it
  const size_t n = (size_t)h->nx * h->ny;
  CUDA_OK(h, cudaMemcpyAsync(h->B, T_host, n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
  launch_set_temperature(h, h->B);
  CUDA_OK(h, cudaStreamSynchronize(h->stream));
  CUDA_OK(h, cudaGetLastError());
  return LBM_OK;
}

// circles: minor == theta == NULL; ellipses: full axes diam (the axis at angle theta to x) x minor.
// cos / sin of theta are taken once, here, by the host libm (as the oracle does).
static int add_shapes(lbm_t* h, int n, const double* x, const double* y, const double* diam,
                      const double* minor, const double* theta, const double* rho_ratio,
                      const double* T_w, const double* ux, const double* uy, const double* omega,
                      const unsigned char* fixed) {
  if (!h) return LBM_E_ARG;
  if (n < 0 || (n > 0 && (!x || !y || !diam || !rho_ratio || !T_w)))
    return fail(h, LBM_E_ARG, "add_particles: NULL array or negative count");
  if (h->primed) return fail(h, LBM_E_STATE, "add_particles after the first step");
  DeviceGuard dg(h);
  if (n == 0) return LBM_OK;
  if ((long long)h->np + n > h->P.max_particles)
    return fail(h, LBM_E_CAPACITY, "add_particles: max_particles (%d) exceeded", h->P.max_particles);

  // existing particles (host mirror via a device read; add_particles is a set-up call)
  const int n0 = h->np, nt = n0 + n;
  std::vector<double> X(nt), Y(nt), R(nt), SA(nt), SB(nt), SC(nt), SS(nt);
  if (n0) {
    CUDA_OK(h, cudaMemcpyAsync(SA.data(), h->pa.a, n0 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_OK(h, cudaMemcpyAsync(SB.data(), h->pa.b, n0 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_OK(h, cudaMemcpyAsync(SC.data(), h->pa.cs[h->cur], n0 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_OK(h, cudaMemcpyAsync(SS.data(), h->pa.sn[h->cur], n0 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_OK(h, cudaMemcpyAsync(X.data(), h->pa.x[h->cur], n0 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_OK(h, cudaMemcpyAsync(Y.data(), h->pa.y[h->cur], n0 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_OK(h, cudaMemcpyAsync(R.data(), h->pa.r, n0 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_OK(h, cudaStreamSynchronize(h->stream));
  }
  double dmax = h->d_max;
  for (int k = 0; k < n; ++k) {
    const double sa = 0.5 * diam[k], sb = minor ? 0.5 * minor[k] : sa;
    const double th = theta ? theta[k] : 0.0;
    const bool ell = sa != sb;
    const double r = sa > sb ? sa : sb;   // radius of a circle; largest semi-axis of an ellipse
    if (!(sa > 0.0) || !(sb > 0.0) || !(rho_ratio[k] > 0.0) || !std::isfinite(x[k]) || !std::isfinite(y[k]) ||
        !std::isfinite(r) || !std::isfinite(th) || !std::isfinite(T_w[k]) || (ux && !std::isfinite(ux[k])) ||
        (uy && !std::isfinite(uy[k])) || (omega && !std::isfinite(omega[k])))
      return fail(h, LBM_E_ARG, "add_particles: particle %d has a bad or non-finite value", k);
    const double oc = ell ? std::cos(th) : 1.0, os = ell ? std::sin(th) : 0.0;
    double hx = r, hy = r;                // half extents of the bounding box
    if (ell) {
      const double ac = sa * oc, bs = sb * os, as = sa * os, bc = sb * oc;
      hx = std::sqrt(ac * ac + bs * bs);
      hy = std::sqrt(as * as + bc * bc);
    }
    if (!(y[k] - hy > -0.5) || !(y[k] + hy < h->NY - 0.5))
      return fail(h, LBM_E_ARG, "add_particles: particle %d touches a y wall", k);
    if (!h->P.periodic_x) {
      if (!(x[k] - hx > -0.5) || !(x[k] + hx < h->nx - 0.5))
        return fail(h, LBM_E_ARG, "add_particles: particle %d touches an x wall", k);
    } else if ((int)std::floor(x[k] - r) - 2 < 0 || (int)std::floor(x[k] + r) + 2 > h->nx - 1) {
      return fail(h, LBM_E_ARG, "add_particles: zone of particle %d crosses the periodic seam", k);
    }
    const int Nmax = (int)std::floor(2.0 * r) + 4;   // worst-case N of PAPER.md:258
    if (12 * Nmax - 12 > h->P.max_links_per_particle)
      return fail(h, LBM_E_CAPACITY, "add_particles: 12N-12 = %d exceeds max_links_per_particle = %d",
                  12 * Nmax - 12, h->P.max_links_per_particle);
    X[n0 + k] = x[k];
    Y[n0 + k] = y[k];
    R[n0 + k] = r;
    SA[n0 + k] = sa;
    SB[n0 + k] = sb;
    SC[n0 + k] = oc;
    SS[n0 + k] = os;
    dmax = std::max(dmax, 2.0 * r);
  }
  // overlap test through a host cell grid (cell >= largest diameter): flat cells filled in particle
  // order (counting sort), each new particle tested against the earlier ones in its 3 x 3 cells
  {
    double cell = std::max(dmax, 1.0);
    double xlo = X[0], ylo = Y[0], xhi = X[0], yhi = Y[0];
    for (int k = 1; k < nt; ++k) {
      xlo = std::min(xlo, X[k]); xhi = std::max(xhi, X[k]);
      ylo = std::min(ylo, Y[k]); yhi = std::max(yhi, Y[k]);
    }
    // (a few tiny particles far apart: coarser cells rather than a huge empty grid)
    while ((std::floor((xhi - xlo) / cell) + 1.0) * (std::floor((yhi - ylo) / cell) + 1.0) > 16.0 * nt + 4096.0) cell *= 2.0;
    const int gx = (int)std::floor((xhi - xlo) / cell) + 1, gy = (int)std::floor((yhi - ylo) / cell) + 1;
    std::vector<int> ci(nt), cj(nt), start((size_t)gx * gy + 1, 0), order(nt);
    for (int k = 0; k < nt; ++k) {
      ci[k] = std::min((int)std::floor((X[k] - xlo) / cell), gx - 1);
      cj[k] = std::min((int)std::floor((Y[k] - ylo) / cell), gy - 1);
      start[(size_t)cj[k] * gx + ci[k] + 1]++;
    }
    for (size_t q = 0; q < (size_t)gx * gy; ++q) start[q + 1] += start[q];
    {
      std::vector<int> fill(start.begin(), start.end() - 1);
      for (int k = 0; k < nt; ++k) order[fill[(size_t)cj[k] * gx + ci[k]]++] = k;   // ascending k inside a cell
    }
    // circles: centre distance against r_a + r_b; with an ellipse: the support functions along
    // the line of centres (conservative)
    auto support = [&](int q, double nx, double ny) {
      if (SA[q] == SB[q]) return R[q];
      const double mm = nx * SC[q] + ny * SS[q], ww = ny * SC[q] - nx * SS[q];
      const double am = SA[q] * mm, bw = SB[q] * ww;
      return std::sqrt(am * am + bw * bw);
    };
    for (int k = n0; k < nt; ++k)
      for (int b = std::max(cj[k] - 1, 0); b <= std::min(cj[k] + 1, gy - 1); ++b)
        for (int a = std::max(ci[k] - 1, 0); a <= std::min(ci[k] + 1, gx - 1); ++a)
          for (int q = start[(size_t)b * gx + a]; q < start[(size_t)b * gx + a + 1]; ++q) {
            const int m = order[q];
            if (m >= k) break;                             // (a new particle is tested against the earlier ones)
            const double dx = X[k] - X[m], dy = Y[k] - Y[m];
            const double dist = std::sqrt(dx * dx + dy * dy);
            bool bad;
            if (SA[k] == SB[k] && SA[m] == SB[m]) bad = dist < R[k] + R[m];
            else bad = !(dist > 0.0) || dist < support(k, dx / dist, dy / dist) + support(m, dx / dist, dy / dist);
            if (bad) return fail(h, LBM_E_ARG, "add_particles: particles %d and %d overlap", m, k);
          }
  }
  // upload
  const int c = h->cur;
  std::vector<double> zero(n, 0.0), rr(n);
  for (int k = 0; k < n; ++k) rr[k] = R[n0 + k];
  std::vector<unsigned char> fx(n, 0);
  if (fixed)
    for (int k = 0; k < n; ++k) fx[k] = fixed[k] ? 1 : 0;
  auto up = [&](double* dst, const double* src) {
    return cudaMemcpyAsync(dst + n0, src ? src : zero.data(), n * sizeof(double), cudaMemcpyHostToDevice, h->stream);
  };
  for (int b = 0; b < 2; ++b) {
    CUDA_OK(h, up(h->pa.x[b], x));
    CUDA_OK(h, up(h->pa.y[b], y));
    CUDA_OK(h, up(h->pa.theta[b], theta));
    CUDA_OK(h, up(h->pa.cs[b], SC.data() + n0));
    CUDA_OK(h, up(h->pa.sn[b], SS.data() + n0));
    CUDA_OK(h, up(h->pa.ux[b], ux));
    CUDA_OK(h, up(h->pa.uy[b], uy));
    CUDA_OK(h, up(h->pa.omega[b], omega));
  }
  CUDA_OK(h, up(h->pa.r, rr.data()));
  CUDA_OK(h, up(h->pa.a, SA.data() + n0));
  CUDA_OK(h, up(h->pa.b, SB.data() + n0));
  CUDA_OK(h, up(h->pa.rho_ratio, rho_ratio));
  CUDA_OK(h, up(h->pa.Tw, T_w));
  CUDA_OK(h, up(h->pa.Fx, nullptr));
  CUDA_OK(h, up(h->pa.Fy, nullptr));
  CUDA_OK(h, up(h->pa.Tz, nullptr));
  CUDA_OK(h, cudaMemcpyAsync(h->pa.fixed + n0, fx.data(), n, cudaMemcpyHostToDevice, h->stream));
  CUDA_OK(h, cudaMemsetAsync(h->pa.ovl + n0, 0, n, h->stream));
  // y-slab: a particle whose centre lies in the own rows must be inside the stored rows together
  // with its link stencils (2 rows) and the refill stencils of its newborn nodes (4 rows + the
  // parked values those pull: 2 more), for as long as it is owned: r + 8 rows
  if (h->is_slab && 0.5 * dmax + 8.0 > (double)h->halo)
    return fail(h, LBM_E_ARG, "add_particles: halo of %d rows is too narrow for particles of diameter %.1f (need d/2 + 8)",
                h->halo, dmax);
  h->np = nt;
  for (int k = n0; k < nt; ++k) h->n_ell += (SA[k] != SB[k]) ? 1 : 0;
  h->d_max = dmax;
  size_chain(h);
  h->cell = std::max(dmax + h->P.rep_s, MIN_CELL);
  h->ncx = (int)std::ceil(h->nx / h->cell) + 1;
  h->ncy = (int)std::ceil(h->NY / h->cell) + 1;
  if ((long long)h->ncx * h->ncy > h->max_cells)
    return fail(h, LBM_E_CAPACITY, "add_particles: repulsion grid larger than the workspace allows");
  // flag and owner maps and the repulsion grid of step 0 (primed == 0: every particle, full sweep)
  CUDA_OK(h, cudaMemsetAsync(h->cell_count[c], 0, sizeof(int) * (size_t)h->max_cells, h->stream));
  launch_cover(h, c, h->stream, false);
  h->links_ready = 0;
  CUDA_OK(h, cudaStreamSynchronize(h->stream));
  CUDA_OK(h, cudaGetLastError());
  return LBM_OK;
}

int lbm_add_particles(lbm_t* h, int n, const double* x, const double* y, const double* diam,
                      const double* rho_ratio, const double* T_w, const double* ux,
                      const double* uy, const double* omega, const unsigned char* fixed) {
  return add_shapes(h, n, x, y, diam, nullptr, nullptr, rho_ratio, T_w, ux, uy, omega, fixed);
}

int lbm_add_ellipses(lbm_t* h, int n, const double* x, const double* y, const double* major,
                     const double* minor, const double* theta, const double* rho_ratio,
                     const double* T_w, const double* ux, const double* uy, const double* omega,
                     const unsigned char* fixed) {
  if (h && n > 0 && (!minor || !theta)) return fail(h, LBM_E_ARG, "add_ellipses: NULL array");
  return add_shapes(h, n, x, y, major, minor, theta, rho_ratio, T_w, ux, uy, omega, fixed);
}

// While a graph is being captured: remember the node the last launch on a chain stream became
// (the stream's only capture dependency), so that it can be given the chain's priority afterwards.
static void note_chain_node(lbm* h, cudaStream_t S1) {
  if (!h->cap_nodes) return;
  cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
  const cudaGraphNode_t* deps = nullptr;
  size_t ndeps = 0;
  if (cudaStreamGetCaptureInfo(S1, &st, nullptr, nullptr, &deps, &ndeps) == cudaSuccess &&
      st == cudaStreamCaptureStatusActive && ndeps == 1)
    static_cast<std::vector<cudaGraphNode_t>*>(h->cap_nodes)->push_back(deps[0]);
}

// Step schedule: the resident state A is f+(x,t), g+(x,t), the index array holds
// the links of x_p(t).  Three streams, S0 = the caller's (or the capturing) stream:
//   S1: bounce-back + momentum exchange (parks f_ibar(x_f,t+1) in solid slots of A, sums F, T_z)
//   S0:   after it: fused pull-stream-collide A -> B over every node fluid at t
//   S1: integrate + uncover -> cover -> links of x_p(t+1)        } concurrent with the
//   S2:                        after cover: refill (A -> stash)   } lattice kernel
//   S1: after the lattice kernel and the refill: refill commit (stash -> B, newborn flags cleared)
// S1 is one dependent chain from step to step (the next bounce-back follows the commit), each link
// a programmatic dependent launch.  The caller's stream is joined to it at both ends of a call.
// Enqueues ONE time step (the streams may be capturing) and flips the host-side phase (A/B, cur).
//
// Banded schedule (phase = 0..3, the position of the step in a period of four; phase = -1: the
// plain step above).  At the start of a period (every row in A at the same time t) k_band_plan
// picks Q from the particle positions; for the four steps the rows [0, Q) belong to the two-step
// kernel: with X, Y = A, B at the start of the period,
//   steps 0, 1: band X -> Y (t -> t+2);  rows >= Q: X -> Y -> X as always
//   steps 2, 3: band Y -> X (t+2 -> t+4); rows >= Q: X -> Y -> X
// The band's tile rows of a pair are dealt to its two steps and launched on S0 BEFORE the wait for
// the bounce-back kernel: they fill the time in which that latency-bound kernel leaves the
// memory system idle.  The one-step kernel of the first step of a pair also updates row Q-1 (into
// the spare row of its output copy), which the second step reads there; the band's part of a pair
// is complete before the second step's one-step kernel overwrites the rows Q, Q+1 of X it reads.
static void enqueue_step(lbm* h, int phase, bool plan = true) {
  cudaStream_t S0 = h->stream, S1 = h->chain, S2 = h->side;
  const bool fork = S1 != S0;
  const bool pdl = h->use_pdl != 0;
  const bool banded = phase >= 0;
  h->band_live = banded ? 1 : 0;
  const int sp = h->cur;   // step parity: which newborn counter / repulsion grid this step uses
  double* X = (phase & 1) ? h->B : h->A;   // the copies as they were named at the start of the period
  double* Y = (phase & 1) ? h->A : h->B;
  // h->band3: periods of SIX steps, the band advancing three steps per pass (phases 0-2: X -> Y,
  // 3-5: Y -> X); the band and the rows above it are then in the same copy at the start of every
  // half period, so the band kernel needs no second source and the one-step kernel never computes
  // a band row: it reads row Q-1 in place in the first step of a half period and from the spare
  // row, where the band kernel's top tiles put it, in the other two
  const int half = h->band3 ? 3 : 2;
  double* band_src = phase < half ? X : Y;
  double* band_dst = phase < half ? Y : X;
  if (banded && phase == 0 && plan) {   // one plan serves two periods (k_band_plan allows for 8 steps of motion)
    { Timed tm(h, K_BAND_PLAN, S1); launch_band_plan(h, S1); }
    note_chain_node(h, S1);
    if (fork) {
      cudaEventRecord(h->ev_plan, S1);
      cudaStreamWaitEvent(S0, h->ev_plan, 0);
    }
  }
  if (h->np > 0) {
    { Timed tm(h, K_BOUNCE_BACK, S1); launch_bounce_back(h, S1, pdl); }
    note_chain_node(h, S1);
    if (fork) cudaEventRecord(h->ev_bb, S1);
  }
  if (banded) {
    if (h->band3) {
      Timed tm(h, K_STREAM_COLLIDE_3STEP, S0);
      launch_stream_collide_band3(h, band_src, band_dst, 3, phase % 3);
    } else {
      Timed tm(h, K_STREAM_COLLIDE_2STEP, S0);
      launch_stream_collide_band(h, band_src, X, band_dst, 2, phase & 1);
    }
    // the particle chain holds register space the band kernel's large CTAs need (measured: the band
    // part takes 115 us beside the bounce-back kernel alone, 190 us beside the chain): the chain
    // starts after the band's part and still has the whole one-step kernel to hide under
    if (fork) {
      cudaEventRecord(h->ev_p2, S0);
      cudaStreamWaitEvent(S1, h->ev_p2, 0);
    }
  }
  if (h->np > 0 && fork) cudaStreamWaitEvent(S0, h->ev_bb, 0);
  const int lattice_mode = !banded ? 0 : (h->band3 ? (phase % 3 == 0 ? 3 : 2) : ((phase & 1) ? 2 : 1));
  if (fork || h->np == 0) {
    Timed tm(h, K_STREAM_COLLIDE, S0);
    launch_stream_collide(h, lattice_mode, band_src);
  }
  if (h->np > 0) {
    if (fork) cudaEventRecord(h->ev_sc, S0);
    { Timed tm(h, K_MOVE, S1); launch_move(h, S1, pdl); }
    note_chain_node(h, S1);
    { Timed tm(h, K_COVER, S1); launch_cover(h, sp ^ 1, S1, pdl); }
    note_chain_node(h, S1);
    if (fork) {
      cudaEventRecord(h->ev_cov, S1);
      cudaStreamWaitEvent(S2, h->ev_cov, 0);
    }
    { Timed tm(h, K_REFILL, S2); launch_refill(h, S2); }
    note_chain_node(h, S2);
    if (fork) cudaEventRecord(h->ev_ref, S2);
    { Timed tm(h, K_BUILD_LINKS, S1); launch_build_links(h, sp ^ 1, S1, pdl && fork); }
    note_chain_node(h, S1);
    h->cur ^= 1;
    if (fork) {
      cudaStreamWaitEvent(S1, h->ev_sc, 0);
      cudaStreamWaitEvent(S1, h->ev_ref, 0);
    } else {
      Timed tm(h, K_STREAM_COLLIDE, S0);
      launch_stream_collide(h, lattice_mode, band_src);
    }
    { Timed tm(h, K_REFILL_COMMIT, S1); launch_refill_commit(h, sp, S1, pdl); }
    note_chain_node(h, S1);
  }
  std::swap(h->A, h->B);
}

// Both ends of a run of steps: the chain stream starts after everything already on the caller's
// stream, and the caller's stream continues after the last refill commit.
static void join_in(lbm* h) {
  if (h->np == 0 || h->chain == h->stream) return;
  cudaEventRecord(h->ev_in, h->stream);
  cudaStreamWaitEvent(h->chain, h->ev_in, 0);
}
static void join_out(lbm* h) {
  if (h->np == 0 || h->chain == h->stream) return;
  cudaEventRecord(h->ev_out, h->chain);
  cudaStreamWaitEvent(h->stream, h->ev_out, 0);
}

static void drop_graphs(lbm* h) {
  for (int k = 0; k < h->n_graphs; ++k) cudaGraphExecDestroy(h->graphs[k].exec);
  h->n_graphs = 0;
}

// The graph of `steps` (even) time steps starting in the handle's current phase: looked up, or
// captured now.  Capture runs on the library's own stream pair (the caller's stream may be the
// legacy default stream, which cannot capture); the fork / join events turn into graph edges.
// Returns nullptr if capture is not possible (the caller then launches directly).
static lbm::StepGraph* step_graph(lbm* h, int steps, int banded) {
  for (int k = 0; k < h->n_graphs; ++k) {
    lbm::StepGraph& g = h->graphs[k];
    if (g.A == h->A && g.cur == h->cur && g.steps == steps && g.overlap == h->overlap &&
        g.chain_ctas == h->chain_ctas && g.banded == banded &&
        (!banded || (g.band_hint == h->band_hint && g.band_cap == h->band_cap && g.band_orient == h->band_orient)))
      return &g;
  }
  if (h->n_graphs == LBM_MAX_GRAPHS) drop_graphs(h);
  cudaStream_t user = h->stream, chain = h->chain;
  double *A0 = h->A, *B0 = h->B;
  const int cur0 = h->cur;
  const long long l0 = h->launches;
  cudaStream_t side = h->side;
  h->stream = h->cap_stream;
  if (chain == user) h->chain = h->side = h->cap_stream;
  cudaGraph_t graph = nullptr;
  std::vector<cudaGraphNode_t> chain_nodes;
  cudaError_t e = cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeRelaxed);
  if (e == cudaSuccess) {
    if (h->chain != h->stream) h->cap_nodes = &chain_nodes;
    join_in(h);
    h->band3 = banded == 3 ? 1 : 0;   // (the unit's schedule: plan margins, band kernel, cover's safety net)
    for (int s = 0; s < steps; ++s) enqueue_step(h, banded ? s % (h->band3 ? 6 : 4) : -1, s == 0);
    join_out(h);
    h->cap_nodes = nullptr;
    e = cudaStreamEndCapture(h->cap_stream, &graph);
  }
  // The chain's kernel nodes get the chain stream's priority explicitly: without it the chain
  // would start in the lattice kernel's tail.
  if (e == cudaSuccess)
    for (cudaGraphNode_t nd : chain_nodes) {
      cudaGraphNodeType ty;
      if (cudaGraphNodeGetType(nd, &ty) != cudaSuccess || ty != cudaGraphNodeTypeKernel) continue;
      cudaLaunchAttributeValue v;
      std::memset(&v, 0, sizeof v);
      v.priority = h->chain_priority;
      cudaGraphKernelNodeSetAttribute(nd, cudaLaunchAttributePriority, &v);
    }
  cudaGetLastError();
  const long long per = h->launches - l0;
  h->launches = l0;
  h->stream = user;
  h->chain = chain;
  h->side = side;
  h->A = A0;
  h->B = B0;
  h->cur = cur0;
  cudaGraphExec_t exec = nullptr;
  // per-node priorities are honoured only on request (otherwise every node runs at the priority
  // of the stream the graph is launched into)
  if (e == cudaSuccess) e = cudaGraphInstantiateWithFlags(&exec, graph, cudaGraphInstantiateFlagUseNodePriority);
  if (graph) cudaGraphDestroy(graph);
  if (e != cudaSuccess) {
    cudaGetLastError();
    h->use_graph = 0;   // not available here: direct launches from now on
    return nullptr;
  }
  lbm::StepGraph& g = h->graphs[h->n_graphs++];
  g.exec = exec;
  g.A = h->A;
  g.cur = h->cur;
  g.steps = steps;
  g.overlap = h->overlap;
  g.chain_ctas = h->chain_ctas;
  g.banded = banded;
  g.band_hint = h->band_hint;
  g.band_cap = h->band_cap;
  g.band_orient = h->band_orient;
  g.launches = per;
  return &g;
}

// The banded schedule needs the particle-free two-step kernel, runs in periods of four steps and
// is worth one extra synchronisation per call only for calls of some length: the band is planned
// once at the start of a call, on the caller's stream, so that the host can size the grids -- the
// one-step kernel gets one CTA row per lattice row above (the planned band less a margin, in steps
// of 64 rows), the band kernel's grid covers (the planned band plus a margin, in steps of 16 rows);
// each pair of values is its own graph.  The per-period plans on the device stay below the cap; a
// band that shrinks faster than the margin is caught by the one-step kernel's row loop.
static int plan_call(lbm* h, int nsteps, bool* band_ok_out) {
  bool band_ok = h->np > 0 && h->band_on && h->two_step_ok && nsteps >= LBM_BAND_MIN_STEPS;
  h->band3 = h->want3 = 0;
  if (band_ok) {
    h->band_cap = h->ny;
    h->band_orient = 0;                // under or above the suspension: whichever band is larger
    h->band3 = h->want3 = h->band_steps >= 3 ? 1 : 0;   // (the call-start plan then takes the wider margins)
    launch_band_plan(h, h->stream);
    CUDA_OK(h, cudaMemcpyAsync(h->status_host + 1, h->band, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CUDA_OK(h, cudaStreamSynchronize(h->stream));
    const int q0 = h->status_host[1];                         // > 0: rows [0, q0); < 0: rows [-q0, ny)
    const int rows0 = q0 > 0 ? q0 : (q0 < 0 ? h->ny + q0 : 0);  // rows of the band
    // a band of less than 2^18 nodes costs more in launches than it saves in traffic (config 0)
    if (rows0 <= 0 || (h->band_on < 2 && (long long)rows0 * h->nx < LBM_BAND_MIN_NODES)) band_ok = false;
    else {
      h->band_orient = q0 > 0 ? 1 : -1;                       // fixed for this call: the grids are sized for it
      h->band_hint = std::max(0, ((rows0 - 96) / 64) * 64);   // (32 / 96 / 160 rows of margin: the same step time)
      h->band_l1_rows = h->ny - h->band_hint;                 // the rows outside the band, with that margin
      h->band_cap = std::min(h->ny, ((rows0 + 8 + 15) / 16) * 16);
    }
  }
  if (!band_ok) h->band3 = h->want3 = 0;
  *band_ok_out = band_ok;
  return LBM_OK;
}

// how many steps the next graph launch of a call with `left` steps to go covers, and in which schedule
// With the three-step band (h->want3) a period is six steps -- units of 12 and 6, `banded` = 3 --
// and a remainder of four is a period of the two-step band (`banded` = 1): every even number of
// steps >= 4 is a sum of sixes and fours, so only a unit that would leave exactly two steps is
// passed over (20 = 12 + 4 + 4, 14 = 6 + 4 + 4).
static int graph_unit(const lbm* h, int left, bool band_ok, int* banded) {
  if (band_ok && h->want3) {
    const int even = left & ~1;
    if (even >= 12 && even - 12 != 2) { *banded = 3; return 12; }
    if (even >= 6 && even - 6 != 2) { *banded = 3; return 6; }
    if (even >= 4) { *banded = 1; return 4; }
    *banded = 0;
    return 2;
  }
  *banded = (band_ok && left >= 4) ? 1 : 0;
  return left >= LBM_GRAPH_STEPS ? LBM_GRAPH_STEPS : (*banded ? 4 : 2);
}

int lbm_prepare(lbm_t* h, int nsteps) {
  if (!h) return LBM_E_ARG;
  if (nsteps < 0) return fail(h, LBM_E_ARG, "lbm_prepare: negative step count");
  if (h->is_slab) return fail(h, LBM_E_STATE, "lbm_prepare: not for slab handles");
  DeviceGuard dg(h);
  if (nsteps == 0) return LBM_OK;
  prime(h);
  ensure_links(h);
  bool band_ok = false;
  int rc = plan_call(h, nsteps, &band_ok);
  if (rc) return rc;
  if (h->np > 0 && h->use_graph && !h->prof_on) {
    // every unit of a call is an even number of steps, so all of them start in the current phase
    for (int s = 0; nsteps - s >= 2;) {
      int banded = 0;
      const int unit = graph_unit(h, nsteps - s, band_ok, &banded);
      lbm::StepGraph* g = step_graph(h, unit, banded);
      if (!g) break;
      cudaGraphUpload(g->exec, h->stream);
      s += unit;
    }
  }
  return check_status(h);
}

int lbm_step(lbm_t* h, int nsteps) {
  if (!h) return LBM_E_ARG;
  if (nsteps < 0) return fail(h, LBM_E_ARG, "lbm_step: negative step count");
  if (h->is_slab && nsteps > 0)
    return fail(h, LBM_E_STATE, "lbm_step on a slab: use lbm_slab_forces / lbm_slab_advance and the exchanges between them");
  DeviceGuard dg(h);
  if (nsteps > 0) {
    prime(h);
    ensure_links(h);
  }
  int s = 0;
  bool band_ok = false;
  {
    const int rc = plan_call(h, nsteps, &band_ok);
    if (rc) return rc;
  }
  // lattices with particles: whole periods of the schedule as CUDA graph replays (8 steps per
  // launch while that many remain, then 4 if banded, then 2), the odd last step directly; event
  // profiling needs the direct launches
  if (h->np > 0 && h->use_graph && !h->prof_on) {
    while (nsteps - s >= 2) {
      int banded = 0;
      const int unit = graph_unit(h, nsteps - s, band_ok, &banded);
      lbm::StepGraph* g = step_graph(h, unit, banded);
      if (!g) break;
      CUDA_OK(h, cudaGraphLaunch(g->exec, h->stream));
      h->launches += g->launches;
      h->steps_done += unit;
      s += unit;
    }
  }
  if (s < nsteps) join_in(h);
  const bool direct = s < nsteps;
  while (s < nsteps) {
    if (h->np == 0 && h->two_step >= 2 && nsteps - s >= 3) {
      // particle-free lattice: three time steps per pass
      if (h->use_tma && h->tma_ok) {
        Timed tm(h, K_STREAM_COLLIDE_3STEP_TMA, h->stream);
        launch_stream_collide_3step_tma(h);
      } else {
        Timed tm(h, K_STREAM_COLLIDE_3STEP, h->stream);
        launch_stream_collide_3step(h);
      }
      std::swap(h->A, h->B);
      h->steps_done += 3;
      s += 3;
      continue;
    }
    if (h->np == 0 && h->two_step && nsteps - s >= 2) {
      // particle-free lattice: two time steps per pass over the populations (A -> B)
      { Timed tm(h, K_STREAM_COLLIDE_2STEP, h->stream); launch_stream_collide_2step(h); }
      std::swap(h->A, h->B);
      h->steps_done += 2;
      s += 2;
      continue;
    }
    if (band_ok && nsteps - s >= 4) {
      // direct launches of the unit a graph would replay (same steps, same plans, same kernels)
      int banded = 0;
      const int unit = graph_unit(h, nsteps - s, band_ok, &banded);
      if (banded) {
        h->band3 = banded == 3 ? 1 : 0;
        for (int k = 0; k < unit; ++k) enqueue_step(h, k % (h->band3 ? 6 : 4), k == 0);
        h->steps_done += unit;
        s += unit;
        continue;
      }
    }
    enqueue_step(h, -1);
    h->steps_done++;
    ++s;
  }
  if (direct) join_out(h);
  return check_status(h);
}

int lbm_set_band(lbm_t* h, int on) {
  if (!h) return LBM_E_ARG;
  h->band_on = (on && h->ev_p2 && !h->is_slab) ? (on >= 2 ? 2 : 1) : 0;
  return LBM_OK;
}

int lbm_get_band(lbm_t* h, int* rows) {
  if (!h || !rows) return LBM_E_ARG;
  *rows = (h->np > 0 && h->band_on && h->two_step_ok) ? h->status_host[1] : 0;   // signed, see lbm.h
  return LBM_OK;
}

// ---- y-slabs: one time step in two halves, the two exchanges between them left to the caller ----
// copies `rows` rows of all 14 populations: (src copy, local row sr) -> (dst copy, local row dr);
// the planes are row-major with the same pitch in every slab of a decomposition, so a block of
// rows is one contiguous piece per plane.  buf != nullptr: to / from a packed buffer instead.
static int copy_rows(lbm* hd, double* dstA, int dr, const lbm* hs, const double* srcA, int sr, int rows,
                     double* pack_to, const double* unpack_from, cudaStream_t st) {
  const size_t px = (size_t)hs->px;
  size_t off = 0;
  for (int k = 0; k < 9; ++k) {
    const bool pair = k < 5;
    const size_t cnt = (pair ? 2 : 1) * px * rows;
    const size_t ps_s = (size_t)hs->ps, ps_d = hd ? (size_t)hd->ps : 0;
    const double* src = unpack_from ? unpack_from + off
                                    : srcA + (pair ? 2 * k * ps_s + 2 * px * sr : (k + 5) * ps_s + px * sr);
    double* dst = pack_to ? pack_to + off
                          : dstA + (pair ? 2 * k * ps_d + 2 * px * dr : (k + 5) * ps_d + px * dr);
    cudaError_t e;
    if (hd && hs && hd->device != hs->device && !pack_to && !unpack_from)
      e = cudaMemcpyPeerAsync(dst, hd->device, src, hs->device, cnt * sizeof(double), st);
    else
      e = cudaMemcpyAsync(dst, src, cnt * sizeof(double), cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return -1;
    off += cnt;
  }
  return 0;
}

int lbm_slab_halo_doubles(const lbm_t* h, long long* doubles) {
  if (!h || !doubles) return LBM_E_ARG;
  *doubles = 14LL * h->halo * h->px;
  return LBM_OK;
}

int lbm_slab_forces(lbm_t* h) {
  if (!h) return LBM_E_ARG;
  if (!h->is_slab) return fail(h, LBM_E_STATE, "lbm_slab_forces: not a slab handle");
  DeviceGuard dg(h);
  prime(h);
  ensure_links(h);
  launch_bounce_back(h, h->stream, false);
  launch_slab_forces_out(h);
  return LBM_OK;
}

int lbm_slab_force_buffer(lbm_t* h, double** dev_buf, int* count) {
  if (!h || !dev_buf || !count) return LBM_E_ARG;
  *dev_buf = h->force_buf;
  *count = 3 * h->np;
  return LBM_OK;
}

// Where the rows next to this slab's cuts go in the neighbours' copies of the state being written.
// All slabs of a decomposition step in lockstep and swap their A / B in every advance: a neighbour
// that has already advanced this step holds the new state in its A, one that has not will write it
// to its B.
static HaloPush halo_push(const lbm* h) {
  HaloPush hp = {nullptr, 0, 0, 0, 0, nullptr, 0, 0, 0, 0};
  if (const lbm* p = h->peer_lo) {
    hp.lo = p->steps_done > h->steps_done ? p->A : p->B;
    hp.lo_ps = p->ps;
    hp.lo_shift = h->yoff - p->yoff;            // (global row) - p->yoff = local row + this
    hp.lo_start = h->row0;
    hp.lo_end = h->row0 + h->halo;
  }
  if (const lbm* p = h->peer_hi) {
    hp.hi = p->steps_done > h->steps_done ? p->A : p->B;
    hp.hi_ps = p->ps;
    hp.hi_shift = h->yoff - p->yoff;
    hp.hi_start = h->row1 - h->halo;
    hp.hi_end = h->row1;
  }
  return hp;
}

int lbm_slab_advance(lbm_t* h) {
  if (!h) return LBM_E_ARG;
  if (!h->is_slab) return fail(h, LBM_E_STATE, "lbm_slab_advance: not a slab handle");
  if (!h->primed) return fail(h, LBM_E_STATE, "lbm_slab_advance before lbm_slab_forces");
  DeviceGuard dg(h);
  cudaStream_t S = h->stream;
  const int sp = h->cur;
  h->band_live = 0;
  if (h->np > 0) {
    launch_slab_forces_in(h);
    launch_move(h, S, false);
    launch_cover(h, sp ^ 1, S, false);
    launch_refill(h, S);
    launch_build_links(h, sp ^ 1, S, false);
    h->cur ^= 1;
  }
  // the slab's own rows; with linked peers (lbm_slab_link_peers) the rows next to the cuts are
  // written into the neighbours' ghost rows by the same kernel, and so are the refilled nodes
  const HaloPush hp = halo_push(h);
  launch_stream_collide_slab(h, hp);
  if (h->np > 0) launch_refill_commit(h, sp, S, false, &hp);
  std::swap(h->A, h->B);
  h->steps_done++;
  return LBM_OK;
}

// Slabs of ONE process, ascending row ranges: from now on lbm_slab_advance pushes the halo rows
// straight into the neighbours' ghost rows (peer access is enabled between devices), and
// lbm_slab_fence replaces lbm_slab_exchange_halos.  Every slab must be advanced in every step.
int lbm_slab_link_peers(lbm_t** hs, int n) {
  if (!hs || n < 1) return LBM_E_ARG;
  for (int s = 0; s < n; ++s) {
    if (!hs[s] || !hs[s]->is_slab) return LBM_E_ARG;
    if (s + 1 < n && (hs[s]->own1 != hs[s + 1]->own0 || hs[s]->halo != hs[s + 1]->halo || hs[s]->px != hs[s + 1]->px))
      return fail(hs[s], LBM_E_ARG, "lbm_slab_link_peers: slabs %d and %d do not adjoin", s, s + 1);
  }
  for (int s = 0; s < n; ++s) {
    hs[s]->peer_lo = s > 0 ? hs[s - 1] : nullptr;
    hs[s]->peer_hi = s + 1 < n ? hs[s + 1] : nullptr;
    for (lbm* p : {hs[s]->peer_lo, hs[s]->peer_hi})
      if (p && p->device != hs[s]->device) {
        DeviceGuard dg(hs[s]);
        cudaError_t e = cudaDeviceEnablePeerAccess(p->device, 0);
        if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled)
          return fail(hs[s], LBM_E_CUDA, "lbm_slab_link_peers: no peer access from device %d to %d", hs[s]->device, p->device);
        cudaGetLastError();
      }
  }
  return LBM_OK;
}

// end of a step with linked peers: every slab's kernels (and with them the pushes into its
// neighbours) have completed before anyone starts the next step
int lbm_slab_fence(lbm_t** hs, int n) {
  if (!hs || n < 1) return LBM_E_ARG;
  for (int s = 0; s < n; ++s) {
    if (!hs[s]) return LBM_E_ARG;
    DeviceGuard dg(hs[s]);
    CUDA_OK(hs[s], cudaStreamSynchronize(hs[s]->stream));
  }
  return LBM_OK;
}

int lbm_slab_check(lbm_t* h) {
  if (!h) return LBM_E_ARG;
  DeviceGuard dg(h);
  return check_status(h);
}

// side 0: the slab's lowest `halo` own rows (what the slab below needs), 1: its highest
int lbm_slab_pack(lbm_t* h, int side, double* dev_buf) {
  if (!h || !dev_buf || (side != 0 && side != 1)) return LBM_E_ARG;
  if (!h->is_slab) return fail(h, LBM_E_STATE, "lbm_slab_pack: not a slab handle");
  DeviceGuard dg(h);
  const int sr = side == 0 ? h->row0 : h->row1 - h->halo;
  if (copy_rows(nullptr, nullptr, 0, h, h->A, sr, h->halo, dev_buf, nullptr, h->stream))
    return fail(h, LBM_E_CUDA, "lbm_slab_pack: copy failed");
  return LBM_OK;
}

// side 0: into the ghost rows below the own rows, 1: above
int lbm_slab_unpack(lbm_t* h, int side, const double* dev_buf) {
  if (!h || !dev_buf || (side != 0 && side != 1)) return LBM_E_ARG;
  if (!h->is_slab) return fail(h, LBM_E_STATE, "lbm_slab_unpack: not a slab handle");
  if ((side == 0 && h->row0 == 0) || (side == 1 && h->row1 == h->ny))
    return fail(h, LBM_E_ARG, "lbm_slab_unpack: no ghost rows on that side (cavity wall)");
  DeviceGuard dg(h);
  const int dr = side == 0 ? h->row0 - h->halo : h->row1;
  if (copy_rows(h, h->A, dr, h, nullptr, 0, h->halo, nullptr, dev_buf, h->stream))
    return fail(h, LBM_E_CUDA, "lbm_slab_unpack: copy failed");
  return LBM_OK;
}

// Both exchanges for slabs that live in ONE process (ascending row ranges, e.g. the GPUs of one
// node driven by one process, or several slabs on one GPU in the tests): the halo rows go straight
// from copy to copy (peer copies between devices); the force buffers are added in ascending slab
// order -- each entry is non-zero in exactly one slab, so the sum is that slab's value exactly.
int lbm_slab_exchange_halos(lbm_t** hs, int n) {
  if (!hs || n < 1) return LBM_E_ARG;
  for (int s = 0; s < n; ++s) {
    if (!hs[s] || !hs[s]->is_slab) return LBM_E_ARG;
    CUDA_OK(hs[s], cudaStreamSynchronize(hs[s]->stream));   // every slab's step has completed
  }
  for (int s = 0; s + 1 < n; ++s) {
    lbm *lo = hs[s], *up = hs[s + 1];
    if (lo->own1 != up->own0 || lo->halo != up->halo || lo->px != up->px)
      return fail(lo, LBM_E_ARG, "lbm_slab_exchange_halos: slabs %d and %d do not adjoin", s, s + 1);
    // the lower slab's highest own rows -> the upper slab's ghost rows below, and back
    if (copy_rows(up, up->A, up->row0 - up->halo, lo, lo->A, lo->row1 - lo->halo, lo->halo, nullptr, nullptr, up->stream) ||
        copy_rows(lo, lo->A, lo->row1, up, up->A, up->row0, up->halo, nullptr, nullptr, lo->stream))
      return fail(lo, LBM_E_CUDA, "lbm_slab_exchange_halos: copy failed");
  }
  for (int s = 0; s < n; ++s) CUDA_OK(hs[s], cudaStreamSynchronize(hs[s]->stream));
  return LBM_OK;
}

int lbm_slab_combine_forces(lbm_t** hs, int n) {
  if (!hs || n < 1 || !hs[0]) return LBM_E_ARG;
  const int cnt = 3 * hs[0]->np;
  if (cnt == 0) return LBM_OK;
  for (int s = 0; s < n; ++s) {
    if (!hs[s] || !hs[s]->is_slab || hs[s]->np != hs[0]->np) return LBM_E_ARG;
    DeviceGuard dg(hs[s]);
    CUDA_OK(hs[s], cudaStreamSynchronize(hs[s]->stream));
  }
  // summed on the first slab's device, in ascending slab order; buffers on other devices are read
  // and written through peer access
  DeviceGuard dg(hs[0]);
  cudaStream_t S = hs[0]->stream;
  for (int s = 1; s < n; ++s) {
    if (hs[s]->device != hs[0]->device) {
      cudaError_t e = cudaDeviceEnablePeerAccess(hs[s]->device, 0);
      if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled)
        return fail(hs[0], LBM_E_CUDA, "lbm_slab_combine_forces: no peer access from device %d to %d",
                    hs[0]->device, hs[s]->device);
      cudaGetLastError();
    }
    launch_add_buffer(hs[0]->force_buf, hs[s]->force_buf, cnt, S);
  }
  for (int s = 1; s < n; ++s) {
    if (hs[s]->device != hs[0]->device)
      CUDA_OK(hs[0], cudaMemcpyPeerAsync(hs[s]->force_buf, hs[s]->device, hs[0]->force_buf, hs[0]->device,
                                         cnt * sizeof(double), S));
    else
      CUDA_OK(hs[0], cudaMemcpyAsync(hs[s]->force_buf, hs[0]->force_buf, cnt * sizeof(double),
                                     cudaMemcpyDeviceToDevice, S));
  }
  CUDA_OK(hs[0], cudaStreamSynchronize(S));
  return LBM_OK;
}

int lbm_set_graph(lbm_t* h, int on) {
  if (!h) return LBM_E_ARG;
  h->use_graph = (on && h->cap_stream) ? 1 : 0;
  return LBM_OK;
}

int lbm_set_two_step(lbm_t* h, int on) {
  if (!h) return LBM_E_ARG;
  h->two_step = (on && h->two_step_ok) ? (on >= 3 ? 2 : 1) : 0;   // on: steps per pass (1 = 2: two)
  return LBM_OK;
}

int lbm_set_band_steps(lbm_t* h, int steps) {
  if (!h) return LBM_E_ARG;
  if (steps != 2 && steps != 3) return fail(h, LBM_E_ARG, "lbm_set_band_steps: 2 or 3");
  h->band_steps = steps;
  return LBM_OK;
}

int lbm_set_tma(lbm_t* h, int on) {
  if (!h) return LBM_E_ARG;
  if (on && !h->tma_ok) return fail(h, LBM_E_STATE, "lbm_set_tma: no tensor maps for this handle (periodic x, a slab, or the driver lacks cuTensorMapEncodeTiled)");
  h->use_tma = on ? (on >= 2 ? 2 : 1) : 0;
  return LBM_OK;
}

int lbm_set_overlap(lbm_t* h, int on) {
  if (!h) return LBM_E_ARG;
  DeviceGuard dg(h);
  cudaStreamSynchronize(h->stream);
  if (h->chain_own) cudaStreamSynchronize(h->chain_own);
  if (h->side_own) cudaStreamSynchronize(h->side_own);
  h->overlap = (on && h->chain_own) ? 1 : 0;
  h->chain = h->overlap ? h->chain_own : h->stream;
  h->side = h->overlap ? h->side_own : h->stream;
  return LBM_OK;
}

int lbm_get_fields(lbm_t* h, double* rho, double* ux, double* uy, double* T, double* f, double* g,
                   unsigned char* flag) {
  if (!h) return LBM_E_ARG;
  DeviceGuard dg(h);
  // a slab hands out its OWN rows only (nx * (j1 - j0) values per field, global row j0 first)
  const size_t n = (size_t)h->nx * h->ny;                 // nodes stored
  const size_t m = (size_t)h->nx * (h->row1 - h->row0);   // nodes handed out
  const size_t o0 = (size_t)h->nx * h->row0;
  if (rho || ux || uy || T) {
    // B is dead between steps: use four of its planes as dense scratch
    double* s0 = h->B;
    double* s1 = h->B + h->ps;
    double* s2 = h->B + 2 * h->ps;
    double* s3 = h->B + 3 * h->ps;
    launch_macroscopic(h, s0, s1, s2, s3);
    if (rho) CUDA_OK(h, cudaMemcpyAsync(rho, s0 + o0, m * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    if (ux) CUDA_OK(h, cudaMemcpyAsync(ux, s1 + o0, m * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    if (uy) CUDA_OK(h, cudaMemcpyAsync(uy, s2 + o0, m * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    if (T) CUDA_OK(h, cudaMemcpyAsync(T, s3 + o0, m * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  }
  if (f || g) {
    // f, g are defined as the post-collision populations; before the first step the resident
    // state is still pre-collision and the export kernel collides on the fly.  The dense
    // population-major planes are staged in B (dead between steps; stream order keeps the
    // macroscopic copies above ahead of this overwrite)
    double* fd = h->B;
    double* gd = h->B + 9 * n;
    launch_export(h, f ? fd : nullptr, g ? gd : nullptr);
    if (m == n) {
      if (f) CUDA_OK(h, cudaMemcpyAsync(f, fd, 9 * n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
      if (g) CUDA_OK(h, cudaMemcpyAsync(g, gd, 5 * n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    } else {
      for (int k = 0; f && k < 9; ++k)
        CUDA_OK(h, cudaMemcpyAsync(f + k * m, fd + k * n + o0, m * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
      for (int k = 0; g && k < 5; ++k)
        CUDA_OK(h, cudaMemcpyAsync(g + k * m, gd + k * n + o0, m * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    }
  }
  if (flag)
    CUDA_OK(h, cudaMemcpy2DAsync(flag, h->nx, h->flag + (size_t)h->row0 * h->px, h->px, h->nx,
                                 h->row1 - h->row0, cudaMemcpyDeviceToHost, h->stream));
  CUDA_OK(h, cudaStreamSynchronize(h->stream));
  CUDA_OK(h, cudaGetLastError());
  return LBM_OK;
}

int lbm_get_macroscopic_static(lbm_t* h, double* rho, double* ux, double* uy, double* T) {
  if (!h) return LBM_E_ARG;
  if (h->is_slab) return fail(h, LBM_E_STATE, "lbm_get_macroscopic_static: not for slab handles");
  DeviceGuard dg(h);
  double* s[4] = {nullptr, nullptr, nullptr, nullptr};
  const int rc = launch_macroscopic_static(h, s);
  if (rc == -1)
    return fail(h, LBM_E_CAPACITY, "lbm_get_macroscopic_static: %d x %d nodes exceed the static scratch array (LBM_STATIC_MAX_NODES = %d)",
                h->nx, h->ny, (int)LBM_STATIC_MAX_NODES);
  if (rc != 0) return fail(h, LBM_E_CUDA, "lbm_get_macroscopic_static: cudaGetSymbolAddress failed");
  const size_t bytes = (size_t)h->nx * h->ny * sizeof(double);
  double* out[4] = {rho, ux, uy, T};
  for (int k = 0; k < 4; ++k)
    if (out[k]) CUDA_OK(h, cudaMemcpyAsync(out[k], s[k], bytes, cudaMemcpyDeviceToHost, h->stream));
  CUDA_OK(h, cudaStreamSynchronize(h->stream));
  CUDA_OK(h, cudaGetLastError());
  return LBM_OK;
}

int lbm_get_particles(lbm_t* h, int* n, double* x, double* y, double* theta, double* ux,
                      double* uy, double* omega, double* Fx, double* Fy, double* Tz) {
  if (!h || !n) return h ? fail(h, LBM_E_ARG, "get_particles: n is NULL") : LBM_E_ARG;
  *n = h->np;
  if (h->np == 0) return LBM_OK;
  DeviceGuard dg(h);
  const int c = h->cur;
  const size_t b = (size_t)h->np * sizeof(double);
  auto down = [&](double* dst, const double* src) {
    return dst ? cudaMemcpyAsync(dst, src, b, cudaMemcpyDeviceToHost, h->stream) : cudaSuccess;
  };
  CUDA_OK(h, down(x, h->pa.x[c]));
  CUDA_OK(h, down(y, h->pa.y[c]));
  CUDA_OK(h, down(theta, h->pa.theta[c]));
  CUDA_OK(h, down(ux, h->pa.ux[c]));
  CUDA_OK(h, down(uy, h->pa.uy[c]));
  CUDA_OK(h, down(omega, h->pa.omega[c]));
  CUDA_OK(h, down(Fx, h->pa.Fx));
  CUDA_OK(h, down(Fy, h->pa.Fy));
  CUDA_OK(h, down(Tz, h->pa.Tz));
  CUDA_OK(h, cudaStreamSynchronize(h->stream));
  return LBM_OK;
}

int lbm_get_links(lbm_t* h, long long* n, int* pid, int* i, int* j, int* alpha, double* q) {
  if (!h || !n) return h ? fail(h, LBM_E_ARG, "get_links: n is NULL") : LBM_E_ARG;
  const long long capacity = *n;
  *n = 0;
  if (h->np == 0) return LBM_OK;
  DeviceGuard dg(h);
  ensure_links(h);
  std::vector<int> count(h->np);
  CUDA_OK(h, cudaMemcpyAsync(count.data(), h->la.count, h->np * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  int rc = check_status(h);
  if (rc) return rc;
  long long total = 0;
  for (int c : count) total += c;
  *n = total;
  if (total > capacity) return fail(h, LBM_E_CAPACITY, "get_links: %lld links, capacity %lld", total, capacity);
  const size_t nl = (size_t)h->np * h->la.cap;
  std::vector<int> node(nl);
  std::vector<unsigned char> dir(nl);
  std::vector<double> qq(nl);
  CUDA_OK(h, cudaMemcpyAsync(node.data(), h->la.node, nl * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CUDA_OK(h, cudaMemcpyAsync(dir.data(), h->la.dir, nl, cudaMemcpyDeviceToHost, h->stream));
  CUDA_OK(h, cudaMemcpyAsync(qq.data(), h->la.q, nl * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_OK(h, cudaStreamSynchronize(h->stream));
  long long o = 0;
  for (int p = 0; p < h->np; ++p)
    for (int s = 0; s < count[p]; ++s, ++o) {
      const size_t k = (size_t)p * h->la.cap + s;
      if (pid) pid[o] = p;
      if (i) i[o] = node[k] & 0xffff;
      if (j) j[o] = (int)((unsigned)node[k] >> 16);
      if (alpha) alpha[o] = dir[k] & LINK_DIR_MASK;
      if (q) q[o] = qq[k];
    }
  return LBM_OK;
}

int lbm_profile_enable(lbm_t* h, int on) {
  if (!h) return LBM_E_ARG;
  DeviceGuard dg(h);
  if (on) {
    for (int k = 0; k < K_COUNT; ++k) {
      if (!h->ev0[k]) {
        h->ev0[k] = new cudaEvent_t[LBM_PROFILE_MAX_SAMPLES];
        h->ev1[k] = new cudaEvent_t[LBM_PROFILE_MAX_SAMPLES];
        for (int s = 0; s < LBM_PROFILE_MAX_SAMPLES; ++s) {
          CUDA_OK(h, cudaEventCreate(&h->ev0[k][s]));
          CUDA_OK(h, cudaEventCreate(&h->ev1[k][s]));
        }
      }
      h->ev_n[k] = 0;
    }
  }
  h->prof_on = on ? 1 : 0;
  return LBM_OK;
}

int lbm_profile_kernels(void) { return K_COUNT; }

const char* lbm_profile_kernel_name(int kernel_id) {
  return (kernel_id >= 0 && kernel_id < K_COUNT) ? kKernelNames[kernel_id] : "";
}

int lbm_profile_get(lbm_t* h, int kernel_id, double* total_ms, long long* launches) {
  if (!h || kernel_id < 0 || kernel_id >= K_COUNT) return LBM_E_ARG;
  DeviceGuard dg(h);
  CUDA_OK(h, cudaStreamSynchronize(h->stream));
  if (h->chain != h->stream) CUDA_OK(h, cudaStreamSynchronize(h->chain));
  if (h->side != h->stream) CUDA_OK(h, cudaStreamSynchronize(h->side));
  double tot = 0.0;
  const int n = h->ev0[kernel_id] ? h->ev_n[kernel_id] : 0;
  for (int s = 0; s < n; ++s) {
    float ms = 0.f;
    CUDA_OK(h, cudaEventElapsedTime(&ms, h->ev0[kernel_id][s], h->ev1[kernel_id][s]));
    tot += ms;
  }
  if (total_ms) *total_ms = tot;
  if (launches) *launches = n;
  return LBM_OK;
}

long long lbm_kernel_launches(const lbm_t* h) { return h ? h->launches : -1; }

int lbm_destroy(lbm_t* h) {
  if (!h) return LBM_OK;
  DeviceGuard dg(h);
  // a linked neighbour slab must not push into (or read the step counter of) a handle that is gone
  if (h->peer_lo && h->peer_lo->peer_hi == h) h->peer_lo->peer_hi = nullptr;
  if (h->peer_hi && h->peer_hi->peer_lo == h) h->peer_hi->peer_lo = nullptr;
  cudaStreamSynchronize(h->stream);
  drop_graphs(h);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  if (h->ev_p2) cudaEventDestroy(h->ev_p2);
  if (h->chain_own) {
    cudaStreamSynchronize(h->chain_own);
    cudaStreamDestroy(h->chain_own);
    if (h->side_own) cudaStreamDestroy(h->side_own);
    cudaEvent_t evs[7] = {h->ev_in, h->ev_out, h->ev_bb, h->ev_sc, h->ev_cov, h->ev_ref, h->ev_plan};
    for (cudaEvent_t e : evs) cudaEventDestroy(e);
  }
  for (int k = 0; k < K_COUNT; ++k)
    if (h->ev0[k]) {
      for (int s = 0; s < LBM_PROFILE_MAX_SAMPLES; ++s) {
        cudaEventDestroy(h->ev0[k][s]);
        cudaEventDestroy(h->ev1[k][s]);
      }
      delete[] h->ev0[k];
      delete[] h->ev1[k];
    }
  if (h->status_host) cudaFreeHost(h->status_host);
  delete h;
  return LBM_OK;
}

const char* lbm_last_error(const lbm_t* h) { return h ? h->err : g_create_error; }

} // extern "C"
