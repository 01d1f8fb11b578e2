// stream_collide.cu -- row a1 of SURVEY.md 8(a): ONE fused kernel per time step doing
// pull-streaming (LHS of Eqs. 5, 6), macroscopic moments, Boussinesq forcing, MRT collision of f
// and g, and the cavity-wall boundary conditions; plus the small set-up / read-out kernels.
//
// The paper runs collision f, collision g, streaming f, streaming g, macroscopic T and
// macroscopic u, rho as six OpenACC loop nests; here each population is read
// once and written once per step: 2*(9+5)*8 = 224 B + 1 flag byte per lattice update.
//
// State: A holds the POST-collision populations f+(x,t), g+(x,t).  A fluid node pulls
// f_k(x,t+1) = f+_k(x - e_k, t) whatever x - e_k is: if it is a solid node the bounce-back kernel
// has already parked the bounced value in that slot, so this
// kernel needs no link awareness.  Only the cavity walls are handled here: halfway bounce-back
// f_k(x,t+1) = f+_kbar(x,t); thermal g_k(x,t+1) = -g+_kbar(x,t) + 2 w_k T_wall (Dirichlet) or
// g+_kbar(x,t) (adiabatic)  (DESIGN.md readings; the paper only says "no-slip").
#include "collide.cuh"

namespace {

// lattice tables as constexpr functions so that fully unrolled loops fold them to immediates
__host__ __device__ constexpr int ex_of(int k) { return (k == 1 || k == 5 || k == 8) - (k == 3 || k == 6 || k == 7); }
__host__ __device__ constexpr int ey_of(int k) { return (k == 2 || k == 5 || k == 6) - (k == 4 || k == 7 || k == 8); }
__host__ __device__ constexpr int opp_of(int k) { return k == 0 ? 0 : (k <= 4 ? ((k + 1) % 4) + 1 : ((k - 3) % 4) + 5); }

constexpr int SC_THREADS = 128;

// generic pull with cavity-wall handling; only nodes on the lattice rim take this path.
// Fully unrolled and inlined so that f, g stay in registers.
__device__ __forceinline__ void pull_boundary(const double* __restrict__ A, const LbmConst& c, int i,
                                              int j, double (&f)[9], double (&g)[5]) {
  const long long x = (long long)j * c.px + i;
#pragma unroll
  for (int k = 0; k < 9; ++k) {
    int si = i - ex_of(k), sj = j - ey_of(k);
    bool in = (sj >= 0 && sj < c.ny);
    if (si < 0 || si >= c.nx) {
      if (c.periodic_x) si = (si + c.nx) % c.nx; else in = false;
    }
    f[k] = in ? A[k * c.ps + (long long)sj * c.px + si] : A[opp_of(k) * c.ps + x];
  }
  const double* G = A + 9 * c.ps;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    int si = i - ex_of(k), sj = j - ey_of(k);
    bool in = (sj >= 0 && sj < c.ny);
    int wall = sj < 0 ? 2 : 3;
    if (si < 0 || si >= c.nx) {
      if (c.periodic_x) si = (si + c.nx) % c.nx;
      else { in = false; wall = si < 0 ? 0 : 1; }
    }
    if (in) g[k] = G[k * c.ps + (long long)sj * c.px + si];
    else {
      const double gb = G[opp_of(k) * c.ps + x];
      g[k] = c.wall_type[wall] == 1 ? (2.0 * c.wT * c.wall_T[wall] - gb) : gb;
    }
  }
}

// one lattice update of node (i, j): pull, collide, store
__device__ __forceinline__ void update_node(const double* __restrict__ A, double* __restrict__ B,
                                            const LbmConst& c, int i, int j) {
  const long long x = (long long)j * c.px + i;
  double f[9], g[5];
  if (i >= 1 && i < c.nx - 1 && j >= 1 && j < c.ny - 1) {
    const double* __restrict__ F = A + x;
    const long long ps = c.ps;
    const int px = c.px;
    f[0] = __ldg(F);
    f[1] = __ldg(F + 1 * ps - 1);
    f[2] = __ldg(F + 2 * ps - px);
    f[3] = __ldg(F + 3 * ps + 1);
    f[4] = __ldg(F + 4 * ps + px);
    f[5] = __ldg(F + 5 * ps - px - 1);
    f[6] = __ldg(F + 6 * ps - px + 1);
    f[7] = __ldg(F + 7 * ps + px + 1);
    f[8] = __ldg(F + 8 * ps + px - 1);
    g[0] = __ldg(F + 9 * ps);
    g[1] = __ldg(F + 10 * ps - 1);
    g[2] = __ldg(F + 11 * ps - px);
    g[3] = __ldg(F + 12 * ps + 1);
    g[4] = __ldg(F + 13 * ps + px);
  } else {
    pull_boundary(A, c, i, j, f, g);
  }
  mrt_collide(f, g, c);
  double* __restrict__ O = B + x;
#pragma unroll
  for (int k = 0; k < 9; ++k) O[k * c.ps] = f[k];
#pragma unroll
  for (int k = 0; k < 5; ++k) O[(9 + k) * c.ps] = g[k];
}

// FAR pass: every node outside all particle zones of this step (zstamp != stamp).  Such a node is
// fluid, stays fluid, and none of its upstream neighbours is a solid slot, so this kernel depends
// on nothing the particle chain of the step produces and runs concurrently with it.
__global__ void __launch_bounds__(SC_THREADS)
k_stream_collide(const double* __restrict__ A, double* __restrict__ B,
                 const unsigned char* __restrict__ zstamp, const unsigned char stamp,
                 const LbmConst c) {
  const int i = blockIdx.x * SC_THREADS + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= c.nx) return;
  if (zstamp[(long long)j * c.px + i] == stamp) return;   // near: left to k_stream_collide_near
  update_node(A, B, c, i, j);
}

// NEAR pass: one CTA per particle, after the flag update, at the positions of time t.  Phase 1
// scans the particle's effective zone [INT(xc-r)-1, INT(xc+r)+1]^2 with arithmetic only (the
// same near_disc() predicate that stamped the zone map, so far and near pass partition the
// lattice exactly), reads the flag of the candidates and compacts the nodes that are fluid at t
// and t+1 (flag 0; solid = 1 and newborn = 2 are skipped) into shared memory.  Phase 2 updates
// the compacted nodes, one per thread: ~100 of the 23 x 23 zone nodes at d = 20, so the heavy
// per-node code runs with full warps instead of a 5-pass sweep with 80 % idle lanes.
// Near sets of neighbouring particles may overlap: both CTAs then compute and store
// bit-identical values (same inputs, same code), which is benign.
__global__ void __launch_bounds__(SC_THREADS)
k_stream_collide_near(const double* __restrict__ A, double* __restrict__ B,
                      const unsigned char* __restrict__ flag, const double* __restrict__ px_,
                      const double* __restrict__ py_, const double* __restrict__ pr, int cap,
                      const LbmConst c) {
  extern __shared__ unsigned s_list[];   // cap entries: i | j << 16
  __shared__ int s_n;
  const int p = blockIdx.x;
  const double xc = px_[p], yc = py_[p], r = pr[p];
  int i0, i1, j0, j1;
  zone_of(xc, yc, r, i0, i1, j0, j1);
  const int W = i1 - i0 + 1, total = W * (j1 - j0 + 1);
  if (threadIdx.x == 0) s_n = 0;
  __syncthreads();
  // nodes closer than r - 1 to the centre are inside the disc under any rounding: never flag 0
  const double rin = r > 1.0 ? (r - 1.0) * (r - 1.0) : -1.0;
  for (int t = threadIdx.x; t < total; t += SC_THREADS) {
    const int i = i0 + t % W, j = j0 + t / W;
    if (i < 0 || i >= c.nx || j < 0 || j >= c.ny) continue;
    const double dx = (double)i - xc, dy = (double)j - yc;
    if (dx * dx + dy * dy < rin) continue;
    if (!near_disc((double)i, (double)j, xc, yc, r)) continue;
    if (flag[(long long)j * c.px + i] != 0) continue;
    const int e = atomicAdd(&s_n, 1);
    if (e < cap) s_list[e] = (unsigned)i | ((unsigned)j << 16);
  }
  __syncthreads();
  const int n = min(s_n, cap);
  for (int e = threadIdx.x; e < n; e += SC_THREADS) {
    const unsigned v = s_list[e];
    update_node(A, B, c, (int)(v & 0xffffu), (int)(v >> 16));
  }
}

// first step only: A holds the PRE-collision initial state f(x,0); collide it (in place when
// priming, into the scratch copy when the populations are read out before the first step)
__global__ void __launch_bounds__(SC_THREADS)
k_init_collide(const double* A, double* O, const unsigned char* __restrict__ flag, const LbmConst c) {
  const int i = blockIdx.x * SC_THREADS + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= c.nx) return;
  const long long x = (long long)j * c.px + i;
  if (flag[x] != 0) return;
  double f[9], g[5];
#pragma unroll
  for (int k = 0; k < 9; ++k) f[k] = A[k * c.ps + x];
#pragma unroll
  for (int k = 0; k < 5; ++k) g[k] = A[(9 + k) * c.ps + x];
  mrt_collide(f, g, c);
#pragma unroll
  for (int k = 0; k < 9; ++k) O[k * c.ps + x] = f[k];
#pragma unroll
  for (int k = 0; k < 5; ++k) O[(9 + k) * c.ps + x] = g[k];
}

// f = f_eq(rho0, 0) = w_k rho0, g = g_eq(T0, 0) = wT_k T0 on every node (SURVEY 8(c) "Initial state")
__global__ void k_set_equilibrium(double* __restrict__ A, const LbmConst c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= c.px) return;
  const long long x = (long long)j * c.px + i;
  const double w[9] = {4.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36};
#pragma unroll
  for (int k = 0; k < 9; ++k) A[k * c.ps + x] = w[k] * c.rho0;
  A[9 * c.ps + x] = c.wT0 * c.T0;
#pragma unroll
  for (int k = 1; k < 5; ++k) A[(9 + k) * c.ps + x] = c.wT * c.T0;
}

// g = g_eq(T, u = 0) from a dense nx*ny temperature field (lbm_set_temperature)
__global__ void k_set_temperature(double* __restrict__ A, const double* __restrict__ T, const LbmConst c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= c.nx) return;
  const long long x = (long long)j * c.px + i;
  const double t = T[(long long)j * c.nx + i];
  A[9 * c.ps + x] = c.wT0 * t;
#pragma unroll
  for (int k = 1; k < 5; ++k) A[(9 + k) * c.ps + x] = c.wT * t;
}

// read-out: dense nx*ny outputs
__global__ void k_macroscopic(const double* __restrict__ A, const unsigned char* __restrict__ flag,
                              const int* __restrict__ owner, const double* __restrict__ px_,
                              const double* __restrict__ py_, const double* __restrict__ pux,
                              const double* __restrict__ puy, const double* __restrict__ pom,
                              const double* __restrict__ pTw, int post, double* __restrict__ rho,
                              double* __restrict__ ux, double* __restrict__ uy,
                              double* __restrict__ T, const LbmConst c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= c.nx) return;
  const long long x = (long long)j * c.px + i;
  const long long o = (long long)j * c.nx + i;
  if (flag[x] != 0) {
    const int p = owner[x];
    rho[o] = c.rho0;
    ux[o] = pux[p] - pom[p] * ((double)j - py_[p]);
    uy[o] = puy[p] + pom[p] * ((double)i - px_[p]);
    T[o] = pTw[p];
    return;
  }
  double f[9], g[5];
#pragma unroll
  for (int k = 0; k < 9; ++k) f[k] = A[k * c.ps + x];
#pragma unroll
  for (int k = 0; k < 5; ++k) g[k] = A[(9 + k) * c.ps + x];
  double r, vx, vy, t;
  macroscopic(f, g, c, post, r, vx, vy, t);
  rho[o] = r;
  ux[o] = vx;
  uy[o] = vy;
  T[o] = t;
}

inline dim3 grid_rows(int n, int ny, int threads) { return dim3((n + threads - 1) / threads, ny); }

} // namespace

void launch_stream_collide_far(lbm* h) {
  h->launches++;
  k_stream_collide<<<grid_rows(h->nx, h->ny, SC_THREADS), SC_THREADS, 0, h->stream>>>(
      h->A, h->B, h->zstamp[h->steps_done & 1], zone_stamp(h->steps_done), h->C);
}

void launch_stream_collide_near(lbm* h) {
  if (h->np == 0) return;
  const int old = h->cur ^ 1;   // positions at time t (the integrator has already flipped cur)
  h->launches++;
  k_stream_collide_near<<<h->np, SC_THREADS, h->la.cap * sizeof(unsigned), h->chain>>>(
      h->A, h->B, h->flag, h->pa.x[old], h->pa.y[old], h->pa.r, h->la.cap, h->C);
}

void launch_init_collide(lbm* h, double* dst) {
  h->launches++;
  k_init_collide<<<grid_rows(h->nx, h->ny, SC_THREADS), SC_THREADS, 0, h->stream>>>(h->A, dst, h->flag, h->C);
}

void launch_set_equilibrium(lbm* h) {
  h->launches++;
  k_set_equilibrium<<<grid_rows(h->px, h->ny, 128), 128, 0, h->stream>>>(h->A, h->C);
}

void launch_set_temperature(lbm* h, const double* T_dev_dense) {
  h->launches++;
  k_set_temperature<<<grid_rows(h->nx, h->ny, 128), 128, 0, h->stream>>>(h->A, T_dev_dense, h->C);
}

void launch_macroscopic(lbm* h, double* rho, double* ux, double* uy, double* T) {
  const int c = h->cur;
  h->launches++;
  k_macroscopic<<<grid_rows(h->nx, h->ny, 128), 128, 0, h->stream>>>(
      h->A, h->flag, h->owner, h->pa.x[c], h->pa.y[c], h->pa.ux[c], h->pa.uy[c], h->pa.omega[c],
      h->pa.Tw, h->primed, rho, ux, uy, T, h->C);
}
