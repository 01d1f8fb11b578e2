// particles.cu -- rows a2, a5 and the flag half of a6: link builder, repulsion
// grid + particle integrator, flag/owner-map update.  Compiled with -fmad=false: every decision
// that yields an integer (node inside a disc, which nodes form links, which nodes are uncovered)
// is taken with separately rounded fp64 operations, the same way the paper-order CPU oracle does,
// so link lists are bit-exact ("Hard parts").
//
// a2  PAPER.md:250-258  per-step collection of (i, j, alpha) into a fixed index array: one CTA
//     per particle scans the particle's effective zone [INT(xc-r)-1, INT(xc+r)+1]^2 and compacts
//     the links into the particle's segment with popc + warp-shuffle scan + block prefix.
// a5  PAPER.md:88-97, 142-147  Eqs. (7), (8), (15): one thread per particle; neighbours through
//     a uniform cell grid (cell edge >= d_max + s), visited in ascending particle id so that the
//     sum order is fixed.
// a6  PAPER.md:151  "a solid node may be uncovered by the particle and become a fluid node".
#include "lbm_internal.cuh"

namespace {

__constant__ int p_ex[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1};
__constant__ int p_ey[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1};

constexpr int PT = 128;   // threads per particle CTA

__device__ __forceinline__ bool inside_disc(double xi, double yj, double xc, double yc, double r) {
  const double dx = xi - xc, dy = yj - yc;
  return dx * dx + dy * dy <= r * r;
}

// q = |x_f - x_w|/|x_f - x_b|: smaller root of |x_f + t e - x_c|^2 = r^2
__device__ __forceinline__ double link_q(double xf, double yf, int al, double xc, double yc, double r) {
  const double ex = (double)p_ex[al], ey = (double)p_ey[al];
  const double dx = xf - xc, dy = yf - yc;
  const double a = ex * ex + ey * ey;
  const double b = 2.0 * (ex * dx + ey * dy);
  const double cc = (dx * dx + dy * dy) - r * r;
  double disc = b * b - 4.0 * a * cc;
  if (disc < 0.0) disc = 0.0;
  double t = (-b - sqrt(disc)) / (2.0 * a);
  if (t < 0.0) t = 0.0;
  if (t > 1.0) t = 1.0;
  return t;
}

// ------------------------------------------------------------------------------------------
// a2: link builder.  grid = particles, block = PT.
__global__ void __launch_bounds__(PT)
k_build_links(const double* __restrict__ px_, const double* __restrict__ py_,
              const double* __restrict__ pr, const unsigned char* __restrict__ flag,
              const int* __restrict__ owner, LinkArrays la, int* __restrict__ status,
              const LbmConst c) {
  const int p = blockIdx.x;
  const double xc = px_[p], yc = py_[p], r = pr[p];
  int i0, i1, j0, j1;
  zone_of(xc, yc, r, i0, i1, j0, j1);
  const int W = i1 - i0 + 1, H = j1 - j0 + 1, total = W * H;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  __shared__ int s_warp[PT / 32];
  __shared__ int s_running;
  if (threadIdx.x == 0) s_running = 0;
  __syncthreads();
  const long long base = (long long)p * la.cap;
  const double rfar = (r + 1.5) * (r + 1.5);   // beyond this no neighbour can be inside the disc

  for (int start = 0; start < total; start += PT) {
    const int t = start + threadIdx.x;
    unsigned mask = 0;
    int i = 0, j = 0;
    if (t < total) {
      i = i0 + t % W;
      j = j0 + t / W;
      if (i >= 0 && i < c.nx && j >= 0 && j < c.ny) {
        const double dx = (double)i - xc, dy = (double)j - yc;
        // flag 2 = newborn: a fluid node of the step these links belong to
        if (dx * dx + dy * dy <= rfar && flag[(long long)j * c.px + i] != 1) {
#pragma unroll
          for (int al = 1; al <= 8; ++al) {
            const int bi = i + p_ex[al], bj = j + p_ey[al];
            if (bi >= 0 && bi < c.nx && bj >= 0 && bj < c.ny &&
                owner[(long long)bj * c.px + bi] == p)
              mask |= 1u << al;
          }
        }
      }
    }
    // block exclusive scan of popc(mask)
    const int cnt = __popc(mask);
    int incl = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int v = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += v;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    int woff = 0, btotal = 0;
#pragma unroll
    for (int w = 0; w < PT / 32; ++w) {
      const int v = s_warp[w];
      if (w < warp) woff += v;
      btotal += v;
    }
    int off = s_running + woff + incl - cnt;
    if (cnt) {
      if (off + cnt <= la.cap) {
        const int node = j * c.px + i;
        while (mask) {                         // compaction only; q follows in a balanced pass
          const int al = __ffs(mask) - 1;
          mask &= mask - 1;
          la.node[base + off] = node;
          la.dir[base + off] = (unsigned char)al;
          ++off;
        }
      } else {
        atomicOr(status, ST_LINK_OVERFLOW);
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) s_running += btotal;
    __syncthreads();
  }
  // q and the ladder rung for the compacted links, one link per thread (no divergence over
  // directions): how many of x_f - e, x_f - 2e are fluid nodes inside the cavity
  const int nl = min(s_running, la.cap);
  for (int s = threadIdx.x; s < nl; s += PT) {
    const int node = la.node[base + s];
    const int al = la.dir[base + s];
    const int i = node % c.px, j = node / c.px;
    la.q[base + s] = link_q((double)i, (double)j, al, xc, yc, r);
    int behind = 0;
    int a1 = i - p_ex[al], b1 = j - p_ey[al];
    if (c.periodic_x) a1 = (a1 + c.nx) % c.nx;
    if (a1 >= 0 && a1 < c.nx && b1 >= 0 && b1 < c.ny && flag[(long long)b1 * c.px + a1] != 1) {
      behind = 1;
      int a2 = i - 2 * p_ex[al], b2 = j - 2 * p_ey[al];
      if (c.periodic_x) a2 = (a2 + c.nx) % c.nx;
      if (a2 >= 0 && a2 < c.nx && b2 >= 0 && b2 < c.ny && flag[(long long)b2 * c.px + a2] != 1)
        behind = 2;
    }
    la.dir[base + s] = (unsigned char)(al | (behind << LINK_BEHIND_SHIFT));
  }
  if (threadIdx.x == 0) la.count[p] = nl;
}

// ------------------------------------------------------------------------------------------
// a5: repulsion grid
__global__ void k_cells_build(const double* __restrict__ px_, const double* __restrict__ py_, int np,
                              double cell, int ncx, int ncy, int* __restrict__ cell_count,
                              int* __restrict__ cell_items, int* __restrict__ status,
                              int* __restrict__ nb_count) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= np) return;
  if (p == 0) *nb_count = 0;   // the newborn list of the previous step has been consumed
  int ci = (int)floor(px_[p] / cell), cj = (int)floor(py_[p] / cell);
  ci = min(max(ci, 0), ncx - 1);
  cj = min(max(cj, 0), ncy - 1);
  const int cidx = cj * ncx + ci;
  const int slot = atomicAdd(&cell_count[cidx], 1);
  if (slot < CELL_CAP) cell_items[cidx * CELL_CAP + slot] = p;
  else atomicOr(status, ST_CELL_OVERFLOW);
}

__device__ __forceinline__ double ipow(double x, int p) {
  double r = 1.0;
  for (int k = 0; k < p; ++k) r = r * x;
  return r;
}

// Eq. (15) magnitude: (C/eps_w) ((s - delta)/s)^p for delta <= s
__device__ __forceinline__ double repulsion_mag(double C, const LbmConst& c, double delta) {
  if (!(delta <= c.rep_s)) return 0.0;
  return (C / c.rep_eps) * ipow((c.rep_s - delta) / c.rep_s, c.rep_power);
}

// Eqs. (7), (8), (15): total force = hydrodynamic + weight - buoyancy + repulsion; one step of
// U' = U + F/M, x' = x + (U + U')/2 (DESIGN.md reading), same for Omega, theta.
// One WARP per particle: the lanes fetch the candidates of the 3 x 3 cell neighbourhood in
// parallel (one round of dependent loads instead of a serial walk), each lane evaluates one pair,
// and the non-zero contributions are added in ascending particle id (warp min-reduction picks the
// next one), so the sum order is fixed whatever order the cell slots were filled in.
constexpr int IW = 4;   // warps (particles) per CTA
__global__ void __launch_bounds__(IW * 32)
k_integrate(ParticleArrays pa, int cur, int np, double cell, int ncx, int ncy,
            const int* __restrict__ cell_count, const int* __restrict__ cell_items,
            int* __restrict__ status, const LbmConst c) {
  const int lane = threadIdx.x & 31;
  const int ia = blockIdx.x * IW + (threadIdx.x >> 5);
  if (ia >= np) return;
  const unsigned FULL = 0xffffffffu;
  const int nxt = cur ^ 1;
  const double PI = 3.14159265358979323846;
  const double ax = pa.x[cur][ia], ay = pa.y[cur][ia], ar = pa.r[ia], ratio = pa.rho_ratio[ia];
  const double Ca = PI * ar * ar * (ratio * c.rho0 - c.rho0) * c.g;
  double Fx = pa.Fx[ia], Fy = pa.Fy[ia];
  Fy += -(ratio * c.rho0 - c.rho0) * PI * ar * ar * c.g;
  int ci = (int)floor(ax / cell), cj = (int)floor(ay / cell);
  ci = min(max(ci, 0), ncx - 1);
  cj = min(max(cj, 0), ncy - 1);
  // lanes 0..8: one cell of the neighbourhood each
  int cidx = -1, cnt = 0;
  if (lane < 9) {
    const int a = ci + lane % 3 - 1, b = cj + lane / 3 - 1;
    if (a >= 0 && a < ncx && b >= 0 && b < ncy) {
      cidx = b * ncx + a;
      cnt = min(cell_count[cidx], CELL_CAP);
    }
  }
  int incl = cnt;   // inclusive prefix over lanes 0..8
#pragma unroll
  for (int d = 1; d < 16; d <<= 1) {
    const int v = __shfl_up_sync(FULL, incl, d);
    if (lane >= d) incl += v;
  }
  const int total = __shfl_sync(FULL, incl, 8);
  for (int base = 0; base < total; base += 32) {
    const int k = base + lane;   // candidate number k lives in the cell whose prefix range holds it
    int id = 0x7fffffff;
    double fx = 0.0, fy = 0.0;
    int my_cell = -1, my_slot = 0;
#pragma unroll
    for (int s = 0; s < 9; ++s) {
      const int hi = __shfl_sync(FULL, incl, s), n = __shfl_sync(FULL, cnt, s);
      const int cc = __shfl_sync(FULL, cidx, s);
      if (my_cell < 0 && k < hi && k >= hi - n) { my_cell = cc; my_slot = k - (hi - n); }
    }
    bool has = false;
    if (k < total && my_cell >= 0) {
      const int best = cell_items[my_cell * CELL_CAP + my_slot];
      if (best != ia) {
        const double bx = pa.x[cur][best], by = pa.y[cur][best], br = pa.r[best];
        const double dx = ax - bx, dy = ay - by;
        const double reach = ar + br + c.rep_s;
        if (!(fabs(dx) > reach || fabs(dy) > reach)) {
          const double dist = sqrt(dx * dx + dy * dy);
          const double delta = dist - ar - br;
          if (delta <= c.rep_s && dist > 0.0) {
            const double Cb = PI * br * br * (pa.rho_ratio[best] * c.rho0 - c.rho0) * c.g;
            const double mag = repulsion_mag(0.5 * (Ca + Cb), c, delta);
            fx = mag * (dx / dist);
            fy = mag * (dy / dist);
            id = best;
            has = true;
          }
        }
      }
    }
    // contributions of this batch in ascending id (batches themselves are rare beyond the first:
    // 32 candidates already cover 9 cells of edge >= d_max + s)
    while (__any_sync(FULL, has)) {
      const int m = __reduce_min_sync(FULL, has ? id : 0x7fffffff);
      const int src = __ffs(__ballot_sync(FULL, has && id == m)) - 1;
      Fx += __shfl_sync(FULL, fx, src);
      Fy += __shfl_sync(FULL, fy, src);
      if (lane == src) has = false;
    }
  }
  if (lane != 0) return;
  if (!c.periodic_x) {
    const double dW = (ax + 0.5) - ar;
    if (dW <= c.rep_s) Fx += repulsion_mag(Ca, c, dW);
    const double dE = ((double)c.nx - 0.5 - ax) - ar;
    if (dE <= c.rep_s) Fx -= repulsion_mag(Ca, c, dE);
  }
  const double dS = (ay + 0.5) - ar;
  if (dS <= c.rep_s) Fy += repulsion_mag(Ca, c, dS);
  const double dN = ((double)c.ny - 0.5 - ay) - ar;
  if (dN <= c.rep_s) Fy -= repulsion_mag(Ca, c, dN);

  double x = ax, y = ay, th = pa.theta[cur][ia];
  double ux = pa.ux[cur][ia], uy = pa.uy[cur][ia], om = pa.omega[cur][ia];
  if (!pa.fixed[ia]) {
    const double mass = ratio * c.rho0 * PI * ar * ar;
    const double inertia = 0.5 * mass * ar * ar;
    const double ux1 = ux + Fx / mass;
    const double uy1 = uy + Fy / mass;
    const double om1 = om + pa.Tz[ia] / inertia;
    x = x + 0.5 * (ux + ux1);
    y = y + 0.5 * (uy + uy1);
    th = th + 0.5 * (om + om1);
    ux = ux1;
    uy = uy1;
    om = om1;
  }
  pa.x[nxt][ia] = x;
  pa.y[nxt][ia] = y;
  pa.theta[nxt][ia] = th;
  pa.ux[nxt][ia] = ux;
  pa.uy[nxt][ia] = uy;
  pa.omega[nxt][ia] = om;
  if (!(isfinite(x) && isfinite(y) && isfinite(th) && isfinite(ux) && isfinite(uy) && isfinite(om)))
    atomicOr(status, ST_NONFINITE);
}

// ------------------------------------------------------------------------------------------
// a6, flags.  Phase A: nodes owned by p that the disc at its NEW position no longer covers become
// newborn candidates (flag 2, owner NONE) and are appended to the newborn list.
__global__ void __launch_bounds__(PT)
k_uncover(ParticleArrays pa, int cur, unsigned char* __restrict__ flag, int* __restrict__ owner,
          int* __restrict__ nb_node, int* __restrict__ nb_pid, int* __restrict__ nb_count, int nb_cap,
          int* __restrict__ status, int* __restrict__ cell_count, int ncells, const LbmConst c) {
  const int p = blockIdx.x;
  // the repulsion grid of this step has been consumed by k_integrate: zero it for the next step
  for (int k = p * PT + threadIdx.x; k < ncells; k += gridDim.x * PT) cell_count[k] = 0;
  if (pa.fixed[p]) return;
  const int nxt = cur ^ 1;
  const double xo = pa.x[cur][p], yo = pa.y[cur][p], r = pa.r[p];
  const double xn = pa.x[nxt][p], yn = pa.y[nxt][p];
  int i0, i1, j0, j1;
  zone_of(xo, yo, r, i0, i1, j0, j1);
  const int W = i1 - i0 + 1, total = W * (j1 - j0 + 1);
  for (int t = threadIdx.x; t < total; t += PT) {
    const int i = i0 + t % W, j = j0 + t / W;
    if (i < 0 || i >= c.nx || j < 0 || j >= c.ny) continue;
    if (!inside_disc((double)i, (double)j, xo, yo, r)) continue;
    if (inside_disc((double)i, (double)j, xn, yn, r)) continue;
    const long long x = (long long)j * c.px + i;
    if (owner[x] != p) continue;
    owner[x] = OWNER_NONE;
    flag[x] = 2;
    const int e = atomicAdd(nb_count, 1);
    if (e < nb_cap) {
      nb_node[e] = (int)x;
      nb_pid[e] = p;
    } else {
      atomicOr(status, ST_NEWBORN_OVERFLOW);
    }
  }
}

// Phase B: every node inside the disc at the position in buffer `buf` is solid; the lowest
// particle id wins the owner map (same rule as a from-scratch recomputation).
__global__ void __launch_bounds__(PT)
k_cover(ParticleArrays pa, int buf, int skip_fixed, unsigned char* __restrict__ flag,
        int* __restrict__ owner, const LbmConst c) {
  const int p = blockIdx.x;
  if (skip_fixed && pa.fixed[p]) return;
  const double xn = pa.x[buf][p], yn = pa.y[buf][p], r = pa.r[p];
  int i0, i1, j0, j1;
  zone_of(xn, yn, r, i0, i1, j0, j1);
  const int W = i1 - i0 + 1, total = W * (j1 - j0 + 1);
  for (int t = threadIdx.x; t < total; t += PT) {
    const int i = i0 + t % W, j = j0 + t / W;
    if (i < 0 || i >= c.nx || j < 0 || j >= c.ny) continue;
    if (!inside_disc((double)i, (double)j, xn, yn, r)) continue;
    const long long x = (long long)j * c.px + i;
    if (owner[x] == p) continue;
    const int prev = atomicMin(&owner[x], p);
    if (prev != p) flag[x] = 1;
  }
}

} // namespace

void launch_build_links(lbm* h, int which_buffer, cudaStream_t st) {
  if (h->np == 0) return;
  h->launches++;
  k_build_links<<<h->np, PT, 0, st>>>(h->pa.x[which_buffer], h->pa.y[which_buffer], h->pa.r,
                                      h->flag, h->owner, h->la, h->status_dev, h->C);
}

void launch_cells_and_integrate(lbm* h) {
  if (h->np == 0) return;
  const int blocks = (h->np + 127) / 128;
  h->launches++;
  k_cells_build<<<blocks, 128, 0, h->chain>>>(h->pa.x[h->cur], h->pa.y[h->cur], h->np, h->cell,
                                               h->ncx, h->ncy, h->cell_count, h->cell_items,
                                               h->status_dev, h->newborn_count);
  h->launches++;
  k_integrate<<<(h->np + IW - 1) / IW, IW * 32, 0, h->chain>>>(h->pa, h->cur, h->np, h->cell, h->ncx, h->ncy,
                                             h->cell_count, h->cell_items, h->status_dev, h->C);
}

void launch_uncover(lbm* h) {
  if (h->np == 0) return;
  h->launches++;
  k_uncover<<<h->np, PT, 0, h->chain>>>(h->pa, h->cur, h->flag, h->owner, h->newborn_node,
                                         h->newborn_pid, h->newborn_count, h->newborn_cap,
                                         h->status_dev, h->cell_count, h->ncx * h->ncy, h->C);
}

// after add_particles every particle (fixed ones too) is rasterised; during stepping the fixed
// ones never move
void launch_cover(lbm* h, int which_buffer, cudaStream_t st) {
  if (h->np == 0) return;
  h->launches++;
  k_cover<<<h->np, PT, 0, st>>>(h->pa, which_buffer, h->primed ? 1 : 0, h->flag, h->owner, h->C);
}
