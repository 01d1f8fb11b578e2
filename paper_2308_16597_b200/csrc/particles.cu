// particles.cu -- rows a2, a5 and the flag half of a6: link builder, repulsion
// grid + particle integrator, flag/owner-map update.  Compiled with -fmad=false: every decision
// that yields an integer (node inside a disc, which nodes form links, which nodes are uncovered)
// is taken with separately rounded fp64 operations, the same way the paper-order CPU oracle does,
// so link lists are bit-exact ("Hard parts").
//
// a2  PAPER.md:250-258  per-step collection of (i, j, alpha) into a fixed index array: a CTA per
//     particle enumerates the ring of candidate nodes of the particle's effective zone
//     [INT(xc-r)-1, INT(xc+r)+1]^2 row by row and compacts the links into the particle's segment
//     with popc + a packed warp-shuffle scan + block prefix.
// a5  PAPER.md:88-97, 142-147  Eqs. (7), (8), (15): one warp per particle; neighbours through
//     a uniform cell grid (cell edge >= d_max + s), added in ascending particle id so that the
//     sum order is fixed.
// a6  PAPER.md:151  "a solid node may be uncovered by the particle and become a fluid node".
// Shapes: circles, and ellipses through the Shape helpers below; the kernels
// are templated on whether the simulation holds an ellipse at all.  All four kernels loop over
// the particles (grid-size agnostic): under the lattice kernel they run as a few persistent CTAs
// per SM.
#include "lbm_internal.cuh"

namespace {

__constant__ int p_ex[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1};
__constant__ int p_ey[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1};

// Threads per particle CTA: PT_MAX when a kernel has the GPU to itself (one CTA per particle: the
// single particle's latency counts), PT_THROTTLED for the few persistent CTAs per SM that run
// under the lattice kernel: a chain kernel is bound by the latency of its dependent loads, not by
// threads, and 64-thread CTAs put twice as many particles in flight per register taken from the
// lattice kernel (r28, r33: config 3 538 -> 533 us, config 5 535 -> 520 us; alone, or on the small
// configs, 64 threads are slower: config 2 50.7 -> 54.4 us).
constexpr int PT_MAX = 128;
constexpr int PT_THROTTLED = 64;

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

// ---- shapes.  A particle is a circle (a == b: the formulas above, bit for bit) or an ellipse with
// semi-axes a, b and orientation unit vector (c, s) (DESIGN.md "Elliptical
// particles").  Every expression below is the oracle's, operation for operation (-fmad=false).
struct Shape {
  double x, y, r, a, b, c, s;
  bool ell;
};

// ELL = false: the simulation holds circles only; the shape is then a compile-time circle and
// every ellipse branch of the kernels folds away (same code and registers as before ellipses).
template <bool ELL>
__device__ __forceinline__ Shape load_shape(const ParticleArrays& pa, int buf, int p) {
  Shape S;
  S.x = pa.x[buf][p];
  S.y = pa.y[buf][p];
  S.r = pa.r[p];
  if (ELL) {
    S.a = pa.a[p];
    S.b = pa.b[p];
    S.ell = S.a != S.b;
    S.c = S.ell ? pa.cs[buf][p] : 1.0;
    S.s = S.ell ? pa.sn[buf][p] : 0.0;
  } else {
    S.a = S.r;
    S.b = S.r;
    S.ell = false;
    S.c = 1.0;
    S.s = 0.0;
  }
  return S;
}

__device__ __forceinline__ bool inside_ellipse(double xi, double yj, const Shape& S) {
  const double dx = xi - S.x, dy = yj - S.y;
  const double u = dx * S.c + dy * S.s;
  const double v = dy * S.c - dx * S.s;
  const double ua = u / S.a, vb = v / S.b;
  return ua * ua + vb * vb <= 1.0;
}

__device__ __forceinline__ bool inside_shape(double xi, double yj, const Shape& S) {
  return S.ell ? inside_ellipse(xi, yj, S) : inside_disc(xi, yj, S.x, S.y, S.r);
}

// half extents of the bounding box: r, or sqrt((a c)^2 + (b s)^2), sqrt((a s)^2 + (b c)^2)
__device__ __forceinline__ void half_extents(const Shape& S, double& hx, double& hy) {
  if (!S.ell) {
    hx = S.r;
    hy = S.r;
    return;
  }
  const double ac = S.a * S.c, bs = S.b * S.s, as = S.a * S.s, bc = S.b * S.c;
  hx = sqrt(ac * ac + bs * bs);
  hy = sqrt(as * as + bc * bc);
}

// effective zone [INT(xc-hx)-1, INT(xc+hx)+1] x [INT(yc-hy)-1, INT(yc+hy)+1]
__device__ __forceinline__ void zone_shape(const Shape& S, int& i0, int& i1, int& j0, int& j1) {
  double hx, hy;
  half_extents(S, hx, hy);
  i0 = (int)floor(S.x - hx) - 1;
  i1 = (int)floor(S.x + hx) + 1;
  j0 = (int)floor(S.y - hy) - 1;
  j1 = (int)floor(S.y + hy) + 1;
}

// q of a link towards an ellipse: smaller root of the ray-ellipse quadratic in the body frame
__device__ __forceinline__ double link_q_ellipse(double xf, double yf, int al, const Shape& S) {
  const double ex = (double)p_ex[al], ey = (double)p_ey[al];
  const double dx = xf - S.x, dy = yf - S.y;
  const double u = dx * S.c + dy * S.s, v = dy * S.c - dx * S.s;
  const double eu = ex * S.c + ey * S.s, ev = ey * S.c - ex * S.s;
  const double ua = u / S.a, vb = v / S.b, ea = eu / S.a, eb = ev / S.b;
  const double A = ea * ea + eb * eb;
  const double B = 2.0 * (ua * ea + vb * eb);
  const double C = (ua * ua + vb * vb) - 1.0;
  double disc = B * B - 4.0 * A * C;
  if (disc < 0.0) disc = 0.0;
  double t = (-B - sqrt(disc)) / (2.0 * A);
  if (t < 0.0) t = 0.0;
  if (t > 1.0) t = 1.0;
  return t;
}

// support function along the unit vector (nx, ny)
__device__ __forceinline__ double support_shape(const Shape& S, double nx, double ny) {
  if (!S.ell) return S.r;
  const double m = nx * S.c + ny * S.s;
  const double w = ny * S.c - nx * S.s;
  const double am = S.a * m, bw = S.b * w;
  return sqrt(am * am + bw * bw);
}

// ------------------------------------------------------------------------------------------
// a2: link builder.  grid = particles (or fewer persistent CTAs), block = LB_WARPS warps.
//
// A fluid node can carry a link of particle p only in the ring r^2 < d^2 <= (r + 1.5)^2 around
// the centre, so the work is made proportional to the perimeter, not to the area of the zone:
//   0. one thread per zone row turns the ring into at most two column segments of that row
//      (square roots only bracket them: each end is padded by one node and every candidate is
//      then decided by the exact, separately rounded predicate that rasterised the disc); a block
//      prefix over the rows numbers the candidates in row-major order;
//   1. candidates are dealt to the threads, LB_CPT per thread and round, each found by a binary
//      search in the row prefix; arithmetic only: is the node in the ring, which neighbours lie
//      inside the disc;
//   2. the flag bytes of all candidates of the round, requested together (a candidate may be
//      inside ANOTHER particle);
//   3. only for a particle whose disc may overlap another one (sticky flag pa.ovl, set by k_cover):
//      the owner of each solid neighbour, lowest id owns the node.  Without
//      overlap every node inside the disc is owned by the particle and the loads are skipped;
//   4. packed block prefix (the LB_CPT counts of a thread in the 16-bit fields of one 64-bit
//      shuffle), emission in row-major order (neighbouring links -> neighbouring nodes for the
//      bounce-back kernel) into shared memory;
//   5. q and the ladder rung per link, one link per thread, both flag bytes requested together.
constexpr int LB_CPT = 4;
template <bool ELL, int LB_WARPS>
__global__ void __launch_bounds__(LB_WARPS * 32)
k_build_links(ParticleArrays pa, int buf, const unsigned char* __restrict__ flag,
              const int* __restrict__ owner, LinkArrays la, int np, int max_rows,
              int* __restrict__ status, int early, const LbmConst c) {
  if (early) pdl_launch_dependents();
  pdl_wait();
  constexpr int LB_T = LB_WARPS * 32;
  extern __shared__ int s_node[];                           // la.cap packed nodes, la.cap dir bytes,
  unsigned char* s_dir = (unsigned char*)(s_node + la.cap); // then the row tables
  int* s_off = s_node + la.cap + (la.cap + 3) / 4;          // max_rows + 1: candidates before row t
  int* s_a1 = s_off + max_rows + 1;                         // first column of segment 1
  int* s_n1 = s_a1 + max_rows;                              // its length
  int* s_a2 = s_n1 + max_rows;                              // first column of segment 2
  __shared__ int s_warp[LB_WARPS];
  __shared__ unsigned long long s_wpk[LB_WARPS];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned FULL = 0xffffffffu;
  for (int p = blockIdx.x; p < np; p += gridDim.x) {   // grid-size agnostic
  const Shape S = load_shape<ELL>(pa, buf, p);
  const double xc = S.x, yc = S.y, r = S.r;
  const bool check_owner = pa.ovl[p] != 0;
  int i0, i1, j0, j1;
  zone_shape(S, i0, i1, j0, j1);
  const int H = min(j1 - j0 + 1, max_rows);
  const double r2 = r * r;
  const double rfar = (r + 1.5) * (r + 1.5);   // beyond this no neighbour can be inside the disc
  const int ilo = max(i0, 0), ihi = min(i1, c.nx - 1);

  // ---- 0. ring segments per row and their prefix
  int carry = 0;
  for (int t0 = 0; t0 < H; t0 += LB_T) {
    const int t = t0 + threadIdx.x;
    int cnt = 0;
    if (t < H) {
      const int j = j0 + t;
      int a1 = 0, n1 = 0, a2 = 0, n2 = 0;
      const double dy = (double)j - yc, dy2 = dy * dy;
      if (S.ell) {                                // first version: every column of the zone row
        if (row_here(c, j) && ihi >= ilo) { a1 = ilo; n1 = ihi - ilo + 1; }
      } else if (row_here(c, j) && dy2 <= rfar) {
        const double wo = sqrt(rfar - dy2);
        const int oa = max((int)floor(xc - wo) - 1, ilo), ob = min((int)floor(xc + wo) + 2, ihi);
        int ha = ob + 1, hb = ob;                 // hole = columns certainly inside the disc
        if (dy2 < r2) {
          const double wi = sqrt(r2 - dy2);
          ha = (int)floor(xc - wi) + 2;
          hb = (int)floor(xc + wi) - 1;
        }
        if (ha <= hb && ha > oa && hb < ob) {     // two segments around the hole
          a1 = oa; n1 = ha - oa;
          a2 = hb + 1; n2 = ob - hb;
        } else if (ob >= oa) {                    // one segment
          a1 = oa; n1 = ob - oa + 1;
        }
      }
      s_a1[t] = a1; s_n1[t] = n1; s_a2[t] = a2;
      cnt = n1 + n2;
    }
    int incl = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int v = __shfl_up_sync(FULL, incl, d);
      if (lane >= d) incl += v;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    int woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < LB_WARPS; ++w) {
      const int v = s_warp[w];
      if (w < warp) woff += v;
      tot += v;
    }
    if (t < H) s_off[t] = carry + woff + incl - cnt;
    carry += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) s_off[H] = carry;
  __syncthreads();
  const int ncand = carry;
  int running = 0;                             // links emitted by earlier rounds (same in all threads)

  for (int first = 0; first < ncand; first += LB_T * LB_CPT) {
    unsigned mask[LB_CPT];
    int node[LB_CPT];
    // ---- 1. arithmetic
#pragma unroll
    for (int k = 0; k < LB_CPT; ++k) {
      mask[k] = 0;
      node[k] = 0;
      const int cnd = first + k * LB_T + threadIdx.x;
      if (cnd >= ncand) continue;
      int lo = 0, hi = H - 1;                  // last row whose prefix is <= cnd
      while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (s_off[mid] <= cnd) lo = mid; else hi = mid - 1;
      }
      const int l = cnd - s_off[lo], n1 = s_n1[lo];
      const int i = l < n1 ? s_a1[lo] + l : s_a2[lo] + (l - n1), j = j0 + lo;
      // coordinates of the 3 x 3 neighbourhood: integers are exact in fp64, so xi + 1.0 is
      // (double)(i + 1) bit for bit and the disc test below is the rasteriser's
      const double xi = (double)i, yj = (double)j;
      if (S.ell) {
        if (inside_ellipse(xi, yj, S)) continue;
        const bool wi = i > 0, ei = i < c.nx - 1, so = j > 0, no = j < c.NY - 1;
        unsigned m = 0;
        if (ei && inside_ellipse(xi + 1.0, yj, S)) m |= 1u << 1;
        if (no && inside_ellipse(xi, yj + 1.0, S)) m |= 1u << 2;
        if (wi && inside_ellipse(xi - 1.0, yj, S)) m |= 1u << 3;
        if (so && inside_ellipse(xi, yj - 1.0, S)) m |= 1u << 4;
        if (ei && no && inside_ellipse(xi + 1.0, yj + 1.0, S)) m |= 1u << 5;
        if (wi && no && inside_ellipse(xi - 1.0, yj + 1.0, S)) m |= 1u << 6;
        if (wi && so && inside_ellipse(xi - 1.0, yj - 1.0, S)) m |= 1u << 7;
        if (ei && so && inside_ellipse(xi + 1.0, yj - 1.0, S)) m |= 1u << 8;
        mask[k] = m;
        node[k] = (int)((unsigned)i | ((unsigned)j << 16));
        continue;
      }
      const double dx0 = xi - xc, dy0 = yj - yc;
      const double sx0 = dx0 * dx0, sy0 = dy0 * dy0;
      const double d2 = sx0 + sy0;
      if (!(d2 > r2) || !(d2 <= rfar)) continue;
      const double dxm = (xi - 1.0) - xc, dxp = (xi + 1.0) - xc;
      const double dym = (yj - 1.0) - yc, dyp = (yj + 1.0) - yc;
      const double sxm = dxm * dxm, sxp = dxp * dxp, sym = dym * dym, syp = dyp * dyp;
      const bool wi = i > 0, ei = i < c.nx - 1, so = j > 0, no = j < c.NY - 1;
      unsigned m = 0;
      if (ei && sxp + sy0 <= r2) m |= 1u << 1;
      if (no && sx0 + syp <= r2) m |= 1u << 2;
      if (wi && sxm + sy0 <= r2) m |= 1u << 3;
      if (so && sx0 + sym <= r2) m |= 1u << 4;
      if (ei && no && sxp + syp <= r2) m |= 1u << 5;
      if (wi && no && sxm + syp <= r2) m |= 1u << 6;
      if (wi && so && sxm + sym <= r2) m |= 1u << 7;
      if (ei && so && sxp + sym <= r2) m |= 1u << 8;
      mask[k] = m;
      node[k] = (int)((unsigned)i | ((unsigned)j << 16));
    }
    // ---- 2. flags of the candidates (flag 2 = newborn: a fluid node of the step the links are for)
    unsigned char fl[LB_CPT];
#pragma unroll
    for (int k = 0; k < LB_CPT; ++k)
      fl[k] = mask[k] ? flag[node_index(c, node[k] & 0xffff, (int)((unsigned)node[k] >> 16))] : 1;
#pragma unroll
    for (int k = 0; k < LB_CPT; ++k)
      if (fl[k] == 1) mask[k] = 0;
    // ---- 3. ownership of the solid neighbours, only if discs may overlap
    if (check_owner) {
#pragma unroll
      for (int k = 0; k < LB_CPT; ++k) {
        const int i = node[k] & 0xffff, j = (int)((unsigned)node[k] >> 16);
        unsigned keep = 0;
        for (unsigned t = mask[k]; t; t &= t - 1) {
          const int al = __ffs(t) - 1;
          // (a solid neighbour in a row this slab does not store: the link's parked value is not
          // needed here and the particle's force is summed by the slab that owns it)
          if (row_here(c, j + p_ey[al]) && owner[node_index(c, i + p_ex[al], j + p_ey[al])] == p) keep |= 1u << al;
        }
        mask[k] = keep;
      }
    }
    // ---- 4. prefix in candidate order: (k, warp, lane)
    unsigned long long pk = 0;                 // 16-bit link counts of this thread's candidates
#pragma unroll
    for (int k = 0; k < LB_CPT; ++k) pk |= (unsigned long long)__popc(mask[k]) << (16 * k);
    unsigned long long incl = pk;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const unsigned long long v = __shfl_up_sync(FULL, incl, d);
      if (lane >= d) incl += v;
    }
    if (lane == 31) s_wpk[warp] = incl;        // per-warp totals, still packed (<= 256 per field)
    __syncthreads();
    int before[LB_CPT];                        // links of earlier warps, per k
    int total[LB_CPT];
#pragma unroll
    for (int k = 0; k < LB_CPT; ++k) before[k] = total[k] = 0;
#pragma unroll
    for (int w = 0; w < LB_WARPS; ++w) {
      const unsigned long long v = s_wpk[w];
#pragma unroll
      for (int k = 0; k < LB_CPT; ++k) {
        const int n = (int)((v >> (16 * k)) & 0xffffu);
        if (w < warp) before[k] += n;
        total[k] += n;
      }
    }
    const unsigned long long excl = incl - pk;
    int btotal = 0;
#pragma unroll
    for (int k = 0; k < LB_CPT; ++k) btotal += total[k];
    if (running + btotal <= la.cap) {
      int kbase = running;
#pragma unroll
      for (int k = 0; k < LB_CPT; ++k) {
        unsigned m = mask[k];
        int off = kbase + before[k] + (int)((excl >> (16 * k)) & 0xffffu);
        kbase += total[k];
        while (m) {
          const int al = __ffs(m) - 1;
          m &= m - 1;
          s_node[off] = node[k];
          s_dir[off] = (unsigned char)al;
          ++off;
        }
      }
    } else if (threadIdx.x == 0) {
      atomicOr(status, ST_LINK_OVERFLOW);
    }
    running += btotal;
    __syncthreads();
  }
  // ---- 5. q and the ladder rung, one link per thread: how many of x_f - e, x_f - 2e are fluid
  // nodes inside the cavity (both flag bytes requested before either is tested)
  const int nl = running <= la.cap ? running : 0;
  const long long base = (long long)p * la.cap;
  for (int s = threadIdx.x; s < nl; s += LB_T) {
    const int nd = s_node[s];
    const int al = s_dir[s];
    const int i = nd & 0xffff, j = (int)((unsigned)nd >> 16);
    int a1 = i - p_ex[al], b1 = j - p_ey[al], a2 = i - 2 * p_ex[al], b2 = j - 2 * p_ey[al];
    if (c.periodic_x) {
      a1 = (a1 + c.nx) % c.nx;
      a2 = (a2 + c.nx) % c.nx;
    }
    const bool in1 = a1 >= 0 && a1 < c.nx && row_here(c, b1);
    const bool in2 = a2 >= 0 && a2 < c.nx && row_here(c, b2);
    const unsigned char f1 = in1 ? flag[node_index(c, a1, b1)] : 1;
    const unsigned char f2 = in2 ? flag[node_index(c, a2, b2)] : 1;
    const int behind = f1 == 1 ? 0 : (f2 == 1 ? 1 : 2);
    la.q[base + s] = S.ell ? link_q_ellipse((double)i, (double)j, al, S)
                           : link_q((double)i, (double)j, al, xc, yc, r);
    la.node[base + s] = nd;
    la.dir[base + s] = (unsigned char)(al | (behind << LINK_BEHIND_SHIFT));
  }
  if (threadIdx.x == 0) la.count[p] = nl;
  __syncthreads();   // the shared list is reused by the next particle
  }
}

// ------------------------------------------------------------------------------------------
// a5: repulsion grid
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
// the non-zero contributions of all batches are collected and then added in ascending particle id
// (warp min-reduction picks the next one), so the sum order is fixed whatever order the cell slots
// were filled in and however many candidates the nine cells hold.
// Called by warp 0 of the particle's CTA (k_move); s_cid / s_cfx / s_cfy: 32 entries each.
template <bool ELL>
__device__ __forceinline__ void integrate_particle(const ParticleArrays& pa, int cur, int ia, double cell,
                                                   int ncx, int ncy, const int* __restrict__ cell_count,
                                                   const int* __restrict__ cell_items,
                                                   int* __restrict__ status, const LbmConst& c,
                                                   int* s_cid, double* s_cfx, double* s_cfy) {
  const int lane = threadIdx.x & 31;
  const unsigned FULL = 0xffffffffu;
  const int nxt = cur ^ 1;
  const double PI = 3.14159265358979323846;
  const Shape SA = load_shape<ELL>(pa, cur, ia);
  const double ax = SA.x, ay = SA.y, ar = SA.r, ratio = pa.rho_ratio[ia];
  const double Ca = PI * SA.a * SA.b * (ratio * c.rho0 - c.rho0) * c.g;   // area pi a b
  double Fx = pa.Fx[ia], Fy = pa.Fy[ia];
  Fy += -(ratio * c.rho0 - c.rho0) * PI * SA.a * SA.b * c.g;
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
  int ncontrib = 0;
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
        const Shape SB = load_shape<ELL>(pa, cur, best);
        const double bx = SB.x, by = SB.y, br = SB.r;
        const double dx = ax - bx, dy = ay - by;
        const double reach = ar + br + c.rep_s;
        if (!(fabs(dx) > reach || fabs(dy) > reach)) {
          const double dist = sqrt(dx * dx + dy * dy);
          // gap along the line of centres through the support functions (two circles: ra + rb)
          double delta = dist - ar - br;
          if ((SA.ell || SB.ell) && dist > 0.0) {
            const double nxh = dx / dist, nyh = dy / dist;
            delta = dist - support_shape(SA, nxh, nyh) - support_shape(SB, nxh, nyh);
          }
          if (delta <= c.rep_s && dist > 0.0) {
            const double Cb = PI * SB.a * SB.b * (pa.rho_ratio[best] * c.rho0 - c.rho0) * c.g;
            const double mag = repulsion_mag(0.5 * (Ca + Cb), c, delta);
            fx = mag * (dx / dist);
            fy = mag * (dy / dist);
            id = best;
            has = true;
          }
        }
      }
    }
    // the non-zero contributions are parked in the warp's shared list (batch after batch, in slot
    // order); the sum itself waits until every batch has been seen
    const unsigned hm = __ballot_sync(FULL, has);
    if (has) {
      const int slot = ncontrib + __popc(hm & ((1u << lane) - 1u));
      if (slot < 32) {
        s_cid[slot] = id;
        s_cfx[slot] = fx;
        s_cfy[slot] = fy;
      }
    }
    ncontrib += __popc(hm);
  }
  // Sum in ascending particle id over ALL neighbours, whatever batch or cell slot they came from
  // (the slot order is the atomicAdd order of k_cover and varies from run to run): the oracle's
  // order, and the same bits on every run.  A disc has at most a handful of neighbours within the
  // repulsion range; more than 32 is reported as a capacity error.
  if (ncontrib > 32) {
    if (lane == 0) atomicOr(status, ST_CELL_OVERFLOW);
    ncontrib = 32;
  }
  __syncwarp();
  if (ncontrib > 0) {
    bool has = lane < ncontrib;
    const int id = has ? s_cid[lane] : 0x7fffffff;
    const double fx = has ? s_cfx[lane] : 0.0, fy = has ? s_cfy[lane] : 0.0;
    while (__any_sync(FULL, has)) {
      const int m = __reduce_min_sync(FULL, has ? id : 0x7fffffff);
      const int src = __ffs(__ballot_sync(FULL, has && id == m)) - 1;
      Fx += __shfl_sync(FULL, fx, src);
      Fy += __shfl_sync(FULL, fy, src);
      if (lane == src) has = false;
    }
  }
  if (lane != 0) return;
  double ahx, ahy;
  half_extents(SA, ahx, ahy);
  if (!c.periodic_x) {
    const double dW = (ax + 0.5) - ahx;
    if (dW <= c.rep_s) Fx += repulsion_mag(Ca, c, dW);
    const double dE = ((double)c.nx - 0.5 - ax) - ahx;
    if (dE <= c.rep_s) Fx -= repulsion_mag(Ca, c, dE);
  }
  const double dS = (ay + 0.5) - ahy;
  if (dS <= c.rep_s) Fy += repulsion_mag(Ca, c, dS);
  const double dN = ((double)c.NY - 0.5 - ay) - ahy;
  if (dN <= c.rep_s) Fy -= repulsion_mag(Ca, c, dN);

  double x = ax, y = ay, th = pa.theta[cur][ia];
  double ux = pa.ux[cur][ia], uy = pa.uy[cur][ia], om = pa.omega[cur][ia];
  double oc = SA.c, os = SA.s;
  if (!pa.fixed[ia]) {
    const double mass = ratio * c.rho0 * PI * SA.a * SA.b;
    const double inertia = SA.ell ? 0.25 * mass * (SA.a * SA.a + SA.b * SA.b) : 0.5 * mass * ar * ar;
    const double ux1 = ux + Fx / mass;
    const double uy1 = uy + Fy / mass;
    const double om1 = om + pa.Tz[ia] / inertia;
    if (SA.ell) {
      // orientation unit vector advanced by the Cayley rotation of the angle increment
      // (only +, -, *, /, sqrt: the oracle's operations)
      const double t = 0.5 * (0.5 * (om + om1));
      const double den = 1.0 + t * t;
      const double cr = (1.0 - t * t) / den, sr = (2.0 * t) / den;
      const double c1 = oc * cr - os * sr, s1 = os * cr + oc * sr;
      const double nrm = sqrt(c1 * c1 + s1 * s1);
      oc = c1 / nrm;
      os = s1 / nrm;
    }
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
  pa.cs[nxt][ia] = oc;
  pa.sn[nxt][ia] = os;
  pa.ux[nxt][ia] = ux;
  pa.uy[nxt][ia] = uy;
  pa.omega[nxt][ia] = om;
  if (!(isfinite(x) && isfinite(y) && isfinite(th) && isfinite(ux) && isfinite(uy) && isfinite(om)))
    atomicOr(status, ST_NONFINITE);
}

// ------------------------------------------------------------------------------------------
// a6, flags.  Zone sweep shared by both phases: rows dealt to the warps, lanes across x (no
// integer division for zones up to 32 nodes wide).
template <typename F>
__device__ __forceinline__ void for_zone(int i0, int i1, int j0, int j1, const LbmConst& c, F f) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int j = j0 + warp; j <= j1; j += (int)(blockDim.x >> 5)) {
    if (!row_here(c, j)) continue;
    for (int i = i0 + lane; i <= i1; i += 32)
      if (i >= 0 && i < c.nx) f(i, j);
  }
}

// a5 + first half of a6 in ONE kernel, one CTA per particle (grid-size agnostic): warp 0 integrates
// the particle (it needs only the OLD positions of its neighbours, the repulsion grid of this step
// and the particle's own force), then the whole CTA sweeps the particle's old zone:
// Phase A of the flag update: nodes owned by p that the disc at its NEW position no longer covers
// become newborn candidates (flag 2, owner NONE) and are appended to the newborn list.
// The repulsion grid and the newborn counter are double-buffered by the particle buffer index, so
// that nothing this kernel resets is still being read inside it: it zeroes the grid of buffer
// cur ^ 1 (last read by the previous step's integration; k_cover of this step refills it with the
// new positions) and appends to the newborn counter of this step (zeroed by the previous step's
// k_refill_commit).
template <bool ELL>
__global__ void __launch_bounds__(PT_MAX, 12)
k_move(ParticleArrays pa, int cur, int np, double cell, int ncx, int ncy,
       const int* __restrict__ cell_count_cur, const int* __restrict__ cell_items_cur,
       int* __restrict__ cell_count_nxt, int ncells,
       unsigned char* __restrict__ flag, int* __restrict__ owner,
       int* __restrict__ nb_node, int* __restrict__ nb_pid, int* __restrict__ nb_count, int nb_cap,
       int* __restrict__ status, int early, const LbmConst c) {
  __shared__ int s_cid[32];
  __shared__ double s_cfx[32], s_cfy[32];
  if (early) pdl_launch_dependents();
  pdl_wait();
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < ncells; k += gridDim.x * blockDim.x) cell_count_nxt[k] = 0;
  const int nxt = cur ^ 1;
  for (int p = blockIdx.x; p < np; p += gridDim.x) {   // grid-size agnostic
  if (threadIdx.x < 32)
    integrate_particle<ELL>(pa, cur, p, cell, ncx, ncy, cell_count_cur, cell_items_cur, status, c,
                            s_cid, s_cfx, s_cfy);
  __syncthreads();   // the new state (global memory, written by lane 0) is visible to the CTA
  if (pa.fixed[p]) continue;
  const Shape So = load_shape<ELL>(pa, cur, p), Sn = load_shape<ELL>(pa, nxt, p);
  int i0, i1, j0, j1;
  zone_shape(So, i0, i1, j0, j1);
  for_zone(i0, i1, j0, j1, c, [&](int i, int j) {
    if (!inside_shape((double)i, (double)j, So)) return;
    if (inside_shape((double)i, (double)j, Sn)) return;
    const long long x = node_index(c, i, j);
    if (owner[x] != p) return;
    owner[x] = OWNER_NONE;
    flag[x] = 2;
    const int e = atomicAdd(nb_count, 1);
    if (e < nb_cap) {
      nb_node[e] = (int)x;
      nb_pid[e] = p;
    } else {
      atomicOr(status, ST_NEWBORN_OVERFLOW);
    }
  });
  }
}

// Phase B: every node inside the disc at the position in buffer `buf` is solid; the lowest
// particle id wins the owner map (same rule as a from-scratch recomputation).
//
// Invariant: every node inside the disc of a particle with pa.ovl == 0 is owned by it.  Such a
// particle therefore only has to claim the nodes its move has newly covered (inside the new
// disc, outside the old one -- arithmetic), not re-read the owner of its whole disc.  The flag is
// sticky and is raised whenever two discs share a node: by the particle that finds a node of its
// disc owned by a lower id, and for the particle a lower id takes a node from.  A flagged particle
// (and every particle at set-up, `all` = 1) sweeps its whole disc, which also re-claims nodes
// another particle has just uncovered.
// Thread 0 also enters the particle into the repulsion grid of the step that will use this
// position (the grid of buffer `buf`; k_move has zeroed its counts).
template <bool ELL>
__global__ void __launch_bounds__(PT_MAX, 12)
k_cover(ParticleArrays pa, int buf, int np, int all, unsigned char* __restrict__ flag,
        int* __restrict__ owner, double cell, int ncx, int ncy, int* __restrict__ cell_count,
        int* __restrict__ cell_items, int* __restrict__ status, const int* __restrict__ bandp,
        int guard, int early, const LbmConst c) {
  if (early) pdl_launch_dependents();
  pdl_wait();
  const int Q = *bandp;   // > 0: band [0, Q); < 0: band [-Q, ny)
  for (int p = blockIdx.x; p < np; p += gridDim.x) {   // grid-size agnostic
  const Shape Sn = load_shape<ELL>(pa, buf, p);
  const double xn = Sn.x, yn = Sn.y;
  if (threadIdx.x == 0) {
    // safety net of the two-step band: no solid node within 4 rows of it (k_band_plan's margins
    // make this unreachable for any |U|, dU the method is stable at)
    if (Q > 0 && (int)floor(yn - Sn.r) < Q + guard) atomicOr(status, ST_BAND_REACHED);
    if (Q < 0 && (int)ceil(yn + Sn.r) > -Q - guard - 1) atomicOr(status, ST_BAND_REACHED);
    int ci = (int)floor(xn / cell), cj = (int)floor(yn / cell);
    ci = min(max(ci, 0), ncx - 1);
    cj = min(max(cj, 0), ncy - 1);
    const int cidx = cj * ncx + ci;
    const int slot = atomicAdd(&cell_count[cidx], 1);
    if (slot < CELL_CAP) cell_items[cidx * CELL_CAP + slot] = p;
    else atomicOr(status, ST_CELL_OVERFLOW);
  }
  if (!all && pa.fixed[p]) continue;
  const bool sweep = all || pa.ovl[p] != 0;
  const Shape So = load_shape<ELL>(pa, buf ^ 1, p);
  int i0, i1, j0, j1;
  zone_shape(Sn, i0, i1, j0, j1);
  for_zone(i0, i1, j0, j1, c, [&](int i, int j) {
    if (!inside_shape((double)i, (double)j, Sn)) return;
    if (!sweep && inside_shape((double)i, (double)j, So)) return;   // already ours
    const long long x = node_index(c, i, j);
    if (owner[x] == p) return;
    const int prev = atomicMin(&owner[x], p);
    if (prev != p) flag[x] = 1;
    if (prev < p) pa.ovl[p] = 1;                              // a lower id keeps the node
    else if (prev != OWNER_NONE) pa.ovl[prev] = 1;            // taken from a higher id
  });
  }
}

// ------------------------------------------------------------------------------------------
// Two-step band: the rows [0, Q) below the
// lowest particle are advanced two time steps per pass by k_stream_collide_2step for the next
// BAND_PERIOD steps (two periods of the banded schedule).  Within those steps no solid node, no link stencil (x_f - 2 e_i) and no refill
// stencil (x_new + 3 e_c and its upstream neighbours) may reach below row Q: with the lowest solid
// row >= floor(min_p(y_p - r_p)) that needs Q + 4 <= lowest solid row, plus what the particle can
// fall in BAND_PERIOD steps (its speed now, two nodes for its acceleration -- the stiffest
// repulsion of Eq. 15 gives 32 a = 1.7 -- one in reserve); k_cover checks it every step.
// A band of fewer than BAND_MIN rows is not worth its seam: Q = 0 (no band).  One CTA.
// Three steps per pass (h->band3; bands under the suspension only): the band kernel reads one more
// row above Q and a plan serves two periods of SIX steps: period 12, margin 8 instead of 8 and 7,
// and k_cover's safety net moves up by one row.
constexpr int BAND_PERIOD = 8;
constexpr int BAND_MIN = 28;
// orient: +1 only a band under the suspension (rows [0, Q), band[0] = Q), -1 only a band above
// it (rows [Q, ny), band[0] = -Q: a settled bed leaves the rows under the lid free), 0 whichever is
// larger (the plan at the start of a call; the orientation then stays fixed for the call, because
// the grids are sized for it).  qcap: most rows the band may have (the band kernel's grid).
__global__ void __launch_bounds__(1024)
k_band_plan(ParticleArrays pa, int cur, int np, int ny, int orient, int qcap, int period, int margin,
            int* __restrict__ band) {
  __shared__ double s_min[32], s_max[32];
  double low = 1.0e300, high = -1.0e300;
  for (int p = threadIdx.x; p < np; p += blockDim.x) {
    const double uy = pa.fixed[p] ? 0.0 : pa.uy[cur][p];
    low = fmin(low, pa.y[cur][p] - pa.r[p] - (double)period * fmax(-uy, 0.0));
    high = fmax(high, pa.y[cur][p] + pa.r[p] + (double)period * fmax(uy, 0.0));
  }
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    low = fmin(low, __shfl_xor_sync(0xffffffffu, low, d));
    high = fmax(high, __shfl_xor_sync(0xffffffffu, high, d));
  }
  if ((threadIdx.x & 31) == 0) {
    s_min[threadIdx.x >> 5] = low;
    s_max[threadIdx.x >> 5] = high;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) {
      low = fmin(low, s_min[w]);
      high = fmax(high, s_max[w]);
    }
    int below = 0, above = 0;   // rows of the two candidate bands
    int Qb = 0, Qt = ny;
    if (low == low && low < 1.0e9 && low > -1.0e9) {
      Qb = min((int)floor(low) - margin, ny - 8);
      below = Qb >= BAND_MIN ? min(Qb, qcap) : 0;
    }
    if (high == high && high < 1.0e9 && high > -1.0e9) {
      Qt = max((int)ceil(high) + margin, 8);
      above = ny - Qt >= BAND_MIN ? min(ny - Qt, qcap) : 0;
    }
    if (orient > 0) above = 0;
    if (orient < 0) below = 0;
    band[0] = (below == 0 && above == 0) ? 0 : (below >= above ? below : -(ny - above));
  }
}

// ------------------------------------------------------------------------------------------
// y-slabs: the force combine.  Every slab runs the bounce-back kernel on the links it can see, but
// only the slab whose own rows [own0, own1) hold a particle's centre sees ALL of its links (the
// halo is wider than r + 8): that slab's sum, in the single domain's order, is the particle's
// force; every other slab contributes zero.  buf = Fx[np], Fy[np], Tz[np].
__global__ void k_slab_forces_out(ParticleArrays pa, int cur, int np, int own0, int own1,
                                  double* __restrict__ buf) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= np) return;
  const double y = pa.y[cur][p];
  const bool mine = y >= (double)own0 && y < (double)own1;
  buf[p] = mine ? pa.Fx[p] : 0.0;
  buf[np + p] = mine ? pa.Fy[p] : 0.0;
  buf[2 * np + p] = mine ? pa.Tz[p] : 0.0;
}

__global__ void k_slab_forces_in(ParticleArrays pa, int np, const double* __restrict__ buf) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= np) return;
  pa.Fx[p] = buf[p];
  pa.Fy[p] = buf[np + p];
  pa.Tz[p] = buf[2 * np + p];
}

__global__ void k_add_buffer(double* __restrict__ dst, const double* __restrict__ src, int n) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) dst[k] = dst[k] + src[k];
}

} // namespace

// CTAs of a particle-chain kernel.  On the library's own stream (concurrent with the lattice
// kernel) the chain is throttled to h->chain_ctas CTAs: the lattice kernel keeps its full speed
// when it loses up to two of its nine CTA slots per SM to other work and the chain has the whole
// lattice kernel to hide under.  Alone on the caller's stream
// (set-up, sequential mode) a kernel gets one CTA per work item.
static int chain_grid(const lbm* h, int items, cudaStream_t st) {
  if (st == h->chain_own && h->chain_ctas > 0) return items < h->chain_ctas ? items : h->chain_ctas;
  return items;
}

// threads of a chain CTA: see PT_MAX / PT_THROTTLED
static int chain_threads(const lbm* h, int items, cudaStream_t st) {
  return (st == h->chain_own && h->chain_ctas > 0 && items > h->chain_ctas) ? PT_THROTTLED : PT_MAX;
}

// Programmatic dependent launch along the chain: every chain kernel waits for its predecessor in
// griddepcontrol.wait; whether it also lets its successor's CTAs come up at once
// (launch_dependents at its start).  On the library's chain stream it does not: the waiting CTAs
// of the queued kernels hold SM slots the lattice kernel -- or, with few particles, the running
// chain kernel itself -- needs (measured: config 2 50.7 -> 61.6 us with it).  Only set-up launches
// on the caller's stream and the sequential schedule pass 1 (harmless without the launch attribute).
static int chain_early(const lbm* h, cudaStream_t st) {
  return (st == h->chain_own && h->chain_ctas > 0) ? 0 : 1;
}

// rows of the largest effective zone the capacity admits (12N - 12 <= cap) and the
// dynamic shared memory of the link builder: the compacted list + four row tables
static int link_rows(const lbm* h) { return (h->la.cap + 12) / 12 + 2; }
static size_t link_smem(const lbm* h) {
  return ((size_t)h->la.cap + ((size_t)h->la.cap + 3) / 4 + 4 * (size_t)link_rows(h) + 4) * sizeof(int);
}

void launch_build_links(lbm* h, int which_buffer, cudaStream_t st, bool pdl) {
  if (h->np == 0) return;
  h->launches++;
  const int max_rows = link_rows(h);
  const int threads = chain_threads(h, h->np, st);
  auto kernel = threads == PT_MAX ? (h->n_ell ? k_build_links<true, PT_MAX / 32> : k_build_links<false, PT_MAX / 32>)
                                  : (h->n_ell ? k_build_links<true, PT_THROTTLED / 32> : k_build_links<false, PT_THROTTLED / 32>);
  launch_k(kernel, dim3(chain_grid(h, h->np, st)), dim3(threads), link_smem(h), st, pdl, h->pa, which_buffer, (const unsigned char*)h->flag, (const int*)h->owner,
           h->la, h->np, max_rows, h->status_dev, chain_early(h, st), h->C);
}

// The dynamic shared memory limit of the link builder is a per-function (per-device) attribute:
// it is only ever raised, to the largest need any live handle on this device has had, so a later
// handle with a smaller index array cannot take it away from an earlier one.
int particles_configure(lbm* h) {
  static size_t raised[64] = {0};
  const size_t smem = link_smem(h);
  const int dev = (h->device >= 0 && h->device < 64) ? h->device : 0;
  if (smem <= 48 * 1024 || smem <= raised[dev]) return 0;
  if (cudaFuncSetAttribute(k_build_links<false, PT_MAX / 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
      cudaFuncSetAttribute(k_build_links<true, PT_MAX / 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
      cudaFuncSetAttribute(k_build_links<false, PT_THROTTLED / 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
      cudaFuncSetAttribute(k_build_links<true, PT_THROTTLED / 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  raised[dev] = smem;
  return 0;
}

// integrator + phase A of the flag update for the particle buffer h->cur -> h->cur ^ 1
void launch_move(lbm* h, cudaStream_t st, bool pdl) {
  if (h->np == 0) return;
  h->launches++;
  const int c = h->cur;
  launch_k(h->n_ell ? k_move<true> : k_move<false>, dim3(chain_grid(h, h->np, st)), dim3(chain_threads(h, h->np, st)), 0, st, pdl,
           h->pa, c, h->np, h->cell, h->ncx, h->ncy, (const int*)h->cell_count[c],
           (const int*)h->cell_items[c], h->cell_count[c ^ 1], h->ncx * h->ncy, h->flag, h->owner,
           h->newborn_node, h->newborn_pid, h->newborn_count + c, h->newborn_cap, h->status_dev,
           chain_early(h, st), h->C);
}

// after add_particles every particle (fixed ones too) is rasterised with a full sweep; during
// stepping the fixed ones never move
void launch_cover(lbm* h, int which_buffer, cudaStream_t st, bool pdl) {
  if (h->np == 0) return;
  h->launches++;
  launch_k(h->n_ell ? k_cover<true> : k_cover<false>, dim3(chain_grid(h, h->np, st)), dim3(chain_threads(h, h->np, st)), 0, st, pdl,
           h->pa, which_buffer, h->np, h->primed ? 0 : 1, h->flag, h->owner, h->cell, h->ncx, h->ncy,
           h->cell_count[which_buffer], h->cell_items[which_buffer], h->status_dev,
           (const int*)(h->band_live ? h->band : h->band + 1), h->band3 ? 5 : 4, chain_early(h, st), h->C);
}

// rows [0, h->band[0]) of the next BAND_PERIOD steps go to the two-step kernel (positions of
// buffer h->cur); a plain launch: it starts after everything before it in `st` has completed
void launch_band_plan(lbm* h, cudaStream_t st) {
  h->launches++;
  k_band_plan<<<1, 1024, 0, st>>>(h->pa, h->cur, h->np, h->ny, h->band_orient, h->band_cap,
                                  h->band3 ? 12 : BAND_PERIOD, h->band3 ? 8 : 7, h->band);
}

void launch_slab_forces_out(lbm* h) {
  if (h->np == 0) return;
  h->launches++;
  k_slab_forces_out<<<(h->np + 255) / 256, 256, 0, h->stream>>>(h->pa, h->cur, h->np, h->own0, h->own1, h->force_buf);
}

void launch_slab_forces_in(lbm* h) {
  if (h->np == 0) return;
  h->launches++;
  k_slab_forces_in<<<(h->np + 255) / 256, 256, 0, h->stream>>>(h->pa, h->np, h->force_buf);
}

void launch_add_buffer(double* dst, const double* src, int n, cudaStream_t st) {
  if (n > 0) k_add_buffer<<<(n + 255) / 256, 256, 0, st>>>(dst, src, n);
}
