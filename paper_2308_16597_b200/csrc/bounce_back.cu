// bounce_back.cu -- rows a3, a4 and the refill half of a6.
//
// a3  Eqs. (9)/(10) PAPER.md:101-113: quadratic interpolated bounce-back with moving wall;
//     Eqs. (11)/(12) PAPER.md:119-126: thermal curved-wall bounce-back; fallback ladders of
//     DESIGN.md "Readings" when x_f - e_i or x_f - 2 e_i is not a fluid node.
// a4  Eqs. (13)/(14) PAPER.md:134-139: Galilean-invariant momentum exchange, summed per particle
//     in a fixed order: per-thread strided partial sums, warp xor-shuffle tree, then the four
//     warp partials in order -- no floating-point atomics, so the result is reproducible.
// a6  Eqs. (16)/(17) PAPER.md:151-163: normal quadratic extrapolation + MRT momentum constraint
//     for f, equilibrium for g, on nodes uncovered this step.
//
// Solid-slot parking: the bounced population f_ibar(x_f, t+1) is stored in slot
// A_ibar(x_b), x_b = x_f + e_i being the solid node of the link.  The fused stream-collide kernel
// pulls direction ibar at x_f from exactly that slot, and nothing else reads or writes it, so the
// link kernel and the lattice kernel never conflict and the lattice kernel needs no link list.
#include "collide.cuh"

namespace {

__constant__ int b_ex[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1};
__constant__ int b_ey[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1};
__constant__ int b_opp[9] = {0, 3, 4, 1, 2, 7, 8, 5, 6};
__constant__ double b_w[9] = {4.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9,
                              1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36};

constexpr int BT = 128;

// index of node (i+di, j+dj) or -1 if outside the cavity (x wraps when periodic)
__device__ __forceinline__ long long node_at(const LbmConst& c, int i, int j, int di, int dj) {
  int a = i + di, b = j + dj;
  if (b < 0 || b >= c.ny) return -1;
  if (a < 0 || a >= c.nx) {
    if (!c.periodic_x) return -1;
    a = (a + c.nx) % c.nx;
  }
  return (long long)b * c.px + a;
}

__global__ void __launch_bounds__(BT)
k_bounce_back(double* __restrict__ A, LinkArrays la, ParticleArrays pa, int cur, const LbmConst c) {
  const int p = blockIdx.x;
  const int n = la.count[p];
  const long long base = (long long)p * la.cap;
  const double xc = pa.x[cur][p], yc = pa.y[cur][p];
  const double Ux = pa.ux[cur][p], Uy = pa.uy[cur][p], Om = pa.omega[cur][p], Tw = pa.Tw[p];
  double Fx = 0.0, Fy = 0.0, Tz = 0.0;
  for (int s = threadIdx.x; s < n; s += BT) {
    const int xf = la.node[base + s];
    const int db = la.dir[base + s];
    const double q = la.q[base + s];
    const int al = db & LINK_DIR_MASK;
    const int nbehind = db >> LINK_BEHIND_SHIFT;   // fluid nodes behind x_f (link builder)
    const int ab = b_opp[al];
    const int i = xf % c.px, j = xf / c.px;
    const int ex = b_ex[al], ey = b_ey[al];
    // every population the ladder can ask for is fetched up front (independent loads in flight
    // together); a node that is not there is replaced by x_f and its value is not used
    const long long x1 = nbehind >= 1 ? node_at(c, i, j, -ex, -ey) : (long long)xf;
    const long long x2 = nbehind == 2 ? node_at(c, i, j, -2 * ex, -2 * ey) : (long long)xf;
    const double* Fi = A + (long long)al * c.ps;
    const double* Fb = A + (long long)ab * c.ps;
    const double fi0 = Fi[xf];
    const double fb0 = Fb[xf];
    const double fi1 = Fi[x1];
    const double fi2 = Fi[x2];
    const double fb1 = Fb[x1];
    double gi0 = 0.0, gb0 = 0.0, gi1 = 0.0;
    if (al <= 4) {
      const double* Gi = A + (long long)(9 + al) * c.ps;
      const double* Gb = A + (long long)(9 + ab) * c.ps;
      gi0 = Gi[xf];
      gb0 = Gb[xf];
      gi1 = Gi[x1];
    }
    // wall point and wall velocity u_w = U_c + Omega x (x_w - x_c)
    const double rwx = ((double)i + q * ex) - xc;
    const double rwy = ((double)j + q * ey) - yc;
    const double uwx = Ux - Om * rwy;
    const double uwy = Uy + Om * rwx;
    const double wall = 6.0 * b_w[al] * c.rho0 * ((double)b_ex[ab] * uwx + (double)b_ey[ab] * uwy);
    double fbb;
    if (q <= 0.5) {
      if (nbehind == 2)
        fbb = q * (2.0 * q + 1.0) * fi0 + (1.0 - 4.0 * q * q) * fi1 - q * (1.0 - 2.0 * q) * fi2 + wall;
      else if (nbehind == 1)
        fbb = 2.0 * q * fi0 + (1.0 - 2.0 * q) * fi1 + wall;
      else
        fbb = fi0 + wall;
    } else {
      if (nbehind >= 1) {
        const double cq = 1.0 / (q * (2.0 * q + 1.0));
        fbb = cq * fi0 + ((2.0 * q - 1.0) / q) * fb0 - ((2.0 * q - 1.0) / (2.0 * q + 1.0)) * fb1 + cq * wall;
      } else {
        fbb = (fi0 + (2.0 * q - 1.0) * fb0) / (2.0 * q) + wall / (2.0 * q);
      }
    }
    const long long xb = (long long)(j + ey) * c.px + (i + ex);   // solid node of the link
    A[(long long)ab * c.ps + xb] = fbb;                           // parked for the pull at x_f
    if (al <= 4) {
      double cd2 = 0.0, cd4 = 1.0;
      if (nbehind >= 1) {
        cd2 = (2.0 * q - 1.0) / (2.0 * q + 1.0);
        cd4 = 2.0 / (2.0 * q + 1.0);
      } else {
        gi1 = 0.0;
      }
      const double gbb = (-gi0 + cd2 * gi1 + cd2 * gb0) + cd4 * (2.0 * c.wT * Tw);
      A[(long long)(9 + ab) * c.ps + xb] = gbb;
    }
    // Eqs. (13), (14)
    const double dpx = fi0 * ((double)ex - uwx) - fbb * ((double)b_ex[ab] - uwx);
    const double dpy = fi0 * ((double)ey - uwy) - fbb * ((double)b_ey[ab] - uwy);
    Fx += dpx;
    Fy += dpy;
    Tz += rwx * dpy - rwy * dpx;
  }
  // deterministic reduction
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    Fx += __shfl_xor_sync(0xffffffffu, Fx, d);
    Fy += __shfl_xor_sync(0xffffffffu, Fy, d);
    Tz += __shfl_xor_sync(0xffffffffu, Tz, d);
  }
  __shared__ double s_red[3][BT / 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) {
    s_red[0][warp] = Fx;
    s_red[1][warp] = Fy;
    s_red[2][warp] = Tz;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0, t = 0.0;
#pragma unroll
    for (int w = 0; w < BT / 32; ++w) {
      a += s_red[0][w];
      b += s_red[1][w];
      t += s_red[2][w];
    }
    pa.Fx[p] = a;
    pa.Fy[p] = b;
    pa.Tz[p] = t;
  }
}

// f_k(y, t+1) for every k at a node y that was fluid at t: the same pull the lattice kernel does
__device__ __forceinline__ void pull_f(const double* __restrict__ A, const LbmConst& c, int i, int j,
                                       double (&f)[9]) {
  const long long y = (long long)j * c.px + i;
#pragma unroll
  for (int k = 0; k < 9; ++k) {
    const long long s = node_at(c, i, j, -b_ex[k], -b_ey[k]);
    f[k] = s >= 0 ? A[(long long)k * c.ps + s] : A[(long long)b_opp[k] * c.ps + y];
  }
}

__global__ void k_refill(const double* __restrict__ A, double* __restrict__ B,
                         const unsigned char* __restrict__ flag, const int* __restrict__ nb_node,
                         const int* __restrict__ nb_pid, const int* __restrict__ nb_count, int nb_cap,
                         ParticleArrays pa, int cur, const LbmConst c) {
  const int n = min(*nb_count, nb_cap);
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const int x = nb_node[e];
    if (flag[x] != 2) continue;   // covered again by another particle in the same step
    const int p = nb_pid[e];
    const int i = x % c.px, j = x / c.px;
    // state at t+1 (cur already points at the new buffer)
    const double dxn = (double)i - pa.x[cur][p], dyn = (double)j - pa.y[cur][p];
    // e_c maximises n . e_alpha/|e_alpha|, ties -> lowest alpha; separately rounded operations
    int ec = 1;
    double best = -1.0e300;
#pragma unroll
    for (int a = 1; a <= 8; ++a) {
      double s = __dadd_rn(__dmul_rn(dxn, (double)b_ex[a]), __dmul_rn(dyn, (double)b_ey[a]));
      if (a >= 5) s = __dmul_rn(s, 0.70710678118654752440);
      if (s > best) { best = s; ec = a; }
    }
    const double uwx = pa.ux[cur][p] - pa.omega[cur][p] * dyn;
    const double uwy = pa.uy[cur][p] + pa.omega[cur][p] * dxn;
    int nvalid = 0;
    int si[3], sj[3];
    for (int k = 1; k <= 3; ++k) {
      const long long s = node_at(c, i, j, k * b_ex[ec], k * b_ey[ec]);
      if (s < 0 || flag[s] != 0) break;   // must be fluid at t and at t+1
      si[k - 1] = (int)(s % c.px);
      sj[k - 1] = (int)(s / c.px);
      nvalid = k;
    }
    double f[9], g[5];
    if (nvalid == 0) {
      const double u2 = uwx * uwx + uwy * uwy;
#pragma unroll
      for (int k = 0; k < 9; ++k) {
        const double eu = (double)b_ex[k] * uwx + (double)b_ey[k] * uwy;
        f[k] = b_w[k] * c.rho0 * (1.0 + 3.0 * eu + 4.5 * eu * eu - 1.5 * u2);
      }
    } else {
      double f1[9];
      pull_f(A, c, si[0], sj[0], f1);
      if (nvalid == 1) {
#pragma unroll
        for (int k = 0; k < 9; ++k) f[k] = f1[k];
      } else {
        double f2[9];
        pull_f(A, c, si[1], sj[1], f2);
        if (nvalid == 2) {
#pragma unroll
          for (int k = 0; k < 9; ++k) f[k] = 2.0 * f1[k] - f2[k];
        } else {
          double f3[9];
          pull_f(A, c, si[2], sj[2], f3);
#pragma unroll
          for (int k = 0; k < 9; ++k) f[k] = 3.0 * f1[k] - 3.0 * f2[k] + f3[k];   // Eq. (16)
        }
      }
    }
    // MRT velocity constraint: set j = rho_new u_w, all other moments unchanged:
    // f += M^-1 (dj_x e_jx + dj_y e_jy), rows j_x, j_y of M have norm^2 6
    double rho = 0.0, jx = 0.0, jy = 0.0;
#pragma unroll
    for (int k = 0; k < 9; ++k) {
      rho += f[k];
      jx += (double)b_ex[k] * f[k];
      jy += (double)b_ey[k] * f[k];
    }
    const double djx = (rho * uwx - jx) * (1.0 / 6.0), djy = (rho * uwy - jy) * (1.0 / 6.0);
#pragma unroll
    for (int k = 1; k < 9; ++k) f[k] += (double)b_ex[k] * djx + (double)b_ey[k] * djy;
    // Eq. (17): g = g_eq(T_w, u_w)
    const double Tw = pa.Tw[p];
    g[0] = c.wT0 * Tw;
#pragma unroll
    for (int k = 1; k < 5; ++k) g[k] = c.wT * Tw + 0.5 * ((double)b_ex[k] * uwx + (double)b_ey[k] * uwy) * Tw;
    // the resident state is post-collision: collide the refilled node now
    mrt_collide(f, g, c);
#pragma unroll
    for (int k = 0; k < 9; ++k) B[(long long)k * c.ps + x] = f[k];
#pragma unroll
    for (int k = 0; k < 5; ++k) B[(long long)(9 + k) * c.ps + x] = g[k];
    // flag[x] stays 2 until k_newborn_clear: other threads of this kernel still test their
    // stencil nodes against it
  }
}

// newborn nodes are ordinary fluid nodes from the next step on
__global__ void k_newborn_clear(unsigned char* __restrict__ flag, const int* __restrict__ nb_node,
                                const int* __restrict__ nb_count, int nb_cap) {
  const int n = min(*nb_count, nb_cap);
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const int x = nb_node[e];
    if (flag[x] == 2) flag[x] = 0;
  }
}

} // namespace

void launch_bounce_back(lbm* h) {
  if (h->np == 0) return;
  h->launches++;
  k_bounce_back<<<h->np, BT, 0, h->stream>>>(h->A, h->la, h->pa, h->cur, h->C);
}

void launch_refill(lbm* h) {
  if (h->np == 0) return;
  int blocks = (h->np * 4 + 127) / 128;   // a handful of newborn nodes per particle and step
  if (blocks > 1184) blocks = 1184;
  h->launches++;
  k_refill<<<blocks, 128, 0, h->stream>>>(h->A, h->B, h->flag, h->newborn_node, h->newborn_pid,
                                          h->newborn_count, h->newborn_cap, h->pa, h->cur, h->C);
  h->launches++;
  k_newborn_clear<<<blocks, 128, 0, h->stream>>>(h->flag, h->newborn_node, h->newborn_count,
                                                 h->newborn_cap);
}
