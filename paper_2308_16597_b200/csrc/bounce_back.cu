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

// memory index of node (i+di, j+dj), j a GLOBAL row, or -1 if it lies outside the cavity (x wraps
// when periodic) or in a row this handle does not store (y-slabs: such a node is farther from the
// slab's own rows than anything the slab's own results depend on)
__device__ __forceinline__ long long node_at(const LbmConst& c, int i, int j, int di, int dj) {
  int a = i + di, b = j + dj;
  if (!row_here(c, b)) return -1;
  if (a < 0 || a >= c.nx) {
    if (!c.periodic_x) return -1;
    a = (a + c.nx) % c.nx;
  }
  return node_index(c, a, b);
}

__global__ void __launch_bounds__(BT, 8)
k_bounce_back(double* __restrict__ A, LinkArrays la, ParticleArrays pa, int cur, int np, int early,
              const LbmConst c) {
  if (early) pdl_launch_dependents();
  pdl_wait();   // the previous step's refill commit (and, through it, everything before)
  __shared__ double s_red[3][BT / 32];
  for (int p = blockIdx.x; p < np; p += gridDim.x) {   // grid-size agnostic (one CTA per particle, or fewer)
  const int n = la.count[p];
  const long long base = (long long)p * la.cap;
  const double xc = pa.x[cur][p], yc = pa.y[cur][p];
  const double Ux = pa.ux[cur][p], Uy = pa.uy[cur][p], Om = pa.omega[cur][p], Tw = pa.Tw[p];
  double Fx = 0.0, Fy = 0.0, Tz = 0.0;
  for (int s = threadIdx.x; s < n; s += BT) {
    const int nd = la.node[base + s];
    const int db = la.dir[base + s];
    const double q = la.q[base + s];
    const int al = db & LINK_DIR_MASK;
    const int nbehind = db >> LINK_BEHIND_SHIFT;   // fluid nodes behind x_f (link builder)
    const int ab = b_opp[al];
    const int i = nd & 0xffff, j = (int)((unsigned)nd >> 16);
    const int xf = (int)node_index(c, i, j);
    const int ex = b_ex[al], ey = b_ey[al];
    // the populations this link's rung of the ladder needs, all requested before the first use
    // (independent loads in flight together); q <= 1/2 interpolates upstream of x_f in plane
    // alpha, q > 1/2 downstream of the wall in plane alpha-bar
    const bool lo = q <= 0.5;
    const long long x1 = nbehind >= 1 ? node_at(c, i, j, -ex, -ey) : (long long)xf;
    const long long x2 = nbehind == 2 ? node_at(c, i, j, -2 * ex, -2 * ey) : (long long)xf;
    // Axis directions (alpha <= 4) live in pair planes (f_k, g_k): one 16-byte access brings the
    // flow and the temperature population of a node and direction together, and the bounced pair
    // is parked with one 16-byte store.
    double fi0, fa, fc, gi0 = 0.0, gb0 = 0.0, gi1 = 0.0;
    if (al <= 4) {
      const double* Pi = A + 2 * (long long)al * c.ps;
      const double* Pb = A + 2 * (long long)ab * c.ps;
      const double2 a0 = *reinterpret_cast<const double2*>(Pi + 2 * (long long)xf);
      const double2 b0 = *reinterpret_cast<const double2*>(Pb + 2 * (long long)xf);
      const double2 a1 = *reinterpret_cast<const double2*>(Pi + 2 * x1);
      fc = lo ? Pi[2 * x2] : Pb[2 * x1];        // f_i(x_f - 2 e_i)  | f_ibar(x_f - e_i)
      fi0 = a0.x;
      fa = lo ? a1.x : b0.x;                    // f_i(x_f - e_i)    | f_ibar(x_f)
      gi0 = a0.y;
      gb0 = b0.y;
      gi1 = a1.y;
    } else {
      const double* Fi = A + (long long)(al + 5) * c.ps;
      const double* Fb = A + (long long)(ab + 5) * c.ps;
      fi0 = Fi[xf];
      fa = lo ? Fi[x1] : Fb[xf];
      fc = lo ? Fi[x2] : Fb[x1];
    }
    // wall point and wall velocity u_w = U_c + Omega x (x_w - x_c)
    const double rwx = ((double)i + q * ex) - xc;
    const double rwy = ((double)j + q * ey) - yc;
    const double uwx = Ux - Om * rwy;
    const double uwy = Uy + Om * rwx;
    const double wall = 6.0 * b_w[al] * c.rho0 * ((double)b_ex[ab] * uwx + (double)b_ey[ab] * uwy);
    // two reciprocals serve every coefficient of Eqs. (10)-(12) (within an ulp of the quotients)
    const double inv = 1.0 / (2.0 * q + 1.0);
    const double tq = 2.0 * q - 1.0;
    double fbb;
    if (lo) {
      if (nbehind == 2)
        fbb = q * (2.0 * q + 1.0) * fi0 + (1.0 - 4.0 * q * q) * fa - q * (1.0 - 2.0 * q) * fc + wall;
      else if (nbehind == 1)
        fbb = 2.0 * q * fi0 + (1.0 - 2.0 * q) * fa + wall;
      else
        fbb = fi0 + wall;
    } else {
      const double rq = 1.0 / q;
      if (nbehind >= 1) {
        const double cq = rq * inv;
        fbb = cq * fi0 + (tq * rq) * fa - (tq * inv) * fc + cq * wall;
      } else {
        fbb = (fi0 + tq * fa + wall) * (0.5 * rq);
      }
    }
    const long long xb = node_index(c, i + ex, j + ey);   // solid node of the link
    const bool park = row_here(c, j + ey);                // (always, except on a slab's outermost ghost row)
    if (al <= 4) {
      double cd2 = 0.0, cd4 = 1.0;
      if (nbehind >= 1) {
        cd2 = tq * inv;
        cd4 = 2.0 * inv;
      } else {
        gi1 = 0.0;
      }
      const double gbb = (-gi0 + cd2 * gi1 + cd2 * gb0) + cd4 * (2.0 * c.wT * Tw);
      // parked for the pull at x_f: the pair (f_ibar, g_ibar) of the solid node
      if (park) *reinterpret_cast<double2*>(A + 2 * (long long)ab * c.ps + 2 * xb) = make_double2(fbb, gbb);
    } else if (park) {
      A[(long long)(ab + 5) * c.ps + xb] = fbb;
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
  __syncthreads();   // s_red is reused by the next particle
  }
}

// a6: one WARP per newborn node.  Lane l < 27 fetches population k = l % 9 of stencil node
// s = l / 9, i.e. f_k(x_new + (s+1) e_c, t+1) = the same pull the lattice kernel does at a node
// that was fluid at t (upstream slot of A, which holds a parked value where the upstream node is
// solid; the node's own opposite slot at a cavity wall), so the 27 gathers are in flight
// together; the extrapolation, the momentum constraint, Eq. (17) and the collision are then
// evaluated redundantly by every lane and lane k < 14 stores population k -- into the stash
// record of the list entry, not into B: the kernel reads only A, the flags and the particle state
// of t+1, so it runs in the particle chain UNDER the lattice kernel, whose zero fill of non-fluid
// lanes may still touch the node's slots in B; k_refill_commit copies the record into B after it.
constexpr int RW = 8;   // warps (newborn nodes) per CTA
__global__ void __launch_bounds__(RW * 32, 4)
k_refill(const double* __restrict__ A, double* __restrict__ stash,
         const unsigned char* __restrict__ flag, int* __restrict__ nb_node,
         const int* __restrict__ nb_pid, const int* __restrict__ nb_count, int nb_cap,
         ParticleArrays pa, int cur, const LbmConst c) {
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int n = min(*nb_count, nb_cap);
  for (int e = blockIdx.x * RW + (threadIdx.x >> 5); e < n; e += gridDim.x * RW) {
    const int x = nb_node[e];
    if (flag[x] != 2) {           // covered again by another particle in the same step:
      if (lane == 0) nb_node[e] = -1;   // the commit kernel skips the entry without a flag load
      continue;
    }
    const int p = nb_pid[e];
    const int i = x % c.px, j = x / c.px + c.yoff;   // j: global row
    // state at t+1 (cur already points at the new buffer)
    const double dxn = (double)i - pa.x[cur][p], dyn = (double)j - pa.y[cur][p];
    // e_c maximises n . e_alpha/|e_alpha|, ties -> lowest alpha; separately rounded operations
    // outward normal of the wall at the node: radial for a circle; for an ellipse the gradient of
    // (u/a)^2 + (v/b)^2 turned back into the lattice frame (explicitly rounded, as the oracle)
    double nrx = dxn, nry = dyn;
    {
      const double ea = pa.a[p], eb = pa.b[p];
      if (ea != eb) {
        const double oc = pa.cs[cur][p], os = pa.sn[cur][p];
        const double u = __dadd_rn(__dmul_rn(dxn, oc), __dmul_rn(dyn, os));
        const double v = __dsub_rn(__dmul_rn(dyn, oc), __dmul_rn(dxn, os));
        const double gu = __ddiv_rn(__ddiv_rn(u, ea), ea), gv = __ddiv_rn(__ddiv_rn(v, eb), eb);
        nrx = __dsub_rn(__dmul_rn(gu, oc), __dmul_rn(gv, os));
        nry = __dadd_rn(__dmul_rn(gu, os), __dmul_rn(gv, oc));
      }
    }
    int ec = 1;
    double best = -1.0e300;
#pragma unroll
    for (int a = 1; a <= 8; ++a) {
      double s = __dadd_rn(__dmul_rn(nrx, (double)b_ex[a]), __dmul_rn(nry, (double)b_ey[a]));
      if (a >= 5) s = __dmul_rn(s, 0.70710678118654752440);
      if (s > best) { best = s; ec = a; }
    }
    const double uwx = pa.ux[cur][p] - pa.omega[cur][p] * dyn;
    const double uwy = pa.uy[cur][p] + pa.omega[cur][p] * dxn;
    const double Tw = pa.Tw[p];
    // stencil node of this lane and whether it is fluid at t and at t+1 (flag 0)
    const int st = lane / 9, k = lane % 9;
    const long long snode = lane < 27 ? node_at(c, i, j, (st + 1) * b_ex[ec], (st + 1) * b_ey[ec]) : -1;
    const bool ok = snode >= 0 && flag[snode] == 0;
    const unsigned okm = __ballot_sync(FULL, ok);
    int nvalid = 0;                                   // leading run of valid stencil nodes
    if (okm & 1u) { nvalid = 1; if (okm & (1u << 9)) { nvalid = 2; if (okm & (1u << 18)) nvalid = 3; } }
    double v = 0.0;
    if (lane < 27 && st < nvalid) {
      const int ci = (int)(snode % c.px), cj = (int)(snode / c.px) + c.yoff;
      const long long src = node_at(c, ci, cj, -b_ex[k], -b_ey[k]);
      v = src >= 0 ? A[f_at(k, src, c.ps)] : A[f_at(b_opp[k], snode, c.ps)];
    }
    double f[9], g[5];
#pragma unroll
    for (int kk = 0; kk < 9; ++kk) {
      const double f1 = __shfl_sync(FULL, v, kk);
      const double f2 = __shfl_sync(FULL, v, 9 + kk);
      const double f3 = __shfl_sync(FULL, v, 18 + kk);
      if (nvalid == 3) f[kk] = 3.0 * f1 - 3.0 * f2 + f3;   // Eq. (16)
      else if (nvalid == 2) f[kk] = 2.0 * f1 - f2;
      else f[kk] = f1;
    }
    if (nvalid == 0) {
      const double u2 = uwx * uwx + uwy * uwy;
#pragma unroll
      for (int kk = 0; kk < 9; ++kk) {
        const double eu = (double)b_ex[kk] * uwx + (double)b_ey[kk] * uwy;
        f[kk] = b_w[kk] * c.rho0 * (1.0 + 3.0 * eu + 4.5 * eu * eu - 1.5 * u2);
      }
    }
    // MRT velocity constraint: set j = rho_new u_w, all other moments unchanged:
    // f += M^-1 (dj_x e_jx + dj_y e_jy), rows j_x, j_y of M have norm^2 6
    double rho = 0.0, jx = 0.0, jy = 0.0;
#pragma unroll
    for (int kk = 0; kk < 9; ++kk) {
      rho += f[kk];
      jx += (double)b_ex[kk] * f[kk];
      jy += (double)b_ey[kk] * f[kk];
    }
    const double djx = (rho * uwx - jx) * (1.0 / 6.0), djy = (rho * uwy - jy) * (1.0 / 6.0);
#pragma unroll
    for (int kk = 1; kk < 9; ++kk) f[kk] += (double)b_ex[kk] * djx + (double)b_ey[kk] * djy;
    // Eq. (17): g = g_eq(T_w, u_w)
    g[0] = c.wT0 * Tw;
#pragma unroll
    for (int kk = 1; kk < 5; ++kk)
      g[kk] = c.wT * Tw + 0.5 * ((double)b_ex[kk] * uwx + (double)b_ey[kk] * uwy) * Tw;
    // the resident state is post-collision: collide the refilled node now
    mrt_collide(f, g, c);
    double out = 0.0;
#pragma unroll
    for (int kk = 0; kk < 9; ++kk) if (lane == kk) out = f[kk];
#pragma unroll
    for (int kk = 0; kk < 5; ++kk) if (lane == 9 + kk) out = g[kk];
    if (lane < 14) stash[(long long)e * 14 + lane] = out;
    // flag[x] stays 2 until k_refill_commit: other warps of this kernel (and the link builder,
    // which counts 2 as fluid) still test it
  }
}

// After the lattice kernel: the refilled populations go into B and the newborn nodes become
// ordinary fluid nodes.  16 threads per list entry (one per population, two idle), all in one warp.
// Entries whose node was covered again in the same step were marked -1 by k_refill.  Also zeroes
// the OTHER newborn counter, the one the next step's k_move appends to.
__global__ void k_refill_commit(double* __restrict__ B, const double* __restrict__ stash,
                                unsigned char* __restrict__ flag, const int* __restrict__ nb_node,
                                const int* __restrict__ nb_count, int* __restrict__ nb_count_next,
                                int nb_cap, int early, const HaloPush hp, const LbmConst c) {
  if (early) pdl_launch_dependents();
  pdl_wait();
  if (blockIdx.x == 0 && threadIdx.x == 0) *nb_count_next = 0;
  const int n = min(*nb_count, nb_cap);
  const long long total = (long long)n * 16;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const int e = (int)(t >> 4), k = (int)(t & 15);
    const int x = nb_node[e];
    if (x < 0) continue;
    if (k < 14) {
      const double v = stash[(long long)e * 14 + k];
      if (k < 9) B[f_at(k, x, c.ps)] = v;
      else B[g_at(k - 9, x, c.ps)] = v;
      // y-slabs: a newborn node in a row next to a cut also goes to the neighbour's ghost row
      const int j = x / c.px;
      if (hp.lo && j >= hp.lo_start && j < hp.lo_end) {
        const long long xp = x + (long long)hp.lo_shift * c.px;
        if (k < 9) hp.lo[f_at(k, xp, hp.lo_ps)] = v; else hp.lo[g_at(k - 9, xp, hp.lo_ps)] = v;
      }
      if (hp.hi && j >= hp.hi_start && j < hp.hi_end) {
        const long long xp = x + (long long)hp.hi_shift * c.px;
        if (k < 9) hp.hi[f_at(k, xp, hp.hi_ps)] = v; else hp.hi[g_at(k - 9, xp, hp.hi_ps)] = v;
      }
    } else if (k == 15) flag[x] = 0;
  }
}

} // namespace

void launch_bounce_back(lbm* h, cudaStream_t st, bool pdl) {
  if (h->np == 0) return;
  h->launches++;
  launch_k(k_bounce_back, dim3(h->np), dim3(BT), 0, st, pdl, h->A, h->la, h->pa, h->cur, h->np,
           h->chain_ctas > 0 ? 0 : 1, h->C);
}

// newborn list of the step whose particle buffer index is h->cur (called before cur is flipped)
void launch_refill(lbm* h, cudaStream_t st) {
  if (h->np == 0) return;
  int blocks = (h->np + RW - 1) / RW;   // a handful of newborn nodes per particle and step
  if (blocks > 1184) blocks = 1184;
  if (st != h->stream && h->chain_ctas > 0 && blocks > h->chain_ctas / 2) blocks = h->chain_ctas / 2;
  h->launches++;
  k_refill<<<blocks, RW * 32, 0, st>>>(h->A, h->stash, h->flag, h->newborn_node, h->newborn_pid,
                                        h->newborn_count + h->cur, h->newborn_cap, h->pa, h->cur ^ 1, h->C);
}

void launch_refill_commit(lbm* h, int step_parity, cudaStream_t st, bool pdl, const HaloPush* hp) {
  if (h->np == 0) return;
  int blocks = (h->np * 16 + 255) / 256;
  if (blocks > 1184) blocks = 1184;
  h->launches++;
  launch_k(k_refill_commit, dim3(blocks), dim3(256), 0, st, pdl, h->B, (const double*)h->stash, h->flag,
           (const int*)h->newborn_node, (const int*)(h->newborn_count + step_parity),
           h->newborn_count + (step_parity ^ 1), h->newborn_cap, h->chain_ctas > 0 ? 0 : 1,
           hp ? *hp : HaloPush{nullptr, 0, 0, 0, 0, nullptr, 0, 0, 0, 0}, h->C);
}
