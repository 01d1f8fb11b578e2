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
#include <algorithm>
#include <cstring>

#include <cuda.h>   // CUtensorMap and the encoder's signature; the entry point is looked up at run time

#include "collide.cuh"

namespace {

// lattice tables as constexpr functions so that fully unrolled loops fold them to immediates
__host__ __device__ constexpr int ex_of(int k) { return (k == 1 || k == 5 || k == 8) - (k == 3 || k == 6 || k == 7); }
__host__ __device__ constexpr int ey_of(int k) { return (k == 2 || k == 5 || k == 6) - (k == 4 || k == 7 || k == 8); }
__host__ __device__ constexpr int opp_of(int k) { return k == 0 ? 0 : (k <= 4 ? ((k + 1) % 4) + 1 : ((k - 3) % 4) + 5); }

constexpr int SC_THREADS = 128;

// Where the rows of the state a node pulls from live.  Normally every row j sits in one copy of
// the populations at node index j*px + i.  Along the seam of a two-step band (DESIGN.md "Two steps
// per pass below the suspension") the rows below the seam row Q come from elsewhere: from the
// band's own copy (which runs two steps behind / ahead of the rest), or, for the single row Q-1 at
// the intermediate time, from the spare row ny of the same copy.
struct RowsPlain {
  const double* A;
  int px;
  __device__ __forceinline__ const double* base(int) const { return A; }
  __device__ __forceinline__ long long row0(int sj) const { return (long long)sj * px; }
};
struct RowsSeam {
  const double* top;   // rows outside the band
  const double* low;   // rows of the band: [0, Q), or [Q, ny) for a band under the lid (upper)
  int Q;
  int low_row;         // >= 0: every band row is stored as this row of `low` (the spare row)
  int px;
  bool upper;
  __device__ __forceinline__ bool inband(int sj) const { return upper ? sj >= Q : sj < Q; }
  __device__ __forceinline__ const double* base(int sj) const { return inband(sj) ? low : top; }
  __device__ __forceinline__ long long row0(int sj) const {
    return (long long)((inband(sj) && low_row >= 0) ? low_row : sj) * px;
  }
};

// generic pull with cavity-wall handling; nodes on the lattice rim and the rows along a band seam
// take this path.  Fully unrolled and inlined so that f, g stay in registers.
template <typename Rows>
__device__ __forceinline__ void pull_boundary(const Rows& R, const LbmConst& c, int i,
                                              int j, double (&f)[9], double (&g)[5]) {
  const double* __restrict__ Aj = R.base(j);
  const long long x = R.row0(j) + i;
#pragma unroll
  for (int k = 0; k < 9; ++k) {
    int si = i - ex_of(k), sj = j - ey_of(k);
    bool in = (sj >= 0 && sj < c.ny);
    if (si < 0 || si >= c.nx) {
      if (c.periodic_x) si = (si + c.nx) % c.nx; else in = false;
    }
    f[k] = in ? R.base(sj)[f_at(k, R.row0(sj) + si, c.ps)] : Aj[f_at(opp_of(k), x, c.ps)];
  }
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    int si = i - ex_of(k), sj = j - ey_of(k);
    bool in = (sj >= 0 && sj < c.ny);
    int wall = sj < 0 ? 2 : 3;
    if (si < 0 || si >= c.nx) {
      if (c.periodic_x) si = (si + c.nx) % c.nx;
      else { in = false; wall = si < 0 ? 0 : 1; }
    }
    if (in) g[k] = R.base(sj)[g_at(k, R.row0(sj) + si, c.ps)];
    else {
      const double gb = Aj[g_at(opp_of(k), x, c.ps)];
      g[k] = c.wall_type[wall] == 1 ? (2.0 * c.wT * c.wall_T[wall] - gb) : gb;
    }
  }
}

__device__ __forceinline__ double2 ldg2(const double* p) {
  return __ldg(reinterpret_cast<const double2*>(p));
}

// f_k(x, t+1), g_k(x, t+1) of node (i, j) pulled from the post-collision state A.  Interior nodes:
// five 16-byte loads of the (f_k, g_k) pairs of the axis directions and four 8-byte loads of the
// diagonal f_k, each coalesced across the warp (the pair planes shifted by one node stay 16-byte
// aligned); rim nodes take the wall path.
__device__ __forceinline__ void pull_node(const double* __restrict__ A, const LbmConst& c, int i, int j,
                                          double (&f)[9], double (&g)[5]) {
  if (i >= 1 && i < c.nx - 1 && j >= 1 && j < c.ny - 1) {
    const long long x = (long long)j * c.px + i;
    const long long ps = c.ps;
    const int px = c.px;
    const double* __restrict__ P = A + 2 * x;           // pair planes: node x at doubles 2x, 2x+1
    const double2 p0 = ldg2(P);
    const double2 p1 = ldg2(P + 2 * ps - 2);
    const double2 p2 = ldg2(P + 4 * ps - 2 * px);
    const double2 p3 = ldg2(P + 6 * ps + 2);
    const double2 p4 = ldg2(P + 8 * ps + 2 * px);
    const double* __restrict__ D = A + 10 * ps + x;     // diagonal planes f5..f8
    f[5] = __ldg(D - px - 1);
    f[6] = __ldg(D + ps - px + 1);
    f[7] = __ldg(D + 2 * ps + px + 1);
    f[8] = __ldg(D + 3 * ps + px - 1);
    f[0] = p0.x; g[0] = p0.y;
    f[1] = p1.x; g[1] = p1.y;
    f[2] = p2.x; g[2] = p2.y;
    f[3] = p3.x; g[3] = p3.y;
    f[4] = p4.x; g[4] = p4.y;
  } else {
    pull_boundary(RowsPlain{A, c.px}, c, i, j, f, g);
  }
}

// the same nine accesses as stores (ps, px: plane stride and row pitch of the copy written to)
__device__ __forceinline__ void store_node_at(double* __restrict__ B, long long ps, int px, int i, int j,
                                              const double (&f)[9], const double (&g)[5]) {
  const long long x = (long long)j * px + i;   // j: the row of the copy the node is stored in
  double* __restrict__ O = B + 2 * x;
#pragma unroll
  for (int k = 0; k < 5; ++k) *reinterpret_cast<double2*>(O + 2 * k * ps) = make_double2(f[k], g[k]);
  double* __restrict__ Q = B + 10 * ps + x;
#pragma unroll
  for (int k = 0; k < 4; ++k) Q[k * ps] = f[5 + k];
}
__device__ __forceinline__ void store_node(double* __restrict__ B, const LbmConst& c, int i, int j,
                                           const double (&f)[9], const double (&g)[5]) {
  store_node_at(B, c.ps, c.px, i, j, f, g);
}

// one lattice update of node (i, j): pull, collide, store
__device__ __forceinline__ void update_node(const double* __restrict__ A, double* __restrict__ B,
                                            const LbmConst& c, int i, int j) {
  double f[9], g[5];
  pull_node(A, c, i, j, f, g);
  mrt_collide(f, g, c);
  store_node(B, c, i, j, f, g);
}

// One thread per node, 128-thread CTAs along x.  Solid (1) and newborn (2) nodes do no lattice
// update.  DRAM moves whole 32-byte sectors, and a partially written sector costs a read-modify-
// write there, so a non-fluid lane stores zeros into every plane in which its aligned 32-byte
// sector (2 lanes of a pair plane, 4 lanes of a diagonal plane) also holds a fluid lane: slots of
// non-fluid nodes in B are don't-care (a parked value is written by the NEXT step's bounce-back
// kernel, a newborn node by this step's refill kernel, both ordered after this kernel), and every
// store of the kernel then covers complete sectors.  Measured on config 3 (plain schedule, kernel
// alone): no fill 572 us; groups of 8 lanes in every plane 522 us; 4 lanes 518 us; one sector per
// plane type (2 / 4 lanes) 516 us; half a sector (1 / 2 lanes) 536 us.
//
// The flag update of this step (k_uncover / k_cover on the chain stream) may run concurrently:
// a node it covers (0 -> 1) was fluid at t, so updating it or not are both fine (its B slot is
// don't-care from t+1 on); a node it uncovers (1 -> 2) is skipped under either value.
//
// Two-step band: rows [0, Q), Q = *bandp,
// belong to k_stream_collide_2step, which advances them two steps per pass; this kernel covers
// the rows from Q + delta up.  In the first step of a pair (delta = -1) it also updates row Q-1,
// whose result -- the one row of the band the second step needs at the intermediate time -- goes
// to the spare row ny of B; rows below Q are read from the band's copy Alow.  In the second step
// (delta = 0, Alow = nullptr) row Q-1 is read from the spare row of A.  Rows Q-1 and Q take the
// generic pull; everything above is untouched by the band.  Q = 0: no band.
constexpr int SC_FILL_PAIR = 2;   // lanes of one 32-byte sector of a pair plane (16 B per node)
constexpr int SC_FILL_DIAG = 4;   // lanes of one 32-byte sector of a diagonal plane (8 B per node)
__global__ void __launch_bounds__(SC_THREADS, 9)
k_stream_collide(const double* __restrict__ A, double* __restrict__ B,
                 const unsigned char* __restrict__ flag, const double* __restrict__ Alow,
                 const int* __restrict__ bandp, int delta, int row0, int row1, const LbmConst c) {
  // programmatic dependent launch along the caller's stream: the next lattice kernel's CTAs may
  // come up as this grid's last wave drains; every kernel waits here for its predecessor's data
  pdl_launch_dependents();
  pdl_wait();
  // band[0] > 0: rows [0, Q) are the band; < 0: rows [Q, ny) with Q = -band[0] (a band under the
  // lid, above a settled bed: the same scheme mirrored -- this kernel then covers the rows BELOW
  // Q, and in the first step of a pair also row Q, into the spare row); 0: none
  const int Qs = *bandp;
  const bool upper = Qs < 0;
  const int Q = upper ? -Qs : Qs;
  const int i = blockIdx.x * SC_THREADS + threadIdx.x;
  int jfirst = row0, jend = row1;
  if (Q > 0) {
    if (upper) jend = min(row1, Q - delta);
    else jfirst = max(row0, Q + delta);
  }
  // The grid has one CTA row per lattice row the host EXPECTS this launch to cover (it knows the
  // band height of the previous lbm_step call); the loop takes care of a band that has shrunk
  // since (normally it runs once).
  // [row0, row1): the rows this launch may update at all (the whole lattice; a y-slab: its own rows)
  for (int j = blockIdx.y + jfirst; j < jend; j += gridDim.y) {
    const bool fluid = i < c.nx && flag[(long long)j * c.px + i] == 0;
    if (Q > 0 && (upper ? j >= Q - 1 : j <= Q)) {   // the two rows along the seam (all fluid)
      if (fluid) {
        double f[9], g[5];
        const RowsSeam R{A, Alow ? Alow : A, Q, Alow ? -1 : c.ny, c.px, upper};
        pull_boundary(R, c, i, j, f, g);
        mrt_collide(f, g, c);
        store_node(B, c, i, R.inband(j) ? c.ny : j, f, g);
      }
      continue;
    }
    const unsigned m = __ballot_sync(0xffffffffu, fluid);
    if (fluid) {
      update_node(A, B, c, i, j);
      continue;
    }
    const unsigned lane = threadIdx.x & 31u;
    if (i >= c.px) continue;
    const long long x = (long long)j * c.px + i;
    // pair planes: SC_FILL_PAIR lanes x 16 B; diagonal planes: SC_FILL_DIAG lanes x 8 B
    if ((m >> (lane & ~(unsigned)(SC_FILL_PAIR - 1))) & ((1u << SC_FILL_PAIR) - 1u)) {
      double* __restrict__ O = B + 2 * x;
#pragma unroll
      for (int k = 0; k < 5; ++k) *reinterpret_cast<double2*>(O + 2 * k * c.ps) = make_double2(0.0, 0.0);
    }
    if ((m >> (lane & ~(unsigned)(SC_FILL_DIAG - 1))) & ((1u << SC_FILL_DIAG) - 1u)) {
      double* __restrict__ Q4 = B + 10 * c.ps + x;
#pragma unroll
      for (int k = 0; k < 4; ++k) Q4[k * c.ps] = 0.0;
    }
  }
}

// y-slabs: the lattice kernel of a slab updates its own rows [row0, row1) and, fused into the same
// pass, PUSHES the rows next to a cut into the neighbour slab's ghost rows (HaloPush: peer copies
// in the same process -- the same GPU in the tests, another GPU over NVLink with peer access): the
// halo exchange is the epilogue of the kernel that produces the data, not a separate copy.
__global__ void __launch_bounds__(SC_THREADS)
k_stream_collide_slab(const double* __restrict__ A, double* __restrict__ B,
                      const unsigned char* __restrict__ flag, int row0, int row1, const HaloPush hp,
                      const LbmConst c) {
  pdl_launch_dependents();
  pdl_wait();
  const int i = blockIdx.x * SC_THREADS + threadIdx.x;
  const int j = blockIdx.y + row0;
  if (j >= row1) return;
  const bool fluid = i < c.nx && flag[(long long)j * c.px + i] == 0;
  const unsigned m = __ballot_sync(0xffffffffu, fluid);
  if (fluid) {
    double f[9], g[5];
    pull_node(A, c, i, j, f, g);
    mrt_collide(f, g, c);
    store_node(B, c, i, j, f, g);
    if (hp.lo && j < hp.lo_end) store_node_at(hp.lo, hp.lo_ps, c.px, i, j + hp.lo_shift, f, g);
    if (hp.hi && j >= hp.hi_start) store_node_at(hp.hi, hp.hi_ps, c.px, i, j + hp.hi_shift, f, g);
    return;
  }
  const unsigned lane = threadIdx.x & 31u;
  if (i >= c.px) return;
  const long long x = (long long)j * c.px + i;
  if ((m >> (lane & ~(unsigned)(SC_FILL_PAIR - 1))) & ((1u << SC_FILL_PAIR) - 1u)) {
    double* __restrict__ O = B + 2 * x;
#pragma unroll
    for (int k = 0; k < 5; ++k) *reinterpret_cast<double2*>(O + 2 * k * c.ps) = make_double2(0.0, 0.0);
  }
  if ((m >> (lane & ~(unsigned)(SC_FILL_DIAG - 1))) & ((1u << SC_FILL_DIAG) - 1u)) {
    double* __restrict__ Q4 = B + 10 * c.ps + x;
#pragma unroll
    for (int k = 0; k < 4; ++k) Q4[k * c.ps] = 0.0;
  }
}

// ---- mbarrier helpers (shared memory, CTA scope)
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, unsigned parity) {
  const unsigned a = smem_u32(bar);
  unsigned ok;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(a), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void mbar_arrive(void* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// Row-wise hand-over between the warps (= tile rows) of a multi-step kernel.
// rb: row barriers [rows][2] (mbarriers, one arrival each): phases 1 and 3 of a tile
// complete [row][0], phases 2 and 4 [row][1], so that two completions of one barrier are always
// separated by the neighbours' observation of the first (a row cannot publish phase p + 2 before
// both neighbours have published p + 1, i.e. have seen p) and the parity wait stays unambiguous
// (mbarrier.arrive is a release at CTA scope: the warp's shared-memory reads and writes before it --
// __syncwarp orders the other lanes' -- are performed before a waiter that acquires it goes on)
__device__ __forceinline__ void row_publish(unsigned long long* rb, int row, int phase) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0)
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(rb + 2 * row + ((phase - 1) & 1))) : "memory");
}
__device__ __forceinline__ void row_wait(unsigned long long* rb, int row, int phase, int rows) {
  const unsigned parity = (unsigned)((phase - 1) >> 1) & 1u;   // two completions per barrier and tile
  if (row > 0) mbar_wait(rb + 2 * (row - 1) + ((phase - 1) & 1), parity);
  if (row < rows - 1) mbar_wait(rb + 2 * (row + 1) + ((phase - 1) & 1), parity);
}

// TWO time steps per pass over particle-free rows (traffic below 224 B per
// update).  A CTA owns a TB_X x TB_Y tile of output nodes.  Phase 1: its TB_W x TB_H threads
// update the tile plus a one-node halo from the state at t (the same pull + collide as the
// one-step kernel) and keep the result f+(x, t+1), g+(x, t+1) in shared memory, population-major.
// Phase 2: the tile's nodes pull from shared memory (walls as in pull_boundary, on tile-local
// indices, so the periodic wrap needs no arithmetic), collide again and store f+(x, t+2).  Per two
// updates a node costs (TB_W+2)(TB_H+2)/(TB_X TB_Y) = 1.46 reads and one write of its 112 B:
// 138 B per update instead of 224 B (the halo re-reads hit L2: 111 B of DRAM traffic measured);
// the arithmetic is the one-step kernel's, so the result is the same bit for bit.
//
// The kernel updates the rows [0, Q), Q = *bandp (bandp == nullptr: the whole lattice, the
// particle-free case).  Rows below Q are read from Aband, the rows Q and Q+1 the top tiles' halo
// needs from Atop; the band is written to Bband.  The tile rows are split into `nparts` contiguous
// shares, one per launch (part = which of them this is), so that the band's work can be spread
// over the steps of the pair it advances.
constexpr int TB_X = 30, TB_Y = 14;   // TB_W = 32: one warp per tile row
constexpr int TB_W = TB_X + 2, TB_H = TB_Y + 2;
constexpr int TB_THREADS = TB_W * TB_H;   // 512 = 16 warps
constexpr int TB_SMEM = 14 * TB_THREADS * (int)sizeof(double) + TB_H * 8;   // + one mbarrier per tile row

__global__ void __launch_bounds__(TB_THREADS)
k_stream_collide_2step(const double* __restrict__ Aband, const double* __restrict__ Atop,
                       double* __restrict__ Bband, const int* __restrict__ bandp, int nparts,
                       int part, const LbmConst c) {
  extern __shared__ double s_pop[];   // [14][TB_H][TB_W], then TB_H mbarriers
  unsigned long long* const rowbar = reinterpret_cast<unsigned long long*>(s_pop + 14 * TB_THREADS);
  pdl_launch_dependents();
  if (threadIdx.x < TB_H) mbar_init(rowbar + threadIdx.x, 1);
  __syncthreads();                    // (under the predecessor's tail: nothing of its data is touched yet)
  pdl_wait();
  const int Qs = bandp ? *bandp : c.ny;
  const bool upper = Qs < 0;                       // the band is [Q, ny) instead of [0, Q)
  const int Q = upper ? -Qs : min(Qs, c.ny);
  // part p owns the p-th contiguous share of the band's tile rows (neighbouring tile rows of one
  // launch share their halo rows through L2)
  const int tr0 = upper ? Q / TB_Y : 0;            // first tile row that holds band rows
  const int ntr = (upper ? (c.ny + TB_Y - 1) / TB_Y : (Q + TB_Y - 1) / TB_Y) - tr0;
  const int per_part = (ntr + nparts - 1) / nparts;
  if ((int)blockIdx.y >= per_part) return;
  const int tile_j0 = (tr0 + part * per_part + blockIdx.y) * TB_Y;
  if (upper ? tile_j0 >= c.ny : tile_j0 >= Q) return;
  const int tx = threadIdx.x % TB_W, ty = threadIdx.x / TB_W;
  const int i = blockIdx.x * TB_X - 1 + tx, j = tile_j0 - 1 + ty;
  // phase 1: node (i, j) of the halo'd tile, wrapped in x when periodic
  int iw = i;
  if (c.periodic_x) iw = i < 0 ? i + c.nx : (i >= c.nx ? i - c.nx : i);
  const bool exists = iw >= 0 && iw < c.nx && j >= 0 && j < c.ny && (upper ? j >= Q - 1 : j <= Q);
  double f[9], g[5];
  if (exists) {
    if (upper ? j - 1 >= Q : (j + 1 < Q || Q == c.ny)) pull_node(Aband, c, iw, j, f, g);
    else pull_boundary(RowsSeam{Atop, Aband, Q, -1, c.px, upper}, c, iw, j, f, g);   // rows Q-1, Q (warp-uniform)
    mrt_collide(f, g, c);
#pragma unroll
    for (int k = 0; k < 9; ++k) s_pop[k * TB_THREADS + threadIdx.x] = f[k];
#pragma unroll
    for (int k = 0; k < 5; ++k) s_pop[(9 + k) * TB_THREADS + threadIdx.x] = g[k];
  }
  // A warp is a tile row, and phase 2 of row ty pulls from rows ty - 1, ty, ty + 1 only: instead of
  // a CTA-wide barrier each row signals its own mbarrier and waits for its two neighbours', so the
  // sixteen warps drift apart and some rows' loads run under other rows' second collision.
  __syncwarp();
  if (tx == 0) mbar_arrive(rowbar + ty);
  if (ty == 0 || ty == TB_H - 1) return;             // halo rows have no phase 2
  mbar_wait(rowbar + ty - 1, 0);
  mbar_wait(rowbar + ty + 1, 0);
  // phase 2: the tile's own nodes
  if (tx < 1 || tx > TB_X || ty < 1 || ty > TB_Y || i >= c.nx || j >= c.ny || (upper ? j < Q : j >= Q)) return;
  if (i >= 1 && i < c.nx - 1 && j >= 1 && j < c.ny - 1) {
    // interior: every upstream neighbour is a node of the tile's halo'd image
    const double* __restrict__ S = s_pop + threadIdx.x;
#pragma unroll
    for (int k = 0; k < 9; ++k) f[k] = S[k * TB_THREADS - ey_of(k) * TB_W - ex_of(k)];
#pragma unroll
    for (int k = 0; k < 5; ++k) g[k] = S[(9 + k) * TB_THREADS - ey_of(k) * TB_W - ex_of(k)];
  } else {
#pragma unroll
    for (int k = 0; k < 9; ++k) {
      const int si = i - ex_of(k), sj = j - ey_of(k);
      bool in = (sj >= 0 && sj < c.ny);
      if ((si < 0 || si >= c.nx) && !c.periodic_x) in = false;
      f[k] = in ? s_pop[k * TB_THREADS + (ty - ey_of(k)) * TB_W + (tx - ex_of(k))]
                : s_pop[opp_of(k) * TB_THREADS + threadIdx.x];
    }
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      const int si = i - ex_of(k), sj = j - ey_of(k);
      bool in = (sj >= 0 && sj < c.ny);
      int wall = sj < 0 ? 2 : 3;
      if ((si < 0 || si >= c.nx) && !c.periodic_x) { in = false; wall = si < 0 ? 0 : 1; }
      if (in) g[k] = s_pop[(9 + k) * TB_THREADS + (ty - ey_of(k)) * TB_W + (tx - ex_of(k))];
      else {
        const double gb = s_pop[(9 + opp_of(k)) * TB_THREADS + threadIdx.x];
        g[k] = c.wall_type[wall] == 1 ? (2.0 * c.wT * c.wall_T[wall] - gb) : gb;
      }
    }
  }
  mrt_collide(f, g, c);
  store_node(Bband, c, i, j, f, g);
}

// THREE time steps per pass over a particle-free lattice: the same idea one level deeper.  A CTA
// of T3_W x T3_H threads owns a T3_X x T3_Y tile of output nodes and its two-node halo.  Level 1:
// every thread pulls its node of the halo'd tile from A and collides (state t+1) into its slot of
// ONE shared buffer.  Level 2: the threads of the tile dilated by one node pull from their
// neighbours' slots, and -- once the neighbour rows have pulled too, so that nobody reads those
// level-1 values any more -- write their collided result (t+2) back IN PLACE.  Level 3: the tile's own nodes pull level 2, collide and
// store f+(x, t+3) to B.  Per three updates a node costs (T3_W+2)(T3_H+2)/(T3_X T3_Y) = 1.82 reads
// and one write of its 112 B: 105 B per update requested (less from DRAM: the halo re-reads hit
// L2) against 137 B for two steps per pass and 224 B for one, for 1.26 collisions per update
// against 1.11.  Same pull, same collision: bit-identical to three passes of the one-step kernel.
constexpr int T3_X = 28, T3_Y = 12;
constexpr int T3_W = T3_X + 4, T3_H = T3_Y + 4;   // 32 x 16: one warp per row of the halo'd tile
constexpr int T3_THREADS = T3_W * T3_H;
constexpr int T3_SMEM = 14 * T3_THREADS * (int)sizeof(double) + 2 * T3_H * 8;   // + two mbarriers per tile row

// f_k, g_k of the node in slot `tid` (lattice column iw -- wrapped when periodic --, row j) pulled
// from the slots of its neighbours in the tile image s_pop[14][T3_THREADS]; cavity walls as in
// pull_boundary, with the node's own slot standing in for its own populations
__device__ __forceinline__ void pull_tile3(const double* s_pop, int tid, int iw, int j, const LbmConst& c,
                                           double (&f)[9], double (&g)[5]) {
  if (iw >= 1 && iw < c.nx - 1 && j >= 1 && j < c.ny - 1) {
    const double* __restrict__ S = s_pop + tid;
#pragma unroll
    for (int k = 0; k < 9; ++k) f[k] = S[k * T3_THREADS - ey_of(k) * T3_W - ex_of(k)];
#pragma unroll
    for (int k = 0; k < 5; ++k) g[k] = S[(9 + k) * T3_THREADS - ey_of(k) * T3_W - ex_of(k)];
    return;
  }
#pragma unroll
  for (int k = 0; k < 9; ++k) {
    const int si = iw - ex_of(k), sj = j - ey_of(k);
    bool in = (sj >= 0 && sj < c.ny);
    if ((si < 0 || si >= c.nx) && !c.periodic_x) in = false;
    f[k] = in ? s_pop[k * T3_THREADS + tid - ey_of(k) * T3_W - ex_of(k)]
              : s_pop[opp_of(k) * T3_THREADS + tid];
  }
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const int si = iw - ex_of(k), sj = j - ey_of(k);
    bool in = (sj >= 0 && sj < c.ny);
    int wall = sj < 0 ? 2 : 3;
    if ((si < 0 || si >= c.nx) && !c.periodic_x) { in = false; wall = si < 0 ? 0 : 1; }
    if (in) g[k] = s_pop[(9 + k) * T3_THREADS + tid - ey_of(k) * T3_W - ex_of(k)];
    else {
      const double gb = s_pop[(9 + opp_of(k)) * T3_THREADS + tid];
      g[k] = c.wall_type[wall] == 1 ? (2.0 * c.wT * c.wall_T[wall] - gb) : gb;
    }
  }
}

//
// BAND: the kernel advances the rows
// [0, Q), Q = *bandp, of a lattice WITH particles from the period's state t (every row of A at time
// t) to t+3 in B.  The rows Q .. Q+2 it needs as halo are ordinary fluid rows of the same copy
// (three steps per pass keep the band and the rows above it in the same copy at the start of every
// half period, so there is no seam inside this kernel): level 1 covers the rows up to Q+1, level 2
// up to Q, level 3 stores the rows below Q.  What the one-step kernel above the band needs at the
// intermediate times -- row Q-1 at t+1 and at t+2 -- is written by the tile that owns row Q-1 into
// the spare row ny: level 1's into B's (read by the second step of the half period), level 2's
// into A's (read by the third).  The tile rows are dealt to the three steps FROM THE TOP (part 0 =
// the top third): the rows >= Q of A are overwritten by the second step's one-step kernel, which
// runs after the parts 0 and 1 of the pass (stream order); part 2 only reads rows below Q.
template <bool BAND>
__global__ void __launch_bounds__(T3_THREADS, 2)
k_stream_collide_3step(const double* __restrict__ A, double* __restrict__ B, double* __restrict__ Aspare,
                       const int* __restrict__ bandp, int nparts, int part, const LbmConst c) {
  extern __shared__ double s_pop[];   // [14][T3_H][T3_W], then the row barriers [T3_H][2]
  unsigned long long* const rb = reinterpret_cast<unsigned long long*>(s_pop + 14 * T3_THREADS);
  pdl_launch_dependents();
  if (threadIdx.x < 2 * T3_H) mbar_init(rb + threadIdx.x, 1);
  __syncthreads();                    // (under the predecessor's tail)
  pdl_wait();
  const int tid = threadIdx.x;
  const int tx = tid % T3_W, ty = tid / T3_W;
  // A band under the lid (Qs < 0: rows [Q, ny), Q = -Qs, above a settled bed) is the same scheme
  // mirrored: halo rows Q-3 .. Q-1, row Q handed over, the parts dealt from the bottom.
  int Q = c.ny, tile_row = blockIdx.y;
  bool upper = false;
  if (BAND) {
    const int Qs = *bandp;
    if (Qs == 0) return;
    upper = Qs < 0;
    Q = upper ? -Qs : min(Qs, c.ny);
    const int tr0 = upper ? Q / T3_Y : 0;            // first tile row that holds band rows
    const int ntr = (upper ? (c.ny + T3_Y - 1) / T3_Y : (Q + T3_Y - 1) / T3_Y) - tr0;
    const int per_part = (ntr + nparts - 1) / nparts;
    if ((int)blockIdx.y >= per_part) return;
    tile_row = upper ? tr0 + part * per_part + (int)blockIdx.y
                     : tr0 + ntr - (part + 1) * per_part + (int)blockIdx.y;
    if (tile_row < tr0 || tile_row >= tr0 + ntr) return;
  }
  const int i = blockIdx.x * T3_X - 2 + tx, j = tile_row * T3_Y - 2 + ty;
  // the band's row next to the seam, in the tile that owns it, hands its levels 1 and 2 to the
  // rows outside the band
  const bool hand = BAND && j == (upper ? Q : Q - 1) && ty >= 2 && ty <= T3_H - 3 && tx >= 2 && tx <= T3_W - 3 &&
                    i >= 0 && i < c.nx;
  // rows of the band's side that level 1 / 2 / 3 cover
  const bool in1 = !BAND || (upper ? j >= Q - 2 : j <= Q + 1);
  const bool in2 = !BAND || (upper ? j >= Q - 1 : j <= Q);
  const bool in3 = !BAND || (upper ? j >= Q : j < Q);
  // periodic x: the columns -2, -1 and nx, nx+1 are images of nx-2, nx-1 and 0, 1
  int iw = i;
  if (c.periodic_x) iw = i < 0 ? i + c.nx : (i >= c.nx ? i - c.nx : i);
  const bool col1 = c.periodic_x ? (i >= -2 && i <= c.nx + 1 && iw >= 0 && iw < c.nx) : (i >= 0 && i < c.nx);
  const bool ex1 = col1 && j >= 0 && j < c.ny && in1;
  double f[9], g[5];
  // level 1: t -> t+1, from global memory
  if (ex1) {
    pull_node(A, c, iw, j, f, g);
    mrt_collide(f, g, c);
#pragma unroll
    for (int k = 0; k < 9; ++k) s_pop[k * T3_THREADS + tid] = f[k];
#pragma unroll
    for (int k = 0; k < 5; ++k) s_pop[(9 + k) * T3_THREADS + tid] = g[k];
    if (hand) store_node_at(B, c.ps, c.px, i, c.ny, f, g);
  }
  // No CTA-wide barriers: a warp is a tile row and hands over to its two neighbour rows only
  // (phase 1: level 1 written; 2: level 1 pulled; 3: level 2 written)
  row_publish(rb, ty, 1);
  row_wait(rb, ty, 1, T3_H);
  // level 2: t+1 -> t+2 on the tile dilated by one node, written back in place
  const bool ex2 = ex1 && tx >= 1 && tx <= T3_W - 2 && ty >= 1 && ty <= T3_H - 2 &&
                   (!c.periodic_x || (i >= -1 && i <= c.nx)) && in2;
  if (ex2) pull_tile3(s_pop, tid, iw, j, c, f, g);
  row_publish(rb, ty, 2);
  if (ex2) mrt_collide(f, g, c);
  row_wait(rb, ty, 2, T3_H);          // the neighbour rows have read this row's level-1 values
  if (ex2) {
    if (hand) store_node_at(Aspare, c.ps, c.px, i, c.ny, f, g);
#pragma unroll
    for (int k = 0; k < 9; ++k) s_pop[k * T3_THREADS + tid] = f[k];
#pragma unroll
    for (int k = 0; k < 5; ++k) s_pop[(9 + k) * T3_THREADS + tid] = g[k];
  }
  row_publish(rb, ty, 3);
  row_wait(rb, ty, 3, T3_H);
  // level 3: t+2 -> t+3 on the tile's own nodes, to global memory
  if (!(ex2 && tx >= 2 && tx <= T3_W - 3 && ty >= 2 && ty <= T3_H - 3 && i >= 0 && i < c.nx && in3)) return;
  pull_tile3(s_pop, tid, iw, j, c, f, g);
  mrt_collide(f, g, c);
  store_node(B, c, i, j, f, g);
}

// THREE time steps per pass, TMA-fed and persistent (the multi-step kernel IS a
// tile-movement kernel).  One CTA per SM for the whole launch; it walks the tiles b, b + G, b + 2G,
// ... (G = gridDim.x, x fastest: the ~148 tiles in flight are neighbours in a tile row, so their
// overlapping halos meet in L2).  A tile's input -- the state at t on the T3_X x T3_Y tile plus a
// three-node halo, as a TP_IW x TP_IH node image of all 14 populations in the HBM layout (pair
// planes interleaved) -- is fetched by TWO 3-D tensor copies (cp.async.bulk.tensor: box 72 x 18 x 5
// doubles of the pair planes, 36 x 18 x 4 of the diagonal planes; four extra columns on the left
// keep the box 16-byte aligned) into a ring of TP_STAGES images that signal an mbarrier each;
// rows and columns outside the lattice are zero-filled by the copy engine and never used (walls as
// in pull_boundary, the node's own slot standing in).  No thread computes a global load address.
//
// The 1024 threads are two groups of 512, each of which takes every other tile of the CTA's
// sequence and runs the three levels of k_stream_collide_3step on its image IN PLACE: pull from
// the neighbours' slots, (neighbours have pulled) collide, write back to the own slot, (neighbours
// have written) next level -- level 1 on the 32 x 16 nodes of the tile dilated by two, level 2 on
// 30 x 14, level 3 on 28 x 12 and from registers to B.  ROWSYNC (the default): the hand-over in
// brackets is per row -- a warp owns a tile row and waits for its two neighbour rows' mbarriers
// (row_publish / row_wait above); otherwise it is a named barrier of the whole group.  When a
// group has pulled level 3 its image is free: the group's warp 0 collects the other warps'
// arrivals (an mbarrier per stage with ROWSYNC, where the warps of a group may be tiles apart;
// bar.arrive / bar.sync otherwise) and one lane issues the copies for the CTA's tile after next but
// one into it, which land while both groups compute -- the loads of tile m + 3 overlap the
// arithmetic of tiles m + 1 and m + 2 instead of alternating with it.
// Same pull, same collision, same order: bit-identical to three passes of the one-step kernel.
constexpr int TP_IW = T3_W + 4, TP_IH = T3_H + 2;       // 36 x 18 node image
constexpr int TP_PLANE = TP_IW * TP_IH;
constexpr int TP_PAIR_DOUBLES = 5 * 2 * TP_PLANE;       // pair planes: (f_k, g_k) interleaved
constexpr int TP_IMG_DOUBLES = 14 * TP_PLANE;
constexpr int TP_IMG_BYTES = TP_IMG_DOUBLES * (int)sizeof(double);   // 72,576 = 567 x 128
constexpr int TP_STAGES = 3, TP_GROUPS = 2;
constexpr int TP_THREADS = TP_GROUPS * T3_THREADS;
constexpr int TP_SMEM = TP_STAGES * TP_IMG_BYTES + 80 + TP_GROUPS * 2 * T3_H * 8;   // + the stage and the row mbarriers

__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, void* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void group_sync(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(T3_THREADS) : "memory"); }
__device__ __forceinline__ void group_arrive(int id) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "n"(T3_THREADS) : "memory"); }

// f_k, g_k of the node in slot s of an image (lattice column i, row j) pulled from its neighbours'
// slots; cavity walls as in pull_boundary (closed cavity only: the kernel is not used with periodic x)
__device__ __forceinline__ void pull_img(const double* img, int s, int i, int j, const LbmConst& c,
                                         double (&f)[9], double (&g)[5]) {
  if (i >= 1 && i < c.nx - 1 && j >= 1 && j < c.ny - 1) {
    const double2* __restrict__ P = reinterpret_cast<const double2*>(img) + s;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      const double2 v = P[k * TP_PLANE - ey_of(k) * TP_IW - ex_of(k)];
      f[k] = v.x;
      g[k] = v.y;
    }
    const double* __restrict__ D = img + TP_PAIR_DOUBLES + s;
#pragma unroll
    for (int k = 5; k < 9; ++k) f[k] = D[(k - 5) * TP_PLANE - ey_of(k) * TP_IW - ex_of(k)];
    return;
  }
#pragma unroll
  for (int k = 0; k < 9; ++k) {
    const int si = i - ex_of(k), sj = j - ey_of(k);
    const bool in = sj >= 0 && sj < c.ny && si >= 0 && si < c.nx;
    const int kk = in ? k : opp_of(k);
    const int ss = in ? s - ey_of(k) * TP_IW - ex_of(k) : s;
    f[k] = kk <= 4 ? img[2 * (kk * TP_PLANE + ss)] : img[TP_PAIR_DOUBLES + (kk - 5) * TP_PLANE + ss];
  }
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const int si = i - ex_of(k), sj = j - ey_of(k);
    bool in = (sj >= 0 && sj < c.ny);
    int wall = sj < 0 ? 2 : 3;
    if (si < 0 || si >= c.nx) { in = false; wall = si < 0 ? 0 : 1; }
    if (in) g[k] = img[2 * (k * TP_PLANE + s - ey_of(k) * TP_IW - ex_of(k)) + 1];
    else {
      const double gb = img[2 * (opp_of(k) * TP_PLANE + s) + 1];
      g[k] = c.wall_type[wall] == 1 ? (2.0 * c.wT * c.wall_T[wall] - gb) : gb;
    }
  }
}
__device__ __forceinline__ void put_img(double* img, int s, const double (&f)[9], const double (&g)[5]) {
  double2* __restrict__ P = reinterpret_cast<double2*>(img) + s;
#pragma unroll
  for (int k = 0; k < 5; ++k) P[k * TP_PLANE] = make_double2(f[k], g[k]);
  double* __restrict__ D = img + TP_PAIR_DOUBLES + s;
#pragma unroll
  for (int k = 0; k < 4; ++k) D[k * TP_PLANE] = f[5 + k];
}

// Row-wise hand-over inside a group (ROWSYNC): warp w of a group owns row w of the dilated tile,
// and a level's pull of row r reads only rows r-1, r, r+1 of the level below, so instead of four
// group-wide barriers per tile each warp publishes how far it has come (two mbarriers per row,
// row_publish / row_wait; plain counters with st.release / ld.acquire cost a MEMBAR per store
// and lost) and waits for its two neighbours only: before writing its row back in place, that
// they have pulled; before pulling the next level, that they have written.  Neighbouring rows stay within one phase of each other, the sixteen
// warps of a group spread over the phases, and shared-memory phases of some warps run under the
// fp64 phases of others.
template <bool ROWSYNC>
__global__ void __launch_bounds__(TP_THREADS, 1)
k_stream_collide_3step_tma(const __grid_constant__ CUtensorMap tm_pair, const __grid_constant__ CUtensorMap tm_diag,
                           double* __restrict__ B, int ntx, int ntiles, const LbmConst c) {
  extern __shared__ __align__(128) unsigned char s_raw[];
  double* const imgs = reinterpret_cast<double*>(s_raw);
  unsigned long long* const full = reinterpret_cast<unsigned long long*>(s_raw + TP_STAGES * TP_IMG_BYTES);
  pdl_launch_dependents();
  const int grp = threadIdx.x / T3_THREADS, tid = threadIdx.x % T3_THREADS;
  const int tx = tid % T3_W, ty = tid / T3_W;
  const int s = (ty + 1) * TP_IW + tx + 2;               // the thread's slot in every image
  // tile m of this CTA's sequence -> stage m % TP_STAGES; one thread arms the stage's mbarrier with
  // the byte count and issues the two box copies
  auto fetch = [&](int m) {
    const int tile = blockIdx.x + m * gridDim.x;
    if (tile >= ntiles) return;
    const int st = m % TP_STAGES;
    const int i0 = (tile % ntx) * T3_X - 4, j0 = (tile / ntx) * T3_Y - 3;
    double* img = imgs + st * TP_IMG_DOUBLES;
    // One "full" barrier per stage AND consuming group (tile m belongs to group m % 2): with the
    // row-wise hand-over a warp can be more than three tiles of its group ahead of the slowest one,
    // i.e. at the stage's NEXT BUT ONE use -- on a barrier shared by both groups that use has the
    // parity of the one still in progress and the wait would pass on the old image (seen as one
    // corrupted run in 150-250).  Per group, consecutive completions are six tiles apart.
    unsigned long long* bar = full + st + TP_STAGES * (m % TP_GROUPS);
    mbar_expect_tx(bar, TP_IMG_BYTES);
    tma_load_3d(img, &tm_pair, 2 * i0, j0, 0, bar);
    tma_load_3d(img + TP_PAIR_DOUBLES, &tm_diag, i0, j0, 0, bar);
  };
  unsigned long long* const empty = full + 6;                   // ROWSYNC: image handed back (16 warps)
  unsigned long long* const rb = full + 10 + grp * (2 * T3_H);  // the group's row barriers [row][2]
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < TP_STAGES * TP_GROUPS; ++k) mbar_init(full + k, 1);
    if (ROWSYNC) {
      for (int st = 0; st < TP_STAGES; ++st) mbar_init(empty + st, T3_THREADS / 32);
      for (int k = 0; k < TP_GROUPS * 2 * T3_H; ++k) mbar_init(full + 10 + k, 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  pdl_wait();                                            // the previous pass has written A
  if (threadIdx.x == 0) {
#pragma unroll
    for (int m = 0; m < TP_STAGES; ++m) fetch(m);
  }
  for (int m = grp;; m += TP_GROUPS) {
    const int tile = blockIdx.x + m * gridDim.x;
    if (tile >= ntiles) break;
    const int st = m % TP_STAGES;
    double* img = imgs + st * TP_IMG_DOUBLES;
    const int i = (tile % ntx) * T3_X - 2 + tx, j = (tile / ntx) * T3_Y - 2 + ty;
    const bool ex1 = i >= 0 && i < c.nx && j >= 0 && j < c.ny;
    const bool ex2 = ex1 && tx >= 1 && tx <= T3_W - 2 && ty >= 1 && ty <= T3_H - 2;
    const bool ex3 = ex2 && tx >= 2 && tx <= T3_W - 3 && ty >= 2 && ty <= T3_H - 3;
    double f[9], g[5];
    mbar_wait(full + st + TP_STAGES * grp, (unsigned)(m / (TP_STAGES * TP_GROUPS)) & 1u);
    if (ROWSYNC) {
      // level 1: t -> t+1
      if (ex1) pull_img(img, s, i, j, c, f, g);
      row_publish(rb, ty, 1);                              // (release: the pulls are ordered before it)
      if (ex1) mrt_collide(f, g, c);
      row_wait(rb, ty, 1, T3_H);                                 // the neighbour rows have pulled
      if (ex1) put_img(img, s, f, g);
      row_publish(rb, ty, 2);
      // level 2: t+1 -> t+2
      row_wait(rb, ty, 2, T3_H);                                 // ... have written level 1
      if (ex2) pull_img(img, s, i, j, c, f, g);
      row_publish(rb, ty, 3);
      if (ex2) mrt_collide(f, g, c);
      row_wait(rb, ty, 3, T3_H);
      if (ex2) put_img(img, s, f, g);
      row_publish(rb, ty, 4);
      // level 3: t+2 -> t+3
      row_wait(rb, ty, 4, T3_H);
      if (ex3) pull_img(img, s, i, j, c, f, g);
    } else {
      // level 1: t -> t+1
      if (ex1) pull_img(img, s, i, j, c, f, g);
      group_sync(1 + grp);
      if (ex1) {
        mrt_collide(f, g, c);
        put_img(img, s, f, g);
      }
      group_sync(1 + grp);
      // level 2: t+1 -> t+2
      if (ex2) pull_img(img, s, i, j, c, f, g);
      group_sync(1 + grp);
      if (ex2) {
        mrt_collide(f, g, c);
        put_img(img, s, f, g);
      }
      group_sync(1 + grp);
      // level 3: t+2 -> t+3
      if (ex3) pull_img(img, s, i, j, c, f, g);
    }
    // ... to global memory; the image is free once everybody has pulled
    if (ROWSYNC) {
      // the warps of a group may be tiles apart here, so the image is handed back through an
      // mbarrier of its own (one arrival per warp; a named barrier would count a fast warp twice)
      __syncwarp();
      if ((tid & 31) == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(empty + st)) : "memory");
      if (tid < 32) {
        mbar_wait(empty + st, (unsigned)(m / TP_STAGES) & 1u);
        if (tid == 0) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          fetch(m + TP_STAGES);
        }
      }
    } else if (tid < 32) {
      group_sync(3 + grp);                               // every warp of the group has pulled
      if (tid == 0) {
        // the group's reads and in-place writes of this image (ordered before this point by the
        // barrier) come before the copy engine's writes into it
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        fetch(m + TP_STAGES);
      }
    } else {
      group_arrive(3 + grp);
    }
    if (ex3) {
      mrt_collide(f, g, c);
      store_node(B, c, i, j, f, g);
    }
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
  for (int k = 0; k < 9; ++k) f[k] = A[f_at(k, x, c.ps)];
#pragma unroll
  for (int k = 0; k < 5; ++k) g[k] = A[g_at(k, x, c.ps)];
  mrt_collide(f, g, c);
#pragma unroll
  for (int k = 0; k < 9; ++k) O[f_at(k, x, c.ps)] = f[k];
#pragma unroll
  for (int k = 0; k < 5; ++k) O[g_at(k, x, c.ps)] = g[k];
}

// f = f_eq(rho0, 0) = w_k rho0, g = g_eq(T0, 0) = wT_k T0 on every node (SURVEY 8(c) "Initial state")
__global__ void k_set_equilibrium(double* __restrict__ A, const LbmConst c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= c.px) return;
  const long long x = (long long)j * c.px + i;
  const double w[9] = {4.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36};
#pragma unroll
  for (int k = 0; k < 9; ++k) A[f_at(k, x, c.ps)] = w[k] * c.rho0;
  A[g_at(0, x, c.ps)] = c.wT0 * c.T0;
#pragma unroll
  for (int k = 1; k < 5; ++k) A[g_at(k, x, c.ps)] = c.wT * c.T0;
}

// g = g_eq(T, u = 0) from a dense nx*ny temperature field (lbm_set_temperature)
__global__ void k_set_temperature(double* __restrict__ A, const double* __restrict__ T, const LbmConst c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= c.nx) return;
  const long long x = (long long)j * c.px + i;
  const double t = T[(long long)j * c.nx + i];
  A[g_at(0, x, c.ps)] = c.wT0 * t;
#pragma unroll
  for (int k = 1; k < 5; ++k) A[g_at(k, x, c.ps)] = c.wT * t;
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
    ux[o] = pux[p] - pom[p] * ((double)(j + c.yoff) - py_[p]);
    uy[o] = puy[p] + pom[p] * ((double)i - px_[p]);
    T[o] = pTw[p];
    return;
  }
  double f[9], g[5];
#pragma unroll
  for (int k = 0; k < 9; ++k) f[k] = A[f_at(k, x, c.ps)];
#pragma unroll
  for (int k = 0; k < 5; ++k) g[k] = A[g_at(k, x, c.ps)];
  double r, vx, vy, t;
  macroscopic(f, g, c, post, r, vx, vy, t);
  rho[o] = r;
  ux[o] = vx;
  uy[o] = vy;
  T[o] = t;
}

// read-out of the populations: dense population-major planes f[9][ny*nx], g[5][ny*nx] (the
// layout lbm_get_fields hands out) from the paired device layout; `collide` = 1 before the first
// step, when the resident state is still pre-collision
__global__ void k_export(const double* __restrict__ A, const unsigned char* __restrict__ flag,
                         int collide, double* __restrict__ fo, double* __restrict__ go, const LbmConst c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= c.nx) return;
  const long long x = (long long)j * c.px + i;
  const long long o = (long long)j * c.nx + i, n = (long long)c.nx * c.ny;
  double f[9], g[5];
#pragma unroll
  for (int k = 0; k < 9; ++k) f[k] = A[f_at(k, x, c.ps)];
#pragma unroll
  for (int k = 0; k < 5; ++k) g[k] = A[g_at(k, x, c.ps)];
  if (collide && flag[x] == 0) mrt_collide(f, g, c);
  if (fo) {
#pragma unroll
    for (int k = 0; k < 9; ++k) fo[k * n + o] = f[k];
  }
  if (go) {
#pragma unroll
    for (int k = 0; k < 5; ++k) go[k * n + o] = g[k];
  }
}

inline dim3 grid_rows(int n, int ny, int threads) { return dim3((n + threads - 1) / threads, ny); }

} // namespace

// band == 0: the plain step (every row).  band == 1 / 2: first / second step of a pair of the
// banded schedule (lbm_capi.cu): rows from *h->band - 1 resp. *h->band up; low = the band's copy
// (first step only).  band == 3: first step of a half period of the three-step band (rows from
// *h->band up, the band's rows read in place from low = h->A; the later steps of the half period
// are band == 2: row Q-1 from the spare row).
void launch_stream_collide(lbm* h, int band, const double* low) {
  h->launches++;
  // banded steps: one CTA row per lattice row above the band as the host last saw it
  // (h->band_hint, 0 = unknown); the kernel's row loop covers whatever the band has lost since
  const int rows = band ? h->band_l1_rows : h->row1 - h->row0;
  launch_k(k_stream_collide, grid_rows(h->px, rows, SC_THREADS), dim3(SC_THREADS), 0, h->stream, h->use_pdl != 0,
           (const double*)h->A, h->B, (const unsigned char*)h->flag,
           (band == 1 || band == 3) ? low : (const double*)nullptr,
           (const int*)(band ? h->band : h->band + 1), band == 1 ? -1 : 0, h->row0, h->row1, h->C);
}

void launch_stream_collide_slab(lbm* h, const HaloPush& hp) {
  h->launches++;
  launch_k(k_stream_collide_slab, grid_rows(h->px, h->row1 - h->row0, SC_THREADS), dim3(SC_THREADS), 0, h->stream,
           h->use_pdl != 0, (const double*)h->A, h->B, (const unsigned char*)h->flag, h->row0, h->row1, hp, h->C);
}

int stream_collide_configure() {
  return (cudaFuncSetAttribute(k_stream_collide_2step, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               TB_SMEM) == cudaSuccess &&
          cudaFuncSetAttribute(k_stream_collide_3step<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               T3_SMEM) == cudaSuccess &&
          cudaFuncSetAttribute(k_stream_collide_3step<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               T3_SMEM) == cudaSuccess) ? 0 : -1;
}

// Tensor maps of the two copies of the populations for k_stream_collide_3step_tma: per copy one
// 3-D map of the five pair planes (2*px x ny x 5 doubles; rows and planes strided) and one of the
// four diagonal planes (px x ny x 4).  The spare row ny is outside the maps.  cuTensorMapEncodeTiled
// is a driver entry point; it is looked up through the runtime, so the library does not link libcuda.
// 0 = ok (h->tma_ok set), -1 = not available (the plain three-step kernel is used instead).
int stream_collide_tma_setup(lbm* h) {
  h->tma_ok = 0;
  if (h->C.periodic_x || h->is_slab) return -1;
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn encode = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess) {
      cudaGetLastError();
      p = nullptr;
    }
    return (encode_fn)p;
  }();
  if (!encode) return -1;
  if (cudaFuncSetAttribute(k_stream_collide_3step_tma<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TP_SMEM) !=
          cudaSuccess ||
      cudaFuncSetAttribute(k_stream_collide_3step_tma<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, TP_SMEM) !=
          cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  double* base[2] = {h->A, h->B};
  for (int cpy = 0; cpy < 2; ++cpy) {
    CUtensorMap tm;
    const cuuint32_t ones[3] = {1, 1, 1};
    {
      const cuuint64_t dims[3] = {(cuuint64_t)2 * h->px, (cuuint64_t)h->ny, 5};
      const cuuint64_t strides[2] = {(cuuint64_t)h->px * 16, (cuuint64_t)h->ps * 16};
      const cuuint32_t box[3] = {2 * TP_IW, TP_IH, 5};
      if (encode(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base[cpy], dims, strides, box, ones,
                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return -1;
      static_assert(sizeof(tm) == sizeof(h->tmaps[0]), "CUtensorMap is 128 bytes");
      std::memcpy(h->tmaps[2 * cpy], &tm, sizeof(tm));
    }
    {
      const cuuint64_t dims[3] = {(cuuint64_t)h->px, (cuuint64_t)h->ny, 4};
      const cuuint64_t strides[2] = {(cuuint64_t)h->px * 8, (cuuint64_t)h->ps * 8};
      const cuuint32_t box[3] = {TP_IW, TP_IH, 4};
      if (encode(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base[cpy] + 10 * h->ps, dims, strides, box, ones,
                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return -1;
      std::memcpy(h->tmaps[2 * cpy + 1], &tm, sizeof(tm));
    }
    h->tma_base[cpy] = base[cpy];
  }
  h->tma_ok = 1;
  return 0;
}

// particle-free closed cavity: every row, A -> B, three time steps, persistent TMA-fed kernel
void launch_stream_collide_3step_tma(lbm* h) {
  h->launches++;
  const int cpy = h->A == h->tma_base[0] ? 0 : 1;
  alignas(64) CUtensorMap tp, td;
  std::memcpy(&tp, h->tmaps[2 * cpy], sizeof(tp));
  std::memcpy(&td, h->tmaps[2 * cpy + 1], sizeof(td));
  const int ntx = (h->nx + T3_X - 1) / T3_X, nty = (h->ny + T3_Y - 1) / T3_Y;
  const int ntiles = ntx * nty;
  // One CTA per SM -- but not a grid that shares a factor with the tiles per row: a CTA would then
  // keep returning to the same few tile columns, and a launch in which every CTA stays in ONE
  // column takes 20 % longer (4096^2, 147 tiles per row: 1103 us with 147 CTAs against 898 us with
  // 148; 2048^2, 74 per row: 286 us with 148 against 234 us with 147; 1024^2, 37 per row: 80
  // against 68 us).  The largest grid coprime to ntx costs a few SMs at most.
  int grid = std::min(ntiles, h->sm_count > 0 ? h->sm_count : 148);
  auto gcd = [](int a, int b) { while (b) { const int t = a % b; a = b; b = t; } return a; };
  while (grid > 1 && ntx > 1 && gcd(grid, ntx) != 1) --grid;
  if (h->use_tma >= 2)
    launch_k(k_stream_collide_3step_tma<true>, dim3(grid), dim3(TP_THREADS), TP_SMEM, h->stream, h->use_pdl != 0, tp,
             td, h->B, ntx, ntiles, h->C);
  else
    launch_k(k_stream_collide_3step_tma<false>, dim3(grid), dim3(TP_THREADS), TP_SMEM, h->stream, h->use_pdl != 0, tp,
             td, h->B, ntx, ntiles, h->C);
}

// particle-free lattice: every row, A -> B, three time steps
void launch_stream_collide_3step(lbm* h) {
  h->launches++;
  const dim3 grid((h->nx + T3_X - 1) / T3_X, (h->ny + T3_Y - 1) / T3_Y);
  launch_k(k_stream_collide_3step<false>, grid, dim3(T3_THREADS), T3_SMEM, h->stream, h->use_pdl != 0,
           (const double*)h->A, h->B, (double*)nullptr, (const int*)nullptr, 1, 0, h->C);
}

// the band rows [0, *h->band) of a lattice with particles, three steps per pass: the part-th of
// nparts shares of the tile rows, counted from the top; src: the copy that holds every row at the
// start of the half period, dst: the other one
void launch_stream_collide_band3(lbm* h, double* src, double* dst, int nparts, int part) {
  h->launches++;
  const int tile_rows = (std::min(h->band_cap, h->ny) + T3_Y - 1) / T3_Y + 1;
  const dim3 grid((h->nx + T3_X - 1) / T3_X, (tile_rows + nparts - 1) / nparts);
  launch_k(k_stream_collide_3step<true>, grid, dim3(T3_THREADS), T3_SMEM, h->stream, h->use_pdl != 0,
           (const double*)src, dst, src, (const int*)h->band, nparts, part, h->C);
}

// particle-free lattice: every row, A -> B
void launch_stream_collide_2step(lbm* h) {
  h->launches++;
  const dim3 grid((h->nx + TB_X - 1) / TB_X, (h->ny + TB_Y - 1) / TB_Y);
  launch_k(k_stream_collide_2step, grid, dim3(TB_THREADS), TB_SMEM, h->stream, h->use_pdl != 0,
           (const double*)h->A, (const double*)h->A, h->B, (const int*)nullptr, 1, 0, h->C);
}

// the band rows [0, *h->band) of a lattice with particles: the part-th of nparts contiguous shares
void launch_stream_collide_band(lbm* h, const double* src_band, const double* src_top, double* dst_band,
                                int nparts, int part) {
  h->launches++;
  // CTAs of this kernel are expensive to launch even when they exit at once (512 threads, 57 KB):
  // the grid covers the band as the host last saw it plus a margin (k_band_plan keeps Q below it)
  // h->band_cap: the most rows the band may have in this call (k_band_plan clamps to it)
  const int tile_rows = (std::min(h->band_cap, h->ny) + TB_Y - 1) / TB_Y + 1;
  const dim3 grid((h->nx + TB_X - 1) / TB_X, (tile_rows + nparts - 1) / nparts);
  launch_k(k_stream_collide_2step, grid, dim3(TB_THREADS), TB_SMEM, h->stream, h->use_pdl != 0, src_band, src_top,
           dst_band, (const int*)h->band, nparts, part, h->C);
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

void launch_export(lbm* h, double* f_dense, double* g_dense) {
  h->launches++;
  k_export<<<grid_rows(h->nx, h->ny, 128), 128, 0, h->stream>>>(h->A, h->flag, h->primed ? 0 : 1,
                                                                f_dense, g_dense, h->C);
}

// ---- read-out that allocates nothing and touches none of the caller's workspace ----
// lbm_get_fields stages its dense outputs in the dead copy B of the workspace.  For callers that
// must not allocate and want the workspace left alone (include/lbm.h lbm_get_macroscopic_static)
// the same kernel writes into this file-scope array instead: 4 fields x LBM_STATIC_MAX_NODES
// doubles = 32 MiB, held by every GPU that loads the library until the process exits.  Every call
// shares it and it keeps the last call's contents; k_macroscopic writes every node of the
// nx x ny outputs it is asked for, so nothing has to start at zero.  Calls that overlap on the
// GPU (two handles on different streams) race on it.
static __device__ __align__(256) double g_static_fields[4 * (size_t)LBM_STATIC_MAX_NODES];

// The array's name is a host-side stand-in here, not a device address: the address is looked up
// once per device, with that device current (the caller's DeviceGuard), and handed to the kernel.
// 0 = ok, -1 = lattice too large, -2 = cudaGetSymbolAddress failed.
int launch_macroscopic_static(lbm* h, double** fields4) {
  static double* addr[64] = {nullptr};
  if ((long long)h->nx * h->ny > (long long)LBM_STATIC_MAX_NODES) return -1;
  const int dev = (h->device >= 0 && h->device < 64) ? h->device : 0;
  if (!addr[dev]) {
    double* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_static_fields) != cudaSuccess || !p) {
      cudaGetLastError();
      return -2;
    }
    addr[dev] = p;
  }
  double* base = addr[dev];
  const size_t n = (size_t)LBM_STATIC_MAX_NODES;
  const int c = h->cur;
  h->launches++;
  k_macroscopic<<<grid_rows(h->nx, h->ny, 128), 128, 0, h->stream>>>(
      h->A, h->flag, h->owner, h->pa.x[c], h->pa.y[c], h->pa.ux[c], h->pa.uy[c], h->pa.omega[c],
      h->pa.Tw, h->primed, base, base + n, base + 2 * n, base + 3 * n, h->C);
  for (int k = 0; k < 4; ++k) fields4[k] = base + k * n;
  return 0;
}

void launch_macroscopic(lbm* h, double* rho, double* ux, double* uy, double* T) {
  const int c = h->cur;
  h->launches++;
  k_macroscopic<<<grid_rows(h->nx, h->ny, 128), 128, 0, h->stream>>>(
      h->A, h->flag, h->owner, h->pa.x[c], h->pa.y[c], h->pa.ux[c], h->pa.uy[c], h->pa.omega[c],
      h->pa.Tw, h->primed, rho, ux, uy, T, h->C);
}
