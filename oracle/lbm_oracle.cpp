/*
 * lbm_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT.  See lbm_oracle.h.
 *
 * Plain single-threaded C++17, fp64, build with -O2 -ffp-contract=off (no FMA contraction, so
 * that the integer decisions -- solid test, e_c choice -- are taken with separately rounded
 * operations).  No blocking, fusion or reordering: the step below is the
 * list at PAPER.md:347-353 (collide, collect links, stream, fluid-particle interaction,
 * [particle update], refill), one plain loop each, state = PRE-collision f(x,t), g(x,t).
 *
 * Citations: PAPER.md:<line> = the paper; "reading" = a choice the paper leaves open, listed in
 * DESIGN.md "Readings of the paper" (taken over from SURVEY.md 8(c)).
 *
 * Pins (tests/test_oracle_*.py, tests/test_units.py): every formula piece against its algebraic
 * identities; Poiseuille, conduction, thermal decay, mass conservation; brute-force link scans;
 * and the coupled fluid-particle step against Faxen's drag on a cylinder moving between two walls
 * (Eqs. 9, 10, 13, 16) and the conduction shape factor of a hot cylinder between two cold walls
 * (Eqs. 11, 12).  Parity unpinned: the readings no closed form sees (integrator order, fallback
 * ladders in narrow gaps, e_c tie rule, pair repulsion) -- see DESIGN.md section 2.
 */
#include "lbm_oracle.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

namespace {

/* ---- lattice (reading: the paper does not print its numbering; PAPER.md:258 only needs e1
 * along a grid line and e6 along i+j = const) ---- */
const int EX[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1};
const int EY[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1};
const int OPP[9] = {0, 3, 4, 1, 2, 7, 8, 5, 6};
const double W9[9] = {4.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9,
                      1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36};

/* D2Q9 moment matrix M (reading: Lallemand-Luo basis; the paper defers M to refs [27,28,41-43],
 * PAPER.md:84).  Rows: rho, e, eps, jx, qx, jy, qy, pxx, pxy. */
const double MM[9][9] = {
    {1, 1, 1, 1, 1, 1, 1, 1, 1},
    {-4, -1, -1, -1, -1, 2, 2, 2, 2},
    {4, -2, -2, -2, -2, 1, 1, 1, 1},
    {0, 1, 0, -1, 0, 1, -1, -1, 1},
    {0, -2, 0, 2, 0, 1, -1, -1, 1},
    {0, 0, 1, 0, -1, 1, 1, -1, -1},
    {0, 0, -2, 0, 2, 1, 1, -1, -1},
    {0, 1, -1, 1, -1, 0, 0, 0, 0},
    {0, 0, 0, 0, 0, 1, -1, 1, -1}};
const double MNORM[9] = {9, 36, 36, 6, 12, 6, 12, 4, 4}; /* |row|^2: rows are orthogonal */

/* D2Q5 moment matrix N (reading).  Rows: T, e1x-moment, e1y-moment, (-4,1,1,1,1), (0,1,-1,1,-1) */
const double NN[5][5] = {
    {1, 1, 1, 1, 1}, {0, 1, 0, -1, 0}, {0, 0, 1, 0, -1}, {-4, 1, 1, 1, 1}, {0, 1, -1, 1, -1}};
const double NNORM[5] = {5, 2, 2, 20, 4};

const int E_ARG = -1, E_STATE = -2, E_CAPACITY = -3, E_NONFINITE = -5;

struct Particle {
  double x, y, theta, ux, uy, omega;
  double r, rho_ratio, Tw;
  /* ellipse (App. A; reading in DESIGN.md "Elliptical particles"): semi-axes
   * a (along the body x axis), b, and the orientation as a unit vector (c, s) = (cos, sin) of
   * theta, carried on its own so that no cos/sin is evaluated after set-up.  ell = 0: a circle
   * of radius r = a = b, which takes the circle formulas bit for bit. */
  double a, b, c, s;
  int ell;
  double Fx, Fy, Tz; /* hydrodynamic force / torque of the last step, Eqs. (13), (14) */
  int fixed;
};

struct Link {
  int pid, i, j, alpha;
  double q;
};

std::string g_create_error;

} // namespace

static void collide_core(const oracle_params* p, const double* S9, const double* Q5, double aT,
                         const double* f9, const double* g5, double* fpost9, double* gpost5);

struct oracle_lbm {
  int nx = 0, ny = 0;
  long long n = 0;
  oracle_params P{};
  std::vector<double> f, g;         /* pre-collision, f[k*n+idx] */
  std::vector<double> fpost, gpost; /* post-collision f+, g+ */
  std::vector<double> fnew, gnew;   /* f(.,t+1), g(.,t+1) */
  std::vector<int> owner;           /* -1 fluid, else id of the (lowest-numbered) covering particle */
  std::vector<Particle> parts;
  bool have_post = false;           /* fpost/gpost were injected (oracle_set_state): the next step
                                       starts at "collect links", its collision is already done */
  long long steps_done = 0;
  std::string err;
};

namespace {

inline long long IDX(const oracle_lbm* h, int i, int j) { return (long long)j * h->nx + i; }

/* neighbour (i+di, j+dj): returns false if outside the cavity; wraps x if periodic_x */
inline bool neighbour(const oracle_lbm* h, int i, int j, int di, int dj, int* oi, int* oj) {
  int a = i + di, b = j + dj;
  if (b < 0 || b >= h->ny) return false;
  if (a < 0 || a >= h->nx) {
    if (!h->P.periodic_x) return false;
    a = (a + h->nx) % h->nx;
  }
  *oi = a;
  *oj = b;
  return true;
}

inline bool is_fluid(const oracle_lbm* h, int i, int j, int di, int dj) {
  int a, b;
  if (!neighbour(h, i, j, di, dj, &a, &b)) return false;
  return h->owner[IDX(h, a, b)] < 0;
}

/* solid test: dx*dx + dy*dy <= r*r, each operation separately rounded */
inline bool inside(double xi, double yj, double xc, double yc, double r) {
  double dx = xi - xc;
  double dy = yj - yc;
  double d2 = dx * dx + dy * dy;
  double r2 = r * r;
  return d2 <= r2;
}

/* ellipse: body coordinates u = dx c + dy s, v = dy c - dx s; inside iff (u/a)^2 + (v/b)^2 <= 1,
 * each operation separately rounded, in exactly this order */
inline bool inside_ellipse(double xi, double yj, double xc, double yc, double a, double b,
                           double c, double s) {
  double dx = xi - xc;
  double dy = yj - yc;
  double u = dx * c + dy * s;
  double v = dy * c - dx * s;
  double ua = u / a;
  double vb = v / b;
  return ua * ua + vb * vb <= 1.0;
}

inline bool inside_p(const Particle& p, double xi, double yj) {
  return p.ell ? inside_ellipse(xi, yj, p.x, p.y, p.a, p.b, p.c, p.s) : inside(xi, yj, p.x, p.y, p.r);
}

/* half extents of the bounding box of the particle: r, or sqrt((a c)^2 + (b s)^2) etc. */
inline void half_extents(const Particle& p, double* hx, double* hy) {
  if (!p.ell) {
    *hx = p.r;
    *hy = p.r;
    return;
  }
  double ac = p.a * p.c, bs = p.b * p.s, as = p.a * p.s, bc = p.b * p.c;
  *hx = std::sqrt(ac * ac + bs * bs);
  *hy = std::sqrt(as * as + bc * bc);
}

/* effective zone (narrower reading): [INT(xc-hx)-1, INT(xc+hx)+1] x [.. hy ..] */
inline void zone_p(const Particle& p, int* i0, int* i1, int* j0, int* j1) {
  double hx, hy;
  half_extents(p, &hx, &hy);
  *i0 = (int)std::floor(p.x - hx) - 1;
  *i1 = (int)std::floor(p.x + hx) + 1;
  *j0 = (int)std::floor(p.y - hy) - 1;
  *j1 = (int)std::floor(p.y + hy) + 1;
}

inline double q_p(const Particle& p, double xf, double yf, int al) {
  return p.ell ? oracle_link_q_ellipse(xf, yf, al, p.x, p.y, p.a, p.b, p.c, p.s)
               : oracle_link_q(xf, yf, al, p.x, p.y, p.r);
}

/* support function of the particle along the unit vector (nx, ny): half width in that direction */
inline double support_p(const Particle& p, double nx, double ny) {
  if (!p.ell) return p.r;
  double m = nx * p.c + ny * p.s;
  double w = ny * p.c - nx * p.s;
  double am = p.a * m, bw = p.b * w;
  return std::sqrt(am * am + bw * bw);
}

void compute_owner(const oracle_lbm* h, std::vector<int>& own) {
  own.assign((size_t)h->n, -1);
  for (int p = (int)h->parts.size() - 1; p >= 0; --p) { /* descending so the lowest pid wins */
    const Particle& a = h->parts[p];
    int i0, i1, j0, j1;
    zone_p(a, &i0, &i1, &j0, &j1);
    for (int j = j0; j <= j1; ++j) {
      if (j < 0 || j >= h->ny) continue;
      for (int i = i0; i <= i1; ++i) {
        if (i < 0 || i >= h->nx) continue;
        if (inside_p(a, (double)i, (double)j)) own[IDX(h, i, j)] = p;
      }
    }
  }
}

/* a2: scan the particle's effective zone [INT(xc-r)-1, INT(xc+r)+1]^2 */
void build_links(const oracle_lbm* h, std::vector<Link>& links) {
  links.clear();
  for (int p = 0; p < (int)h->parts.size(); ++p) {
    const Particle& a = h->parts[p];
    int i0, i1, j0, j1;
    zone_p(a, &i0, &i1, &j0, &j1);
    for (int al = 1; al <= 8; ++al)
      for (int j = j0; j <= j1; ++j) {
        if (j < 0 || j >= h->ny) continue;
        for (int i = i0; i <= i1; ++i) {
          if (i < 0 || i >= h->nx) continue;
          if (h->owner[IDX(h, i, j)] >= 0) continue; /* x_f must be fluid */
          int bi = i + EX[al], bj = j + EY[al];       /* x_b = x_f + e_alpha (no wrap: zones do
                                                         not cross the periodic seam) */
          if (bi < 0 || bi >= h->nx || bj < 0 || bj >= h->ny) continue;
          if (h->owner[IDX(h, bi, bj)] != p) continue;
          Link L;
          L.pid = p;
          L.i = i;
          L.j = j;
          L.alpha = al;
          L.q = q_p(a, (double)i, (double)j, al);
          links.push_back(L);
        }
      }
  }
}

int copy_links(const std::vector<Link>& links, long long* n, int* pid, int* i, int* j, int* alpha,
               double* q) {
  long long cap = *n;
  *n = (long long)links.size();
  if ((long long)links.size() > cap) return E_CAPACITY;
  for (size_t k = 0; k < links.size(); ++k) {
    if (pid) pid[k] = links[k].pid;
    if (i) i[k] = links[k].i;
    if (j) j[k] = links[k].j;
    if (alpha) alpha[k] = links[k].alpha;
    if (q) q[k] = links[k].q;
  }
  return 0;
}

double ipow(double x, int p) {
  double r = 1.0;
  for (int k = 0; k < p; ++k) r = r * x;
  return r;
}

int fail(oracle_lbm* h, int code, const std::string& msg) {
  h->err = msg;
  return code;
}

/* one time step */
int step_once(oracle_lbm* h) {
  const int nx = h->nx, ny = h->ny;
  const long long n = h->n;
  const oracle_params& P = h->P;
  const double qnan = std::numeric_limits<double>::quiet_NaN();
  double S9[9], Q5[5], aT;
  oracle_relaxation_rates(P.nu, P.kappa, S9, Q5, &aT);
  const double wT = (4.0 + aT) / 20.0; /* thermal weight of directions 1..4 (reading) */

  /* 1-3: macroscopic + collision of f and g on fluid nodes (Eqs. 5, 6) */
  const bool injected = h->have_post;
  h->have_post = false;
  for (int j = 0; j < ny && !injected; ++j)
    for (int i = 0; i < nx; ++i) {
      long long x = IDX(h, i, j);
      if (h->owner[x] >= 0) continue;
      double fi[9], gi[5], fo[9], go[5];
      for (int k = 0; k < 9; ++k) fi[k] = h->f[k * n + x];
      for (int k = 0; k < 5; ++k) gi[k] = h->g[k * n + x];
      collide_core(&P, S9, Q5, aT, fi, gi, fo, go);
      for (int k = 0; k < 9; ++k) h->fpost[k * n + x] = fo[k];
      for (int k = 0; k < 5; ++k) h->gpost[k * n + x] = go[k];
    }

  /* 4: collect the fluid-particle links for positions at time t */
  std::vector<Link> links;
  build_links(h, links);
  {
    std::vector<int> cnt(h->parts.size(), 0);
    for (const Link& L : links) cnt[L.pid]++;
    for (size_t p = 0; p < cnt.size(); ++p)
      if (cnt[p] > P.max_links_per_particle)
        return fail(h, E_CAPACITY, "link count exceeds max_links_per_particle");
  }

  /* 5-6: streaming + cavity walls (LHS of Eqs. 5, 6; walls: reading = halfway bounce-back,
   * thermal anti-bounce-back (Dirichlet) or bounce-back (adiabatic)) */
  for (int k = 0; k < 9; ++k)
    for (long long x = 0; x < n; ++x) h->fnew[k * n + x] = qnan;
  for (int k = 0; k < 5; ++k)
    for (long long x = 0; x < n; ++x) h->gnew[k * n + x] = qnan;
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      long long x = IDX(h, i, j);
      if (h->owner[x] >= 0) continue;
      for (int k = 0; k < 9; ++k) {
        int si, sj;
        if (neighbour(h, i, j, -EX[k], -EY[k], &si, &sj)) {
          long long s = IDX(h, si, sj);
          if (h->owner[s] < 0) h->fnew[k * n + x] = h->fpost[k * n + s];
          /* else: x - e_k is solid -> supplied by the link (x, alpha = opp(k)) below */
        } else {
          h->fnew[k * n + x] = h->fpost[OPP[k] * n + x]; /* f_k(x,t+1) = f+_kbar(x,t) */
        }
      }
      for (int k = 0; k < 5; ++k) {
        int si, sj;
        if (neighbour(h, i, j, -EX[k], -EY[k], &si, &sj)) {
          long long s = IDX(h, si, sj);
          if (h->owner[s] < 0) h->gnew[k * n + x] = h->gpost[k * n + s];
        } else {
          /* which wall did x - e_k cross?  W,E,S,N = 0..3 */
          int wall = (i - EX[k] < 0) ? 0 : (i - EX[k] >= nx) ? 1 : (j - EY[k] < 0) ? 2 : 3;
          double gb = h->gpost[OPP[k] * n + x];
          if (P.wall_T_type[wall] == 1)
            h->gnew[k * n + x] = -gb + 2.0 * wT * P.wall_T[wall];
          else
            h->gnew[k * n + x] = gb;
        }
      }
    }

  /* 7-8: fluid-particle interaction on the links: Eqs. (9)-(12), then Eqs. (13)-(14) summed in
   * stored link order */
  for (Particle& a : h->parts) a.Fx = a.Fy = a.Tz = 0.0;
  for (const Link& L : links) {
    Particle& a = h->parts[L.pid];
    const int al = L.alpha, ab = OPP[al];
    long long xf = IDX(h, L.i, L.j);
    int nbehind = 0;
    long long x1 = -1, x2 = -1;
    {
      int a1, b1, a2, b2;
      if (neighbour(h, L.i, L.j, -EX[al], -EY[al], &a1, &b1) && h->owner[IDX(h, a1, b1)] < 0) {
        nbehind = 1;
        x1 = IDX(h, a1, b1);
        if (neighbour(h, L.i, L.j, -2 * EX[al], -2 * EY[al], &a2, &b2) &&
            h->owner[IDX(h, a2, b2)] < 0) {
          nbehind = 2;
          x2 = IDX(h, a2, b2);
        }
      }
    }
    /* wall point x_w = x_f + q e_alpha, wall velocity u_w = U_c + Omega x (x_w - x_c) */
    double rwx = ((double)L.i + L.q * EX[al]) - a.x;
    double rwy = ((double)L.j + L.q * EY[al]) - a.y;
    double uwx = a.ux - a.omega * rwy;
    double uwy = a.uy + a.omega * rwx;
    double fi0 = h->fpost[al * n + xf];
    double fi1 = nbehind >= 1 ? h->fpost[al * n + x1] : 0.0;
    double fi2 = nbehind >= 2 ? h->fpost[al * n + x2] : 0.0;
    double fb0 = h->fpost[ab * n + xf];
    double fb1 = nbehind >= 1 ? h->fpost[ab * n + x1] : 0.0;
    double fbb = oracle_bounce_back_f(al, L.q, fi0, fi1, fi2, fb0, fb1, nbehind, P.rho0, uwx, uwy);
    h->fnew[ab * n + xf] = fbb;
    if (al <= 4) {
      double gi0 = h->gpost[al * n + xf];
      double gi1 = nbehind >= 1 ? h->gpost[al * n + x1] : 0.0;
      double gb0 = h->gpost[ab * n + xf];
      h->gnew[ab * n + xf] = oracle_bounce_back_g(al, L.q, gi0, gi1, gb0, nbehind, P.kappa, a.Tw);
    }
    double dP[3];
    oracle_momentum_exchange(al, fi0, fbb, uwx, uwy, rwx, rwy, dP);
    a.Fx += dP[0];
    a.Fy += dP[1];
    a.Tz += dP[2];
  }

  /* every population of every fluid node must now have exactly one source */
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      long long x = IDX(h, i, j);
      if (h->owner[x] >= 0) continue;
      for (int k = 0; k < 9; ++k)
        if (std::isnan(h->fnew[k * n + x])) {
          char b[160];
          std::snprintf(b, sizeof b, "step %lld: f_%d(%d,%d) unfilled or NaN", h->steps_done, k, i, j);
          return fail(h, E_NONFINITE, b);
        }
      for (int k = 0; k < 5; ++k)
        if (std::isnan(h->gnew[k * n + x])) {
          char b[160];
          std::snprintf(b, sizeof b, "step %lld: g_%d(%d,%d) unfilled or NaN", h->steps_done, k, i, j);
          return fail(h, E_NONFINITE, b);
        }
    }

  /* 9: particle update, Eqs. (7), (8), (15).  Forces from positions at time t. */
  const double PI = 3.14159265358979323846;
  const int np = (int)h->parts.size();
  std::vector<double> Ftx(np, 0.0), Fty(np, 0.0);
  for (int ia = 0; ia < np; ++ia) {
    const Particle& a = h->parts[ia];
    /* area pi a b of an ellipse; a circle keeps pi r r (same operations, same bits) */
    double Ca = PI * a.a * a.b * (a.rho_ratio * P.rho0 - P.rho0) * P.g; /* Eq. 15's C */
    double Fx = a.Fx, Fy = a.Fy;
    Fy += -(a.rho_ratio * P.rho0 - P.rho0) * PI * a.a * a.b * P.g; /* weight minus buoyancy */
    double ahx, ahy;
    half_extents(a, &ahx, &ahy);
    for (int ib = 0; ib < np; ++ib) {
      if (ib == ia) continue;
      const Particle& b = h->parts[ib];
      double dx = a.x - b.x, dy = a.y - b.y;
      double reach = a.r + b.r + P.rep_s;
      if (std::fabs(dx) > reach || std::fabs(dy) > reach) continue; /* cannot interact */
      double dist = std::sqrt(dx * dx + dy * dy);
      /* gap along the line of centres through the support functions (reading: the paper does
       * not state the pair form; for two circles this is |xa - xb| - ra - rb) */
      double delta;
      if (!a.ell && !b.ell) {
        delta = dist - a.r - b.r;
      } else {
        if (!(dist > 0.0)) continue;
        double nxh = dx / dist, nyh = dy / dist;
        delta = dist - support_p(a, nxh, nyh) - support_p(b, nxh, nyh);
      }
      if (!(delta <= P.rep_s) || !(dist > 0.0)) continue;
      double Cb = PI * b.a * b.b * (b.rho_ratio * P.rho0 - P.rho0) * P.g;
      double mag = oracle_repulsion_mag(0.5 * (Ca + Cb), P.rep_eps, P.rep_s, delta, P.rep_power);
      Fx += mag * (dx / dist);
      Fy += mag * (dy / dist);
    }
    /* walls W,E,S,N at -1/2, nx-1/2, -1/2, ny-1/2 */
    if (!P.periodic_x) {
      double dW = (a.x + 0.5) - ahx;
      if (dW <= P.rep_s) Fx += oracle_repulsion_mag(Ca, P.rep_eps, P.rep_s, dW, P.rep_power);
      double dE = ((double)nx - 0.5 - a.x) - ahx;
      if (dE <= P.rep_s) Fx -= oracle_repulsion_mag(Ca, P.rep_eps, P.rep_s, dE, P.rep_power);
    }
    double dS = (a.y + 0.5) - ahy;
    if (dS <= P.rep_s) Fy += oracle_repulsion_mag(Ca, P.rep_eps, P.rep_s, dS, P.rep_power);
    double dN = ((double)ny - 0.5 - a.y) - ahy;
    if (dN <= P.rep_s) Fy -= oracle_repulsion_mag(Ca, P.rep_eps, P.rep_s, dN, P.rep_power);
    Ftx[ia] = Fx;
    Fty[ia] = Fy;
  }
  for (int ia = 0; ia < np; ++ia) {
    Particle& a = h->parts[ia];
    if (a.fixed) continue;
    double mass = a.rho_ratio * P.rho0 * PI * a.a * a.b;
    double inertia = a.ell ? 0.25 * mass * (a.a * a.a + a.b * a.b) : 0.5 * mass * a.r * a.r;
    double st[6] = {a.x, a.y, a.theta, a.ux, a.uy, a.omega};
    oracle_integrate(st, Ftx[ia], Fty[ia], a.Tz, mass, inertia);
    if (a.ell) oracle_rotate_unit(&a.c, &a.s, 0.5 * (a.omega + st[5]));
    a.x = st[0];
    a.y = st[1];
    a.theta = st[2];
    a.ux = st[3];
    a.uy = st[4];
    a.omega = st[5];
  }

  /* 10: new flags, refill of uncovered nodes (Eqs. 16, 17) */
  std::vector<int> own_new;
  compute_owner(h, own_new);
  struct Born {
    long long x;
    double f[9], g[5];
  };
  std::vector<Born> born;
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      long long x = IDX(h, i, j);
      int p = h->owner[x];
      if (!(p >= 0 && own_new[x] < 0)) continue;
      const Particle& a = h->parts[p]; /* state at t+1 */
      double dxn = (double)i - a.x, dyn = (double)j - a.y;
      /* outward normal of the wall at the newborn node: radial for a circle; for an
       * ellipse the gradient of (u/a)^2 + (v/b)^2 turned back into the lattice frame */
      double nrx = dxn, nry = dyn;
      if (a.ell) oracle_ellipse_normal(dxn, dyn, a.a, a.b, a.c, a.s, &nrx, &nry);
      int c = oracle_refill_direction(nrx, nry);
      int nvalid = 0;
      long long xs[3] = {-1, -1, -1};
      for (int k = 1; k <= 3; ++k) {
        int si, sj;
        if (!neighbour(h, i, j, k * EX[c], k * EY[c], &si, &sj)) break;
        long long s = IDX(h, si, sj);
        if (h->owner[s] >= 0 || own_new[s] >= 0) break; /* must be fluid at t and at t+1 */
        xs[k - 1] = s;
        nvalid = k;
      }
      double f1[9] = {0}, f2[9] = {0}, f3[9] = {0};
      for (int k = 0; k < 9; ++k) {
        if (nvalid >= 1) f1[k] = h->fnew[k * n + xs[0]];
        if (nvalid >= 2) f2[k] = h->fnew[k * n + xs[1]];
        if (nvalid >= 3) f3[k] = h->fnew[k * n + xs[2]];
      }
      double uwx = a.ux - a.omega * dyn;
      double uwy = a.uy + a.omega * dxn;
      Born b;
      b.x = x;
      oracle_refill_f(nvalid, f1, f2, f3, P.rho0, uwx, uwy, b.f);
      oracle_geq(a.Tw, uwx, uwy, P.kappa, b.g); /* Eq. (17) */
      born.push_back(b);
    }
  for (long long x = 0; x < n; ++x) {
    if (own_new[x] >= 0) continue;
    if (h->owner[x] >= 0) continue; /* newborn: written below */
    for (int k = 0; k < 9; ++k) h->f[k * n + x] = h->fnew[k * n + x];
    for (int k = 0; k < 5; ++k) h->g[k * n + x] = h->gnew[k * n + x];
  }
  for (const Born& b : born) {
    for (int k = 0; k < 9; ++k) h->f[k * n + b.x] = b.f[k];
    for (int k = 0; k < 5; ++k) h->g[k * n + b.x] = b.g[k];
  }
  h->owner.swap(own_new);
  h->steps_done++;
  return 0;
}

} // namespace

/* ======================= pieces ======================= */

extern "C" void oracle_moments_f(const double* f9, double* m9) {
  for (int k = 0; k < 9; ++k) {
    double s = 0.0;
    for (int i = 0; i < 9; ++i) s += MM[k][i] * f9[i];
    m9[k] = s;
  }
}

extern "C" void oracle_moments_g(const double* g5, double* n5) {
  for (int k = 0; k < 5; ++k) {
    double s = 0.0;
    for (int i = 0; i < 5; ++i) s += NN[k][i] * g5[i];
    n5[k] = s;
  }
}

/* M^-1 = M^T diag(1/|row|^2) because the rows of M are mutually orthogonal */
extern "C" void oracle_from_moments_f(const double* m9, double* f9) {
  double ms[9];
  for (int k = 0; k < 9; ++k) ms[k] = m9[k] / MNORM[k];
  for (int i = 0; i < 9; ++i) {
    double s = 0.0;
    for (int k = 0; k < 9; ++k) s += MM[k][i] * ms[k];
    f9[i] = s;
  }
}

extern "C" void oracle_from_moments_g(const double* n5, double* g5) {
  double ns[5];
  for (int k = 0; k < 5; ++k) ns[k] = n5[k] / NNORM[k];
  for (int i = 0; i < 5; ++i) {
    double s = 0.0;
    for (int k = 0; k < 5; ++k) s += NN[k][i] * ns[k];
    g5[i] = s;
  }
}

/* reading: s_nu = 1/tau, tau = 3 nu + 1/2; s_e = s_eps = s_nu; s_q = 8(2-s_nu)/(8-s_nu);
 * q_kappa = 3 - sqrt3, q_e = q_nu = 4 sqrt3 - 6, a_T = 20 sqrt3 kappa - 4 */
extern "C" void oracle_relaxation_rates(double nu, double kappa, double* S9, double* Q5,
                                        double* aT) {
  double tau = 3.0 * nu + 0.5;
  double snu = 1.0 / tau;
  double sq = 8.0 * (2.0 - snu) / (8.0 - snu);
  double S[9] = {0.0, snu, snu, 0.0, sq, 0.0, sq, snu, snu};
  for (int k = 0; k < 9; ++k) S9[k] = S[k];
  double r3 = std::sqrt(3.0);
  double Q[5] = {0.0, 3.0 - r3, 3.0 - r3, 4.0 * r3 - 6.0, 4.0 * r3 - 6.0};
  for (int k = 0; k < 5; ++k) Q5[k] = Q[k];
  *aT = 20.0 * r3 * kappa - 4.0;
}

static void meq9(double rho, double ux, double uy, double* m) {
  double u2 = ux * ux + uy * uy;
  m[0] = rho;
  m[1] = rho * (-2.0 + 3.0 * u2);
  m[2] = rho * (1.0 - 3.0 * u2);
  m[3] = rho * ux;
  m[4] = -rho * ux;
  m[5] = rho * uy;
  m[6] = -rho * uy;
  m[7] = rho * (ux * ux - uy * uy);
  m[8] = rho * ux * uy;
}

static void neq5(double T, double ux, double uy, double aT, double* nq) {
  nq[0] = T;
  nq[1] = ux * T;
  nq[2] = uy * T;
  nq[3] = aT * T;
  nq[4] = 0.0;
}

extern "C" void oracle_feq(double rho, double ux, double uy, double* out9) {
  double m[9];
  meq9(rho, ux, uy, m);
  oracle_from_moments_f(m, out9);
}

extern "C" void oracle_geq(double T, double ux, double uy, double kappa, double* out5) {
  double S9[9], Q5[5], aT, nq[5];
  oracle_relaxation_rates(0.1, kappa, S9, Q5, &aT);
  neq5(T, ux, uy, aT, nq);
  oracle_from_moments_g(nq, out5);
}

/* rho = sum f, u = (sum e f + F/2)/rho, F = rho g beta (T - T0) y^, T = sum g
 * (plus the extra uniform body acceleration of the closed-form checks) */
extern "C" void oracle_macroscopic(const oracle_params* p, const double* f9, const double* g5,
                                   double* rho, double* ux, double* uy, double* T) {
  double t = 0.0;
  for (int k = 0; k < 5; ++k) t += g5[k];
  double r = 0.0, jx = 0.0, jy = 0.0;
  for (int k = 0; k < 9; ++k) {
    r += f9[k];
    jx += EX[k] * f9[k];
    jy += EY[k] * f9[k];
  }
  double Fx = r * p->body_ax;
  double Fy = r * (p->body_ay + p->gbeta * (t - p->T0));
  *rho = r;
  *T = t;
  *ux = (jx + 0.5 * Fx) / r;
  *uy = (jy + 0.5 * Fy) / r;
}

/* Eq. (5): f+ = f - M^-1 S (m - m_eq) + dt F'  with  dt F' = M^-1 (I - S/2) M F~ (Guo forcing in
 * moment space, reading);  Eq. (6): g+ = g - N^-1 Q (n - n_eq).  The rates are passed in so that
 * the lattice loop does not recompute them per node. */
static void collide_core(const oracle_params* p, const double* S9, const double* Q5, double aT,
                         const double* f9, const double* g5, double* fpost9, double* gpost5) {
  double rho, ux, uy, T;
  oracle_macroscopic(p, f9, g5, &rho, &ux, &uy, &T);
  double Fx = rho * p->body_ax;
  double Fy = rho * (p->body_ay + p->gbeta * (T - p->T0));

  double m[9], me[9], mp[9];
  oracle_moments_f(f9, m);
  meq9(rho, ux, uy, me);
  double uF = ux * Fx + uy * Fy;
  double MF[9] = {0.0, 6.0 * uF, -6.0 * uF, Fx, -Fx, Fy, -Fy,
                  2.0 * (ux * Fx - uy * Fy), ux * Fy + uy * Fx};
  for (int k = 0; k < 9; ++k) mp[k] = m[k] - S9[k] * (m[k] - me[k]) + (1.0 - 0.5 * S9[k]) * MF[k];
  oracle_from_moments_f(mp, fpost9);

  double nm[5], ne[5], np5[5];
  oracle_moments_g(g5, nm);
  neq5(T, ux, uy, aT, ne);
  for (int k = 0; k < 5; ++k) np5[k] = nm[k] - Q5[k] * (nm[k] - ne[k]);
  oracle_from_moments_g(np5, gpost5);
}

extern "C" void oracle_collide_node(const oracle_params* p, const double* f9, const double* g5,
                                    double* fpost9, double* gpost5) {
  double S9[9], Q5[5], aT;
  oracle_relaxation_rates(p->nu, p->kappa, S9, Q5, &aT);
  collide_core(p, S9, Q5, aT, f9, g5, fpost9, gpost5);
}

/* q = |x_f - x_w| / |x_f - x_b|: smaller root t of |x_f + t e - x_c|^2 = r^2 */
extern "C" double oracle_link_q(double xf, double yf, int alpha, double xc, double yc, double r) {
  double ex = (double)EX[alpha], ey = (double)EY[alpha];
  double dx = xf - xc, dy = yf - yc;
  double a = ex * ex + ey * ey;
  double b = 2.0 * (ex * dx + ey * dy);
  double c = (dx * dx + dy * dy) - r * r;
  double disc = b * b - 4.0 * a * c;
  if (disc < 0.0) disc = 0.0;
  double t = (-b - std::sqrt(disc)) / (2.0 * a);
  if (t < 0.0) t = 0.0;
  if (t > 1.0) t = 1.0;
  return t;
}

/* q for an ellipse: smaller root of the ray-ellipse quadratic in the body frame,
 * |((u + t eu)/a, (v + t ev)/b)|^2 = 1 (definition of q) */
extern "C" double oracle_link_q_ellipse(double xf, double yf, int alpha, double xc, double yc,
                                        double a, double b, double c, double s) {
  double ex = (double)EX[alpha], ey = (double)EY[alpha];
  double dx = xf - xc, dy = yf - yc;
  double u = dx * c + dy * s, v = dy * c - dx * s;
  double eu = ex * c + ey * s, ev = ey * c - ex * s;
  double ua = u / a, vb = v / b, ea = eu / a, eb = ev / b;
  double A = ea * ea + eb * eb;
  double B = 2.0 * (ua * ea + vb * eb);
  double C = (ua * ua + vb * vb) - 1.0;
  double disc = B * B - 4.0 * A * C;
  if (disc < 0.0) disc = 0.0;
  double t = (-B - std::sqrt(disc)) / (2.0 * A);
  if (t < 0.0) t = 0.0;
  if (t > 1.0) t = 1.0;
  return t;
}

/* orientation unit vector advanced by the angle increment d through the Cayley rotation
 * (cr, sr) = ((1 - t^2)/(1 + t^2), 2t/(1 + t^2)), t = d/2 (a rotation by 2 atan(d/2) = d + O(d^3)),
 * then renormalised: only +, -, *, /, sqrt, so both implementations produce the same bits */
extern "C" void oracle_rotate_unit(double* c, double* s, double d) {
  double t = 0.5 * d;
  double den = 1.0 + t * t;
  double cr = (1.0 - t * t) / den;
  double sr = (2.0 * t) / den;
  double c1 = (*c) * cr - (*s) * sr;
  double s1 = (*s) * cr + (*c) * sr;
  double nrm = std::sqrt(c1 * c1 + s1 * s1);
  *c = c1 / nrm;
  *s = s1 / nrm;
}

/* Eq. (9) for q <= 1/2, Eq. (10) for q > 1/2, moving-wall term
 * 2 w_i rho0 (e_ibar . u_w)/c_s^2.  Fallback ladder (reading):
 *  q <= 1/2: nbehind=2 Eq.(9); nbehind=1 linear 2q f_i(x_f) + (1-2q) f_i(x_f-e_i); nbehind=0 halfway
 *  q >  1/2: nbehind>=1 Eq.(10); nbehind=0 linear [f_i(x_f) + (2q-1) f_ibar(x_f)]/(2q), wall/(2q) */
extern "C" double oracle_bounce_back_f(int alpha, double q, double fi_0, double fi_1, double fi_2,
                                       double fib_0, double fib_1, int nbehind, double rho0,
                                       double uwx, double uwy) {
  const int ab = OPP[alpha];
  const double cs2 = 1.0 / 3.0;
  double wall = 2.0 * W9[alpha] * rho0 * ((double)EX[ab] * uwx + (double)EY[ab] * uwy) / cs2;
  if (q <= 0.5) {
    if (nbehind >= 2)
      return q * (2.0 * q + 1.0) * fi_0 + (1.0 - 4.0 * q * q) * fi_1 - q * (1.0 - 2.0 * q) * fi_2 +
             wall;
    if (nbehind == 1) return 2.0 * q * fi_0 + (1.0 - 2.0 * q) * fi_1 + wall;
    return fi_0 + wall;
  }
  if (nbehind >= 1) {
    double c = 1.0 / (q * (2.0 * q + 1.0));
    return c * fi_0 + ((2.0 * q - 1.0) / q) * fib_0 - ((2.0 * q - 1.0) / (2.0 * q + 1.0)) * fib_1 +
           c * wall;
  }
  return (fi_0 + (2.0 * q - 1.0) * fib_0) / (2.0 * q) + wall / (2.0 * q);
}

/* Eq. (11) with Eq. (12) coefficients; omega_i = thermal weight (4+a_T)/20.
 * Fallback (reading): x_f - e_i not fluid -> c_d2 = c_d3 = 0, c_d4 = 1 (anti-bounce-back). */
extern "C" double oracle_bounce_back_g(int alpha, double q, double gi_0, double gi_1, double gib_0,
                                       int nbehind, double kappa, double Tw) {
  (void)alpha;
  double S9[9], Q5[5], aT;
  oracle_relaxation_rates(0.1, kappa, S9, Q5, &aT);
  double w = (4.0 + aT) / 20.0;
  double cd1 = -1.0, cd2, cd3, cd4;
  if (nbehind >= 1) {
    cd2 = (2.0 * q - 1.0) / (2.0 * q + 1.0);
    cd3 = cd2;
    cd4 = 2.0 / (2.0 * q + 1.0);
  } else {
    cd2 = 0.0;
    cd3 = 0.0;
    cd4 = 1.0;
  }
  return (cd1 * gi_0 + cd2 * gi_1 + cd3 * gib_0) + cd4 * (2.0 * w * Tw);
}

/* Eqs. (13), (14), one link:
 * dP = f_i^+(x_f,t)(e_i - u_w) - f_ibar(x_f,t+dt)(e_ibar - u_w);  T_z = (x_w - x_c) x dP */
extern "C" void oracle_momentum_exchange(int alpha, double fi_post, double fibar_new, double uwx,
                                         double uwy, double rwx, double rwy, double* dP3) {
  const int ab = OPP[alpha];
  double px = fi_post * ((double)EX[alpha] - uwx) - fibar_new * ((double)EX[ab] - uwx);
  double py = fi_post * ((double)EY[alpha] - uwy) - fibar_new * ((double)EY[ab] - uwy);
  dP3[0] = px;
  dP3[1] = py;
  dP3[2] = rwx * py - rwy * px;
}

/* Eq. (15) magnitude: (C/eps_w) ((s - delta)/s)^p for delta <= s, 0 beyond */
extern "C" double oracle_repulsion_mag(double C, double eps, double s, double delta, int power) {
  if (!(delta <= s)) return 0.0;
  return (C / eps) * ipow((s - delta) / s, power);
}

/* Eqs. (7), (8) with the fluid's time step.  Reading (integrator not stated):
 * U' = U + F/M, x' = x + (U + U')/2; same for Omega, theta.  2-D: Omega x (I Omega) = 0. */
extern "C" void oracle_integrate(double* s, double Fx, double Fy, double Tz, double mass,
                                 double inertia) {
  double ux1 = s[3] + Fx / mass;
  double uy1 = s[4] + Fy / mass;
  double om1 = s[5] + Tz / inertia;
  s[0] = s[0] + 0.5 * (s[3] + ux1);
  s[1] = s[1] + 0.5 * (s[4] + uy1);
  s[2] = s[2] + 0.5 * (s[5] + om1);
  s[3] = ux1;
  s[4] = uy1;
  s[5] = om1;
}

/* e_c maximises n . e_alpha/|e_alpha| over alpha = 1..8, ties -> lowest alpha (reading; the paper
 * says "maximizes n . e_c").  n need not be normalised (positive scale). */
extern "C" int oracle_refill_direction(double nx_, double ny_) {
  const double INV_SQRT2 = 0.70710678118654752440;
  int best = 1;
  double bs = -std::numeric_limits<double>::infinity();
  for (int a = 1; a <= 8; ++a) {
    double s = (nx_ * (double)EX[a] + ny_ * (double)EY[a]);
    if (a >= 5) s = s * INV_SQRT2;
    if (s > bs) {
      bs = s;
      best = a;
    }
  }
  return best;
}

/* Outward normal (not normalised) of an ellipse at the point (dx, dy) relative to its centre:
 * the gradient of (u/a)^2 + (v/b)^2, u = dx c + dy s, v = dy c - dx s, turned back into the
 * lattice frame.  The "n" of PAPER.md:151 for an elliptical particle (reading, DESIGN.md
 * "Elliptical particles"); for a = b it is parallel to (dx, dy). */
extern "C" void oracle_ellipse_normal(double dx, double dy, double a, double b, double c, double s,
                                      double* nx_, double* ny_) {
  double u = dx * c + dy * s, v = dy * c - dx * s;
  double gu = (u / a) / a, gv = (v / b) / b;
  *nx_ = gu * c - gv * s;
  *ny_ = gu * s + gv * c;
}

/* Eq. (16) f_new = 3 f(1) - 3 f(2) + f(3); fallback (reading): 2 nodes -> 2 f(1) - f(2);
 * 1 node -> f(1); 0 nodes -> f_eq(rho0, u_w).  Then the MRT velocity constraint:
 * m = M f_new, j = rho_new u_w with rho_new = sum f_new, f_new = M^-1 m. */
extern "C" void oracle_refill_f(int nvalid, const double* f1, const double* f2, const double* f3,
                                double rho0, double uwx, double uwy, double* out9) {
  double fn[9];
  if (nvalid >= 3)
    for (int k = 0; k < 9; ++k) fn[k] = 3.0 * f1[k] - 3.0 * f2[k] + f3[k];
  else if (nvalid == 2)
    for (int k = 0; k < 9; ++k) fn[k] = 2.0 * f1[k] - f2[k];
  else if (nvalid == 1)
    for (int k = 0; k < 9; ++k) fn[k] = f1[k];
  else
    oracle_feq(rho0, uwx, uwy, fn);
  double m[9];
  oracle_moments_f(fn, m);
  m[3] = m[0] * uwx;
  m[5] = m[0] * uwy;
  oracle_from_moments_f(m, out9);
}

/* ======================= whole simulation ======================= */

extern "C" int oracle_create(int nx, int ny, const oracle_params* p, oracle_lbm_t** out) {
  if (!out) return E_ARG;
  *out = nullptr;
  if (!p || nx < 4 || ny < 4 || !(p->nu > 0.0) || !(p->kappa > 0.0) || !(p->kappa < 0.144) ||
      !(p->rho0 > 0.0) || p->max_particles < 0 || p->max_links_per_particle < 0 ||
      !(p->rep_s > 0.0) || !(p->rep_eps > 0.0) || p->rep_power < 1) {
    g_create_error = "oracle_create: bad argument";
    return E_ARG;
  }
  oracle_lbm* h = new oracle_lbm;
  h->nx = nx;
  h->ny = ny;
  h->n = (long long)nx * ny;
  h->P = *p;
  size_t n = (size_t)h->n;
  h->f.assign(9 * n, 0.0);
  h->g.assign(5 * n, 0.0);
  h->fpost.assign(9 * n, 0.0);
  h->gpost.assign(5 * n, 0.0);
  h->fnew.assign(9 * n, 0.0);
  h->gnew.assign(5 * n, 0.0);
  h->owner.assign(n, -1);
  double fe[9], ge[5];
  oracle_feq(p->rho0, 0.0, 0.0, fe);
  oracle_geq(p->T0, 0.0, 0.0, p->kappa, ge);
  for (int k = 0; k < 9; ++k)
    for (size_t x = 0; x < n; ++x) h->f[k * n + x] = fe[k];
  for (int k = 0; k < 5; ++k)
    for (size_t x = 0; x < n; ++x) h->g[k * n + x] = ge[k];
  *out = h;
  return 0;
}

extern "C" int oracle_set_temperature(oracle_lbm_t* h, const double* T) {
  if (!h || !T) return E_ARG;
  if (h->steps_done > 0) return fail(h, E_STATE, "set_temperature after the first step");
  for (long long x = 0; x < h->n; ++x) {
    double ge[5];
    oracle_geq(T[x], 0.0, 0.0, h->P.kappa, ge);
    for (int k = 0; k < 5; ++k) h->g[k * h->n + x] = ge[k];
  }
  return 0;
}

/* circles: minor == NULL and theta == NULL; ellipses: full axes 2a = major[k], 2b = minor[k],
 * theta[k] = angle of the a axis to the x axis (cos / sin taken once, here, by the host libm) */
static int add_shapes(oracle_lbm_t* h, int n, const double* x, const double* y, const double* major,
                      const double* minor, const double* theta, const double* rho_ratio,
                      const double* T_w, const double* ux, const double* uy, const double* omega,
                      const unsigned char* fixed) {
  if (!h || n < 0 || (n > 0 && (!x || !y || !major || !rho_ratio || !T_w))) return E_ARG;
  if (h->steps_done > 0) return fail(h, E_STATE, "add_particles after the first step");
  if ((long long)h->parts.size() + n > h->P.max_particles)
    return fail(h, E_CAPACITY, "max_particles exceeded");
  std::vector<Particle> add;
  for (int k = 0; k < n; ++k) {
    Particle a{};
    a.x = x[k];
    a.y = y[k];
    a.a = 0.5 * major[k];
    a.b = minor ? 0.5 * minor[k] : a.a;
    a.theta = theta ? theta[k] : 0.0;
    a.ell = (a.a != a.b);
    a.c = a.ell ? std::cos(a.theta) : 1.0;
    a.s = a.ell ? std::sin(a.theta) : 0.0;
    a.r = a.a > a.b ? a.a : a.b; /* radius of a circle; largest semi-axis of an ellipse */
    a.rho_ratio = rho_ratio[k];
    a.Tw = T_w[k];
    a.ux = ux ? ux[k] : 0.0;
    a.uy = uy ? uy[k] : 0.0;
    a.omega = omega ? omega[k] : 0.0;
    a.fixed = fixed ? (fixed[k] != 0) : 0;
    if (!(a.a > 0.0) || !(a.b > 0.0) || !(a.rho_ratio > 0.0))
      return fail(h, E_ARG, "bad diameter or density");
    if (!std::isfinite(a.x) || !std::isfinite(a.y) || !std::isfinite(a.ux) ||
        !std::isfinite(a.uy) || !std::isfinite(a.omega) || !std::isfinite(a.Tw) ||
        !std::isfinite(a.theta) || !std::isfinite(a.r))
      return fail(h, E_ARG, "non-finite particle input");
    double hx, hy;
    half_extents(a, &hx, &hy);
    /* strictly inside the cavity walls at -1/2 and n-1/2 */
    if (!(a.y - hy > -0.5) || !(a.y + hy < h->ny - 0.5))
      return fail(h, E_ARG, "particle touches a y wall");
    if (!h->P.periodic_x) {
      if (!(a.x - hx > -0.5) || !(a.x + hx < h->nx - 0.5))
        return fail(h, E_ARG, "particle touches an x wall");
    } else {
      if ((int)std::floor(a.x - a.r) - 2 < 0 || (int)std::floor(a.x + a.r) + 2 > h->nx - 1)
        return fail(h, E_ARG, "particle zone crosses the periodic seam");
    }
    int Nmax = (int)std::floor(2.0 * a.r) + 4; /* worst-case N of PAPER.md:258 for this diameter */
    if (12 * Nmax - 12 > h->P.max_links_per_particle)
      return fail(h, E_CAPACITY, "12N-12 exceeds max_links_per_particle");
    auto overlaps = [&](const Particle& b) {
      double dx = a.x - b.x, dy = a.y - b.y;
      double dist = std::sqrt(dx * dx + dy * dy);
      if (!a.ell && !b.ell) return dist < a.r + b.r;
      if (!(dist > 0.0)) return true;
      /* support-function gap along the line of centres (conservative for ellipses) */
      return dist < support_p(a, dx / dist, dy / dist) + support_p(b, dx / dist, dy / dist);
    };
    for (const Particle& b : h->parts)
      if (overlaps(b)) return fail(h, E_ARG, "particles overlap");
    for (const Particle& b : add)
      if (overlaps(b)) return fail(h, E_ARG, "particles overlap");
    add.push_back(a);
  }
  for (const Particle& a : add) h->parts.push_back(a);
  compute_owner(h, h->owner);
  return 0;
}

extern "C" int oracle_add_particles(oracle_lbm_t* h, int n, const double* x, const double* y,
                                    const double* diam, const double* rho_ratio, const double* T_w,
                                    const double* ux, const double* uy, const double* omega,
                                    const unsigned char* fixed) {
  return add_shapes(h, n, x, y, diam, nullptr, nullptr, rho_ratio, T_w, ux, uy, omega, fixed);
}

extern "C" int oracle_add_ellipses(oracle_lbm_t* h, int n, const double* x, const double* y,
                                   const double* major, const double* minor, const double* theta,
                                   const double* rho_ratio, const double* T_w, const double* ux,
                                   const double* uy, const double* omega,
                                   const unsigned char* fixed) {
  if (n > 0 && (!minor || !theta)) return E_ARG;
  return add_shapes(h, n, x, y, major, minor, theta, rho_ratio, T_w, ux, uy, omega, fixed);
}

extern "C" int oracle_step(oracle_lbm_t* h, int nsteps) {
  if (!h || nsteps < 0) return E_ARG;
  for (int s = 0; s < nsteps; ++s) {
    int rc = step_once(h);
    if (rc) return rc;
  }
  for (const Particle& a : h->parts)
    if (!std::isfinite(a.x) || !std::isfinite(a.y) || !std::isfinite(a.ux) ||
        !std::isfinite(a.uy) || !std::isfinite(a.omega) || !std::isfinite(a.theta))
      return fail(h, E_NONFINITE, "particle state is not finite");
  return 0;
}

extern "C" int oracle_get_fields(oracle_lbm_t* h, double* rho, double* ux, double* uy, double* T,
                                 double* f, double* g, unsigned char* flag) {
  if (!h) return E_ARG;
  const long long n = h->n;
  for (int j = 0; j < h->ny; ++j)
    for (int i = 0; i < h->nx; ++i) {
      long long x = IDX(h, i, j);
      int p = h->owner[x];
      if (flag) flag[x] = p >= 0 ? 1 : 0;
      if (p >= 0) {
        const Particle& a = h->parts[p];
        if (rho) rho[x] = h->P.rho0;
        if (ux) ux[x] = a.ux - a.omega * ((double)j - a.y);
        if (uy) uy[x] = a.uy + a.omega * ((double)i - a.x);
        if (T) T[x] = a.Tw;
        if (f)
          for (int k = 0; k < 9; ++k) f[k * n + x] = 0.0;
        if (g)
          for (int k = 0; k < 5; ++k) g[k * n + x] = 0.0;
        continue;
      }
      double fi[9], gi[5];
      for (int k = 0; k < 9; ++k) fi[k] = h->f[k * n + x];
      for (int k = 0; k < 5; ++k) gi[k] = h->g[k * n + x];
      double r, vx, vy, t;
      oracle_macroscopic(&h->P, fi, gi, &r, &vx, &vy, &t);
      if (rho) rho[x] = r;
      if (ux) ux[x] = vx;
      if (uy) uy[x] = vy;
      if (T) T[x] = t;
      if (f || g) {
        double fo[9], go[5];
        oracle_collide_node(&h->P, fi, gi, fo, go);
        if (f)
          for (int k = 0; k < 9; ++k) f[k * n + x] = fo[k];
        if (g)
          for (int k = 0; k < 5; ++k) g[k * n + x] = go[k];
      }
    }
  return 0;
}

/* Test infrastructure of the deep-run parity check: replaces the whole state by one taken from
 * elsewhere (the CUDA path's read-out after many steps): POST-collision populations f+(x,t),
 * g+(x,t) on the fluid nodes -- what lbm_get_fields hands out -- and the particle states; the
 * solid map is rasterised from the positions.  The next oracle_step then starts after the
 * collision ("collect links" onwards).  Circles only keep their exact geometry; an
 * ellipse's orientation vector is re-derived from theta. */
extern "C" int oracle_set_state(oracle_lbm_t* h, const double* fpost, const double* gpost, int n,
                                const double* x, const double* y, const double* theta,
                                const double* ux, const double* uy, const double* omega) {
  if (!h || !fpost || !gpost) return E_ARG;
  if (n != (int)h->parts.size()) return fail(h, E_ARG, "set_state: particle count differs");
  std::memcpy(h->fpost.data(), fpost, sizeof(double) * 9 * (size_t)h->n);
  std::memcpy(h->gpost.data(), gpost, sizeof(double) * 5 * (size_t)h->n);
  for (int k = 0; k < n; ++k) {
    Particle& a = h->parts[k];
    a.x = x[k];
    a.y = y[k];
    a.theta = theta[k];
    a.ux = ux[k];
    a.uy = uy[k];
    a.omega = omega[k];
    if (a.ell) {
      a.c = std::cos(a.theta);
      a.s = std::sin(a.theta);
    }
  }
  compute_owner(h, h->owner);
  h->have_post = true;
  if (h->steps_done == 0) h->steps_done = 1; /* no more set-up calls after this */
  return 0;
}

extern "C" int oracle_get_precollision(oracle_lbm_t* h, double* f, double* g) {
  if (!h) return E_ARG;
  if (f) std::memcpy(f, h->f.data(), sizeof(double) * 9 * (size_t)h->n);
  if (g) std::memcpy(g, h->g.data(), sizeof(double) * 5 * (size_t)h->n);
  return 0;
}

extern "C" int oracle_get_particles(oracle_lbm_t* h, int* n, double* x, double* y, double* theta,
                                    double* ux, double* uy, double* omega, double* Fx, double* Fy,
                                    double* Tz) {
  if (!h || !n) return E_ARG;
  *n = (int)h->parts.size();
  for (int k = 0; k < *n; ++k) {
    const Particle& a = h->parts[k];
    if (x) x[k] = a.x;
    if (y) y[k] = a.y;
    if (theta) theta[k] = a.theta;
    if (ux) ux[k] = a.ux;
    if (uy) uy[k] = a.uy;
    if (omega) omega[k] = a.omega;
    if (Fx) Fx[k] = a.Fx;
    if (Fy) Fy[k] = a.Fy;
    if (Tz) Tz[k] = a.Tz;
  }
  return 0;
}

extern "C" int oracle_get_links(oracle_lbm_t* h, long long* n, int* pid, int* i, int* j,
                                int* alpha, double* q) {
  if (!h || !n) return E_ARG;
  std::vector<Link> links;
  build_links(h, links);
  return copy_links(links, n, pid, i, j, alpha, q);
}

extern "C" int oracle_get_links_bruteforce(oracle_lbm_t* h, long long* n, int* pid, int* i, int* j,
                                           int* alpha, double* q) {
  if (!h || !n) return E_ARG;
  const int np = (int)h->parts.size();
  auto covering = [&](int a, int b) -> int { /* lowest pid whose disc covers node (a,b) */
    for (int p = 0; p < np; ++p)
      if (inside_p(h->parts[p], (double)a, (double)b)) return p;
    return -1;
  };
  std::vector<Link> links;
  for (int p = 0; p < np; ++p)
    for (int al = 1; al <= 8; ++al)
      for (int b = 0; b < h->ny; ++b)
        for (int a = 0; a < h->nx; ++a) {
          if (covering(a, b) >= 0) continue;
          int bi = a + EX[al], bj = b + EY[al];
          if (bi < 0 || bi >= h->nx || bj < 0 || bj >= h->ny) continue;
          if (covering(bi, bj) != p) continue;
          Link L;
          L.pid = p;
          L.i = a;
          L.j = b;
          L.alpha = al;
          L.q = q_p(h->parts[p], (double)a, (double)b, al);
          links.push_back(L);
        }
  return copy_links(links, n, pid, i, j, alpha, q);
}

extern "C" int oracle_destroy(oracle_lbm_t* h) {
  delete h;
  return 0;
}

extern "C" const char* oracle_last_error(const oracle_lbm_t* h) {
  return h ? h->err.c_str() : g_create_error.c_str();
}
