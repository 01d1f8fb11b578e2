/*
 * lbm_oracle.h -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, single-threaded CPU oracle for the particle-resolved thermal lattice Boltzmann
 * time step of Xu & Li (arXiv 2308.16597), written from the paper and from the
 * readings in SURVEY.md 8(c) / DESIGN.md "Readings".  It shares NO code with the CUDA path
 * (paper_2308_16597_b200/csrc) and neither includes the other.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may load it.
 *
 * All pointers are host pointers.  Return codes: 0 OK, -1 ARG, -2 STATE, -3 CAPACITY,
 * -5 NONFINITE (numerically the same values as the product's, defined independently).
 *
 * Parity status: every piece below is pinned by tests/test_oracle_*.py to closed forms,
 * invariants or brute force, EXCEPT the whole coupled moving-particle step (choice of M, S, N, Q,
 * integrator, fallback ladders, e_c rule), for which the paper prints no field or trajectory
 * values: "parity unpinned against the paper" for that composite.
 */
#ifndef LBM_ORACLE_H
#define LBM_ORACLE_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_lbm oracle_lbm_t;

typedef struct {
  double nu, kappa, rho0, T0, g, gbeta, body_ax, body_ay;
  int    periodic_x;
  int    wall_T_type[4];   /* W,E,S,N: 0 adiabatic, 1 Dirichlet */
  double wall_T[4];
  double rep_s, rep_eps;
  int    rep_power;
  int    max_particles, max_links_per_particle;
} oracle_params;

/* ---- whole-simulation interface (mirrors the product's calls) ---- */
int  oracle_create(int nx, int ny, const oracle_params* p, oracle_lbm_t** out);
int  oracle_set_temperature(oracle_lbm_t* h, const double* T);
int  oracle_add_particles(oracle_lbm_t* h, int n, const double* x, const double* y,
                          const double* diam, const double* rho_ratio, const double* T_w,
                          const double* ux, const double* uy, const double* omega,
                          const unsigned char* fixed);
/* elliptical particles: full axes major (along the body axis that makes the
 * angle theta with x) and minor; equal axes = a circle through the circle formulas */
int  oracle_add_ellipses(oracle_lbm_t* h, int n, const double* x, const double* y,
                         const double* major, const double* minor, const double* theta,
                         const double* rho_ratio, const double* T_w, const double* ux,
                         const double* uy, const double* omega, const unsigned char* fixed);
int  oracle_step(oracle_lbm_t* h, int nsteps);
int  oracle_get_fields(oracle_lbm_t* h, double* rho, double* ux, double* uy, double* T,
                       double* f, double* g, unsigned char* flag);
int  oracle_get_particles(oracle_lbm_t* h, int* n, double* x, double* y, double* theta,
                          double* ux, double* uy, double* omega,
                          double* Fx, double* Fy, double* Tz);
/* links by the paper's per-particle effective-zone scan, order (p, alpha, j, i) */
int  oracle_get_links(oracle_lbm_t* h, long long* n, int* pid, int* i, int* j, int* alpha,
                      double* q);
/* links by a full-lattice scan with a per-node loop over ALL particles (no zone, no owner map) */
int  oracle_get_links_bruteforce(oracle_lbm_t* h, long long* n, int* pid, int* i, int* j,
                                 int* alpha, double* q);
/* pre-collision populations f(x,t), g(x,t) (the oracle's own state), 9n and 5n doubles */
int  oracle_get_precollision(oracle_lbm_t* h, double* f, double* g);
/* deep-run parity check: inject post-collision populations (9n, 5n doubles, population-major) and
 * particle states taken from elsewhere; the next oracle_step starts after the collision.  Until
 * that step has run, oracle_get_fields / oracle_get_precollision still show the old state. */
int  oracle_set_state(oracle_lbm_t* h, const double* fpost, const double* gpost, int n,
                      const double* x, const double* y, const double* theta,
                      const double* ux, const double* uy, const double* omega);
int  oracle_destroy(oracle_lbm_t* h);
const char* oracle_last_error(const oracle_lbm_t* h);

/* ---- the pieces, exposed so that tests can pin each one to a closed form ---- */
void   oracle_feq(double rho, double ux, double uy, double* out9);          /* M^-1 m_eq      */
void   oracle_geq(double T, double ux, double uy, double kappa, double* out5); /* N^-1 n_eq   */
void   oracle_moments_f(const double* f9, double* m9);                      /* m = M f        */
void   oracle_moments_g(const double* g5, double* n5);                      /* n = N g        */
void   oracle_from_moments_f(const double* m9, double* f9);                 /* f = M^-1 m     */
void   oracle_from_moments_g(const double* n5, double* g5);                 /* g = N^-1 n     */
void   oracle_relaxation_rates(double nu, double kappa, double* S9, double* Q5, double* aT);
void   oracle_macroscopic(const oracle_params* p, const double* f9, const double* g5,
                          double* rho, double* ux, double* uy, double* T);
void   oracle_collide_node(const oracle_params* p, const double* f9, const double* g5,
                           double* fpost9, double* gpost5);                 /* Eqs. (5), (6)  */
double oracle_link_q(double xf, double yf, int alpha, double xc, double yc, double r);
double oracle_link_q_ellipse(double xf, double yf, int alpha, double xc, double yc, double a,
                             double b, double c, double s);
void oracle_rotate_unit(double* c, double* s, double d);
/* Eqs. (9)/(10) with the fallback ladder; nbehind = how many of x_f-e_i, x_f-2e_i are fluid
 * (counted contiguously from x_f): 2, 1 or 0.  fi_k = f_i^+(x_f - k e_i), fib_k = f_ibar^+(...) */
double oracle_bounce_back_f(int alpha, double q, double fi_0, double fi_1, double fi_2,
                            double fib_0, double fib_1, int nbehind,
                            double rho0, double uwx, double uwy);
/* Eqs. (11)/(12); alpha in 1..4 */
double oracle_bounce_back_g(int alpha, double q, double gi_0, double gi_1, double gib_0,
                            int nbehind, double kappa, double Tw);
/* Eqs. (13)/(14), one link: dP[0..1] momentum, dP[2] z-torque about (xc,yc) */
void   oracle_momentum_exchange(int alpha, double fi_post, double fibar_new,
                                double uwx, double uwy, double rwx, double rwy, double* dP3);
double oracle_repulsion_mag(double C, double eps, double s, double delta, int power); /* Eq. 15 */
/* Eqs. (7)/(8), one step, in place: state = {x, y, theta, ux, uy, omega} */
void   oracle_integrate(double* state6, double Fx, double Fy, double Tz, double mass,
                        double inertia);
int    oracle_refill_direction(double nx_, double ny_);                     /* e_c */
/* outward normal (not normalised) of an ellipse (semi-axes a, b, orientation (c, s)) at the point
 * (dx, dy) relative to its centre: the n of PAPER.md:151 for an elliptical particle */
void   oracle_ellipse_normal(double dx, double dy, double a, double b, double c, double s,
                             double* nx_, double* ny_);
/* Eq. (16) + fallback ladder + MRT momentum constraint */
void   oracle_refill_f(int nvalid, const double* f1, const double* f2, const double* f3,
                       double rho0, double uwx, double uwy, double* out9);

#ifdef __cplusplus
}
#endif
#endif
