// collide.cuh -- per-node macroscopic moments, Boussinesq forcing and MRT collision of the D2Q9
// (flow) and D2Q5 (temperature) populations, in registers.
//
// Eq. (5)  f+ = f - M^-1 S (m - m_eq) + dt F'
// Eq. (6)  g+ = g - N^-1 Q (n - n_eq)
// rho = sum f, u = (sum e f + F/2)/rho, F = rho g beta (T - T0) y^, T = sum g
// M, S, m_eq, N, Q, n_eq and the Guo forcing in moment space are the readings of DESIGN.md
// (Lallemand-Luo basis; D2Q5 basis with a_T = 20 sqrt3 kappa - 4).  The transforms are written
// out as sums/differences of pairs (the rows of M and N are orthogonal, so M^-1 = M^T diag(1/|row|^2)).
#pragma once
#include "lbm_internal.cuh"

// in: pre-collision f[9], g[5] (after streaming).  out: post-collision, in place.
__device__ __forceinline__ void mrt_collide(double (&f)[9], double (&g)[5], const LbmConst& c) {
  // ---- temperature moments
  const double g13 = g[1] + g[3], g24 = g[2] + g[4];
  const double gs = g13 + g24;
  const double T = g[0] + gs;
  const double n1 = g[1] - g[3], n2 = g[2] - g[4];
  const double n3 = gs - 4.0 * g[0];
  const double n4 = g13 - g24;
  // ---- flow moments
  const double s13 = f[1] + f[3], s24 = f[2] + f[4], d13 = f[1] - f[3], d24 = f[2] - f[4];
  const double s57 = f[5] + f[7], s68 = f[6] + f[8], d57 = f[5] - f[7], d68 = f[6] - f[8];
  const double sa = s13 + s24, sd = s57 + s68;
  const double dxx = d57 - d68, dyy = d57 + d68;
  const double rho = f[0] + (sa + sd);
  const double jx = d13 + dxx, jy = d24 + dyy;
  const double e = (2.0 * sd - sa) - 4.0 * f[0];
  const double eps = (sd - 2.0 * sa) + 4.0 * f[0];
  const double qx = dxx - 2.0 * d13, qy = dyy - 2.0 * d24;
  const double pxx = s13 - s24, pxy = s57 - s68;
  // ---- force and velocity
  const double Fx = rho * c.ax;
  const double Fy = rho * (c.ay + c.gbeta * (T - c.T0));
  const double inv = __drcp_rn(rho);
  const double ux = (jx + 0.5 * Fx) * inv;
  const double uy = (jy + 0.5 * Fy) * inv;
  const double uxx = ux * ux, uyy = uy * uy;
  const double usq3 = 3.0 * (uxx + uyy);
  const double uF6 = 6.0 * (ux * Fx + uy * Fy);
  // ---- relaxation + Guo forcing in moment space: m+ = m - S(m - m_eq) + (I - S/2) M F~
  const double ep = e - c.s_e * (e - rho * (usq3 - 2.0)) + (1.0 - 0.5 * c.s_e) * uF6;
  const double epsp = eps - c.s_eps * (eps - rho * (1.0 - usq3)) - (1.0 - 0.5 * c.s_eps) * uF6;
  const double jxp = jx + Fx, jyp = jy + Fy;
  const double hq = 1.0 - 0.5 * c.s_q;
  const double qxp = qx - c.s_q * (qx + rho * ux) - hq * Fx;
  const double qyp = qy - c.s_q * (qy + rho * uy) - hq * Fy;
  const double hn = 1.0 - 0.5 * c.s_nu;
  const double pxxp = pxx - c.s_nu * (pxx - rho * (uxx - uyy)) + hn * 2.0 * (ux * Fx - uy * Fy);
  const double pxyp = pxy - c.s_nu * (pxy - rho * ux * uy) + hn * (ux * Fy + uy * Fx);
  // ---- back to populations: f = M^T diag(1/9,1/36,1/36,1/6,1/12,1/6,1/12,1/4,1/4) m+
  const double a0 = rho * (1.0 / 9.0), a1 = ep * (1.0 / 36.0), a2 = epsp * (1.0 / 36.0);
  const double a3 = jxp * (1.0 / 6.0), a4 = qxp * (1.0 / 12.0);
  const double a5 = jyp * (1.0 / 6.0), a6 = qyp * (1.0 / 12.0);
  const double a7 = pxxp * 0.25, a8 = pxyp * 0.25;
  const double ba = a0 - a1 - 2.0 * a2;
  const double bd = a0 + 2.0 * a1 + a2;
  const double X1 = a3 - 2.0 * a4, Y1 = a5 - 2.0 * a6;
  const double X2 = a3 + a4, Y2 = a5 + a6;
  f[0] = a0 - 4.0 * (a1 - a2);
  f[1] = (ba + a7) + X1;
  f[3] = (ba + a7) - X1;
  f[2] = (ba - a7) + Y1;
  f[4] = (ba - a7) - Y1;
  f[5] = (bd + a8) + (X2 + Y2);
  f[7] = (bd + a8) - (X2 + Y2);
  f[6] = (bd - a8) - (X2 - Y2);
  f[8] = (bd - a8) + (X2 - Y2);
  // ---- temperature: n+ = n - Q(n - n_eq), n_eq = (T, ux T, uy T, a_T T, 0)
  const double n1p = n1 - c.q_k * (n1 - ux * T);
  const double n2p = n2 - c.q_k * (n2 - uy * T);
  const double n3p = n3 - c.q_e * (n3 - c.aT * T);
  const double n4p = n4 - c.q_nu * n4;
  const double b0 = T * 0.2, b1 = 0.5 * n1p, b2 = 0.5 * n2p, b3 = n3p * 0.05, b4 = 0.25 * n4p;
  g[0] = b0 - 4.0 * b3;
  g[1] = (b0 + b3 + b4) + b1;
  g[3] = (b0 + b3 + b4) - b1;
  g[2] = (b0 + b3 - b4) + b2;
  g[4] = (b0 + b3 - b4) - b2;
}

// Macroscopic fields from either state.  post = 1: f, g are POST-collision (the resident state);
// rho and T are collision invariants and sum e f+ = sum e f + F, so u = (sum e f+ - F/2)/rho.
__device__ __forceinline__ void macroscopic(const double (&f)[9], const double (&g)[5],
                                            const LbmConst& c, int post, double& rho, double& ux,
                                            double& uy, double& T) {
  T = g[0] + ((g[1] + g[3]) + (g[2] + g[4]));
  rho = f[0] + (((f[1] + f[3]) + (f[2] + f[4])) + ((f[5] + f[7]) + (f[6] + f[8])));
  const double jx = (f[1] - f[3]) + ((f[5] - f[7]) - (f[6] - f[8]));
  const double jy = (f[2] - f[4]) + ((f[5] - f[7]) + (f[6] - f[8]));
  const double Fx = rho * c.ax;
  const double Fy = rho * (c.ay + c.gbeta * (T - c.T0));
  const double h = post ? -0.5 : 0.5;
  ux = (jx + h * Fx) / rho;
  uy = (jy + h * Fy) / rho;
}
