// Device-side arithmetic of the hot path: stiffened-gas primitives, WENO5-JS, HLLC.
// Hand-written for sm_100a fp64.  Citations are PAPER.md lines; O-/A-/N-numbers refer to DESIGN.md §2-§3.
// This file shares nothing with oracle/ (the CPU oracle is written separately from the paper).
#pragma once
#include <cuda_runtime.h>

namespace mfc {

enum { BC_PERIODIC = 0, BC_EXTRAP = 1, BC_HALO = 2 };
enum { WENO_JS = 0, WENO_M = 1, WENO_Z = 2 };  // nonlinear weights (mfc_weno of include/mfc_b200.h)

// Kernel parameters (passed by value; lives in the constant bank of each launch).
struct KP {
  int n[3];
  int bc_lo[3], bc_hi[3];
  long long ncells;
  double dx[3], inv_dx[3];
  double G[3];   // G_i = 1/(gamma_i - 1)
  double P[3];   // P_i = gamma_i pi_inf_i/(gamma_i - 1)
  double eps4;   // 4 * weno_eps (the smoothness indicators are carried scaled by 4)
  double alpha_floor;
  int clamp;
  double eta;    // uniform shear viscosity of PAPER.md eq.(1); 0 = inviscid
  int kapila;    // 1: add K div(u) to the volume-fraction equations (two fluids)
  double gam[2]; // gamma_i and gamma_i pi_inf_i of the two fluids: rho_i c_i^2 = gamma_i p + gamma_i pi_inf_i (eq. 6)
  double gpi[2];
  int* flag;     // sticky non-physical flag (A19)
  const double* dt_dev;  // if not NULL the RK stages take dt from here (mfc_advance keeps dt on the device) instead of the argument
  // BC_HALO on the last direction (slab decomposition): the three ghost layers beyond each end, [neq][3][plane]
  const double* halo_lo;
  const double* halo_hi;
  // velocities of the ghost layer next to each such end, [D][plane] (viscous terms on a slab)
  const double* vel_halo_lo;
  const double* vel_halo_hi;
};

// O1: logical cell g in [-3, n+2] -> interior cell that supplies its value.
__device__ __forceinline__ int ghost_index(int g, int n, int bc_lo, int bc_hi) {
  if (g < 0) return bc_lo == BC_PERIODIC ? ((g % n) + n) % n : 0;
  if (g >= n) return bc_hi == BC_PERIODIC ? g % n : n - 1;
  return g;
}

// 1/x for normal x: the 2^-23 hardware seed (MUFU.RCP64H) plus one cubically convergent step
// y(1 + e + e^2), e = 1 - x y  ->  relative error ~2^-69 before the final rounding.
__device__ __forceinline__ double frcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);
  const double t = fma(e, e, e);
  return fma(y, t, y);
}

// O5-K (eq.(5) with the sign of reading A13): K of the alpha_1 equation for two fluids,
//   K = (A2 - A1)/(A1/alpha_1 + A2/alpha_2) = alpha_1 alpha_2 (A2 - A1)/(alpha_2 A1 + alpha_1 A2),  A_i = rho_i c_i^2 = gamma_i (p + pi_inf_i);
// the second form has one reciprocal and is 0, not 0/0, when a volume fraction vanishes.
__device__ __forceinline__ double kapila_K(const KP& kp, double p, double a1, double a2) {
  const double A1 = fma(kp.gam[0], p, kp.gpi[0]), A2 = fma(kp.gam[1], p, kp.gpi[1]);
  const double den = fma(a2, A1, a1 * A2);
  return ((a1 * a2) * (A2 - A1)) * frcp(den);
}

// sqrt(a/b) for a b > 0 without forming the quotient: a * rsqrt(a b), the hardware rsqrt seed y refined by one cubically
// convergent step y (1 + e/2 + 3 e^2/8), e = 1 - (a b) y^2.  Measured on B200 (mfc_sqrt_ratio_values,
// tests/test_gpu_parity.py::test_sqrt_ratio_unit_entry_point, 2^18 pairs over 280 decades of a b): the seed's relative error
// is at most 2^-20.1 (rsqrt.approx.ftz.f64 looks at the upper half of its operand), so e <= 2^-19 and the neglected e^3 term
// is ~2^-59; with the roundings of t y, the two FMAs and the final product the result is within 1.86 ulp of the correctly
// rounded sqrt(a/b).  8 FP64 instructions and one MUFU where reciprocal + multiply + square root took 12 and two.
// RANGE: the PRODUCT t = a b must be a normal double — it has half the exponent range of the quotient.  t flushed to zero
// (ftz) fails the callers' `ct > 0` test and the face is flagged non-physical; t overflowing to +inf would pass that test
// and give 0.  For the sound speed t ~ p Gamma rho, 1e3..1e14 in SI units (1e-2..1e3 nondimensional): far inside.
__device__ __forceinline__ double fsqrt_ratio(double a, double t /* = a b */) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(t));
  const double e = fma(-(t * y), y, 1.0);
  const double pe = fma(0.375, e, 0.5) * e;
  return a * fma(y, pe, y);
}

// O2 (eq.(4), 117, 165): conservative cell -> primitive cell.
// Pi and Gamma are summed with individually rounded products in fluid order (N1): with water
// (P_i = 7.8e8) at p = 1e5 the energy carries p in its last digits, so (E - Pi) must see the same Pi
// bits as any other evaluation of this definition.  EXACT additionally uses IEEE division and unfused
// squares (mfc_prim_from_cons, mfc_cfl_dt: bandwidth-bound kernels); the sweeps use the fast reciprocal.
// Returns true if rho is not positive (A19).
template <int N, int D, bool EXACT>
__device__ __forceinline__ bool prim_cell(const KP& kp, const double* q, double* w) {
  constexpr int IM = N, IE = N + D, IA = N + D + 1;
  double rho = q[0];
#pragma unroll
  for (int i = 1; i < N; ++i) rho = __dadd_rn(rho, q[i]);
  double usq;
  if (EXACT) {
#pragma unroll
    for (int d = 0; d < D; ++d) {
      const double u = __ddiv_rn(q[IM + d], rho);
      w[IM + d] = u;
      usq = d == 0 ? __dmul_rn(u, u) : __dadd_rn(usq, __dmul_rn(u, u));
    }
  } else {
    const double rr = frcp(rho);
#pragma unroll
    for (int d = 0; d < D; ++d) {
      double u = q[IM + d] * rr;
      u = fma(fma(-rho, u, q[IM + d]), rr, u);  // one residual step: the quotient to ~1/2 ulp (N2)
      w[IM + d] = u;
      usq = d == 0 ? u * u : fma(u, u, usq);
    }
  }
  double Gam = __dmul_rn(q[IA], kp.G[0]), Pi = __dmul_rn(q[IA], kp.P[0]);
#pragma unroll
  for (int i = 1; i < N; ++i) {
    Gam = __dadd_rn(Gam, __dmul_rn(q[IA + i], kp.G[i]));
    Pi = __dadd_rn(Pi, __dmul_rn(q[IA + i], kp.P[i]));
  }
  const double ke = __dmul_rn(__dmul_rn(0.5, rho), usq);
  const double num = __dadd_rn(__dadd_rn(q[IE], -Pi), -ke);
  w[IE] = EXACT ? __ddiv_rn(num, Gam) : num * frcp(Gam);
#pragma unroll
  for (int i = 0; i < N; ++i) {
    w[i] = q[i];
    w[IA + i] = q[IA + i];
  }
  return !(rho > 0.0);
}

// O3 (Jiang-Shu coefficients, A3).  Stencil (a,b,c,d,e) = w_{i-2..i+2}.
// L = left-biased value at i+1/2 (q^L of face i+1/2), R = right-biased value at i-1/2 (q^R of face i-1/2).
// Same definition as the plain formula, arranged for the FP64 pipe:
//   * everything in first differences d1..d4, so each candidate is c + (combination of differences)/6
//     and, since the weights sum to one, value = c + sum_r a_r P_r / sum_r a_r;
//   * the smoothness indicators are carried scaled by 4 (13/3 t^2 + s^2 + 4 eps) — a common factor of
//     the three a_r cancels in the normalisation;
//   * product form of the weights: a_r = d_r /(beta_r+eps)^2 is multiplied through by
//     prod_j (beta_j+eps)^2, which leaves ONE reciprocal per reconstructed value and no other division;
//   * beta_r and the three products are shared by the two values of the cell.
// Split in two so that the y/z sweeps, which march along the stencil direction, can carry the per-cell
// pieces (first differences d_k and u_k = 13/3 t_k^2 + 4 eps of the second differences t_k) from step to step
// instead of recomputing them: weno5_u forms one u_k, weno5_core takes (c; d1..d4; u0..u2).
// The coefficients live in constant memory so that they reach the FP64 instructions as constant-bank
// operands: as literals ptxas re-materialises each of them with two UMOVs per loop iteration (measured in round 1:
// slower), instructions the loop does not need.
enum { W_C133, W_03, W_06, W_01, W_5_60, W_M2_60, W_02, W_M005, W_M02, W_005, W_M01, W_2_60, W_M5_60, W_COUNT };
__constant__ double WC[W_COUNT] = {13.0 / 3.0, 0.3, 0.6, 0.1, 5.0 / 60.0, -2.0 / 60.0, 0.2, -0.05, -0.2, 0.05, -0.1,
                                   2.0 / 60.0, -5.0 / 60.0};
#define WCV(i) WC[i]

__device__ __forceinline__ double weno5_u(double t, double eps4) { return fma(WCV(W_C133) * t, t, eps4); }

// Both face values of a cell from its centre value c, the first differences d1..d4 of its stencil and
// u_k = 13/3 t_k^2 + 4 eps of its three second differences; WV = WENO_JS / WENO_M / WENO_Z selects the nonlinear weights.
template <int WV>
__device__ __forceinline__ void weno5_core(double c, double d1, double d2, double d3, double d4, double u0, double u1,
                                           double u2, double& L, double& R) {
  const double s0 = fma(3.0, d2, -d1), s1 = d2 + d3, s2 = fma(-3.0, d3, d4);
  const double b0 = fma(s0, s0, u0);  // 4 (beta_r + eps)
  const double b1 = fma(s1, s1, u1);
  const double b2 = fma(s2, s2, u2);
  // E_jk: the weight of stencil r multiplied through by the product of all three denominators
  //   JS: a_r = d_r/(beta_r+eps)^2                  ->  d_r (b_j b_k)^2
  //   Z  (q = 1): a_r = d_r (1 + tau/(beta_r+eps)) = d_r (b_r + tau4)/b_r  ->  d_r (b_r + tau4) b_j b_k,
  //      tau4 = |b0 - b2| = 4 tau (eps cancels in the difference)
  //   M: the JS weights, normalised, then Henrick's map (below)
  double E12, E02, E01;
  if (WV == WENO_Z) {
    const double tau = fabs(b0 - b2);
    const double p12 = b1 * b2, p02 = b0 * b2, p01 = b0 * b1;
    const double P = b0 * p12;
    E12 = fma(tau, p12, P);
    E02 = fma(tau, p02, P);
    E01 = fma(tau, p01, P);
  } else {
    const double e0 = b0 * b0, e1 = b1 * b1, e2 = b2 * b2;
    E12 = e1 * e2, E02 = e0 * e2, E01 = e0 * e1;
  }
  if (WV != WENO_M) {
    const double S6 = WCV(W_06) * E02;  // the middle stencil has the ideal weight 6/10 in both values
    {  // ideal weights (1/10, 6/10, 3/10); candidates c + (5 d2 - 2 d1)/6, c + (d2 + 2 d3)/6, c + (4 d3 - d4)/6
      const double S = fma(WCV(W_03), E01, fma(WCV(W_01), E12, S6));
      const double X = WCV(W_02) * d3;  // shared by Q1 and Q2
      const double Q0 = fma(WCV(W_5_60), d2, WCV(W_M2_60) * d1);
      const double Q1 = fma(WCV(W_01), d2, X);
      const double Q2 = fma(WCV(W_M005), d4, X);
      const double num = fma(E01, Q2, fma(E02, Q1, E12 * Q0));
      L = fma(num, frcp(S), c);
    }
    {  // mirror image: ideal weights (3/10, 6/10, 1/10); c + (d1 - 4 d2)/6, c - (2 d2 + d3)/6, c + (2 d4 - 5 d3)/6
      const double S = fma(WCV(W_01), E01, fma(WCV(W_03), E12, S6));
      const double Y = WCV(W_M02) * d2;  // shared by Q0 and Q1
      const double Q0 = fma(WCV(W_005), d1, Y);
      const double Q1 = fma(WCV(W_M01), d3, Y);
      const double Q2 = fma(WCV(W_2_60), d4, WCV(W_M5_60) * d3);
      const double num = fma(E01, Q2, fma(E02, Q1, E12 * Q0));
      R = fma(num, frcp(S), c);
    }
  } else {
    // Henrick's map g_r(w) = w (d_r + d_r^2 - 3 d_r w + w^2)/(d_r^2 + w (1 - 2 d_r)) = n_r/m_r of the normalised JS weights
    // w_r, then omega_r = g_r / sum g.  Multiplied through by m_0 m_1 m_2: A_r = n_r m_j m_k, one more reciprocal.
    // The candidate deviations are P_r = (.)/6 with the 1/6 folded into the constants.
    constexpr double C16 = 1.0 / 6.0, C26 = 2.0 / 6.0, C46 = 4.0 / 6.0, C56 = 5.0 / 6.0;
    auto mapped = [&](double dA, double dB, double dC, double P0, double P1, double P2) {
      // dA, dB, dC: ideal weights of stencils 0, 1, 2
      const double a0 = dA * E12, a1 = dB * E02, a2 = dC * E01;
      const double inv = frcp((a0 + a1) + a2);
      const double w0 = a0 * inv, w1 = a1 * inv, w2 = a2 * inv;
      const double n0 = w0 * fma(w0, w0 - 3.0 * dA, dA + dA * dA);
      const double n1 = w1 * fma(w1, w1 - 3.0 * dB, dB + dB * dB);
      const double n2 = w2 * fma(w2, w2 - 3.0 * dC, dC + dC * dC);
      const double m0 = fma(w0, 1.0 - 2.0 * dA, dA * dA);
      const double m1 = fma(w1, 1.0 - 2.0 * dB, dB * dB);
      const double m2 = fma(w2, 1.0 - 2.0 * dC, dC * dC);
      const double A0 = n0 * (m1 * m2), A1 = n1 * (m0 * m2), A2 = n2 * (m0 * m1);
      const double num = fma(A2, P2, fma(A1, P1, A0 * P0));
      return fma(num, frcp((A0 + A1) + A2), c);
    };
    L = mapped(0.1, 0.6, 0.3, fma(C56, d2, -C26 * d1), fma(C16, d2, C26 * d3), fma(C46, d3, -C16 * d4));
    R = mapped(0.3, 0.6, 0.1, fma(-C46, d2, C16 * d1), fma(-C26, d2, -C16 * d3), fma(C26, d4, -C56 * d3));
  }
}

template <int WV>
__device__ __forceinline__ void weno5(double a, double b, double c, double d, double e, double eps4, double& L,
                                      double& R) {
  const double d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
  weno5_core<WV>(c, d1, d2, d3, d4, weno5_u(d2 - d1, eps4), weno5_u(d3 - d2, eps4), weno5_u(d4 - d3, eps4), L, R);
}

// O4 (S_L,S_R 653-654; S* 664; rho* 668; A5-A8): HLLC at one face with normal direction
// DIR from the reconstructed primitives wL, wR.  Writes the flux F[neq] and the face velocity uf
// (A7: the HLLC flux of a unit scalar).  Returns true if a face state is non-physical.
//
// Branch-free form of the four-way selection (first match in the printed order, A8):
//   side K = L if (S_L >= 0 or S* >= 0) else R;  star = (K = L) ? !(S_L >= 0) : (S_R > 0).
// With ds = S* - u_K (0 outside the fan), r = 1/(S_K - S*), chi - 1 = ds r, the star-state correction
// S_K (q*_K - q_K) collapses to
//   alpha_i rho_i, alpha_i, rho u_t :  q u_f,           u_f = u_K + S_K (chi - 1) = chi S*
//   rho u_n :  rho u_K^2 + p + S_K rho (chi ds + (chi-1) u_K)
//   E       :  (E + p) u_K + S_K ((chi-1) E + chi ds rho S* + ds p r)        [uses chi/(S_K-u_K) = r]
template <int N, int D, int DIR>
__device__ __forceinline__ bool hllc(const KP& kp, const double* wL, const double* wR, double* F, double& uf) {
  constexpr int IM = N, IE = N + D, IA = N + D + 1, NEQ = 2 * N + D + 1;
  double rho[2], E[2], c[2], un[2], p[2];
  bool bad = false;
#pragma unroll
  for (int K = 0; K < 2; ++K) {
    const double* w = K ? wR : wL;
    double r = w[0], Gam = w[IA] * kp.G[0], Pi = w[IA] * kp.P[0];
#pragma unroll
    for (int i = 1; i < N; ++i) {
      r += w[i];
      Gam = fma(w[IA + i], kp.G[i], Gam);
      Pi = fma(w[IA + i], kp.P[i], Pi);
    }
    double usq = w[IM] * w[IM];
#pragma unroll
    for (int d = 1; d < D; ++d) usq = fma(w[IM + d], w[IM + d], usq);
    rho[K] = r;
    p[K] = w[IE];
    un[K] = w[IM + DIR];
    E[K] = fma(0.5 * r, usq, fma(Gam, p[K], Pi));
    const double cn = fma(Gam + 1.0, p[K], Pi), ct = cn * (Gam * r);  // A5: c^2 = cn / (Gamma rho); ct has the sign of c^2
    bad = bad || !(r > 0.0) || !(ct > 0.0);
    c[K] = fsqrt_ratio(cn, ct);
  }
  const double SL = fmin(un[0] - c[0], un[1] - c[1]);
  const double SR = fmax(un[0] + c[0], un[1] + c[1]);
  const double mL = rho[0] * (SL - un[0]), mR = rho[1] * (SR - un[1]);
  const double Ss = fma(mL, un[0], fma(-mR, un[1], p[1] - p[0])) * frcp(mL - mR);
  const bool useL = (SL >= 0.0) || (Ss >= 0.0);
  const bool star = useL ? !(SL >= 0.0) : (SR > 0.0);
  const double rhoK = useL ? rho[0] : rho[1];
  const double unK = useL ? un[0] : un[1];
  const double pK = useL ? p[0] : p[1];
  const double EK = useL ? E[0] : E[1];
  const double SK = useL ? SL : SR;
  const double r = frcp(SK - Ss);
  const double ds = star ? (Ss - unK) : 0.0;
  const double chim1 = ds * r;
  const double chi = 1.0 + chim1;
  // u_f = u_K + S_K (chi - 1) = chi S* inside the fan (no cancellation in this form), u_K outside
  uf = star ? fma(chim1, Ss, Ss) : unK;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    F[i] = (useL ? wL[i] : wR[i]) * uf;
    F[IA + i] = (useL ? wL[IA + i] : wR[IA + i]) * uf;
  }
  const double rhoSK = rhoK * SK;
#pragma unroll
  for (int d = 0; d < D; ++d) {
    if (d == DIR) {
      F[IM + d] = fma(rhoSK, fma(chi, ds, chim1 * unK), fma(rhoK * unK, unK, pK));
    } else {
      F[IM + d] = (rhoK * (useL ? wL[IM + d] : wR[IM + d])) * uf;
    }
  }
  const double corr = fma(chim1, EK, fma(chi * ds, rhoK * Ss, (ds * pK) * r));
  F[IE] = fma(SK, corr, (EK + pK) * unK);
  (void)NEQ;
  return bad;
}

}  // namespace mfc
