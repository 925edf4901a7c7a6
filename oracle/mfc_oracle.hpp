// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, CPU implementation of the finite-volume right-hand side of the
// 5-equation (Allaire) multi-component model with stiffened-gas EOS, WENO5-JS +
// HLLC, SSP-RK3, written step by step from /root/reference/PAPER.md (MFC 5.0,
// arxiv 2503.07953).  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may use it.  It shares no code with the
// CUDA path under paper_2503_07953_b200/csrc and neither includes the other.
//
// Passages followed (PAPER.md line : section/equation):
//   57-61   §2.1.1 five-equation model            76  eq.(4) mixture rules
//   117     §2.2   stiffened-gas EOS              133-143 eqs.(9),(10), div u
//   151-165 §3.2.1 reconstruction of primitives   187-199 §3.2.2 HLLC
//   203     §3.3   ghost ("buffer") cells         207-211 §3.4 SSP-RK3
//   653-654, 664, 668 (§4.2.5) wave-speed, S_M and rho* formulas
// Readings of silent/garbled points carry the A-numbers of DESIGN.md §3.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): prim round trip and pure-fluid
// closed form (O2); WENO linear/closed-form/ENO/mirror/order-5 (O3); HLLC
// consistency, upwinding, stationary contact, mirror (O4); Sod and water/air
// exact Riemann solutions, uniform-state, conservation, interface equilibrium,
// alpha==1 (O2-O6); third-order convergence in dt and the amplification polynomial
// 1 + z + z^2/2 + z^3/6 of rk3_step (O6, tests/test_oracle_rk3.py).  cfl_dt (A9) and
// the clamp (A10) are defined by BASELINE.json only, not by the paper: "parity
// unpinned" beyond their closed-form definition tests.
//
// Everything is a template on the scalar T so that the same text gives the
// fp64 oracle, a long double adjudicator and an operation-counting build.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <vector>

namespace mfc_oracle {

constexpr int kMaxFluids = 4;
constexpr int kMaxEq = 2 * kMaxFluids + 3 + 1;

enum { BC_PERIODIC = 0, BC_EXTRAP = 1 };
// RECON_WENO5_M: mapped weights of Henrick et al. (the paper's ref. [30]);
// RECON_WENO5_Z: WENO-Z weights (§4.2.2) with q = 1.
// MODEL_ALLAIRE: d(alpha_i)/dt + u.grad(alpha_i) = 0 ("the model reduces to that of Allaire et al.");
// MODEL_KAPILA: ... = K_i div(u) with eq.(5), two fluids.
enum { MODEL_ALLAIRE = 0, MODEL_KAPILA = 1 };
enum { RECON_PIECEWISE_CONSTANT = 1, RECON_WENO5_JS = 5, RECON_WENO5_M = 6, RECON_WENO5_Z = 7 };
// FORM_DIFFERENCE: O3 and O4 evaluated as DESIGN.md readings N2 / N3 write them (deviations from the cell value in first
// differences; star-state jump with chi - 1 formed directly) — what every parity bar is measured against.
// FORM_TEXTBOOK: the same definitions typed as the paper prints them: f = sum_r omega_r f^(r) with the
// Jiang-Shu candidate polynomials, F = F_K + S_K (q*_K - q_K) with q*_K formed first (668).  A second,
// independent evaluation of the same mathematics: tests use it to show that the CUDA path agrees with the paper's text as
// closely as that text's own fp64 rounding allows, whatever form the first oracle is written in.
enum { FORM_DIFFERENCE = 0, FORM_TEXTBOOK = 1 };

// generic helpers so that T may be double, long double or the counting type
template <class T> inline T o_sqrt(const T& x) { using std::sqrt; return sqrt(x); }
template <class T> inline T o_abs(const T& x) { return x < T(0) ? T(0) - x : x; }
template <class T> inline T o_min(const T& a, const T& b) { return b < a ? b : a; }
template <class T> inline T o_max(const T& a, const T& b) { return a < b ? b : a; }
// a rational constant a/b of the scheme, formed in T (so that long double gets it to full precision)
template <class T> inline T o_ratio(int a, int b) { return T(a) / T(b); }

template <class T>
struct Params {
  int ndim = 1;            // D, 1..3
  int n[3] = {1, 1, 1};    // cells; n[d] = 1 for d >= D
  T dx[3] = {T(1), T(1), T(1)};
  int nfluids = 1;         // N
  T gamma[kMaxFluids];     // gamma_i
  T pi_inf[kMaxFluids];    // pi_inf_i
  int bc_lo[3] = {0, 0, 0}, bc_hi[3] = {0, 0, 0};
  T weno_eps = T(1e-16);   // A4
  T alpha_floor = T(1e-6); // A10
  int clamp = 0;           // A10
  int recon = RECON_WENO5_JS;
  int model = MODEL_ALLAIRE;
  T eta = T(0);            // uniform shear viscosity of eq.(1) (A22); 0 = inviscid
  int form = FORM_DIFFERENCE;  // evaluation form of O3 / O4 (WENO5-JS and HLLC): readings N2, N3 or the textbook text

  int neq() const { return 2 * nfluids + ndim + 1; }  // PAPER.md:704 "two advected species (8 PDEs)" in 3D
  std::size_t cells() const { return std::size_t(n[0]) * n[1] * n[2]; }
  // variable slots, identical for q and w (PAPER.md:165 lists them in this order)
  int i_arho(int i) const { return i; }
  int i_mom(int d) const { return nfluids + d; }
  int i_E() const { return nfluids + ndim; }
  int i_alpha(int i) const { return nfluids + ndim + 1 + i; }
  // G_i = 1/(gamma_i-1), P_i = gamma_i pi_inf_i/(gamma_i-1)   (from PAPER.md:117 with eq.(4)),
  // formed once by derive() after gamma/pi_inf are set.
  T Gc[kMaxFluids], Pc[kMaxFluids];
  void derive() {
    for (int i = 0; i < nfluids; ++i) {
      Gc[i] = T(1) / (gamma[i] - T(1));
      Pc[i] = (gamma[i] * pi_inf[i]) / (gamma[i] - T(1));
    }
  }
  const T& G(int i) const { return Gc[i]; }
  const T& P(int i) const { return Pc[i]; }
};

// O1: ghost cell g in [-3, n+2] -> interior cell supplying its value.
inline int ghost_index(int g, int n, int bc_lo, int bc_hi) {
  if (g < 0) return bc_lo == BC_PERIODIC ? ((g % n) + n) % n : 0;
  if (g >= n) return bc_hi == BC_PERIODIC ? g % n : n - 1;
  return g;
}

// O2 (eq.(4), 117, 165): conservative cell -> primitive cell.
// rho e = Gamma p + Pi with Gamma = sum alpha_i G_i, Pi = sum alpha_i P_i; E = rho e + ke.
// Returns 0, or 1 if rho <= 0 / not finite (A19).
template <class T>
int prim_from_cons_cell(const Params<T>& P, const T* q, T* w) {
  const int N = P.nfluids, D = P.ndim;
  T rho = T(0);
  for (int i = 0; i < N; ++i) rho = rho + q[P.i_arho(i)];
  T usq = T(0);
  for (int d = 0; d < D; ++d) {
    T u = q[P.i_mom(d)] / rho;
    w[P.i_mom(d)] = u;
    usq = usq + u * u;
  }
  T Gam = T(0), Pi = T(0);
  for (int i = 0; i < N; ++i) {
    Gam = Gam + q[P.i_alpha(i)] * P.G(i);
    Pi = Pi + q[P.i_alpha(i)] * P.P(i);
  }
  T ke = (T(0.5) * rho) * usq;
  w[P.i_E()] = ((q[P.i_E()] - Pi) - ke) / Gam;
  for (int i = 0; i < N; ++i) {
    w[P.i_arho(i)] = q[P.i_arho(i)];
    w[P.i_alpha(i)] = q[P.i_alpha(i)];
  }
  return (rho > T(0)) ? 0 : 1;
}

// mixture sound speed squared at frozen alpha (A5): c^2 = ((Gamma+1) p + Pi)/(Gamma rho);
// reduces to eq.(6) gamma (p+pi_inf)/rho for a pure fluid.
template <class T>
T sound_speed_sq(const T& Gam, const T& Pi, const T& p, const T& rho) {
  return ((Gam + T(1)) * p + Pi) / (Gam * rho);
}

// O5-K (eqs.(5),(6)): the coefficient K of the K div(u) term of the alpha_1 equation for two
// fluids, from the cell's pressure and volume fractions.  With rho_i c_i^2 = gamma_i (p + pi_inf_i) (eq. 6)
//   K = (rho_2 c_2^2 - rho_1 c_1^2) / (rho_1 c_1^2/alpha_1 + rho_2 c_2^2/alpha_2).
// The paper prints a "+" in the numerator; it must be "-" (reading A13): that is what
// isentropic compression of each phase at common pressure gives (pinned in tests/test_oracle_kapila.py), and
// only then does K vanish for two identical fluids.  The alpha_2 equation takes -K, so that sum alpha_i stays 1.
template <class T>
T kapila_K(const Params<T>& P, const T& p, const T& alpha1, const T& alpha2) {
  const T A1 = P.gamma[0] * (p + P.pi_inf[0]);
  const T A2 = P.gamma[1] * (p + P.pi_inf[1]);
  return (A2 - A1) / (A1 / alpha1 + A2 / alpha2);
}

// O3 (Jiang-Shu coefficients of the paper's refs [30],[70], A3).
// Stencil (a,b,c,d,e) = w_{i-2..i+2}.  *left = left-biased value at i+1/2 (q^L of
// face i+1/2), *right = right-biased value at i-1/2 (q^R of face i-1/2).
// Evaluation form (reading N2): PAPER.md:163 defines f = sum_r omega_r f^(r) with
// sum_r omega_r = 1, hence f = c + sum_r omega_r (f^(r) - c); the candidate deviations f^(r) - c are
// written in the first differences d1..d4 of the stencil:
//   left :  (2a-7b+11c)/6 - c = (5 d2 - 2 d1)/6,  (-b+5c+2d)/6 - c = (d2 + 2 d3)/6,  (2c+5d-e)/6 - c = (4 d3 - d4)/6
//   right:  (-a+5b+2c)/6 - c = (d1 - 4 d2)/6,     (2b+5c-d)/6 - c = -(2 d2 + d3)/6,  (11c-7d+2e)/6 - c = (2 d4 - 5 d3)/6
// Same polynomials as the textbook form, but the rounding error is ~1/2 ulp of the value instead of 3-4 ulp
// (pinned in tests/test_oracle_units.py against the 80-bit evaluation and against the textbook form).
template <class T>
void weno5_js(const T& a, const T& b, const T& c, const T& d, const T& e, const T& eps, T* left, T* right) {
  const T c1312 = o_ratio<T>(13, 12), c14 = o_ratio<T>(1, 4);
  T t0 = a - T(2) * b + c, t1 = b - T(2) * c + d, t2 = c - T(2) * d + e;
  T s0 = a - T(4) * b + T(3) * c, s1 = b - d, s2 = T(3) * c - T(4) * d + e;
  T b0 = c1312 * (t0 * t0) + c14 * (s0 * s0);
  T b1 = c1312 * (t1 * t1) + c14 * (s1 * s1);
  T b2 = c1312 * (t2 * t2) + c14 * (s2 * s2);
  T d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
  // left-biased, ideal weights (1/10, 6/10, 3/10)
  {
    T P0 = (T(5) * d2 - T(2) * d1) / T(6);
    T P1 = (d2 + T(2) * d3) / T(6);
    T P2 = (T(4) * d3 - d4) / T(6);
    T a0 = o_ratio<T>(1, 10) / ((b0 + eps) * (b0 + eps));
    T a1 = o_ratio<T>(6, 10) / ((b1 + eps) * (b1 + eps));
    T a2 = o_ratio<T>(3, 10) / ((b2 + eps) * (b2 + eps));
    T s = a0 + a1 + a2;
    *left = c + ((a0 / s) * P0 + (a1 / s) * P1 + (a2 / s) * P2);
  }
  // right-biased (mirror image), ideal weights (3/10, 6/10, 1/10), same beta
  {
    T P0 = (d1 - T(4) * d2) / T(6);
    T P1 = (T(0) - (T(2) * d2 + d3)) / T(6);
    T P2 = (T(2) * d4 - T(5) * d3) / T(6);
    T a0 = o_ratio<T>(3, 10) / ((b0 + eps) * (b0 + eps));
    T a1 = o_ratio<T>(6, 10) / ((b1 + eps) * (b1 + eps));
    T a2 = o_ratio<T>(1, 10) / ((b2 + eps) * (b2 + eps));
    T s = a0 + a1 + a2;
    *right = c + ((a0 / s) * P0 + (a1 / s) * P1 + (a2 / s) * P2);
  }
}

// O3-M / O3-Z: the same candidates, smoothness indicators and ideal weights as weno5_js; only the step from
// (d_r, beta_r) to the nonlinear weights omega_r differs.
//   RECON_WENO5_JS  alpha_r = d_r/(beta_r+eps)^2,                 omega_r = alpha_r / sum alpha
//   RECON_WENO5_M   omega*_r = the JS weights; g_r(w) = w (d_r + d_r^2 - 3 d_r w + w^2) / (d_r^2 + w (1 - 2 d_r));
//                   omega_r = g_r(omega*_r) / sum_s g_s(omega*_s)    ("mapped weights, following Henrick et al.",
//                   PAPER.md:165; the map itself is not printed in the paper, reading A20)
//   RECON_WENO5_Z   tau = |beta_0 - beta_2|, alpha_r = d_r (1 + (tau/(beta_r+eps))^q), q = 1,
//                   omega_r = alpha_r / sum alpha
template <class T>
void weno5_weights(int recon, const T dr[3], const T beta[3], const T& eps, T omega[3]) {
  T al[3];
  if (recon == RECON_WENO5_Z) {
    const T tau = o_abs(beta[0] - beta[2]);
    for (int r = 0; r < 3; ++r) al[r] = dr[r] * (T(1) + tau / (beta[r] + eps));
  } else {
    for (int r = 0; r < 3; ++r) al[r] = dr[r] / ((beta[r] + eps) * (beta[r] + eps));
  }
  T s = al[0] + al[1] + al[2];
  for (int r = 0; r < 3; ++r) omega[r] = al[r] / s;
  if (recon == RECON_WENO5_M) {
    T g[3];
    for (int r = 0; r < 3; ++r) {
      const T w = omega[r], d = dr[r];
      g[r] = (w * (d + d * d - T(3) * d * w + w * w)) / (d * d + w * (T(1) - T(2) * d));
    }
    T sg = g[0] + g[1] + g[2];
    for (int r = 0; r < 3; ++r) omega[r] = g[r] / sg;
  }
}

// Stencil, outputs and evaluation form exactly as weno5_js (which it reproduces for recon = RECON_WENO5_JS up to
// the order of two roundings: here omega_r is formed before it multiplies the candidate).
template <class T>
void weno5(int recon, const T& a, const T& b, const T& c, const T& d, const T& e, const T& eps, T* left, T* right) {
  const T c1312 = o_ratio<T>(13, 12), c14 = o_ratio<T>(1, 4);
  T t0 = a - T(2) * b + c, t1 = b - T(2) * c + d, t2 = c - T(2) * d + e;
  T s0 = a - T(4) * b + T(3) * c, s1 = b - d, s2 = T(3) * c - T(4) * d + e;
  T beta[3] = {c1312 * (t0 * t0) + c14 * (s0 * s0), c1312 * (t1 * t1) + c14 * (s1 * s1),
               c1312 * (t2 * t2) + c14 * (s2 * s2)};
  T d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
  {  // left-biased value at i+1/2, ideal weights (1/10, 6/10, 3/10)
    const T dr[3] = {o_ratio<T>(1, 10), o_ratio<T>(6, 10), o_ratio<T>(3, 10)};
    T P0 = (T(5) * d2 - T(2) * d1) / T(6), P1 = (d2 + T(2) * d3) / T(6), P2 = (T(4) * d3 - d4) / T(6);
    T om[3];
    weno5_weights(recon, dr, beta, eps, om);
    *left = c + (om[0] * P0 + om[1] * P1 + om[2] * P2);
  }
  {  // right-biased value at i-1/2 (mirror image), ideal weights (3/10, 6/10, 1/10), same beta
    const T dr[3] = {o_ratio<T>(3, 10), o_ratio<T>(6, 10), o_ratio<T>(1, 10)};
    T P0 = (d1 - T(4) * d2) / T(6), P1 = (T(0) - (T(2) * d2 + d3)) / T(6), P2 = (T(2) * d4 - T(5) * d3) / T(6);
    T om[3];
    weno5_weights(recon, dr, beta, eps, om);
    *right = c + (om[0] * P0 + om[1] * P1 + om[2] * P2);
  }
}

// O4 (S_L,S_R 653-654; S* 664; rho* 668; A5-A8): HLLC at one face with
// normal direction dir, from reconstructed primitives wL, wR.  Writes F[neq] and the face
// velocity u_f.  Returns 0, or 1 if a face state is non-physical (A19).
template <class T>
int hllc_face(const Params<T>& P, int dir, const T* wL, const T* wR, T* F, T* uf) {
  const int N = P.nfluids, D = P.ndim, neq = P.neq();
  const T* w[2] = {wL, wR};
  T rho[2], Gam[2], Pi[2], E[2], c[2], un[2], p[2];
  int bad = 0;
  for (int K = 0; K < 2; ++K) {
    rho[K] = T(0); Gam[K] = T(0); Pi[K] = T(0);
    for (int i = 0; i < N; ++i) rho[K] = rho[K] + w[K][P.i_arho(i)];
    for (int i = 0; i < N; ++i) {
      Gam[K] = Gam[K] + w[K][P.i_alpha(i)] * P.G(i);
      Pi[K] = Pi[K] + w[K][P.i_alpha(i)] * P.P(i);
    }
    T usq = T(0);
    for (int d = 0; d < D; ++d) usq = usq + w[K][P.i_mom(d)] * w[K][P.i_mom(d)];
    p[K] = w[K][P.i_E()];
    un[K] = w[K][P.i_mom(dir)];
    E[K] = Gam[K] * p[K] + Pi[K] + (T(0.5) * rho[K]) * usq;
    T c2 = sound_speed_sq(Gam[K], Pi[K], p[K], rho[K]);
    if (!(rho[K] > T(0)) || !(c2 > T(0))) bad = 1;
    c[K] = o_sqrt(c2);
  }
  const T SL = o_min(un[0] - c[0], un[1] - c[1]);
  const T SR = o_max(un[0] + c[0], un[1] + c[1]);
  const T Sstar = (p[1] - p[0] + rho[0] * un[0] * (SL - un[0]) - rho[1] * un[1] * (SR - un[1])) /
                  (rho[0] * (SL - un[0]) - rho[1] * (SR - un[1]));
  // physical flux of side K, then the star correction S_K (q*_K - q_K).
  // Evaluation form (reading N3): with chi = (S_K - u_K)/(S_K - S*) the jump q*_K - q_K is written
  // out per component with  chi - 1 = (S* - u_K)/(S_K - S*)  formed directly,
  //   alpha_i rho_i, alpha_i, rho u_t :  (chi - 1) q_K
  //   rho u_n                         :  chi rho_K S* - rho_K u_K = rho_K ((chi - 1) S* + (S* - u_K))
  //   E                               :  (chi - 1) E_K + chi (S* - u_K)(rho_K S* + p_K/(S_K - u_K))
  // instead of forming q*_K and subtracting q_K: the same algebra, without the cancellation of two numbers of
  // size |q| (7.8e8 for the energy of water) whose difference is of size |q| * Mach.
  auto side_flux = [&](int K, bool star, const T& SK) {
    const T chi = star ? (SK - un[K]) / (SK - Sstar) : T(1);
    const T chim1 = star ? (Sstar - un[K]) / (SK - Sstar) : T(0);
    for (int v = 0; v < neq; ++v) F[v] = T(0);
    for (int i = 0; i < N; ++i) {
      T qv = w[K][P.i_arho(i)];
      F[P.i_arho(i)] = qv * un[K];
      if (star) F[P.i_arho(i)] = F[P.i_arho(i)] + SK * (chim1 * qv);
      T av = w[K][P.i_alpha(i)];
      F[P.i_alpha(i)] = av * un[K];
      if (star) F[P.i_alpha(i)] = F[P.i_alpha(i)] + SK * (chim1 * av);  // A7
    }
    for (int d = 0; d < D; ++d) {
      T qv = rho[K] * w[K][P.i_mom(d)];
      F[P.i_mom(d)] = qv * un[K] + (d == dir ? p[K] : T(0));
      if (star) {
        T dq = (d == dir) ? rho[K] * (chim1 * Sstar + (Sstar - un[K])) : chim1 * qv;
        F[P.i_mom(d)] = F[P.i_mom(d)] + SK * dq;
      }
    }
    F[P.i_E()] = (E[K] + p[K]) * un[K];
    if (star) {
      T dE = chim1 * E[K] + chi * ((Sstar - un[K]) * (rho[K] * Sstar + p[K] / (SK - un[K])));
      F[P.i_E()] = F[P.i_E()] + SK * dE;
    }
    *uf = star ? un[K] + SK * chim1 : un[K];  // HLLC flux of a unit scalar (A7)
  };
  // first match in the printed order (A8)
  if (SL >= T(0)) side_flux(0, false, SL);
  else if (Sstar >= T(0)) side_flux(0, true, SL);
  else if (SR > T(0)) side_flux(1, true, SR);
  else side_flux(1, false, SR);
  return bad;
}

// O3, textbook form (f = sum_r omega_r f^(r); Jiang-Shu candidates and indicators, A3).  Same inputs and
// outputs as weno5_js.
template <class T>
void weno5_js_textbook(const T& a, const T& b, const T& c, const T& d, const T& e, const T& eps, T* left, T* right) {
  const T c1312 = o_ratio<T>(13, 12), c14 = o_ratio<T>(1, 4);
  T t0 = a - T(2) * b + c, t1 = b - T(2) * c + d, t2 = c - T(2) * d + e;
  T s0 = a - T(4) * b + T(3) * c, s1 = b - d, s2 = T(3) * c - T(4) * d + e;
  T b0 = c1312 * (t0 * t0) + c14 * (s0 * s0);
  T b1 = c1312 * (t1 * t1) + c14 * (s1 * s1);
  T b2 = c1312 * (t2 * t2) + c14 * (s2 * s2);
  {  // left-biased value at i+1/2: candidates of stencils (i-2..i), (i-1..i+1), (i..i+2), ideal weights (1/10, 6/10, 3/10)
    T p0 = (T(2) * a - T(7) * b + T(11) * c) / T(6);
    T p1 = (T(5) * c - b + T(2) * d) / T(6);
    T p2 = (T(2) * c + T(5) * d - e) / T(6);
    T a0 = o_ratio<T>(1, 10) / ((b0 + eps) * (b0 + eps));
    T a1 = o_ratio<T>(6, 10) / ((b1 + eps) * (b1 + eps));
    T a2 = o_ratio<T>(3, 10) / ((b2 + eps) * (b2 + eps));
    T s = a0 + a1 + a2;
    *left = (a0 / s) * p0 + (a1 / s) * p1 + (a2 / s) * p2;
  }
  {  // right-biased value at i-1/2: the mirror image, ideal weights (3/10, 6/10, 1/10), same indicators
    T p0 = (T(5) * b - a + T(2) * c) / T(6);
    T p1 = (T(2) * b + T(5) * c - d) / T(6);
    T p2 = (T(11) * c - T(7) * d + T(2) * e) / T(6);
    T a0 = o_ratio<T>(3, 10) / ((b0 + eps) * (b0 + eps));
    T a1 = o_ratio<T>(6, 10) / ((b1 + eps) * (b1 + eps));
    T a2 = o_ratio<T>(1, 10) / ((b2 + eps) * (b2 + eps));
    T s = a0 + a1 + a2;
    *right = (a0 / s) * p0 + (a1 / s) * p1 + (a2 / s) * p2;
  }
}

// O4, textbook form: the star state q*_K of PAPER.md:668 is formed first (alpha_i carried like a passive density, A7) and
// the flux is F_K + S_K (q*_K - q_K).  Same inputs, outputs, wave speeds and selection as hllc_face.
template <class T>
int hllc_face_textbook(const Params<T>& P, int dir, const T* wL, const T* wR, T* F, T* uf) {
  const int N = P.nfluids, D = P.ndim, neq = P.neq();
  const T* w[2] = {wL, wR};
  T rho[2], Gam[2], Pi[2], E[2], c[2], un[2], p[2];
  int bad = 0;
  for (int K = 0; K < 2; ++K) {
    rho[K] = T(0); Gam[K] = T(0); Pi[K] = T(0);
    for (int i = 0; i < N; ++i) rho[K] = rho[K] + w[K][P.i_arho(i)];
    for (int i = 0; i < N; ++i) {
      Gam[K] = Gam[K] + w[K][P.i_alpha(i)] * P.G(i);
      Pi[K] = Pi[K] + w[K][P.i_alpha(i)] * P.P(i);
    }
    T usq = T(0);
    for (int d = 0; d < D; ++d) usq = usq + w[K][P.i_mom(d)] * w[K][P.i_mom(d)];
    p[K] = w[K][P.i_E()];
    un[K] = w[K][P.i_mom(dir)];
    E[K] = Gam[K] * p[K] + Pi[K] + (T(0.5) * rho[K]) * usq;
    T c2 = sound_speed_sq(Gam[K], Pi[K], p[K], rho[K]);
    if (!(rho[K] > T(0)) || !(c2 > T(0))) bad = 1;
    c[K] = o_sqrt(c2);
  }
  const T SL = o_min(un[0] - c[0], un[1] - c[1]);
  const T SR = o_max(un[0] + c[0], un[1] + c[1]);
  const T Sstar = (p[1] - p[0] + rho[0] * un[0] * (SL - un[0]) - rho[1] * un[1] * (SR - un[1])) /
                  (rho[0] * (SL - un[0]) - rho[1] * (SR - un[1]));
  auto side_flux = [&](int K, bool star, const T& SK) {
    const T chi = star ? (SK - un[K]) / (SK - Sstar) : T(1);
    for (int v = 0; v < neq; ++v) F[v] = T(0);
    for (int i = 0; i < N; ++i) {
      T qv = w[K][P.i_arho(i)];
      F[P.i_arho(i)] = qv * un[K];
      if (star) F[P.i_arho(i)] = F[P.i_arho(i)] + SK * (chi * qv - qv);
      T av = w[K][P.i_alpha(i)];
      F[P.i_alpha(i)] = av * un[K];
      if (star) F[P.i_alpha(i)] = F[P.i_alpha(i)] + SK * (chi * av - av);  // A7
    }
    for (int d = 0; d < D; ++d) {
      T qv = rho[K] * w[K][P.i_mom(d)];
      F[P.i_mom(d)] = qv * un[K] + (d == dir ? p[K] : T(0));
      if (star) {
        T qs = (d == dir) ? chi * rho[K] * Sstar : chi * qv;
        F[P.i_mom(d)] = F[P.i_mom(d)] + SK * (qs - qv);
      }
    }
    F[P.i_E()] = (E[K] + p[K]) * un[K];
    if (star) {
      T Es = chi * (E[K] + (Sstar - un[K]) * (rho[K] * Sstar + p[K] / (SK - un[K])));
      F[P.i_E()] = F[P.i_E()] + SK * (Es - E[K]);
    }
    *uf = star ? un[K] + SK * (chi - T(1)) : un[K];  // HLLC flux of a unit scalar (A7)
  };
  if (SL >= T(0)) side_flux(0, false, SL);  // first match in the printed order (A8)
  else if (Sstar >= T(0)) side_flux(0, true, SL);
  else if (SR > T(0)) side_flux(1, true, SR);
  else side_flux(1, false, SR);
  return bad;
}

// A10: positivity / volume-fraction clamp applied to one cell after each RK stage.
template <class T>
void clamp_cell(const Params<T>& P, T* q) {
  const int N = P.nfluids;
  for (int i = 0; i < N; ++i) q[P.i_arho(i)] = o_max(q[P.i_arho(i)], T(0));
  bool marked = false;
  for (int i = 0; i < N; ++i)
    if (q[P.i_alpha(i)] < P.alpha_floor) { q[P.i_alpha(i)] = P.alpha_floor; marked = true; }
  if (marked) {
    T s = T(0);
    for (int i = 0; i < N; ++i) s = s + q[P.i_alpha(i)];
    for (int i = 0; i < N; ++i) q[P.i_alpha(i)] = q[P.i_alpha(i)] / s;
  }
}

template <class T>
struct Solver {
  Params<T> P;
  explicit Solver(const Params<T>& p) : P(p) { P.derive(); }

  std::size_t idx(int v, int i, int j, int k) const {
    return ((std::size_t(v) * P.n[2] + k) * P.n[1] + j) * P.n[0] + i;
  }

  // mfc_prim_from_cons over the whole grid. Returns the number of cells flagged (A19).
  long prim_from_cons(const T* q, T* w) const {
    const int neq = P.neq();
    const std::size_t nc = P.cells();
    long bad = 0;
#pragma omp parallel for reduction(+ : bad) schedule(static)
    for (long c = 0; c < (long)nc; ++c) {
      T qc[kMaxEq], wc[kMaxEq];
      for (int v = 0; v < neq; ++v) qc[v] = q[std::size_t(v) * nc + c];
      bad += prim_from_cons_cell(P, qc, wc);
      for (int v = 0; v < neq; ++v) w[std::size_t(v) * nc + c] = wc[v];
    }
    return bad;
  }

  // O5: rhs = L(q).  dir_mask selects directions (bit d), default all.
  long rhs(const T* q, T* rhs_out, int dir_mask = 7) const {
    const int neq = P.neq(), N = P.nfluids;
    const std::size_t nc = P.cells();
    for (std::size_t t = 0; t < nc * neq; ++t) rhs_out[t] = T(0);
    long bad = 0;
    for (int dir = 0; dir < P.ndim; ++dir) {
      if (!((dir_mask >> dir) & 1)) continue;
      const int n = P.n[dir];
      const int d1 = (dir + 1) % 3, d2 = (dir + 2) % 3;  // the two transverse index directions
      const long nlines = long(P.n[d1]) * P.n[d2];
#pragma omp parallel for reduction(+ : bad) schedule(static)
      for (long line = 0; line < nlines; ++line) {
        int ijk[3];
        ijk[d1] = int(line % P.n[d1]);
        ijk[d2] = int(line / P.n[d1]);
        // primitives along the line with 3 ghost cells each side: wl[(g+3)*neq + v], g = -3..n+2
        std::vector<T> wl(std::size_t(n + 6) * neq), WL(std::size_t(n + 2) * neq), WR(std::size_t(n + 2) * neq);
        std::vector<T> Ff(std::size_t(n + 1) * neq), uf(n + 1);
        for (int g = -3; g < n + 3; ++g) {
          ijk[dir] = ghost_index(g, n, P.bc_lo[dir], P.bc_hi[dir]);
          T qc[kMaxEq];
          for (int v = 0; v < neq; ++v) qc[v] = q[idx(v, ijk[0], ijk[1], ijk[2])];
          bad += prim_from_cons_cell(P, qc, &wl[std::size_t(g + 3) * neq]);
        }
        // reconstruction in cells i = -1..n: WL[i] -> face i+1/2, WR[i] -> face i-1/2
        for (int i = -1; i <= n; ++i) {
          for (int v = 0; v < neq; ++v) {
            const T* c = &wl[std::size_t(i + 3) * neq + v];
            T l, r;
            if (P.recon == RECON_WENO5_JS && P.form == FORM_TEXTBOOK) {
              weno5_js_textbook(c[-2 * neq], c[-neq], c[0], c[neq], c[2 * neq], P.weno_eps, &l, &r);
            } else if (P.recon == RECON_WENO5_JS) {
              weno5_js(c[-2 * neq], c[-neq], c[0], c[neq], c[2 * neq], P.weno_eps, &l, &r);
            } else if (P.recon == RECON_WENO5_M || P.recon == RECON_WENO5_Z) {
              weno5(P.recon, c[-2 * neq], c[-neq], c[0], c[neq], c[2 * neq], P.weno_eps, &l, &r);
            } else {  // PAPER.md:155-157 piecewise constant
              l = c[0]; r = c[0];
            }
            WL[std::size_t(i + 1) * neq + v] = l;
            WR[std::size_t(i + 1) * neq + v] = r;
          }
        }
        // faces f = i+1/2, i = -1..n-1: left state from cell i, right state from cell i+1
        for (int i = -1; i < n; ++i)
          bad += P.form == FORM_TEXTBOOK
                     ? hllc_face_textbook(P, dir, &WL[std::size_t(i + 1) * neq], &WR[std::size_t(i + 2) * neq],
                                          &Ff[std::size_t(i + 1) * neq], &uf[i + 1])
                     : hllc_face(P, dir, &WL[std::size_t(i + 1) * neq], &WR[std::size_t(i + 2) * neq],
                                 &Ff[std::size_t(i + 1) * neq], &uf[i + 1]);
        // eq.(10): flux difference and the alpha_i div(u) source with the cell-centre alpha_i
        for (int i = 0; i < n; ++i) {
          ijk[dir] = i;
          for (int v = 0; v < neq; ++v) {
            std::size_t t = idx(v, ijk[0], ijk[1], ijk[2]);
            rhs_out[t] = rhs_out[t] + (Ff[std::size_t(i) * neq + v] - Ff[std::size_t(i + 1) * neq + v]) / P.dx[dir];
          }
          for (int f = 0; f < N; ++f) {
            std::size_t t = idx(P.i_alpha(f), ijk[0], ijk[1], ijk[2]);
            rhs_out[t] = rhs_out[t] + q[t] * (uf[i + 1] - uf[i]) / P.dx[dir];
          }
          if (P.model == MODEL_KAPILA && N == 2) {  // K div(u), direction by direction, cell-centre K
            const T* wc = &wl[std::size_t(i + 3) * neq];
            const T K = kapila_K(P, wc[P.i_E()], wc[P.i_alpha(0)], wc[P.i_alpha(1)]);
            std::size_t t1 = idx(P.i_alpha(0), ijk[0], ijk[1], ijk[2]), t2 = idx(P.i_alpha(1), ijk[0], ijk[1], ijk[2]);
            rhs_out[t1] = rhs_out[t1] + K * (uf[i + 1] - uf[i]) / P.dx[dir];
            rhs_out[t2] = rhs_out[t2] - K * (uf[i + 1] - uf[i]) / P.dx[dir];
          }
        }
      }
    }
    if (P.eta > T(0) && dir_mask == 7) add_viscous(q, rhs_out);
    return bad;
  }

  // O8 (eqs.(1),(2); reading A22): viscous part of the momentum and energy equations,
  //   d(rho u_m)/dt += d/dx_d T_md,   dE/dt += d/dx_d (T_md u_m),   T = 2 eta (D - tr(D) I/3),  D = (grad u + grad u^T)/2,
  // i.e. T_md = eta (du_m/dx_d + du_d/dx_m) - (2/3) eta delta_md div u, with one uniform eta.  The paper prints no
  // discretisation; the reading is the second-order central one at face centres (the paper's ref. [7]): at the face
  // between cells i and i+1 along d
  //   du_m/dx_d = (u_m[i+1] - u_m[i])/dx_d,
  //   du_m/dx_e = mean over the two cells of (u_m[.,e+1] - u_m[.,e-1])/(2 dx_e)   (e != d),
  //   u_m(face) = (u_m[i] + u_m[i+1])/2,
  // and the cell gets (flux at i+1/2 - flux at i-1/2)/dx_d.  Ghost velocities by the index map O1 in every direction.
  T vel(const T* q, int m, int i, int j, int k) const {
    int c[3] = {i, j, k};
    for (int d = 0; d < 3; ++d) c[d] = d < P.ndim ? ghost_index(c[d], P.n[d], P.bc_lo[d], P.bc_hi[d]) : 0;
    T rho = T(0);
    for (int f = 0; f < P.nfluids; ++f) rho = rho + q[idx(P.i_arho(f), c[0], c[1], c[2])];
    return q[idx(P.i_mom(m), c[0], c[1], c[2])] / rho;
  }

  // viscous flux through the face between cell (i,j,k) and its neighbour one step up in direction d:
  // Tm[m] = T_md, *G = sum_m T_md u_m(face)
  void viscous_face(const T* q, int d, int i, int j, int k, T* Tm, T* G) const {
    const int D = P.ndim;
    int a[3] = {i, j, k}, b[3] = {i, j, k};
    b[d] += 1;
    T grad[3][3];  // grad[m][e] = du_m/dx_e at the face
    T uf[3];
    for (int m = 0; m < D; ++m) {
      const T ua = vel(q, m, a[0], a[1], a[2]), ub = vel(q, m, b[0], b[1], b[2]);
      uf[m] = (ua + ub) / T(2);
      for (int e = 0; e < D; ++e) {
        if (e == d) {
          grad[m][e] = (ub - ua) / P.dx[d];
        } else {
          int ap[3] = {a[0], a[1], a[2]}, am[3] = {a[0], a[1], a[2]}, bp[3] = {b[0], b[1], b[2]}, bm[3] = {b[0], b[1], b[2]};
          ap[e] += 1; am[e] -= 1; bp[e] += 1; bm[e] -= 1;
          const T ga = (vel(q, m, ap[0], ap[1], ap[2]) - vel(q, m, am[0], am[1], am[2])) / (T(2) * P.dx[e]);
          const T gb = (vel(q, m, bp[0], bp[1], bp[2]) - vel(q, m, bm[0], bm[1], bm[2])) / (T(2) * P.dx[e]);
          grad[m][e] = (ga + gb) / T(2);
        }
      }
    }
    T div = T(0);
    for (int m = 0; m < D; ++m) div = div + grad[m][m];
    *G = T(0);
    for (int m = 0; m < D; ++m) {
      Tm[m] = P.eta * (grad[m][d] + grad[d][m]);
      if (m == d) Tm[m] = Tm[m] - (T(2) * P.eta / T(3)) * div;
      *G = *G + Tm[m] * uf[m];
    }
  }

  void add_viscous(const T* q, T* rhs_out) const {
    const int D = P.ndim;
#pragma omp parallel for schedule(static)
    for (long k = 0; k < P.n[2]; ++k)
      for (int j = 0; j < P.n[1]; ++j)
        for (int i = 0; i < P.n[0]; ++i)
          for (int d = 0; d < D; ++d) {
            int lo[3] = {i, j, (int)k};
            lo[d] -= 1;
            T Tp[3], Tm_[3], Gp, Gm;
            viscous_face(q, d, i, j, (int)k, Tp, &Gp);
            viscous_face(q, d, lo[0], lo[1], lo[2], Tm_, &Gm);
            for (int m = 0; m < D; ++m) {
              std::size_t t = idx(P.i_mom(m), i, j, (int)k);
              rhs_out[t] = rhs_out[t] + (Tp[m] - Tm_[m]) / P.dx[d];
            }
            std::size_t t = idx(P.i_E(), i, j, (int)k);
            rhs_out[t] = rhs_out[t] + (Gp - Gm) / P.dx[d];
          }
  }

  void clamp_all(T* q) const {
    if (!P.clamp) return;
    const int neq = P.neq();
    const std::size_t nc = P.cells();
#pragma omp parallel for schedule(static)
    for (long c = 0; c < (long)nc; ++c) {
      T qc[kMaxEq];
      for (int v = 0; v < neq; ++v) qc[v] = q[std::size_t(v) * nc + c];
      clamp_cell(P, qc);
      for (int v = 0; v < neq; ++v) q[std::size_t(v) * nc + c] = qc[v];
    }
  }

  // O6: one SSP-RK3 step, q updated in place.
  long rk3_step(T* q, const T& dt) const {
    const std::size_t tot = P.cells() * P.neq();
    std::vector<T> q1(tot), L(tot);
    long bad = 0;
    bad += rhs(q, L.data());
#pragma omp parallel for schedule(static)
    for (long t = 0; t < (long)tot; ++t) q1[t] = q[t] + dt * L[t];
    clamp_all(q1.data());
    bad += rhs(q1.data(), L.data());
#pragma omp parallel for schedule(static)
    for (long t = 0; t < (long)tot; ++t) q1[t] = T(0.75) * q[t] + T(0.25) * (q1[t] + dt * L[t]);
    clamp_all(q1.data());
    bad += rhs(q1.data(), L.data());
#pragma omp parallel for schedule(static)
    for (long t = 0; t < (long)tot; ++t) q[t] = o_ratio<T>(1, 3) * q[t] + o_ratio<T>(2, 3) * (q1[t] + dt * L[t]);
    clamp_all(q);
    return bad;
  }

  // O7 / A9: dt = cfl / max_cells sum_d (|u_d| + c)/dx_d
  T cfl_dt(const T* q, const T& cfl) const {
    const int neq = P.neq(), N = P.nfluids;
    const std::size_t nc = P.cells();
    T smax = T(0);
    for (std::size_t c = 0; c < nc; ++c) {
      T qc[kMaxEq], w[kMaxEq];
      for (int v = 0; v < neq; ++v) qc[v] = q[std::size_t(v) * nc + c];
      prim_from_cons_cell(P, qc, w);
      T rho = T(0), Gam = T(0), Pi = T(0);
      for (int i = 0; i < N; ++i) rho = rho + w[P.i_arho(i)];
      for (int i = 0; i < N; ++i) {
        Gam = Gam + w[P.i_alpha(i)] * P.G(i);
        Pi = Pi + w[P.i_alpha(i)] * P.P(i);
      }
      T cs = o_sqrt(sound_speed_sq(Gam, Pi, w[P.i_E()], rho));
      T s = T(0);
      for (int d = 0; d < P.ndim; ++d) s = s + (o_abs(w[P.i_mom(d)]) + cs) / P.dx[d];
      smax = o_max(smax, s);
    }
    return cfl / smax;
  }
};

}  // namespace mfc_oracle
