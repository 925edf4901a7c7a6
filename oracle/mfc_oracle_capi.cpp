// ORACLE — TEST INFRASTRUCTURE ONLY (see mfc_oracle.hpp).
// C entry points over host pointers for the fp64 oracle, a long-double adjudicator
// and an operation-counting instantiation.  Built by oracle/build.py into
// oracle/libmfc_oracle.so; loaded with ctypes by oracle/oracle.py.
#include "mfc_oracle.hpp"

#include <cstring>
#ifdef _OPENMP
#include <omp.h>
#endif

using namespace mfc_oracle;

extern "C" {

typedef struct {
  int ndim;
  int n[3];
  double dx[3];
  int nfluids;
  double gamma[kMaxFluids];
  double pi_inf[kMaxFluids];
  int bc_lo[3];
  int bc_hi[3];
  double weno_eps;
  double alpha_floor;
  int clamp;
  int recon;
  int model;
  double eta;
  int form;  /* FORM_DIFFERENCE (0) or FORM_TEXTBOOK (1) */
} oracle_params;

}  // extern "C"

namespace {

template <class T>
Params<T> convert(const oracle_params* p) {
  Params<T> P;
  P.ndim = p->ndim;
  P.nfluids = p->nfluids;
  for (int d = 0; d < 3; ++d) {
    P.n[d] = p->n[d];
    P.dx[d] = T(p->dx[d]);
    P.bc_lo[d] = p->bc_lo[d];
    P.bc_hi[d] = p->bc_hi[d];
  }
  for (int i = 0; i < kMaxFluids; ++i) {
    P.gamma[i] = T(p->gamma[i]);
    P.pi_inf[i] = T(p->pi_inf[i]);
  }
  P.weno_eps = T(p->weno_eps);
  P.alpha_floor = T(p->alpha_floor);
  P.clamp = p->clamp;
  P.recon = p->recon;
  P.model = p->model;
  P.eta = T(p->eta);
  P.form = p->form;
  P.derive();
  return P;
}

// --- operation-counting scalar: every arithmetic operation of the plain definition is tallied ---
struct Counts { long long add = 0, mul = 0, div = 0, sqrt = 0, cmp = 0; };
Counts g_counts;

struct CD {
  double v;
  CD() : v(0) {}
  CD(double x) : v(x) {}
  CD(int x) : v(x) {}
};
inline CD operator+(const CD& a, const CD& b) { ++g_counts.add; return CD(a.v + b.v); }
inline CD operator-(const CD& a, const CD& b) { ++g_counts.add; return CD(a.v - b.v); }
inline CD operator*(const CD& a, const CD& b) { ++g_counts.mul; return CD(a.v * b.v); }
inline CD operator/(const CD& a, const CD& b) { ++g_counts.div; return CD(a.v / b.v); }
inline bool operator<(const CD& a, const CD& b) { ++g_counts.cmp; return a.v < b.v; }
inline bool operator>(const CD& a, const CD& b) { ++g_counts.cmp; return a.v > b.v; }
inline bool operator>=(const CD& a, const CD& b) { ++g_counts.cmp; return a.v >= b.v; }
inline CD sqrt(const CD& a) { ++g_counts.sqrt; return CD(std::sqrt(a.v)); }

}  // namespace

namespace mfc_oracle {
// constants of the scheme are not operations of the method: not tallied
template <> inline CD o_ratio<CD>(int a, int b) { return CD(double(a) / double(b)); }
}  // namespace mfc_oracle

extern "C" {

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

int oracle_num_eqns(const oracle_params* p) { return 2 * p->nfluids + p->ndim + 1; }

int oracle_ghost_index(int g, int n, int bc_lo, int bc_hi) { return ghost_index(g, n, bc_lo, bc_hi); }

long oracle_prim_from_cons(const oracle_params* p, const double* q, double* w) {
  return Solver<double>(convert<double>(p)).prim_from_cons(q, w);
}

long oracle_rhs(const oracle_params* p, const double* q, double* rhs, int dir_mask) {
  return Solver<double>(convert<double>(p)).rhs(q, rhs, dir_mask);
}

long oracle_rk3_step(const oracle_params* p, double* q, double dt) {
  return Solver<double>(convert<double>(p)).rk3_step(q, dt);
}

double oracle_cfl_dt(const oracle_params* p, const double* q, double cfl) {
  return Solver<double>(convert<double>(p)).cfl_dt(q, cfl);
}

void oracle_weno5_js(const double* s, double eps, double* left, double* right) {
  weno5_js<double>(s[0], s[1], s[2], s[3], s[4], eps, left, right);
}

// the same text in 80-bit arithmetic, result rounded to double (pins the rounding error of the fp64 form, N2)
void oracle_weno5_js_ld(const double* s, double eps, double* left, double* right) {
  long double l, r;
  weno5_js<long double>(s[0], s[1], s[2], s[3], s[4], (long double)eps, &l, &r);
  *left = double(l);
  *right = double(r);
}

// weights variant `recon` (RECON_WENO5_JS / _M / _Z) of the general routine, fp64 and 80-bit
void oracle_weno5(int recon, const double* s, double eps, double* left, double* right) {
  weno5<double>(recon, s[0], s[1], s[2], s[3], s[4], eps, left, right);
}

void oracle_weno5_ld(int recon, const double* s, double eps, double* left, double* right) {
  long double l, r;
  weno5<long double>(recon, s[0], s[1], s[2], s[3], s[4], (long double)eps, &l, &r);
  *left = double(l);
  *right = double(r);
}

// the weights step alone: omega[3] from ideal weights dr[3] and smoothness indicators beta[3]
void oracle_weno5_weights(int recon, const double* dr, const double* beta, double eps, double* omega) {
  weno5_weights<double>(recon, dr, beta, eps, omega);
}

double oracle_kapila_K(const oracle_params* p, double pres, double alpha1, double alpha2) {
  return kapila_K<double>(convert<double>(p), pres, alpha1, alpha2);
}

// p->form selects the evaluation form, as Solver::rhs does: FORM_DIFFERENCE -> hllc_face, FORM_TEXTBOOK -> hllc_face_textbook
int oracle_hllc_face(const oracle_params* p, int dir, const double* wL, const double* wR, double* F, double* uf) {
  if (p->form == FORM_TEXTBOOK) return hllc_face_textbook<double>(convert<double>(p), dir, wL, wR, F, uf);
  return hllc_face<double>(convert<double>(p), dir, wL, wR, F, uf);
}

// O3 typed as PAPER.md:163 prints it (weno5_js_textbook), fp64 and 80-bit
void oracle_weno5_js_textbook(const double* s, double eps, double* left, double* right) {
  weno5_js_textbook<double>(s[0], s[1], s[2], s[3], s[4], eps, left, right);
}

void oracle_weno5_js_textbook_ld(const double* s, double eps, double* left, double* right) {
  long double l, r;
  weno5_js_textbook<long double>(s[0], s[1], s[2], s[3], s[4], (long double)eps, &l, &r);
  *left = double(l);
  *right = double(r);
}

void oracle_clamp_cell(const oracle_params* p, double* q) { clamp_cell<double>(convert<double>(p), q); }

// long-double adjudicator: same text evaluated in x87 80-bit; inputs/outputs converted at the edges.
long oracle_rhs_ld(const oracle_params* p, const double* q, double* rhs, int dir_mask) {
  Params<long double> P = convert<long double>(p);
  const std::size_t tot = P.cells() * P.neq();
  std::vector<long double> ql(tot), rl(tot);
  for (std::size_t t = 0; t < tot; ++t) ql[t] = q[t];
  long bad = Solver<long double>(P).rhs(ql.data(), rl.data(), dir_mask);
  for (std::size_t t = 0; t < tot; ++t) rhs[t] = double(rl[t]);
  return bad;
}

long oracle_rk3_steps_ld(const oracle_params* p, double* q, double dt, int nsteps) {
  Params<long double> P = convert<long double>(p);
  const std::size_t tot = P.cells() * P.neq();
  std::vector<long double> ql(tot);
  for (std::size_t t = 0; t < tot; ++t) ql[t] = q[t];
  long bad = 0;
  Solver<long double> S(P);
  for (int s = 0; s < nsteps; ++s) bad += S.rk3_step(ql.data(), (long double)dt);
  for (std::size_t t = 0; t < tot; ++t) q[t] = double(ql[t]);
  return bad;
}

// counts[0..4] = add/sub, mul, div, sqrt, compare for ONE rhs evaluation of the plain definition
// (single thread; used to state the algorithmic flop count in DESIGN.md / bench.py).
void oracle_count_rhs(const oracle_params* p, const double* q, long long* counts) {
  Params<CD> P = convert<CD>(p);
  const std::size_t tot = P.cells() * P.neq();
  std::vector<CD> ql(tot), rl(tot);
  for (std::size_t t = 0; t < tot; ++t) ql[t] = CD(q[t]);
#ifdef _OPENMP
  int nt = omp_get_max_threads();
  omp_set_num_threads(1);
#endif
  g_counts = Counts();
  Solver<CD>(P).rhs(ql.data(), rl.data(), 7);
  Counts c = g_counts;
#ifdef _OPENMP
  omp_set_num_threads(nt);
#endif
  counts[0] = c.add; counts[1] = c.mul; counts[2] = c.div; counts[3] = c.sqrt; counts[4] = c.cmp;
}

}  // extern "C"
