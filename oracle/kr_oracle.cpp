// kr_oracle.cpp -- CPU ORACLE of the per-cell implicit thermochemistry step.  TEST INFRASTRUCTURE.
//
// What it is: a plain, slow, obviously-correct, single-threaded C++17 restatement of
//   PAPER.md:143-150 (eq. 15, the ODE system), 158-163 (eq. 16, Arrhenius; reading R4),
//   173-187 (eqs. 18-20, analytic Jacobian), 199 (T limits), 212-218 (post-processing stages 1-3: readings
//   R12 / R23; revert on persistent failure: R13), 236-276 (Algorithm 1: Crout LU with implicit-scaled row pivoting; reading R14),
//   423 (7-coefficient thermo polynomials),
// in the order and notation of SURVEY.md 8(c) steps 1-9 (= DESIGN.md "Algorithm").  Dense N x N arrays,
// reaction-index summation order, no blocking, no fusion, no reordering.  `double` throughout; the same
// template instantiated with `long double` is the witness, and with std::complex<double> the
// complex-step evaluator used by pin P6.
//
// Who may use it: tests/, __graft_entry__.smoke(), bench.py's cpu_baseline / --impl reference legs.
// It shares no code with the CUDA path (paper_2504_04941_b200/csrc) and neither includes the other.
//
// Pins (tests/test_oracle_pins.py): P1 linear relaxation closed form, P2 A+A->A2 quadratic root,
// P3 detailed balance against K_c recomputed in numpy, P4 element conservation, P5 LU vs
// numpy.linalg.solve / Cramer, P6 analytic J vs complex-step, P7 H ionisation-balance quadratic
// (eq. 35 with eq. 36 coefficients), P8 K=1 equals u_n + h (I-hJ)^-1 f(u_n),
// P9 adiabatic energy drift O(h^2), P10 long-double witness, P11 post-processing stages 1-3 (exact fractions on a
// five-species network, row totals, minimal disintegration, charged compounds left alone), P12 the retry procedure
// (R24: closed form of A + A -> A2, counter bookkeeping, both-fail revert).
// Parity unpinned: the controller constants of step 8 and the choice of Jacobian
// approximations (dropped dC terms) and the retry parameters of R24 -- the paper does not publish them.
#include "kr_oracle.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstring>
#include <limits>
#include <string>
#include <thread>
#include <vector>

namespace {

constexpr double K_B = 1.380649e-16;        // erg/K
constexpr double M_U = 1.66053906660e-24;   // g
constexpr double P0 = 1.01325e6;            // dyn/cm^2
constexpr double T_REF = 300.0;             // K
constexpr double EXP_CLAMP = 690.0;         // R18

enum : int32_t { F_REV = 1, F_TB = 2, F_CONST = 4, F_AUX = 8 };
enum : int32_t { ST_REJECTED_ONCE = 1, ST_CLAMPED_NEG = 2, ST_FAILED_REVERTED = 8, ST_T_CLAMPED = 16,
                 ST_NO_RESERVOIR = 32, ST_NEEDS_STAGE3 = 64, ST_STAGE3 = 128, ST_RETRIED = 256 };

template <class R> struct real_of { using type = R; };
template <class R> struct real_of<std::complex<R>> { using type = R; };
template <class R> inline R re(const R& x) { return x; }
template <class R> inline R re(const std::complex<R>& x) { return x.real(); }

}  // namespace

struct kr_oracle_network {
  int E = 0, S = 0, R = 0, N = 0, energy = 0;
  std::vector<double> elem_mass;
  std::vector<int32_t> comp;                       // [E*S]
  std::vector<int32_t> ridx, rnu, pidx, pnu;       // [R*3]
  std::vector<double> A, beta, Ea;
  std::vector<int32_t> flags, aux_index;
  std::vector<double> tb_eff;                      // [R*S] (all 1 when not given)
  std::vector<double> q_ext;                       // [R]
  std::vector<double> nasa_lo, nasa_hi, T_mid;
  double T_lo = 0, T_hi = 0;
  int n_aux_needed = 0;
  std::vector<int> reservoir_candidates;           // per row: list encoded as [E][S] flags
  kr_oracle_opts opts;
};

namespace {

kr_oracle_opts default_opts() {
  kr_oracle_opts o;
  o.max_newton = 8; o.fixed_newton = 0; o.h0_mode = 1;
  o.rtol = 1e-8; o.atol_y = 1e-20; o.atol_T = 1e-8; o.neg_tol = 1e-12; o.eta = 0.1; o.y_floor = 1e-12;
  o.shrink = 0.25; o.grow_fast = 8.0; o.grow_mid = 2.0; o.chg_floor = 1e-12;
  o.chg_max = std::numeric_limits<double>::infinity();
  o.it_fast = 3; o.it_mid = 5; o.max_substeps = 4096; o.finalize = 1; o.h_min_rel = 1e-12; o.bail_ratio = 10.0;
  o.retry = 0; o.retry_h0 = 0.01; o.cons_tol = 1e-13;
  return o;
}

// ---------------------------------------------------------------------------------------------
// Step 2: thermo at T (7-coefficient form, reading R7).
//   cp/R = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4
//   h/RT = a1 + a2 T/2 + a3 T^2/3 + a4 T^3/4 + a5 T^4/5 + a6/T
//   s/R  = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7
//   ghat = h/RT - s/R ; uhat = h/RT - 1 ; chat = cp/R - 1
// ---------------------------------------------------------------------------------------------
template <class Real>
void thermo(const kr_oracle_network& n, Real T, Real* ghat, Real* uhat, Real* chat) {
  using std::log;
  const Real T2 = T * T, T3 = T2 * T, T4 = T3 * T;
  const Real lnT = log(T);
  for (int s = 0; s < n.S; ++s) {
    const double* a = (re(T) <= n.T_mid[s]) ? &n.nasa_lo[7 * s] : &n.nasa_hi[7 * s];
    const Real cp = Real(a[0]) + Real(a[1]) * T + Real(a[2]) * T2 + Real(a[3]) * T3 + Real(a[4]) * T4;
    const Real h = Real(a[0]) + Real(a[1]) * T / Real(2) + Real(a[2]) * T2 / Real(3) + Real(a[3]) * T3 / Real(4) +
                   Real(a[4]) * T4 / Real(5) + Real(a[5]) / T;
    const Real sR = Real(a[0]) * lnT + Real(a[1]) * T + Real(a[2]) * T2 / Real(2) + Real(a[3]) * T3 / Real(3) +
                    Real(a[4]) * T4 / Real(4) + Real(a[6]);
    ghat[s] = h - sR;
    uhat[s] = h - Real(1);
    chat[s] = cp - Real(1);
  }
}

template <class Real>
inline Real exp_clamped(Real lnk) {
  using std::exp;
  if (re(lnk) > EXP_CLAMP) return exp(Real(EXP_CLAMP));
  return exp(lnk);
}

// ---------------------------------------------------------------------------------------------
// Step 3: rate constants (eq. 16 with reading R4; R5 detailed balance; R16/R17 unary).
// ---------------------------------------------------------------------------------------------
template <class Real>
void rate_constants(const kr_oracle_network& n, Real T, const double* aux_cell, const Real* ghat, const Real* uhat,
                    Real* kf, Real* kr, Real* dlnkf, Real* dlnkr) {
  using std::log;
  const Real lnT = log(T);
  for (int r = 0; r < n.R; ++r) {
    const int32_t fl = n.flags[r];
    kr[r] = Real(0); dlnkf[r] = Real(0); dlnkr[r] = Real(0);
    if (fl & F_CONST) { kf[r] = Real(n.A[r]); continue; }
    if (fl & F_AUX) { kf[r] = Real(n.A[r] * aux_cell[n.aux_index[r]]); continue; }
    const Real lnkf = Real(std::log(n.A[r])) + Real(n.beta[r]) * (lnT - Real(std::log(T_REF))) - Real(n.Ea[r]) / T;
    kf[r] = exp_clamped(lnkf);
    dlnkf[r] = (Real(n.beta[r]) + Real(n.Ea[r]) / T) / T;
    if (fl & F_REV) {
      Real sum_g = Real(0), sum_u = Real(0);
      int dnu = 0;
      for (int k = 0; k < 3; ++k)
        if (n.ridx[3 * r + k] >= 0) {
          const int s = n.ridx[3 * r + k], nu = n.rnu[3 * r + k];
          sum_g -= Real(nu) * ghat[s]; sum_u -= Real(nu) * uhat[s]; dnu -= nu;
        }
      for (int k = 0; k < 3; ++k)
        if (n.pidx[3 * r + k] >= 0) {
          const int s = n.pidx[3 * r + k], nu = n.pnu[3 * r + k];
          sum_g += Real(nu) * ghat[s]; sum_u += Real(nu) * uhat[s]; dnu += nu;
        }
      const Real lnKc = -sum_g + Real(dnu) * log(Real(P0) / (Real(K_B) * T));
      const Real lnkr = lnkf - lnKc;
      kr[r] = exp_clamped(lnkr);
      dlnkr[r] = dlnkf[r] - sum_u / T;
    }
  }
}

template <class Real>
inline Real ipow(Real x, int e) {
  Real p = Real(1);
  for (int i = 0; i < e; ++i) p *= x;
  return p;
}

// scratch for one cell
template <class Real>
struct Scratch {
  std::vector<Real> ghat, uhat, chat, kf, kr, dlnkf, dlnkr, nd, ydot_sum, dqdn, f, J, M, G, delta, u, un, uin, v;
  std::vector<int32_t> perm;
  explicit Scratch(const kr_oracle_network& n)
      : ghat(n.S), uhat(n.S), chat(n.S), kf(n.R), kr(n.R), dlnkf(n.R), dlnkr(n.R), nd(n.S), ydot_sum(n.S),
        dqdn(n.S), f(n.N), J(size_t(n.N) * n.N), M(size_t(n.N) * n.N), G(n.N), delta(n.N), u(n.N), un(n.N),
        uin(n.N), v(n.N), perm(n.N) {}
};

// ---------------------------------------------------------------------------------------------
// Steps 4 and 5: rates of progress, f = (ydot[, Tdot]) and, when J != nullptr, the analytic Jacobian
// with EXACTLY the terms of SURVEY.md 8(c) step 5 (eq. 19 mass action, eq. 20 thermal
// coupling, dC terms neglected per PAPER.md:185).  u = (y_1..y_S[, T]).
// ---------------------------------------------------------------------------------------------
template <class Real>
void eval_f_J(const kr_oracle_network& n, Real Ncal, const Real* y, Real T, Scratch<Real>& w, Real* f, Real* J) {
  const int S = n.S, N = n.N;
  for (int s = 0; s < S; ++s) { w.nd[s] = Ncal * y[s]; w.ydot_sum[s] = Real(0); }
  if (J) std::fill(J, J + size_t(N) * N, Real(0));
  Real heat_sum = Real(0);                               // sum_r (q_ext/k_B) q_r
  std::vector<Real> heat_dn(J && n.energy ? S : 0, Real(0));   // sum_r (q_ext/k_B) dq_r/dn_m
  Real heat_dT = Real(0);                                // sum_r (q_ext/k_B) dq_r/dT
  std::vector<Real> JsT_sum(J && n.energy ? S : 0, Real(0));   // sum_r dnu_rs dq_r/dT

  for (int r = 0; r < n.R; ++r) {
    const int32_t fl = n.flags[r];
    Real Mtb = Real(1);
    if (fl & F_TB) {
      Mtb = Real(0);
      for (int s = 0; s < S; ++s) Mtb += Real(n.tb_eff[size_t(r) * S + s]) * w.nd[s];
    }
    Real Pf = Real(1), Pr = Real(1);
    for (int k = 0; k < 3; ++k)
      if (n.ridx[3 * r + k] >= 0) Pf *= ipow(w.nd[n.ridx[3 * r + k]], n.rnu[3 * r + k]);
    for (int k = 0; k < 3; ++k)
      if (n.pidx[3 * r + k] >= 0) Pr *= ipow(w.nd[n.pidx[3 * r + k]], n.pnu[3 * r + k]);
    const Real qhat = w.kf[r] * Pf - w.kr[r] * Pr;
    const Real q = Mtb * qhat;
    // dnu_rs q_r accumulated in reaction-index order (R21)
    for (int k = 0; k < 3; ++k)
      if (n.ridx[3 * r + k] >= 0) w.ydot_sum[n.ridx[3 * r + k]] -= Real(n.rnu[3 * r + k]) * q;
    for (int k = 0; k < 3; ++k)
      if (n.pidx[3 * r + k] >= 0) w.ydot_sum[n.pidx[3 * r + k]] += Real(n.pnu[3 * r + k]) * q;
    const Real qk = Real(n.q_ext[r] / K_B);
    heat_sum += qk * q;

    if (!J) continue;
    // dq_r/dn_m for every species m
    std::fill(w.dqdn.begin(), w.dqdn.end(), Real(0));
    for (int k = 0; k < 3; ++k)
      if (n.ridx[3 * r + k] >= 0) {
        const int m = n.ridx[3 * r + k], e = n.rnu[3 * r + k];
        Real others = Real(1);
        for (int k2 = 0; k2 < 3; ++k2)
          if (k2 != k && n.ridx[3 * r + k2] >= 0) others *= ipow(w.nd[n.ridx[3 * r + k2]], n.rnu[3 * r + k2]);
        w.dqdn[m] += Mtb * (w.kf[r] * Real(e) * ipow(w.nd[m], e - 1) * others);
      }
    for (int k = 0; k < 3; ++k)
      if (n.pidx[3 * r + k] >= 0) {
        const int m = n.pidx[3 * r + k], e = n.pnu[3 * r + k];
        Real others = Real(1);
        for (int k2 = 0; k2 < 3; ++k2)
          if (k2 != k && n.pidx[3 * r + k2] >= 0) others *= ipow(w.nd[n.pidx[3 * r + k2]], n.pnu[3 * r + k2]);
        w.dqdn[m] -= Mtb * (w.kr[r] * Real(e) * ipow(w.nd[m], e - 1) * others);
      }
    if (fl & F_TB)
      for (int m = 0; m < S; ++m) w.dqdn[m] += Real(n.tb_eff[size_t(r) * S + m]) * qhat;
    // J_{s,m} += dnu_rs dq_r/dn_m   (the 1/Ncal of ydot and the Ncal of dn/dy cancel)
    for (int side = 0; side < 2; ++side)
      for (int k = 0; k < 3; ++k) {
        const int s = side ? n.pidx[3 * r + k] : n.ridx[3 * r + k];
        if (s < 0) continue;
        const Real dnu = side ? Real(n.pnu[3 * r + k]) : -Real(n.rnu[3 * r + k]);
        for (int m = 0; m < S; ++m) J[size_t(s) * N + m] += dnu * w.dqdn[m];
      }
    if (n.energy) {
      const Real dqdT = Mtb * (w.kf[r] * w.dlnkf[r] * Pf - w.kr[r] * w.dlnkr[r] * Pr);
      for (int k = 0; k < 3; ++k)
        if (n.ridx[3 * r + k] >= 0) JsT_sum[n.ridx[3 * r + k]] -= Real(n.rnu[3 * r + k]) * dqdT;
      for (int k = 0; k < 3; ++k)
        if (n.pidx[3 * r + k] >= 0) JsT_sum[n.pidx[3 * r + k]] += Real(n.pnu[3 * r + k]) * dqdT;
      for (int m = 0; m < S; ++m) heat_dn[m] += qk * w.dqdn[m];
      heat_dT += qk * dqdT;
    }
  }
  for (int s = 0; s < S; ++s) f[s] = w.ydot_sum[s] / Ncal;
  if (!n.energy) return;

  Real C = Real(0), su = Real(0), sc = Real(0);
  for (int s = 0; s < S; ++s) { C += y[s] * w.chat[s]; su += w.uhat[s] * f[s]; sc += w.chat[s] * f[s]; }
  f[S] = (heat_sum / Ncal - T * su) / C;
  if (!J) return;
  for (int s = 0; s < S; ++s) J[size_t(s) * N + S] = JsT_sum[s] / Ncal;
  for (int m = 0; m < S; ++m) {
    Real acc = Real(0);
    for (int s = 0; s < S; ++s) acc += w.uhat[s] * J[size_t(s) * N + m];
    J[size_t(S) * N + m] = (heat_dn[m] - T * acc) / C;
  }
  Real accT = Real(0);
  for (int s = 0; s < S; ++s) accT += w.uhat[s] * J[size_t(s) * N + S];
  J[size_t(S) * N + S] = (heat_dT / Ncal - T * accT - sc) / C;
}

// ---------------------------------------------------------------------------------------------
// Step 7: LU (Algorithm 1, reconstructed per reading R14): Crout's column-by-column
// elimination, implicit row scaling v_i = max_j |M_ij|, pivot i* = argmax_{i>=j} |M_ij| / v_i (ties ->
// smallest i), rows and scales swapped, p_j = i*, sub-column divided by the pivot (unit-diagonal L).
// Returns false on a zero row or |pivot| < 1e-300.
// ---------------------------------------------------------------------------------------------
template <class Real>
bool lu_factor(int n, Real* a, Real* v, int32_t* p) {
  using std::abs;
  for (int i = 0; i < n; ++i) {
    Real big = Real(0);
    for (int j = 0; j < n; ++j) big = std::max(big, Real(abs(a[size_t(i) * n + j])));
    if (!(big > Real(0))) return false;
    v[i] = big;
  }
  for (int j = 0; j < n; ++j) {
    // eliminate with the already-final rows/columns: U part (i < j), then the sub-column (i >= j)
    for (int i = 0; i < j; ++i) {
      Real sum = a[size_t(i) * n + j];
      for (int k = 0; k < i; ++k) sum -= a[size_t(i) * n + k] * a[size_t(k) * n + j];
      a[size_t(i) * n + j] = sum;
    }
    Real best = Real(-1);
    int imax = j;
    for (int i = j; i < n; ++i) {
      Real sum = a[size_t(i) * n + j];
      for (int k = 0; k < j; ++k) sum -= a[size_t(i) * n + k] * a[size_t(k) * n + j];
      a[size_t(i) * n + j] = sum;
      const Real t = Real(abs(sum)) / v[i];
      if (t > best) { best = t; imax = i; }      // strict '>' keeps the smallest i on ties
    }
    if (imax != j) {
      for (int k = 0; k < n; ++k) std::swap(a[size_t(imax) * n + k], a[size_t(j) * n + k]);
      std::swap(v[imax], v[j]);
    }
    p[j] = imax;
    const Real piv = a[size_t(j) * n + j];
    if (!(Real(abs(piv)) >= Real(1e-300))) return false;
    for (int i = j + 1; i < n; ++i) a[size_t(i) * n + j] /= piv;
  }
  return true;
}

template <class Real>
void lu_substitute(int n, const Real* a, const int32_t* p, Real* b) {
  for (int j = 0; j < n; ++j) std::swap(b[j], b[p[j]]);       // apply the recorded row exchanges in order
  for (int i = 0; i < n; ++i) {                                // forward, unit-diagonal L
    Real sum = b[i];
    for (int k = 0; k < i; ++k) sum -= a[size_t(i) * n + k] * b[k];
    b[i] = sum;
  }
  for (int i = n - 1; i >= 0; --i) {                           // back, U
    Real sum = b[i];
    for (int k = i + 1; k < n; ++k) sum -= a[size_t(i) * n + k] * b[k];
    b[i] = sum / a[size_t(i) * n + i];
  }
}

template <class Real>
inline bool finite_all(const Real* x, int n) {
  for (int i = 0; i < n; ++i)
    if (!std::isfinite(x[i])) return false;
  return true;
}

struct Counters { int64_t acc = 0, rej = 0, newton = 0, lu = 0, rate = 0, failed = 0; };

template <class Real> int finalize_state(const kr_oracle_network& n, const Real* uin, Real* un, double* margin);

inline void margin_update(double* m, double a, double b) {
  if (!m) return;
  const double den = std::max(std::fabs(a), std::fabs(b));
  if (den == 0.0 || !std::isfinite(den)) return;
  *m = std::min(*m, std::fabs(a - b) / den);
}

// ---------------------------------------------------------------------------------------------
// Step 6: one backward-Euler sub-step of size h from u_n (reading R1; Newton, R3 convergence test, R11).
// Returns true when the iteration ran to its end (no LU failure, no non-finite iterate, no bail-out);
// e = last e_k, it = first k with e_k <= 1 (K+1 if none).  rates_valid: isothermal cells keep the rate
// constants computed once per cell.
// ---------------------------------------------------------------------------------------------
template <class Real>
bool be_substep(const kr_oracle_network& n, Real Ncal, const double* aux_cell, Real T_iso, Real h, Scratch<Real>& w,
                Real& e_out, int& it_out, Counters& c, double* margin, double* amp = nullptr) {
  using std::abs;
  const int S = n.S, N = n.N, K = n.opts.max_newton;
  const kr_oracle_opts& o = n.opts;
  for (int i = 0; i < N; ++i) w.u[i] = w.un[i];
  Real e_prev = Real(0), e = std::numeric_limits<Real>::infinity();
  int it = K + 1;
  for (int k = 1; k <= K; ++k) {
    const Real T = n.energy ? w.u[S] : T_iso;
    if (n.energy) {                                    // steps 2-3 at u^{k-1}
      thermo(n, T, w.ghat.data(), w.uhat.data(), w.chat.data());
      rate_constants(n, T, aux_cell, w.ghat.data(), w.uhat.data(), w.kf.data(), w.kr.data(), w.dlnkf.data(),
                     w.dlnkr.data());
      c.rate++;
    }
    eval_f_J(n, Ncal, w.u.data(), T, w, w.f.data(), w.J.data());   // steps 4-5
    for (int i = 0; i < N; ++i) w.G[i] = w.u[i] - w.un[i] - h * w.f[i];
    for (int i = 0; i < N; ++i)
      for (int j = 0; j < N; ++j) w.M[size_t(i) * N + j] = (i == j ? Real(1) : Real(0)) - h * w.J[size_t(i) * N + j];
    c.newton++; c.lu++;
    if (!lu_factor(N, w.M.data(), w.v.data(), w.perm.data())) { e_out = e; it_out = it; return false; }
    for (int i = 0; i < N; ++i) w.delta[i] = -w.G[i];
    lu_substitute(N, w.M.data(), w.perm.data(), w.delta.data());
    for (int i = 0; i < N; ++i) w.u[i] = w.u[i] + w.delta[i];
    if (!finite_all(w.u.data(), N)) { e_out = e; it_out = it; return false; }
    if (amp)                                              // diagnostic only: cancellation in the update (see kr_oracle.h)
      for (int i = 0; i < N; ++i)
        *amp = std::max(*amp, double(abs(w.delta[i])) / (double(abs(w.u[i])) + (i < S ? 1e-20 : 0.0)));
    e = Real(0);
    for (int i = 0; i < N; ++i) {
      const Real atol = (i < S) ? Real(o.atol_y) : Real(o.atol_T);
      e = std::max(e, Real(abs(w.delta[i])) / (Real(o.rtol) * Real(abs(w.u[i])) + atol));
    }
    margin_update(margin, double(e), 1.0);
    if (it == K + 1 && e <= Real(1)) it = k;
    if (!o.fixed_newton) {
      if (e <= Real(1)) break;
      if (k >= 2) {
        margin_update(margin, double(e), double(Real(o.bail_ratio) * e_prev));
        if (e > Real(o.bail_ratio) * e_prev) { e_out = e; it_out = it; return false; }   // bail out: diverging
      }
    }
    e_prev = e;
  }
  e_out = e; it_out = it;
  return true;
}

// ---------------------------------------------------------------------------------------------
// Steps 1-9 for one cell.  In/out: T, y (double); returns the status bits.
// ---------------------------------------------------------------------------------------------
// One attempt at the cell with the options `o`; h0_scale multiplies the first sub-step (1 for the first attempt).
template <class Real>
int32_t step_attempt(const kr_oracle_network& n, const kr_oracle_opts& o, double h0_scale, bool count_failure, double rho,
                     double& T_io, double* y_io, double dt, const double* aux_cell, Scratch<Real>& w, Counters& c,
                     double* margin, double* amp = nullptr) {
  using std::abs;
  const int S = n.S, N = n.N;
  int32_t st = 0;
  const Real Ncal = Real(rho) / Real(M_U);

  // step 1
  double Tc = T_io;
  if (Tc < n.T_lo) { Tc = n.T_lo; st |= ST_T_CLAMPED; }
  if (Tc > n.T_hi) { Tc = n.T_hi; st |= ST_T_CLAMPED; }
  for (int s = 0; s < S; ++s) w.uin[s] = Real(y_io[s]);
  if (n.energy) w.uin[S] = Real(Tc);
  for (int i = 0; i < N; ++i) w.un[i] = w.uin[i];
  const Real T_iso = Real(Tc);
  Real t = Real(0), h = Real(dt);
  const Real dtR = Real(dt);

  if (!n.energy) {                                       // isothermal: steps 2-3 once per cell
    thermo(n, T_iso, w.ghat.data(), w.uhat.data(), w.chat.data());
    rate_constants(n, T_iso, aux_cell, w.ghat.data(), w.uhat.data(), w.kf.data(), w.kr.data(), w.dlnkf.data(),
                   w.dlnkr.data());
    c.rate++;
  }
  if (o.h0_mode == 1) {
    if (n.energy) {
      thermo(n, T_iso, w.ghat.data(), w.uhat.data(), w.chat.data());
      rate_constants(n, T_iso, aux_cell, w.ghat.data(), w.uhat.data(), w.kf.data(), w.kr.data(), w.dlnkf.data(),
                     w.dlnkr.data());
      c.rate++;
    }
    eval_f_J<Real>(n, Ncal, w.un.data(), T_iso, w, w.f.data(), nullptr);
    Real big = Real(0);
    for (int s = 0; s < S; ++s) big = std::max(big, Real(abs(w.f[s])) / (Real(abs(w.un[s])) + Real(o.y_floor)));
    if (big > Real(0) && std::isfinite(big)) h = std::min(dtR, Real(o.eta) / big);
  }
  h = h * Real(h0_scale);

  bool failed = false;
  int64_t n_acc = 0, n_rej = 0;
  const Real h_floor = Real(o.h_min_rel) * std::min(h, dtR);      // relative to the first sub-step size
  for (;;) {
    // trim so that t lands on dt exactly (R22)
    const Real rem = dtR - t;
    if (h != rem) margin_update(margin, double(h), double(rem));   // an exact tie is taken identically everywhere
    bool last = false;
    if (h >= rem) { h = rem; last = true; }
    if (h < h_floor || n_acc + n_rej > o.max_substeps) { failed = true; break; }

    Real e; int it;
    const bool ran = be_substep<Real>(n, Ncal, aux_cell, T_iso, h, w, e, it, c, margin, amp);
    // step 8: accept / reject
    bool ok = ran && finite_all(w.u.data(), N) && (e <= Real(1));
    if (ok) {
      Real miny = w.u[0];
      for (int s = 1; s < S; ++s) miny = std::min(miny, w.u[s]);
      if (miny < Real(0)) margin_update(margin, double(-miny), o.neg_tol);
      if (!(miny >= -Real(o.neg_tol))) ok = false;
    }
    if (ok && n.energy) {
      margin_update(margin, double(w.u[S]), n.T_lo);
      margin_update(margin, double(w.u[S]), n.T_hi);
      if (!(w.u[S] >= Real(n.T_lo) && w.u[S] <= Real(n.T_hi))) ok = false;
    }
    if (ok && std::isfinite(o.chg_max)) {
      Real chg = Real(0);
      for (int s = 0; s < S; ++s) chg = std::max(chg, Real(abs(w.u[s] - w.un[s])) / (Real(abs(w.un[s])) + Real(o.chg_floor)));
      if (n.energy) chg = std::max(chg, Real(abs(w.u[S] - w.un[S])) / w.un[S]);
      margin_update(margin, double(chg), o.chg_max);
      if (!(chg <= Real(o.chg_max))) ok = false;
    }
    if (ok) {
      n_acc++;
      for (int i = 0; i < N; ++i) w.un[i] = w.u[i];
      if (last) break;
      t = t + h;
      if (it <= o.it_fast) h = h * Real(o.grow_fast);
      else if (it <= o.it_mid) h = h * Real(o.grow_mid);
    } else {
      n_rej++;
      st |= ST_REJECTED_ONCE;
      h = h * Real(o.shrink);
    }
  }
  c.acc += n_acc; c.rej += n_rej;

  if (failed) {                                          // R13: revert, never abort
    if (count_failure) c.failed++;
    return st | ST_FAILED_REVERTED;                      // T_io, y_io untouched
  }

  if (o.finalize) st |= finalize_state<Real>(n, w.uin.data(), w.un.data(), margin);
  for (int s = 0; s < S; ++s) y_io[s] = double(w.un[s]);
  if (n.energy) T_io = double(w.un[S]);
  return st;
}

// The retry procedure of PAPER.md:218 (reading R24): a cell whose first attempt fails is tried once more "using identical
// initial conditions but with reduced initial time step size and enhanced step size control parameters" -- first
// sub-step x retry_h0, shrink -> shrink^2, grow_fast -> grow_mid, grow_mid -> 1 -- before it is reverted (R13).  The
// work counters add up over both attempts; the status is the second attempt's with RETRIED set.
template <class Real>
int32_t step_cell(const kr_oracle_network& n, double rho, double& T_io, double* y_io, double dt, const double* aux_cell,
                  Scratch<Real>& w, Counters& c, double* margin, double* amp = nullptr) {
  const kr_oracle_opts& o = n.opts;
  int32_t st = step_attempt<Real>(n, o, 1.0, !o.retry, rho, T_io, y_io, dt, aux_cell, w, c, margin, amp);
  if ((st & ST_FAILED_REVERTED) && o.retry) {
    kr_oracle_opts o2 = o;
    o2.shrink = o.shrink * o.shrink; o2.grow_fast = o.grow_mid; o2.grow_mid = 1.0;
    st = step_attempt<Real>(n, o2, o.retry_h0, true, rho, T_io, y_io, dt, aux_cell, w, c, margin, amp) | ST_RETRIED;
  }
  return st;
}

// Step 9: post-processing of the final state (readings R12 / R23 of DESIGN.md).
//   Stage 1: negatives -> 0.
//   Stage 2: "Abundances of elements are calculated for the initial and final states of thermochemical
//     evolution.  In the final state, the abundances in the single-element species are adjusted to compensate the
//     differences.  This step corrects the violation in element abundances brought by step 1."  For every conservation
//     row nu:  D_nu = sum_s N_{nu,s} (y_in,s - y_s)  with y already clamped (the paper's initial-minus-final totals),
//     C_nu = sum_s N_{nu,s} min(y_s, 0) before clamping (the part of D_nu that stage 1 brought), and
//     tot_nu = sum_s |N_{nu,s}| |y_in,s|.  The row is compensated by D_nu when |D_nu| > cons_tol tot_nu (a violation
//     above rounding level: the literal text), else by C_nu (only what stage 1 brought: the solver's own drift below
//     cons_tol is rounding noise and is not pushed into a possibly trace reservoir).  The compensation goes to the row's
//     reservoir: the single-row species with the largest abundance (ties -> smallest index); no such species -> bit.
//   Stage 3 (reading R23): "if step 2 causes negative abundances in some single-element species, the
//     most abundant compound species is disintegrated into elements just sufficiently to correct this".  For every
//     element row whose reservoir went negative, in row order: need = -y_res N_{nu,res} atoms; the neutral compound
//     (>= 2 non-zero rows, no entry on a signed row) with the largest abundance that contains the element gives up
//     z = min(y_c, need / N_{nu,c}); its atoms of every row go to that row's reservoir; repeated with the next most
//     abundant compound until the need is met (the reservoir then ends at exactly 0) or no compound is left.
//   NEEDS_STAGE3 is evaluated at the very end: set iff some row's reservoir is still negative (a reservoir that a LATER
//   row's disintegration refilled does not keep the flag).  Every row total is unchanged by stage 3 by construction.
// Returns the status bits it sets.  uin / un have S entries (abundances only); uin == nullptr means "the state itself"
// (D_nu = C_nu: the entry point kr_oracle_finalize with no initial state).
template <class Real>
int finalize_state(const kr_oracle_network& n, const Real* uin, Real* un, double* margin) {
  using std::abs;
  const int E = n.E, S = n.S;
  int st = 0;
  std::vector<Real> C(E, Real(0)), D(E, Real(0)), tot(E, Real(0));
  std::vector<int> res_of(E, -1);
  for (int s = 0; s < S; ++s)
    if (un[s] < Real(0)) {
      for (int nu = 0; nu < E; ++nu) C[nu] += Real(n.comp[size_t(nu) * S + s]) * un[s];
      un[s] = Real(0); st |= ST_CLAMPED_NEG;
    }
  for (int nu = 0; nu < E; ++nu) {
    if (!uin) { D[nu] = C[nu]; continue; }
    for (int s = 0; s < S; ++s) {
      D[nu] += Real(n.comp[size_t(nu) * S + s]) * (uin[s] - un[s]);
      tot[nu] += Real(abs(n.comp[size_t(nu) * S + s])) * Real(abs(uin[s]));
    }
  }
  auto reservoir = [&](int nu, int* second_out) {
    int res = -1, second = -1;
    for (int s = 0; s < S; ++s) {
      if (!n.reservoir_candidates[size_t(nu) * S + s]) continue;
      if (res < 0 || un[s] > un[res]) { second = res; res = s; }
      else if (second < 0 || un[s] > un[second]) second = s;
    }
    if (second_out) *second_out = second;
    return res;
  };
  for (int nu = 0; nu < E; ++nu) {
    Real delta = C[nu];
    if (uin) {
      const Real thr = Real(n.opts.cons_tol) * tot[nu];
      // the drift is rounding noise that no two implementations share: a cell whose drift is within a decade of the
      // threshold is not comparable
      if (margin && Real(abs(D[nu])) > Real(0.1) * thr && Real(abs(D[nu])) < Real(10) * thr) *margin = 0.0;
      if (Real(abs(D[nu])) > thr) delta = D[nu];
    }
    if (delta == Real(0)) continue;
    int second = -1;
    const int res = reservoir(nu, &second);
    if (res < 0) { st |= ST_NO_RESERVOIR; continue; }
    if (second >= 0) margin_update(margin, double(un[res]), double(un[second]));
    res_of[nu] = res;
    un[res] = un[res] + delta / Real(n.comp[size_t(nu) * S + res]);
  }
  // stage 3
  std::vector<char> signed_row(E, 0), compound(S, 0);
  for (int nu = 0; nu < E; ++nu)
    for (int s = 0; s < S; ++s)
      if (n.comp[size_t(nu) * S + s] < 0) signed_row[nu] = 1;
  for (int s = 0; s < S; ++s) {
    int rows = 0;
    bool neutral = true;
    for (int nu = 0; nu < E; ++nu)
      if (n.comp[size_t(nu) * S + s] != 0) { rows++; if (signed_row[nu]) neutral = false; }
    compound[s] = (rows >= 2 && neutral) ? 1 : 0;
  }
  for (int nu = 0; nu < E; ++nu) {
    const int res = res_of[nu];
    if (res < 0 || !(un[res] < Real(0))) continue;
    const Real nres = Real(n.comp[size_t(nu) * S + res]);
    if (signed_row[nu] || !(nres > Real(0))) continue;
    Real need = -un[res] * nres;
    for (int iter = 0; iter < S && need > Real(0); ++iter) {
      int c = -1;
      for (int s = 0; s < S; ++s) {
        if (!compound[s] || n.comp[size_t(nu) * S + s] <= 0 || !(un[s] > Real(0))) continue;
        bool placeable = true;                     // every other row of the compound needs a reservoir for its atoms
        for (int mu = 0; mu < E && placeable; ++mu)
          if (mu != nu && n.comp[size_t(mu) * S + s] != 0 && res_of[mu] < 0 && reservoir(mu, nullptr) < 0) placeable = false;
        if (!placeable) continue;
        if (c < 0 || un[s] > un[c]) c = s;
      }
      if (c < 0) break;
      const Real nc = Real(n.comp[size_t(nu) * S + c]);
      Real z = need / nc;
      const bool all = !(z < un[c]);
      if (all) z = un[c];
      un[c] = all ? Real(0) : un[c] - z;
      for (int mu = 0; mu < E; ++mu) {
        const int nm = n.comp[size_t(mu) * S + c];
        if (nm == 0 || mu == nu) continue;
        if (res_of[mu] < 0) res_of[mu] = reservoir(mu, nullptr);
        un[res_of[mu]] = un[res_of[mu]] + Real(nm) * z / Real(n.comp[size_t(mu) * S + res_of[mu]]);
      }
      un[res] = un[res] + nc * z / nres;
      need = all ? need - nc * z : Real(0);
      st |= ST_STAGE3;
    }
    if (!(need > Real(0))) un[res] = Real(0);      // "just sufficiently": the reservoir ends at exactly zero
  }
  for (int nu = 0; nu < E; ++nu)
    if (res_of[nu] >= 0 && un[res_of[nu]] < Real(0)) st |= ST_NEEDS_STAGE3;
  return st;
}

template <class Real>
void run_range(const kr_oracle_network* n, int64_t lo, int64_t hi, int64_t n_cells, const double* rho, double* T,
               double* y, double dt, const double* aux, int32_t n_aux, int32_t* status, Counters* cnt, double* margins,
               double* amps) {
  Scratch<Real> w(*n);
  std::vector<double> aux_cell(std::max(1, n_aux));
  for (int64_t c = lo; c < hi; ++c) {
    for (int a = 0; a < n_aux; ++a) aux_cell[a] = aux[size_t(a) * n_cells + c];
    double m = std::numeric_limits<double>::infinity(), am = 0.0;
    double Tc = T[c];
    const int32_t st = step_cell<Real>(*n, rho[c], Tc, y + size_t(c) * n->S, dt, aux_cell.data(), w, *cnt,
                                       margins ? &m : nullptr, amps ? &am : nullptr);
    if (amps) amps[c] = am;
    if (n->energy && !(st & ST_FAILED_REVERTED)) T[c] = Tc;
    if (status) status[c] = st;
    if (margins) margins[c] = m;
  }
}

template <class Real>
int run_step(kr_oracle_network* n, int64_t n_cells, const double* rho, double* T, double* y, double dt, const double* aux,
             int32_t n_aux, int32_t* status, kr_oracle_stats* stats, double* margins, int32_t n_threads,
             double* amps = nullptr) {
  if (!n || n_cells < 0 || (n_cells > 0 && (!rho || !T || !y)) || !(dt > 0)) return -1;
  if (n->n_aux_needed > n_aux || (n_aux > 0 && !aux)) return -1;
  n_threads = std::max(1, n_threads);
  std::vector<Counters> cnt(n_threads);
  if (n_threads == 1 || n_cells < 2 * n_threads) {
    run_range<Real>(n, 0, n_cells, n_cells, rho, T, y, dt, aux, n_aux, status, &cnt[0], margins, amps);
  } else {
    std::vector<std::thread> th;
    for (int t = 0; t < n_threads; ++t) {
      const int64_t lo = n_cells * t / n_threads, hi = n_cells * (t + 1) / n_threads;
      th.emplace_back(run_range<Real>, n, lo, hi, n_cells, rho, T, y, dt, aux, n_aux, status, &cnt[t], margins, amps);
    }
    for (auto& x : th) x.join();
  }
  if (stats) {
    std::memset(stats, 0, sizeof(*stats));
    for (auto& c : cnt) {
      stats->n_substeps += c.acc; stats->n_rejected += c.rej; stats->n_newton += c.newton; stats->n_lu += c.lu;
      stats->n_rate_evals += c.rate; stats->n_failed += c.failed;
    }
  }
  return 0;
}

}  // namespace

extern "C" {

int kr_oracle_network_create(const kr_oracle_desc* d, kr_oracle_network** out) {
  if (!d || !out) return -1;
  const int E = d->n_elem, S = d->n_species, R = d->n_reac;
  if (E <= 0 || S <= 0 || R < 0) return -1;
  auto* n = new kr_oracle_network;
  n->E = E; n->S = S; n->R = R; n->energy = d->energy_equation ? 1 : 0; n->N = S + n->energy;
  n->elem_mass.assign(d->elem_mass, d->elem_mass + E);
  n->comp.assign(d->composition, d->composition + size_t(E) * S);
  n->ridx.assign(d->reac_idx, d->reac_idx + 3 * size_t(R));
  n->rnu.assign(d->reac_nu, d->reac_nu + 3 * size_t(R));
  n->pidx.assign(d->prod_idx, d->prod_idx + 3 * size_t(R));
  n->pnu.assign(d->prod_nu, d->prod_nu + 3 * size_t(R));
  n->A.assign(d->A, d->A + R); n->beta.assign(d->beta, d->beta + R); n->Ea.assign(d->Ea_over_k, d->Ea_over_k + R);
  n->flags.assign(d->flags, d->flags + R);
  n->aux_index.assign(R, -1);
  if (d->aux_index) n->aux_index.assign(d->aux_index, d->aux_index + R);
  n->tb_eff.assign(size_t(R) * S, 1.0);
  if (d->tb_eff) n->tb_eff.assign(d->tb_eff, d->tb_eff + size_t(R) * S);
  n->q_ext.assign(R, 0.0);
  if (d->q_ext) n->q_ext.assign(d->q_ext, d->q_ext + R);
  n->nasa_lo.assign(d->nasa_lo, d->nasa_lo + 7 * size_t(S));
  n->nasa_hi.assign(d->nasa_hi, d->nasa_hi + 7 * size_t(S));
  n->T_mid.assign(d->T_mid, d->T_mid + S);
  n->T_lo = d->T_lo; n->T_hi = d->T_hi;
  n->opts = default_opts();
  // validation: indices, order <= 3 per side (R20), element conservation N . dnu_r = 0
  for (int r = 0; r < R; ++r) {
    int order_r = 0, order_p = 0;
    std::vector<long> tot(E, 0);
    for (int k = 0; k < 3; ++k) {
      const int a = n->ridx[3 * r + k], b = n->pidx[3 * r + k];
      if (a >= S || b >= S) { delete n; return -2; }
      if (a >= 0) { if (n->rnu[3 * r + k] <= 0) { delete n; return -2; } order_r += n->rnu[3 * r + k];
        for (int e = 0; e < E; ++e) tot[e] -= long(n->comp[size_t(e) * S + a]) * n->rnu[3 * r + k]; }
      if (b >= 0) { if (n->pnu[3 * r + k] <= 0) { delete n; return -2; } order_p += n->pnu[3 * r + k];
        for (int e = 0; e < E; ++e) tot[e] += long(n->comp[size_t(e) * S + b]) * n->pnu[3 * r + k]; }
    }
    if (order_r < 1 || order_r > 3 || order_p > 3) { delete n; return -2; }
    for (int e = 0; e < E; ++e) if (tot[e] != 0) { delete n; return -3; }
    if (n->flags[r] & F_AUX) {
      if (n->aux_index[r] < 0) { delete n; return -2; }
      n->n_aux_needed = std::max(n->n_aux_needed, n->aux_index[r] + 1);
    }
    if ((n->flags[r] & (F_CONST | F_AUX)) && (n->flags[r] & (F_REV | F_TB))) { delete n; return -2; }
    if (!(n->flags[r] & (F_CONST | F_AUX)) && !(n->A[r] > 0)) { delete n; return -2; }
  }
  // reservoir candidates of row nu: species whose composition has only row nu non-zero (step 9)
  n->reservoir_candidates.assign(size_t(E) * S, 0);
  for (int nu = 0; nu < E; ++nu)
    for (int s = 0; s < S; ++s) {
      bool only = n->comp[size_t(nu) * S + s] != 0;
      for (int mu = 0; mu < E && only; ++mu)
        if (mu != nu && n->comp[size_t(mu) * S + s] != 0) only = false;
      n->reservoir_candidates[size_t(nu) * S + s] = only ? 1 : 0;
    }
  *out = n;
  return 0;
}

void kr_oracle_network_destroy(kr_oracle_network* n) { delete n; }

int kr_oracle_set_options(kr_oracle_network* n, const kr_oracle_opts* o) {
  if (!n || !o) return -1;
  if (o->max_newton < 1 || !(o->rtol > 0) || !(o->shrink > 0 && o->shrink < 1) || o->max_substeps < 1) return -1;
  n->opts = *o;
  return 0;
}

int kr_oracle_thermochem_step_ex(kr_oracle_network* n, int64_t n_cells, const double* rho, double* T, double* y, double dt,
                                 const double* aux, int32_t n_aux, int32_t* status, kr_oracle_stats* stats,
                                 double* margins, int32_t n_threads) {
  return run_step<double>(n, n_cells, rho, T, y, dt, aux, n_aux, status, stats, margins, n_threads);
}

int kr_oracle_thermochem_step_diag(kr_oracle_network* n, int64_t n_cells, const double* rho, double* T, double* y, double dt,
                                   const double* aux, int32_t n_aux, int32_t* status, kr_oracle_stats* stats,
                                   double* margins, double* amps, int32_t n_threads) {
  return run_step<double>(n, n_cells, rho, T, y, dt, aux, n_aux, status, stats, margins, n_threads, amps);
}

int kr_oracle_witness_step_ex(kr_oracle_network* n, int64_t n_cells, const double* rho, double* T, double* y, double dt,
                              const double* aux, int32_t n_aux, int32_t* status, kr_oracle_stats* stats,
                              int32_t n_threads) {
  return run_step<long double>(n, n_cells, rho, T, y, dt, aux, n_aux, status, stats, nullptr, n_threads);
}

int kr_oracle_rate_constants(kr_oracle_network* n, double T, const double* aux_cell, double* kf, double* kr) {
  if (!n) return -1;
  Scratch<double> w(*n);
  thermo<double>(*n, T, w.ghat.data(), w.uhat.data(), w.chat.data());
  rate_constants<double>(*n, T, aux_cell, w.ghat.data(), w.uhat.data(), kf, kr, w.dlnkf.data(), w.dlnkr.data());
  return 0;
}

int kr_oracle_eval_rhs(kr_oracle_network* n, double rho, double T, const double* y, const double* aux_cell, double* f) {
  if (!n) return -1;
  Scratch<double> w(*n);
  thermo<double>(*n, T, w.ghat.data(), w.uhat.data(), w.chat.data());
  rate_constants<double>(*n, T, aux_cell, w.ghat.data(), w.uhat.data(), w.kf.data(), w.kr.data(), w.dlnkf.data(),
                         w.dlnkr.data());
  eval_f_J<double>(*n, rho / M_U, y, T, w, f, nullptr);
  return 0;
}

int kr_oracle_eval_rhs_complex(kr_oracle_network* n, double rho, double T_re, double T_im, const double* y_re,
                               const double* y_im, const double* aux_cell, double* f_re, double* f_im) {
  if (!n) return -1;
  using C = std::complex<double>;
  Scratch<C> w(*n);
  const C T(T_re, T_im);
  std::vector<C> y(n->S), f(n->N);
  for (int s = 0; s < n->S; ++s) y[s] = C(y_re[s], y_im[s]);
  thermo<C>(*n, T, w.ghat.data(), w.uhat.data(), w.chat.data());
  rate_constants<C>(*n, T, aux_cell, w.ghat.data(), w.uhat.data(), w.kf.data(), w.kr.data(), w.dlnkf.data(),
                    w.dlnkr.data());
  eval_f_J<C>(*n, C(rho / M_U), y.data(), T, w, f.data(), nullptr);
  for (int i = 0; i < n->N; ++i) { f_re[i] = f[i].real(); f_im[i] = f[i].imag(); }
  return 0;
}

int kr_oracle_eval_jacobian(kr_oracle_network* n, double rho, double T, const double* y, const double* aux_cell, double* J) {
  if (!n) return -1;
  Scratch<double> w(*n);
  thermo<double>(*n, T, w.ghat.data(), w.uhat.data(), w.chat.data());
  rate_constants<double>(*n, T, aux_cell, w.ghat.data(), w.uhat.data(), w.kf.data(), w.kr.data(), w.dlnkf.data(),
                         w.dlnkr.data());
  eval_f_J<double>(*n, rho / M_U, y, T, w, w.f.data(), J);
  return 0;
}

int kr_oracle_lu_solve(int32_t nn, double* M, const double* b, double* x, int32_t* perm) {
  if (nn <= 0 || !M || !b || !x || !perm) return -2;
  std::vector<double> v(nn);
  if (!lu_factor<double>(nn, M, v.data(), perm)) return -1;
  for (int i = 0; i < nn; ++i) x[i] = b[i];
  lu_substitute<double>(nn, M, perm, x);
  return 0;
}

int kr_oracle_finalize(kr_oracle_network* n, const double* y_in, double* y, int32_t* status) {
  if (!n || !y) return -1;
  const int st = finalize_state<double>(*n, y_in, y, nullptr);
  if (status) *status = st;
  return 0;
}

int kr_oracle_be_substep(kr_oracle_network* n, double rho, double T, const double* y, const double* aux_cell, double h,
                         double* u_out, double* e_out, int32_t* it_out) {
  if (!n) return -1;
  Scratch<double> w(*n);
  Counters c;
  for (int s = 0; s < n->S; ++s) w.un[s] = y[s];
  if (n->energy) w.un[n->S] = T;
  if (!n->energy) {
    thermo<double>(*n, T, w.ghat.data(), w.uhat.data(), w.chat.data());
    rate_constants<double>(*n, T, aux_cell, w.ghat.data(), w.uhat.data(), w.kf.data(), w.kr.data(), w.dlnkf.data(),
                           w.dlnkr.data());
  }
  double e; int it;
  const bool ran = be_substep<double>(*n, rho / M_U, aux_cell, T, h, w, e, it, c, nullptr);
  for (int i = 0; i < n->N; ++i) u_out[i] = w.u[i];
  if (e_out) *e_out = e;
  if (it_out) *it_out = it;
  return ran ? 0 : 1;
}

}  // extern "C"
