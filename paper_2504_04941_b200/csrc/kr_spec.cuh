// kr_spec.cuh -- network-SPECIALISED thread-per-cell solve kernel (small systems, N <= 12).
//
// This file is compiled at kr_network_create time (NVRTC, sm_100a) against a generated `struct KrNet` that
// holds the network as constexpr tables (reaction records, Arrhenius and thermo coefficients, composition).
// Every loop over species / reactions / matrix entries is unrolled at compile time (kr_static_for), so all
// per-cell vectors are statically indexed and live in REGISTERS; only the N x N matrix and u_n live in
// shared memory as [entry][lane] (conflict-free 64-bit accesses).  Same algorithm as DESIGN.md steps 1-9
// (eq. 15, 158-171 eqs. 16-17, 173-187 eqs. 18-20, 199, 212-218, 236-276 Algorithm 1):
//   reaction pass : k_f, k_r (detailed balance), q_r, f, dq/dT                       (steps 2-4)
//   column pass   : column m of J built in registers -- each dq_r/dn_m formed once and applied to the
//                   participating rows (eq. 19) -- then M[:,m] = delta - h J[:,m] stored, row scales kept
//   LU            : left-looking by column with the multipliers L in registers, scaled row pivoting by
//                   compile-time select chains (no dynamic register index), U stored back to shared memory,
//                   right-hand side carried along, back substitution                  (Algorithm 1, R14)
// Persistent kernel: one Newton iteration is the unit of lock-step; finished lanes refill from the global
// work counter (a8).  The unrolled iteration body is ~10^4 instructions, far beyond the instruction caches, so the
// kernel runs ONE block of 8 warps per SM that walks the body in lock-step (block barriers, no divergent code in
// the body): every instruction fetched from L2 serves all resident warps.
#pragma once
#include "kr_tables.h"
#include "kr_math.cuh"
#include "kr_post.cuh"

template <int I> struct KrIC { static constexpr int value = I; };
template <int B, int E, class F>
__device__ __forceinline__ void kr_static_for(F&& f) {
  if constexpr (B < E) { f(KrIC<B>{}); kr_static_for<B + 1, E>(f); }
}
#define KR_FOR(var, B, E) kr_static_for<(B), (E)>([&](auto var##_ic) { constexpr int var = decltype(var##_ic)::value;
#define KR_END });

__device__ __forceinline__ double krs_ipow(double x, int e) { return e <= 0 ? 1.0 : (e == 1 ? x : (e == 2 ? x * x : x * x * x)); }
__device__ __forceinline__ bool krs_finite(double x) { return fabs(x) <= 1.79769313486231570e308; }
__device__ __forceinline__ double krs_sel(bool p, double a, double b) { return p ? a : b; }

// does species m take part in reaction r (either side)?
__host__ __device__ constexpr bool krs_participates(int r, int m) {
  for (int k = 0; k < 6; ++k)
    if (KrNet::sp[r][k] == m) return true;
  return false;
}
__host__ __device__ constexpr bool krs_col_has(int r, int m) { return krs_participates(r, m) || (KrNet::flags[r] & KR_DF_TB); }

struct KrsShared {
  double* sm;     // already offset by the thread index; entry e of this lane is sm[e * KRS_BLOCK]
  __device__ __forceinline__ double& M(int i, int j) const { return sm[(i * KrNet::N + j) * KRS_BLOCK]; }
  __device__ __forceinline__ double& UN(int i) const { return sm[(KrNet::N * KrNet::N + i) * KRS_BLOCK]; }
};

// ---- steps 2-3: thermo of all species and rate constants of all reactions at T -----------------------------
template <bool DERIV>
__device__ __forceinline__ void krs_rate_constants(double T, double aux0, const double* __restrict__ aux, long long cell,
                                                   long long n_cells, double (&kf)[KrNet::R], double (&kr)[KrNet::R],
                                                   double (&dlf)[KrNet::R], double (&dlr)[KrNet::R],
                                                   double (&uh)[KrNet::S], double (&ch)[KrNet::S]) {
  constexpr int S = KrNet::S, R = KrNet::R;
  const double invT = krs_rcp(T), lnT = log(T);
  double gh[S];
  if constexpr (KrNet::any_rev || KrNet::energy) {
    const double T2 = T * T, T3 = T2 * T, T4 = T3 * T;
    KR_FOR(s, 0, S)
      constexpr double tmid = KrNet::T_mid[s];
      constexpr double l0 = KrNet::nasa[s][0], l1 = KrNet::nasa[s][1], l2 = KrNet::nasa[s][2], l3 = KrNet::nasa[s][3],
                       l4 = KrNet::nasa[s][4], l5 = KrNet::nasa[s][5], l6 = KrNet::nasa[s][6];
      constexpr double h0 = KrNet::nasa[s][7], h1 = KrNet::nasa[s][8], h2 = KrNet::nasa[s][9], h3 = KrNet::nasa[s][10],
                       h4 = KrNet::nasa[s][11], h5 = KrNet::nasa[s][12], h6 = KrNet::nasa[s][13];
      const bool lo = T <= tmid;
      const double a0 = lo ? l0 : h0, a1 = lo ? l1 : h1, a2 = lo ? l2 : h2, a3 = lo ? l3 : h3, a4 = lo ? l4 : h4,
                   a5 = lo ? l5 : h5, a6 = lo ? l6 : h6;
      const double cp = a0 + a1 * T + a2 * T2 + a3 * T3 + a4 * T4;
      const double h = a0 + a1 * T * 0.5 + a2 * T2 * (1.0 / 3.0) + a3 * T3 * 0.25 + a4 * T4 * 0.2 + a5 * invT;
      const double sR = a0 * lnT + a1 * T + a2 * T2 * 0.5 + a3 * T3 * (1.0 / 3.0) + a4 * T4 * 0.25 + a6;
      gh[s] = h - sR; uh[s] = h - 1.0; ch[s] = cp - 1.0;
    KR_END
  }
  KR_FOR(r, 0, R)
    constexpr int fl = KrNet::flags[r];
    kr[r] = 0.0; dlf[r] = 0.0; dlr[r] = 0.0;
    if constexpr (fl & KR_DF_CONST) {
      constexpr double A_r = KrNet::A[r];
      kf[r] = A_r;
    } else if constexpr (fl & KR_DF_AUX) {
      constexpr double A_r = KrNet::A[r];
      constexpr int ai = KrNet::auxi[r];
      kf[r] = A_r * (ai == 0 ? aux0 : aux[(long long)ai * n_cells + cell]);
    } else {
      constexpr double c0_r = KrNet::c0[r], beta_r = KrNet::beta[r], Ea_r = KrNet::Ea[r];
      const double lnkf = c0_r + beta_r * lnT - Ea_r * invT;
      kf[r] = krs_exp(lnkf);
      if constexpr (DERIV) dlf[r] = (beta_r + Ea_r * invT) * invT;
      if constexpr (fl & KR_DF_REV) {
        double sg = 0.0, su = 0.0;
        KR_FOR(k, 0, 6)
          if constexpr (KrNet::sp[r][k] >= 0) {
            constexpr double c = (k < 3) ? -(double)KrNet::nu[r][k] : (double)KrNet::nu[r][k];
            constexpr int sk = KrNet::sp[r][k];
            sg += c * gh[sk];
            if constexpr (DERIV) su += c * uh[sk];
          }
        KR_END
        constexpr double dn_r = (double)KrNet::dnu_tot[r], lpk = KrNet::ln_p0_kB;
        const double lnKc = -sg + dn_r * (lpk - lnT);
        kr[r] = krs_exp(lnkf - lnKc);
        if constexpr (DERIV) dlr[r] = dlf[r] - su * invT;
      }
    }
  KR_END
}

// ---- step 4 (+ the T column of step 5): rates of progress, f, and per-reaction factors for the column pass ---
//   a[r] = M_r k_f, b[r] = M_r k_r, qh[r] = k_f P' - k_r P'' (third-body reactions)
template <bool WANTJ>
__device__ __forceinline__ void krs_reactions(double Ncal, double T, const double (&u)[KrNet::N], const double (&kf)[KrNet::R],
                                              const double (&kr)[KrNet::R], const double (&dlf)[KrNet::R],
                                              const double (&dlr)[KrNet::R], const double (&uh)[KrNet::S],
                                              const double (&ch)[KrNet::S], double (&n)[KrNet::S], double (&f)[KrNet::N],
                                              double (&a)[KrNet::R], double (&b)[KrNet::R], double (&qh)[KrNet::R],
                                              double (&jt)[KrNet::N], double& Cval, double& sc_out) {
  constexpr int S = KrNet::S, R = KrNet::R, N = KrNet::N;
  KR_FOR(s, 0, S) n[s] = Ncal * u[s]; f[s] = 0.0; jt[s] = 0.0; KR_END
  double heat_sum = 0.0, heat_dT = 0.0;
  KR_FOR(r, 0, R)
    constexpr int fl = KrNet::flags[r];
    double Pf = 1.0, Pr = 1.0;
    KR_FOR(k, 0, 6)
      if constexpr (KrNet::sp[r][k] >= 0) {
        constexpr int sk = KrNet::sp[r][k], ek = KrNet::nu[r][k];
        const double p = krs_ipow(n[sk], ek);
        if constexpr (k < 3) Pf *= p; else Pr *= p;
      }
    KR_END
    double Mtb = 1.0;
    if constexpr (fl & KR_DF_TB) {
      Mtb = 0.0;
      KR_FOR(s, 0, S) constexpr double eff = KrNet::tb_eff[r][s]; Mtb += eff * n[s]; KR_END
    }
    const double qhat = kf[r] * Pf - kr[r] * Pr;
    const double q = Mtb * qhat;
    KR_FOR(k, 0, 6)
      if constexpr (KrNet::sp[r][k] >= 0) {
        constexpr int sk = KrNet::sp[r][k];
        constexpr double dn = (k < 3) ? -(double)KrNet::nu[r][k] : (double)KrNet::nu[r][k];
        f[sk] += dn * q;
      }
    KR_END
    constexpr double qk_r = KrNet::qk[r];
    if constexpr (KrNet::any_qext) heat_sum += qk_r * q;
    if constexpr (WANTJ) {
      a[r] = Mtb * kf[r]; b[r] = Mtb * kr[r]; qh[r] = qhat;
      if constexpr (KrNet::energy) {
        const double dqdT = Mtb * (kf[r] * dlf[r] * Pf - kr[r] * dlr[r] * Pr);
        KR_FOR(k, 0, 6)
          if constexpr (KrNet::sp[r][k] >= 0) {
            constexpr int sk = KrNet::sp[r][k];
            constexpr double dn = (k < 3) ? -(double)KrNet::nu[r][k] : (double)KrNet::nu[r][k];
            jt[sk] += dn * dqdT;
          }
        KR_END
        if constexpr (KrNet::any_qext) heat_dT += qk_r * dqdT;
      }
    }
  KR_END
  const double invN = krs_rcp(Ncal);
  KR_FOR(s, 0, S) f[s] *= invN; KR_END
  if constexpr (KrNet::energy) {
    double C = 0.0, su = 0.0, sc = 0.0;
    KR_FOR(s, 0, S) C += u[s] * ch[s]; su += uh[s] * f[s]; sc += ch[s] * f[s]; KR_END
    const double invC = krs_rcp(C);
    f[S] = (heat_sum * invN - T * su) * invC;
    Cval = invC; sc_out = sc;
    if constexpr (WANTJ) {
      double accT = 0.0;
      KR_FOR(s, 0, S) jt[s] *= invN; accT += uh[s] * jt[s]; KR_END
      jt[S] = (heat_dT * invN - T * accT - sc) * invC;
    }
  }
}

// ---- step 5: column m of J in registers (eq. 19), T-row entry, then M[:,m] = delta - h J[:,m] ---------------
template <int m>
__device__ __forceinline__ void krs_column(const KrsShared& sh, double h, double T, double Cval, const double (&n)[KrNet::S],
                                           const double (&a)[KrNet::R], const double (&b)[KrNet::R],
                                           const double (&qh)[KrNet::R], const double (&uh)[KrNet::S],
                                           int (&vh)[KrNet::N]) {
  constexpr int S = KrNet::S, R = KrNet::R, N = KrNet::N;
  double col[N];
  KR_FOR(i, 0, N) col[i] = 0.0; KR_END
  double heat_dn = 0.0;
  KR_FOR(r, 0, R)
    if constexpr (krs_col_has(r, m)) {
      double d = 0.0;
      KR_FOR(k, 0, 6)
        if constexpr (KrNet::sp[r][k] == m && (k < 3 || (KrNet::flags[r] & KR_DF_REV))) {
          constexpr int base = (k < 3) ? 0 : 3;
          double others = 1.0;
          KR_FOR(kk, 0, 3)
            if constexpr (base + kk != k && KrNet::sp[r][base + kk] >= 0) {
              constexpr int so = KrNet::sp[r][base + kk], eo = KrNet::nu[r][base + kk];
              others *= krs_ipow(n[so], eo);
            }
          KR_END
          const double kk2 = (k < 3) ? a[r] : -b[r];
          constexpr int ek = KrNet::nu[r][k];
          d += kk2 * (double)ek * krs_ipow(n[m], ek - 1) * others;
        }
      KR_END
      if constexpr (KrNet::flags[r] & KR_DF_TB) { constexpr double eff = KrNet::tb_eff[r][m]; d += eff * qh[r]; }
      KR_FOR(i, 0, 6)
        if constexpr (KrNet::sp[r][i] >= 0) {
          constexpr int si = KrNet::sp[r][i];
          constexpr double dn = (i < 3) ? -(double)KrNet::nu[r][i] : (double)KrNet::nu[r][i];
          col[si] += dn * d;
        }
      KR_END
      if constexpr (KrNet::energy && KrNet::any_qext) { constexpr double qk_r = KrNet::qk[r]; heat_dn += qk_r * d; }
    }
  KR_END
  if constexpr (KrNet::energy) {
    double acc = 0.0;
    KR_FOR(s, 0, S) acc += uh[s] * col[s]; KR_END
    col[S] = (heat_dn - T * acc) * Cval;      // Cval holds 1 / C
  }
  KR_FOR(i, 0, N)
    const double x = ((i == m) ? 1.0 : 0.0) - h * col[i];
    sh.M(i, m) = x;
    vh[i] = max(vh[i], __double2hiint(x) & 0x7fffffff);
  KR_END
}

// ---- step 7: LU + substitution.  M in shared memory (row i at its physical place), rhs in registers. --------
// Left-looking by column: column j is loaded in the current row order (perm), the known multipliers are
// applied from registers, the scaled pivot is chosen, the exchange is done by select chains on every
// register-resident row quantity (perm, scale, rhs, L rows), U(:,j) goes back to shared memory.
// Row scales: vh[i] is the HIGH WORD of max_j |M_ij| (the scale to 2^-20 relative: the implicit scaling of
// Algorithm 1 only ranks pivot candidates, so a truncated scale changes nothing but exact ties).
__device__ __forceinline__ bool krs_lu_solve(const KrsShared& sh, const int (&vh)[KrNet::N], double (&rhs)[KrNet::N]) {
  constexpr int N = KrNet::N;
  double L[N][N], v[N];        // v[i] = 1 / scale_i
  int perm[N];
  bool ok = true;
  KR_FOR(i, 0, N)
    perm[i] = i;
    ok = ok && (vh[i] >= 0x00100000) && (vh[i] < 0x7ff00000);      // zero / denormal / non-finite row
    v[i] = krs_rcp(__hiloint2double(ok ? vh[i] : 0x3ff00000, 0));
  KR_END
  KR_FOR(j, 0, N)
    double c[N];
    KR_FOR(i, 0, N) c[i] = sh.M(perm[i], j); KR_END
    KR_FOR(k, 0, j)
      KR_FOR(i, k + 1, N) c[i] -= L[i][k] * c[k]; KR_END
    KR_END
    double best = -1.0;
    int imax = j;
    KR_FOR(i, j, N)
      const double t = fabs(c[i]) * v[i];
      if (t > best) { best = t; imax = i; }
    KR_END
    // exchange logical rows j and imax
    {
      double cj = c[j], vj = v[j], rj = rhs[j];
      int pj = perm[j];
      KR_FOR(i, j + 1, N)
        const bool p = (imax == i);
        cj = krs_sel(p, c[i], cj); vj = krs_sel(p, v[i], vj); rj = krs_sel(p, rhs[i], rj); pj = p ? perm[i] : pj;
      KR_END
      KR_FOR(i, j + 1, N)
        const bool p = (imax == i);
        c[i] = krs_sel(p, c[j], c[i]); v[i] = krs_sel(p, v[j], v[i]); rhs[i] = krs_sel(p, rhs[j], rhs[i]);
        perm[i] = p ? perm[j] : perm[i];
      KR_END
      c[j] = cj; v[j] = vj; rhs[j] = rj; perm[j] = pj;
      KR_FOR(k, 0, j)
        double lj = L[j][k];
        KR_FOR(i, j + 1, N) lj = krs_sel(imax == i, L[i][k], lj); KR_END
        KR_FOR(i, j + 1, N) L[i][k] = krs_sel(imax == i, L[j][k], L[i][k]); KR_END
        L[j][k] = lj;
      KR_END
    }
    const double piv = c[j];
    if (!(fabs(piv) >= 1e-300)) ok = false;
    const double rp = krs_rcp(piv);
    KR_FOR(i, j + 1, N) L[i][j] = c[i] * rp; rhs[i] -= L[i][j] * rhs[j]; KR_END
    KR_FOR(i, 0, j) sh.M(i, j) = c[i]; KR_END              // U(0..j-1, j): column j of shared memory is free now
    sh.M(j, j) = rp;                                       // the reciprocal pivot, for the back substitution
  KR_END
  KR_FOR(ii, 0, N)
    constexpr int i = N - 1 - ii;
    double sum = rhs[i];
    KR_FOR(k, i + 1, N) sum -= sh.M(i, k) * rhs[k]; KR_END
    rhs[i] = sum * sh.M(i, i);
  KR_END
  return ok;                                               // no early exit: every lane of the block walks the same code
}

// step 9 on the lane's u_n in shared memory ([entry][lane] layout), out of line: it runs once per cell and only for the
// few cells that need it (a negative abundance, or a conservation row drifting beyond cons_tol)
__device__ __forceinline__ KrPostLists krs_post_lists() {
  return KrPostLists{KrNet::E, KrNet::S, KrNet::post_sp_ptr, KrNet::post_sp_ent, KrNet::post_res_ptr, KrNet::post_res_ent,
                     KrNet::post_cmp_ptr, KrNet::post_cmp_ent, KrNet::signed_row};
}
__device__ __noinline__ int krs_post(double* un0, const double* yin, double cons_tol) {
  return kr_postprocess<KrNet::E>(krs_post_lists(), cons_tol, [&](int s) { return yin[s]; }, [&](int s) -> double& { return un0[s * KRS_BLOCK]; });
}

enum { KRS_FETCH = 0, KRS_RUN = 1, KRS_DONE = 2 };

#if defined(KRS_SYNC) && KRS_SYNC >= 2
#define KRS_ALIGN() __syncthreads()      // keeps the 8 warps of the block on one instruction stream inside the body too
#else
#define KRS_ALIGN() ((void)0)
#endif
#if defined(KRS_SYNC) && KRS_SYNC >= 3   // a barrier between rate constants and reactions keeps all 4 R rate values live
#define KRS_ALIGN_RC() __syncthreads()
#else
#define KRS_ALIGN_RC() ((void)0)
#endif

// One trip of the main loop = one pass of EVERY lane through the same straight-line body: rate constants, reactions,
// Jacobian columns, LU, update, controller.  A lane that has just loaded a cell uses its first pass as the
// preliminary evaluation (rate constants of an isothermal cell, f(u_in) for the first sub-step, DESIGN.md step 1) and
// discards the rest of that pass; idle lanes (no cells left) run the body on dead data.  Nothing in the body
// diverges, so block-wide barriers inside it are legal and every warp of the block fetches the same instructions.
extern "C" __global__ void __launch_bounds__(KRS_BLOCK, KRS_MIN_BLOCKS)
kr_spec_kernel(const KrOptsDev o, const KrStepArgs g) {
  extern __shared__ double kr_sm[];
  constexpr int S = KrNet::S, R = KrNet::R, N = KrNet::N, E = KrNet::E;
  const int K = o.max_newton;
  const int lane = threadIdx.x & 31;
  KrsShared sh;
  sh.sm = kr_sm + threadIdx.x;

  int phase = KRS_FETCH;
  long long cell = -1;
  double u[N];
  double kfi[R], kri[R];                       // isothermal networks: rate constants of the cell (registers)
  double Ncal = 1.0, T_iso = 1.0, aux0 = 0.0, t = 0.0, h = 1.0, h_floor = 0.0, e = 0.0, e_prev = 0.0;
  int k = 0, it = 0, st = 0, n_acc = 0, n_rej = 0;
  bool last = false, pend = false;
  unsigned long long c_acc = 0, c_rej = 0, c_newton = 0, c_rate = 0, c_failed = 0;
  KR_FOR(i, 0, N) u[i] = 1.0; sh.UN(i) = 1.0; KR_END
  KR_FOR(r, 0, R) kfi[r] = 0.0; kri[r] = 0.0; KR_END

  for (;;) {
    __syncwarp();
    const bool need = (phase == KRS_FETCH);
    const unsigned want = __ballot_sync(0xffffffffu, need);
    if (want) {                                                  // step 1: a8 refill + layout-in
      const int leader = __ffs(want) - 1;
      unsigned long long base = 0;
      if (lane == leader) base = atomicAdd(g.counter, (unsigned long long)__popc(want));
      base = __shfl_sync(0xffffffffu, base, leader);
      if (need) {
        cell = (long long)(base + (unsigned long long)__popc(want & ((1u << lane) - 1u)));
        phase = (cell < g.n_cells) ? KRS_RUN : KRS_DONE;
        if (phase == KRS_RUN) {
          st = 0;
          double Tc = g.T[cell];
          constexpr double T_lo = KrNet::T_lo, T_hi = KrNet::T_hi;
          if (Tc < T_lo) { Tc = T_lo; st |= KR_DST_T_CLAMPED; }
          if (Tc > T_hi) { Tc = T_hi; st |= KR_DST_T_CLAMPED; }
          Ncal = g.rho[cell] * (1.0 / KR_M_U);
          KR_FOR(s, 0, S) u[s] = g.y[cell * S + s]; sh.UN(s) = u[s]; KR_END
          if constexpr (KrNet::energy) { u[S] = Tc; sh.UN(S) = Tc; }
          T_iso = Tc;
          aux0 = (KrNet::n_aux > 0) ? g.aux[cell] : 0.0;
          t = 0.0; h = g.dt; n_acc = 0; n_rej = 0; k = 0;
          h_floor = o.h_min_rel * g.dt;
          pend = (o.h0_mode == 1) || !KrNet::energy;
#ifdef KRS_PRELIM_WS
          // isothermal: the preliminary evaluation was done for every cell by kr_spec_prelim_kernel (full warps, no
          // exponentials in this kernel's body, no discarded pass)
          KR_FOR(r, 0, R)
            constexpr int fl = KrNet::flags[r];
            constexpr double A_r = KrNet::A[r];
            if constexpr (fl & KR_DF_CONST) kfi[r] = A_r; else kfi[r] = g.prelim[(long long)r * g.n_cells + cell];
            if constexpr (fl & KR_DF_REV) kri[r] = g.prelim[(long long)(R + r) * g.n_cells + cell]; else kri[r] = 0.0;
          KR_END
          h = g.prelim[(long long)(2 * R) * g.n_cells + cell];
          h_floor = o.h_min_rel * fmin(h, g.dt);
          pend = false;
          c_rate++;
#endif
        }
      }
    }
#ifdef KRS_SYNC
    if (__syncthreads_and(phase == KRS_DONE)) break;
#else
    if (__all_sync(0xffffffffu, phase == KRS_DONE)) break;
#endif
    const bool active = (phase == KRS_RUN);
    const bool prelim = pend;                                    // this pass only evaluates (see above)

    bool fail_cell = false, cell_done = false;
    if (active && !prelim && k == 0) {                           // sub-step start: trim (R22), failure test
      const double rem = g.dt - t;
      last = false;
      if (h >= rem) { h = rem; last = true; }
      if (h < h_floor || n_acc + n_rej > o.max_substeps) fail_cell = true;
      else {
        KR_FOR(i, 0, N) u[i] = sh.UN(i); KR_END
        e_prev = 0.0; e = __longlong_as_double(0x7ff0000000000000LL); it = K + 1; k = 1;
      }
    }
    const bool live = active && !prelim && !fail_cell;           // this pass is a Newton iteration of the lane's cell

    // ---- steps 2-5 ------------------------------------------------------------------------------------------
    const double T = KrNet::energy ? u[N - 1] : T_iso;
    double rhs[N];
    int vh[N];
    {
      double uh[S], ch[S], n[S], f[N], a[R], b[R], qh[R], jt[N], Cv = 1.0, sc = 0.0;
      if constexpr (KrNet::energy) {
        double kf[R], kr[R], dlf[R], dlr[R];
        krs_rate_constants<true>(T, aux0, g.aux, active ? cell : 0, g.n_cells, kf, kr, dlf, dlr, uh, ch);
        if (active && !fail_cell) c_rate++;
        KRS_ALIGN_RC();
        krs_reactions<true>(Ncal, T, u, kf, kr, dlf, dlr, uh, ch, n, f, a, b, qh, jt, Cv, sc);
      } else {
        double dlf[R], dlr[R];
#ifndef KRS_PRELIM_WS
        if (__any_sync(0xffffffffu, active && prelim)) {         // rate constants of freshly loaded isothermal cells
          double kf[R], kr[R];
          krs_rate_constants<false>(T, aux0, g.aux, active ? cell : 0, g.n_cells, kf, kr, dlf, dlr, uh, ch);
          if (active && prelim) {
            KR_FOR(r, 0, R) kfi[r] = kf[r]; kri[r] = kr[r]; KR_END
            c_rate++;
          }
        }
#endif
        KRS_ALIGN_RC();
        krs_reactions<true>(Ncal, T, u, kfi, kri, dlf, dlr, uh, ch, n, f, a, b, qh, jt, Cv, sc);
      }
      if (active && prelim) {                                    // first sub-step from f(u_in) (step 1, h0_mode 1)
        if (o.h0_mode == 1) {
          double big = 0.0;
          KR_FOR(s, 0, S) big = fmax(big, fabs(f[s]) / (fabs(u[s]) + o.y_floor)); KR_END
          if (big > 0.0 && krs_finite(big)) h = fmin(g.dt, o.eta / big);
        }
        h_floor = o.h_min_rel * fmin(h, g.dt);
        pend = false;
      }
      KRS_ALIGN();
      KR_FOR(i, 0, N) vh[i] = 0; KR_END
      KR_FOR(m, 0, S) krs_column<m>(sh, h, T, Cv, n, a, b, qh, uh, vh); KR_END
      if constexpr (KrNet::energy) {                             // T column (eq. 20)
        KR_FOR(i, 0, N)
          const double x = ((i == S) ? 1.0 : 0.0) - h * jt[i];
          sh.M(i, S) = x;
          vh[i] = max(vh[i], __double2hiint(x) & 0x7fffffff);
        KR_END
      }
      KR_FOR(i, 0, N) rhs[i] = -(u[i] - sh.UN(i) - h * f[i]); KR_END
    }
    KRS_ALIGN();
    const bool solved = krs_lu_solve(sh, vh, rhs);               // step 7 (no early exits inside)
    KRS_ALIGN();

    if (live) {                                                  // steps 6-8 for the lanes this pass counts for
      c_newton++;
      bool ran = true, sub_end = false;
      if (!solved) { ran = false; sub_end = true; }
      else {
        bool fin = true;
        double en = 0.0;
        KR_FOR(i, 0, N)
          u[i] += rhs[i];
          fin = fin && krs_finite(u[i]);
          const double w = fabs(rhs[i]) * krs_rcp(o.rtol * fabs(u[i]) + ((i < S) ? o.atol_y : o.atol_T));
          en = (w > en) ? w : en;
        KR_END
        if (!fin) { ran = false; sub_end = true; }
        else {
          e = en;
          if (it == K + 1 && e <= 1.0) it = k;
          if (!o.fixed_newton) {
            if (e <= 1.0) sub_end = true;
            else if (k >= 2 && e > o.bail_ratio * e_prev) { ran = false; sub_end = true; }
          }
          e_prev = e;
          if (k >= K) sub_end = true;
          k++;
        }
      }
      if (sub_end) {                                             // step 8: accept / reject
        bool ok = ran && (e <= 1.0);
        if (ok) {
          double miny = u[0];
          KR_FOR(s, 1, S) miny = fmin(miny, u[s]); KR_END
          if (!(miny >= -o.neg_tol)) ok = false;
        }
        if constexpr (KrNet::energy) {
          constexpr double T_lo = KrNet::T_lo, T_hi = KrNet::T_hi;
          if (ok && !(u[N - 1] >= T_lo && u[N - 1] <= T_hi)) ok = false;
        }
        if (ok && krs_finite(o.chg_max)) {
          double chg = 0.0;
          KR_FOR(i, 0, N)
            const double un = sh.UN(i);
            chg = fmax(chg, fabs(u[i] - un) / ((i < S) ? (fabs(un) + o.chg_floor) : un));
          KR_END
          if (!(chg <= o.chg_max)) ok = false;
        }
        if (ok) {
          n_acc++;
          KR_FOR(i, 0, N) sh.UN(i) = u[i]; KR_END
          if (last) cell_done = true;
          else {
            t = t + h;
            if (it <= o.it_fast) h = h * o.grow_fast;
            else if (it <= o.it_mid) h = h * o.grow_mid;
          }
        } else {
          n_rej++;
          st |= KR_DST_REJECTED;
          h = h * o.shrink;
          KR_FOR(i, 0, N) u[i] = sh.UN(i); KR_END               // keep the lane's state finite
        }
        k = 0;
      }
    }
    if (fail_cell) {                                             // R13: revert (the caller's buffers were never written)
      c_acc += n_acc; c_rej += n_rej;
      if (g.fail_list) g.fail_list[atomicAdd(g.fail_count, 1ull)] = cell;          // second attempt
      else { c_failed++; if (g.status) g.status[cell] = st | KR_DST_FAILED; }
      KR_FOR(i, 0, N) u[i] = 1.0; sh.UN(i) = 1.0; KR_END
      phase = KRS_FETCH;
    } else if (cell_done) {                                      // step 9: finalise + layout-out (u == u_n here)
      c_acc += n_acc; c_rej += n_rej;
      if (o.finalize) {                                          // post-processing stages 1-3
        // screen (unrolled over the composition matrix): a negative abundance, or a row whose initial-minus-final total
        // exceeds cons_tol x its scale
        bool any = false;
        double yin[S];
        KR_FOR(s, 0, S) yin[s] = g.y[cell * S + s]; any = any || (u[s] < 0.0); KR_END
        KR_FOR(nu, 0, KrNet::E)
          double full = 0.0, scale = 0.0;
          KR_FOR(s, 0, S)
            constexpr int c = KrNet::comp[nu][s];
            if constexpr (c != 0) { full += (double)c * (yin[s] - u[s]); scale += fabs((double)c * yin[s]); }
          KR_END
          any = any || (fabs(full) > o.cons_tol * scale);
        KR_END
        if (any) {                                               // rare: the shared routine works on u_n (== u here)
          st |= krs_post(&sh.UN(0), g.y + cell * S, o.cons_tol);
          KR_FOR(s, 0, S) u[s] = sh.UN(s); KR_END
        }
      }
      KR_FOR(s, 0, S) g.y[cell * S + s] = u[s]; KR_END
      if constexpr (KrNet::energy) g.T[cell] = u[N - 1];
      if (g.status) g.status[cell] = st;
      phase = KRS_FETCH;
    }
  }
  unsigned long long c[5] = {c_acc, c_rej, c_newton, c_rate, c_failed};
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    unsigned long long x = c[i];
    for (int off = 16; off > 0; off >>= 1) x += __shfl_xor_sync(0xffffffffu, x, off);
    c[i] = x;
  }
  if (lane == 0) {
    atomicAdd(g.stats + 0, c[0]); atomicAdd(g.stats + 1, c[1]); atomicAdd(g.stats + 2, c[2]);
    atomicAdd(g.stats + 3, c[2]); atomicAdd(g.stats + 4, c[3]); atomicAdd(g.stats + 5, c[4]);
  }
}

#ifdef KRS_PRELIM_WS
// Preliminary evaluation of an isothermal network for every cell (DESIGN.md step 1): rate constants at the clamped T and
// the first sub-step from f(u_in).  One thread per cell, grid-stride, full warps; output as [2R + 1][n_cells].
extern "C" __global__ void __launch_bounds__(256) kr_spec_prelim_kernel(const KrOptsDev o, const KrStepArgs g) {
  constexpr int S = KrNet::S, R = KrNet::R, N = KrNet::N;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x; cell < g.n_cells; cell += stride) {
    double Tc = g.T[cell];
    constexpr double T_lo = KrNet::T_lo, T_hi = KrNet::T_hi;
    Tc = (Tc < T_lo) ? T_lo : ((Tc > T_hi) ? T_hi : Tc);
    const double Ncal = g.rho[cell] * (1.0 / KR_M_U);
    const double aux0 = (KrNet::n_aux > 0) ? g.aux[cell] : 0.0;
    double u[N];
    KR_FOR(s, 0, S) u[s] = g.y[cell * S + s]; KR_END
    double kf[R], kr[R], dlf[R], dlr[R], uh[S], ch[S];
    krs_rate_constants<false>(Tc, aux0, g.aux, cell, g.n_cells, kf, kr, dlf, dlr, uh, ch);
    double h = g.dt;
    if (o.h0_mode == 1) {
      double n[S], f[N], a[R], b[R], qh[R], jt[N], Cv = 1.0, sc = 0.0;
      krs_reactions<false>(Ncal, Tc, u, kf, kr, dlf, dlr, uh, ch, n, f, a, b, qh, jt, Cv, sc);
      double big = 0.0;
      KR_FOR(s, 0, S) big = fmax(big, fabs(f[s]) / (fabs(u[s]) + o.y_floor)); KR_END
      if (big > 0.0 && krs_finite(big)) h = fmin(g.dt, o.eta / big);
    }
    KR_FOR(r, 0, R)
      constexpr int fl = KrNet::flags[r];
      if constexpr (!(fl & KR_DF_CONST)) g.prelim[(long long)r * g.n_cells + cell] = kf[r];
      if constexpr (fl & KR_DF_REV) g.prelim[(long long)(R + r) * g.n_cells + cell] = kr[r];
    KR_END
    g.prelim[(long long)(2 * R) * g.n_cells + cell] = h;
  }
}
#endif
