// kr_tpc.cuh -- thread-per-cell solve kernel (small systems, N <= KR_TPC_MAX_N), table driven.
//
// One lane integrates one cell through DESIGN.md steps 1-9 (eq. 15, 158-171 eqs. 16-17,
// 173-187 eqs. 18-20, 199, 212-218, 236-276 Algorithm 1).  The per-lane vectors and the N x N matrix live
// in shared memory laid out [entry][lane] (species-SoA across the warp: conflict-free, dynamic indexing
// is free there), scalars in registers.  The kernel is persistent: the unit of lock-step is ONE Newton
// iteration; a lane whose cell finishes pulls the next cell from a global work counter (warp-aggregated
// atomic), so lanes never idle while cells remain (a8, "refill").
#pragma once
#include "kr_device.cuh"
#include "kr_post.cuh"

#define KR_TPC_MAX_N 16
#define KR_TPC_BD 64

enum { KR_PH_FETCH = 0, KR_PH_INIT = 1, KR_PH_NEWTON = 2, KR_PH_DONE = 3 };

// number of doubles of shared memory one lane needs
__host__ __device__ inline int kr_tpc_doubles_per_lane(int N, int S, int R, int energy) {
  return 5 * N + N * N + 3 * S + (energy ? 0 : 2 * R);
}

struct KrTpcView {
  double* sm;
  int tid, BD;
  int oU, oUN, oF, oB, oV, oM, oTH, oK;
  __device__ __forceinline__ double& at(int off, int i) const { return sm[(off + i) * BD + tid]; }
};

// thermo of every species at T -> shared ghat[S], uhat[S], chat[S]
__device__ __forceinline__ void kr_tpc_thermo(const KrNetDev& n, const KrTpcView& v, double T, double invT, double lnT) {
  for (int s = 0; s < n.S; ++s) {
    double g, u, c;
    kr_thermo_species(n.nasa + 14 * s, n.T_mid[s], T, invT, lnT, g, u, c);
    v.at(v.oTH, s) = g; v.at(v.oTH, n.S + s) = u; v.at(v.oTH, 2 * n.S + s) = c;
  }
}

// Steps 4-5 at the iterate U (shared): f -> F[0..N), J -> M (row-major N x N) when wantJ.
template <bool ENERGY>
__device__ __forceinline__ void kr_tpc_eval(const KrNetDev& n, const KrTpcView& v, double Ncal, double T, double aux0,
                                            const double* __restrict__ aux, long long cell, long long n_cells,
                                            bool wantJ) {
  const int S = n.S, R = n.R, N = n.N;
  for (int s = 0; s < S; ++s) v.at(v.oF, s) = 0.0;
  if (wantJ)
    for (int i = 0; i < N * N; ++i) v.at(v.oM, i) = 0.0;
  double heat_sum = 0.0, heat_dT = 0.0;
  const double invT = 1.0 / T;
  const double lnT = ENERGY ? log(T) : 0.0;
  for (int r = 0; r < R; ++r) {
    const int fl = n.flags[r];
    double kf, kr, dlf = 0.0, dlr = 0.0;
    if (ENERGY) {
      double ax = aux0;
      if ((fl & KR_DF_AUX) && n.auxi[r] > 0) ax = aux[(long long)n.auxi[r] * n_cells + cell];
      kr_rate_constants(n, r, fl, invT, lnT, ax, [&](int s) { return v.at(v.oTH, s); },
                        [&](int s) { return v.at(v.oTH, S + s); }, kf, kr, dlf, dlr);
    } else {
      kf = v.at(v.oK, r); kr = v.at(v.oK, R + r);
    }
    int sp[6], nu[6];
    double nn[6], pw[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      sp[k] = n.sp[6 * r + k]; nu[k] = n.nu[6 * r + k];
      nn[k] = (sp[k] >= 0) ? Ncal * v.at(v.oU, sp[k]) : 1.0;
      pw[k] = kr_ipow(nn[k], nu[k]);
    }
    double Mtb = 1.0;
    if (fl & KR_DF_TB) {
      Mtb = 0.0;
      for (int s = 0; s < S; ++s) Mtb += n.tb_eff[r * S + s] * (Ncal * v.at(v.oU, s));
    }
    const double Pf = pw[0] * pw[1] * pw[2], Pr = pw[3] * pw[4] * pw[5];
    const double qhat = kf * Pf - kr * Pr;
    const double q = Mtb * qhat;
#pragma unroll
    for (int k = 0; k < 6; ++k)
      if (sp[k] >= 0) v.at(v.oF, sp[k]) += ((k < 3) ? -(double)nu[k] : (double)nu[k]) * q;
    const double qk = n.any_qext ? n.qk[r] : 0.0;
    heat_sum += qk * q;
    if (!wantJ) continue;
    double d[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const int k1 = (k < 3) ? (k + 1) % 3 : 3 + (k - 3 + 1) % 3, k2 = (k < 3) ? (k + 2) % 3 : 3 + (k - 3 + 2) % 3;
      const double others = pw[k1 < k2 ? k1 : k2] * pw[k1 < k2 ? k2 : k1];
      const double kk = (k < 3) ? kf : -kr;
      d[k] = (sp[k] >= 0) ? Mtb * (kk * (double)nu[k] * kr_ipow(nn[k], nu[k] - 1) * others) : 0.0;
    }
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      if (sp[i] < 0) continue;
      const double dnu = (i < 3) ? -(double)nu[i] : (double)nu[i];
#pragma unroll
      for (int j = 0; j < 6; ++j)
        if (sp[j] >= 0) v.at(v.oM, sp[i] * N + sp[j]) += dnu * d[j];
    }
    if (fl & KR_DF_TB) {
      for (int m = 0; m < S; ++m) {
        const double tq = n.tb_eff[r * S + m] * qhat;
#pragma unroll
        for (int i = 0; i < 6; ++i)
          if (sp[i] >= 0) v.at(v.oM, sp[i] * N + m) += ((i < 3) ? -(double)nu[i] : (double)nu[i]) * tq;
        if (ENERGY && qk != 0.0) v.at(v.oM, S * N + m) += qk * tq;
      }
    }
    if (ENERGY) {
      const double dqdT = Mtb * (kf * dlf * Pf - kr * dlr * Pr);
#pragma unroll
      for (int i = 0; i < 6; ++i)
        if (sp[i] >= 0) v.at(v.oM, sp[i] * N + S) += ((i < 3) ? -(double)nu[i] : (double)nu[i]) * dqdT;
      if (qk != 0.0) {
#pragma unroll
        for (int j = 0; j < 6; ++j)
          if (sp[j] >= 0) v.at(v.oM, S * N + sp[j]) += qk * d[j];
        heat_dT += qk * dqdT;
      }
    }
  }
  const double invN = 1.0 / Ncal;
  for (int s = 0; s < S; ++s) v.at(v.oF, s) = v.at(v.oF, s) / Ncal;
  if (!ENERGY) return;
  double C = 0.0, su = 0.0, sc = 0.0;
  for (int s = 0; s < S; ++s) {
    const double fs = v.at(v.oF, s), uh = v.at(v.oTH, S + s), ch = v.at(v.oTH, 2 * S + s);
    C += v.at(v.oU, s) * ch; su += uh * fs; sc += ch * fs;
  }
  v.at(v.oF, S) = (heat_sum / Ncal - T * su) / C;
  if (!wantJ) return;
  (void)invN;
  for (int s = 0; s < S; ++s) v.at(v.oM, s * N + S) = v.at(v.oM, s * N + S) / Ncal;
  for (int m = 0; m < S; ++m) {
    double acc = 0.0;
    for (int s = 0; s < S; ++s) acc += v.at(v.oTH, S + s) * v.at(v.oM, s * N + m);
    v.at(v.oM, S * N + m) = (v.at(v.oM, S * N + m) - T * acc) / C;
  }
  double accT = 0.0;
  for (int s = 0; s < S; ++s) accT += v.at(v.oTH, S + s) * v.at(v.oM, s * N + S);
  v.at(v.oM, S * N + S) = (heat_dT / Ncal - T * accT - sc) / C;
}

// Step 7 (Algorithm 1, reading R14) on the shared N x N matrix with the right-hand side B carried along:
// implicit row scaling, pivot = argmax_{i>=j} |M_ij| / v_i (ties -> smallest i), rows exchanged, elimination,
// then back substitution; B holds the solution.  Returns false on a zero row or |pivot| < 1e-300.
__device__ __forceinline__ bool kr_tpc_lu_solve(const KrTpcView& v, int N) {
  for (int i = 0; i < N; ++i) {
    double big = 0.0;
    for (int j = 0; j < N; ++j) big = fmax(big, fabs(v.at(v.oM, i * N + j)));
    if (!(big > 0.0)) return false;
    v.at(v.oV, i) = big;
  }
  for (int j = 0; j < N; ++j) {
    double best = -1.0;
    int imax = j;
    for (int i = j; i < N; ++i) {
      const double t = fabs(v.at(v.oM, i * N + j)) / v.at(v.oV, i);
      if (t > best) { best = t; imax = i; }
    }
    if (imax != j) {
      for (int k = j; k < N; ++k) {
        const double x = v.at(v.oM, imax * N + k);
        v.at(v.oM, imax * N + k) = v.at(v.oM, j * N + k);
        v.at(v.oM, j * N + k) = x;
      }
      double x = v.at(v.oV, imax); v.at(v.oV, imax) = v.at(v.oV, j); v.at(v.oV, j) = x;
      x = v.at(v.oB, imax); v.at(v.oB, imax) = v.at(v.oB, j); v.at(v.oB, j) = x;
    }
    const double piv = v.at(v.oM, j * N + j);
    if (!(fabs(piv) >= 1e-300)) return false;
    const double bj = v.at(v.oB, j);
    for (int i = j + 1; i < N; ++i) {
      const double l = v.at(v.oM, i * N + j) / piv;
      for (int k = j + 1; k < N; ++k) v.at(v.oM, i * N + k) -= l * v.at(v.oM, j * N + k);
      v.at(v.oB, i) -= l * bj;
    }
  }
  for (int i = N - 1; i >= 0; --i) {
    double sum = v.at(v.oB, i);
    for (int k = i + 1; k < N; ++k) sum -= v.at(v.oM, i * N + k) * v.at(v.oB, k);
    v.at(v.oB, i) = sum / v.at(v.oM, i * N + i);
  }
  return true;
}

template <bool ENERGY>
__global__ void __launch_bounds__(KR_TPC_BD) kr_tpc_kernel(const KrNetDev n, const KrOptsDev o, const KrStepArgs a) {
  extern __shared__ double kr_sm[];
  const int S = n.S, R = n.R, N = n.N, K = o.max_newton;
  const int lane = threadIdx.x & 31;
  KrTpcView v;
  v.sm = kr_sm; v.tid = threadIdx.x; v.BD = blockDim.x;
  v.oU = 0; v.oUN = N; v.oF = 2 * N; v.oB = 3 * N; v.oV = 4 * N; v.oM = 5 * N; v.oTH = 5 * N + N * N; v.oK = v.oTH + 3 * S;

  int phase = KR_PH_FETCH;
  long long cell = -1;
  double Ncal = 1.0, T_iso = 0.0, aux0 = 0.0, t = 0.0, h = 0.0, h_floor = 0.0, e = 0.0, e_prev = 0.0;
  int k = 0, it = 0, st = 0, n_acc = 0, n_rej = 0;
  bool last = false;
  unsigned long long c_acc = 0, c_rej = 0, c_newton = 0, c_rate = 0, c_failed = 0;

  for (;;) {
    __syncwarp();
    const bool need = (phase == KR_PH_FETCH);
    const unsigned want = __ballot_sync(0xffffffffu, need);
    if (want) {
      const int leader = __ffs(want) - 1;
      unsigned long long base = 0;
      if (lane == leader) base = atomicAdd(a.counter, (unsigned long long)__popc(want));
      base = __shfl_sync(0xffffffffu, base, leader);
      if (need) {
        cell = (long long)(base + (unsigned long long)__popc(want & ((1u << lane) - 1u)));
        phase = (cell < a.n_cells) ? KR_PH_INIT : KR_PH_DONE;
      }
    }
    if (__all_sync(0xffffffffu, phase == KR_PH_DONE)) break;

    if (phase == KR_PH_INIT) {                                   // step 1
      st = 0;
      double Tc = a.T[cell];
      if (Tc < n.T_lo) { Tc = n.T_lo; st |= KR_DST_T_CLAMPED; }
      if (Tc > n.T_hi) { Tc = n.T_hi; st |= KR_DST_T_CLAMPED; }
      Ncal = a.rho[cell] / KR_M_U;
      for (int s = 0; s < S; ++s) v.at(v.oUN, s) = a.y[cell * S + s];
      if (ENERGY) v.at(v.oUN, S) = Tc;
      T_iso = Tc;
      aux0 = (n.n_aux > 0) ? a.aux[cell] : 0.0;
      t = 0.0; h = a.dt; n_acc = 0; n_rej = 0;
      const double invT = 1.0 / Tc, lnT = log(Tc);
      if (!ENERGY) {                                             // isothermal: steps 2-3 once per cell
        if (n.any_rev) kr_tpc_thermo(n, v, Tc, invT, lnT);
        for (int r = 0; r < R; ++r) {
          const int fl = n.flags[r];
          double ax = aux0;
          if ((fl & KR_DF_AUX) && n.auxi[r] > 0) ax = a.aux[(long long)n.auxi[r] * a.n_cells + cell];
          double kf, kr, d0, d1;
          kr_rate_constants(n, r, fl, invT, lnT, ax, [&](int s) { return v.at(v.oTH, s); },
                            [&](int s) { return v.at(v.oTH, S + s); }, kf, kr, d0, d1);
          v.at(v.oK, r) = kf; v.at(v.oK, R + r) = kr;
        }
        c_rate++;
      }
      if (o.h0_mode == 1) {
        if (ENERGY) { kr_tpc_thermo(n, v, Tc, invT, lnT); c_rate++; }
        for (int i = 0; i < N; ++i) v.at(v.oU, i) = v.at(v.oUN, i);
        kr_tpc_eval<ENERGY>(n, v, Ncal, Tc, aux0, a.aux, cell, a.n_cells, false);
        double big = 0.0;
        for (int s = 0; s < S; ++s) big = fmax(big, fabs(v.at(v.oF, s)) / (fabs(v.at(v.oUN, s)) + o.y_floor));
        // fmax drops a NaN operand; the oracle's std::max(big, x) keeps big as well
        if (big > 0.0 && kr_finite(big)) h = fmin(a.dt, o.eta / big);
      }
      h_floor = o.h_min_rel * fmin(h, a.dt);
      k = 0;
      phase = KR_PH_NEWTON;
    }
    __syncwarp();

    if (phase == KR_PH_NEWTON) {
      bool fail_cell = false, cell_done = false;
      if (k == 0) {                                              // sub-step start: trim (R22), failure test
        const double rem = a.dt - t;
        last = false;
        if (h >= rem) { h = rem; last = true; }
        if (h < h_floor || n_acc + n_rej > o.max_substeps) fail_cell = true;
        else {
          for (int i = 0; i < N; ++i) v.at(v.oU, i) = v.at(v.oUN, i);
          e_prev = 0.0; e = __longlong_as_double(0x7ff0000000000000LL); it = K + 1; k = 1;
        }
      }
      if (!fail_cell) {                                          // one Newton iteration (step 6)
        const double T = ENERGY ? v.at(v.oU, S) : T_iso;
        if (ENERGY) { kr_tpc_thermo(n, v, T, 1.0 / T, log(T)); c_rate++; }
        kr_tpc_eval<ENERGY>(n, v, Ncal, T, aux0, a.aux, cell, a.n_cells, true);
        for (int i = 0; i < N; ++i) v.at(v.oB, i) = -(v.at(v.oU, i) - v.at(v.oUN, i) - h * v.at(v.oF, i));
        for (int i = 0; i < N; ++i)
          for (int j = 0; j < N; ++j) v.at(v.oM, i * N + j) = ((i == j) ? 1.0 : 0.0) - h * v.at(v.oM, i * N + j);
        c_newton++;
        bool ran = true, sub_end = false;
        if (!kr_tpc_lu_solve(v, N)) { ran = false; sub_end = true; }
        else {
          bool fin = true;
          for (int i = 0; i < N; ++i) {
            const double x = v.at(v.oU, i) + v.at(v.oB, i);
            v.at(v.oU, i) = x;
            fin = fin && kr_finite(x);
          }
          if (!fin) { ran = false; sub_end = true; }
          else {
            double en = 0.0;
            for (int i = 0; i < N; ++i) {
              const double atol = (i < S) ? o.atol_y : o.atol_T;
              const double x = fabs(v.at(v.oB, i)) / (o.rtol * fabs(v.at(v.oU, i)) + atol);
              en = (x > en) ? x : en;
            }
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
        if (sub_end) {                                           // step 8: accept / reject
          bool ok = ran && (e <= 1.0);
          if (ok) {
            double miny = v.at(v.oU, 0);
            for (int s = 1; s < S; ++s) miny = fmin(miny, v.at(v.oU, s));
            if (!(miny >= -o.neg_tol)) ok = false;
          }
          if (ok && ENERGY) {
            const double Tn = v.at(v.oU, S);
            if (!(Tn >= n.T_lo && Tn <= n.T_hi)) ok = false;
          }
          if (ok && kr_finite(o.chg_max)) {
            double chg = 0.0;
            for (int s = 0; s < S; ++s)
              chg = fmax(chg, fabs(v.at(v.oU, s) - v.at(v.oUN, s)) / (fabs(v.at(v.oUN, s)) + o.chg_floor));
            if (ENERGY) chg = fmax(chg, fabs(v.at(v.oU, S) - v.at(v.oUN, S)) / v.at(v.oUN, S));
            if (!(chg <= o.chg_max)) ok = false;
          }
          if (ok) {
            n_acc++;
            for (int i = 0; i < N; ++i) v.at(v.oUN, i) = v.at(v.oU, i);
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
          }
          k = 0;
        }
      }
      if (fail_cell) {                                           // R13: revert (global T, y untouched)
        c_acc += n_acc; c_rej += n_rej;
        if (a.fail_list) a.fail_list[atomicAdd(a.fail_count, 1ull)] = cell;        // second attempt
        else { c_failed++; if (a.status) a.status[cell] = st | KR_DST_FAILED; }
        phase = KR_PH_FETCH;
      } else if (cell_done) {                                    // step 9: finalise + layout-out
        c_acc += n_acc; c_rej += n_rej;
        if (o.finalize) st |= kr_postprocess(kr_post_lists(n), o.cons_tol, [&](int s) { return a.y[cell * S + s]; }, [&](int s) -> double& { return v.at(v.oUN, s); });
        for (int s = 0; s < S; ++s) a.y[cell * S + s] = v.at(v.oUN, s);
        if (ENERGY) a.T[cell] = v.at(v.oUN, S);
        if (a.status) a.status[cell] = st;
        phase = KR_PH_FETCH;
      }
    }
  }
  // counters: warp reduction, one atomic per warp and counter
  unsigned long long c[5] = {c_acc, c_rej, c_newton, c_rate, c_failed};
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    unsigned long long x = c[i];
    for (int off = 16; off > 0; off >>= 1) x += __shfl_xor_sync(0xffffffffu, x, off);
    c[i] = x;
  }
  if (lane == 0) {
    atomicAdd(a.stats + 0, c[0]); atomicAdd(a.stats + 1, c[1]); atomicAdd(a.stats + 2, c[2]);
    atomicAdd(a.stats + 3, c[2]); atomicAdd(a.stats + 4, c[3]); atomicAdd(a.stats + 5, c[4]);
  }
}
