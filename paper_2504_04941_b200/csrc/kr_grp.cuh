// kr_grp.cuh -- group-per-cell solve kernel: one warp (W = 1) or one CTA slice of W warps per cell.
//
// The N x N matrix, the vectors and the per-reaction values of ONE cell live in shared memory; the
// 32 W threads of the group split the work of DESIGN.md steps 2-7 as
//   thermo            : thread <-> species
//   rate constants, q : thread <-> reaction (strided)
//   Jacobian          : thread <-> COLUMN m: each derivative dq_r/dn_m is formed once by the owner of
//                       column m and scattered down that column -- no atomics, fixed summation order
//                       (replaces the atomicAdd accumulation of PAPER.md:232; eq. 19)
//   f, J[:,T]         : thread <-> ROW s, gather over the species' reaction list   (eq. 15, eq. 20)
//   LU                : thread <-> matrix row ("one thread per row"), pivot by group arg-max,
//                       right-looking elimination with the right-hand side carried along (Algorithm 1)
// Controller scalars (t, h, k, e, ...) are replicated in every thread and evolve identically.
// The kernel is persistent: a group that finishes a cell pulls the next one from the global counter.
#pragma once
#include "kr_device.cuh"
#include "kr_post.cuh"

struct KrGrpLayout {
  int oM, oU, oUN, oF, oB, oV, oTH, oKF, oKR, oQ, oDQT, oQH, oMT, oRED, total;   // in doubles
};

__host__ __device__ inline KrGrpLayout kr_grp_layout(int N, int S, int R, int ld, int energy, int any_tb, int W) {
  KrGrpLayout L;
  int o = 0;
  L.oM = o; o += N * ld;
  L.oU = o; o += N;
  L.oUN = o; o += N;
  L.oF = o; o += N;
  L.oB = o; o += N;
  L.oV = o; o += N;
  L.oTH = o; o += 3 * S;
  L.oKF = o; o += R;
  L.oKR = o; o += R;
  L.oQ = o; o += R;
  L.oDQT = o; o += energy ? R : 0;
  L.oQH = o; o += any_tb ? R : 0;
  L.oMT = o; o += any_tb ? R : 0;
  L.oRED = o; o += 8 * W + 2;
  L.total = (o + 1) & ~1;
  return L;
}

template <int W>
struct KrGrp {
  double* red;   // [8 W + 2] scratch
  int g, gl;     // group index in the block, thread index in the group
  __device__ __forceinline__ void sync() const {
    if (W == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(g + 1), "r"(32 * W) : "memory");
  }
  // sum of NV values over the group (fixed order: butterfly inside a warp, then warps in index order)
  template <int NV>
  __device__ __forceinline__ void sum(double (&x)[NV]) const {
#pragma unroll
    for (int i = 0; i < NV; ++i)
      for (int off = 16; off > 0; off >>= 1) x[i] += __shfl_xor_sync(0xffffffffu, x[i], off);
    if (W > 1) {
      const int w = gl >> 5;
      if ((gl & 31) == 0)
        for (int i = 0; i < NV; ++i) red[w * NV + i] = x[i];
      sync();
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        double s = red[i];
        for (int ww = 1; ww < W; ++ww) s += red[ww * NV + i];
        x[i] = s;
      }
      sync();
    }
  }
  // NaN-dropping maximum, the oracle's "if (x > m) m = x"
  __device__ __forceinline__ double max(double x) const {
    for (int off = 16; off > 0; off >>= 1) { const double y = __shfl_xor_sync(0xffffffffu, x, off); x = (y > x) ? y : x; }
    if (W > 1) {
      const int w = gl >> 5;
      if ((gl & 31) == 0) red[w] = x;
      sync();
      double m = red[0];
      for (int ww = 1; ww < W; ++ww) { const double y = red[ww]; m = (y > m) ? y : m; }
      x = m;
      sync();
    }
    return x;
  }
  __device__ __forceinline__ double min(double x) const { return -max(-x); }
  __device__ __forceinline__ bool all(bool p) const {
    int ok = __all_sync(0xffffffffu, p);
    if (W > 1) {
      const int w = gl >> 5;
      if ((gl & 31) == 0) red[w] = ok ? 1.0 : 0.0;
      sync();
      ok = 1;
      for (int ww = 0; ww < W; ++ww) ok = ok && (red[ww] != 0.0);
      sync();
    }
    return ok != 0;
  }
  // arg-max of (val, idx) with ties -> smallest idx; idx < 0 marks "no candidate"
  __device__ __forceinline__ int argmax(double val, int idx) const {
    for (int off = 16; off > 0; off >>= 1) {
      const double v2 = __shfl_xor_sync(0xffffffffu, val, off);
      const int i2 = __shfl_xor_sync(0xffffffffu, idx, off);
      if (i2 >= 0 && (idx < 0 || v2 > val || (v2 == val && i2 < idx))) { val = v2; idx = i2; }
    }
    if (W > 1) {
      const int w = gl >> 5;
      if ((gl & 31) == 0) { red[2 * w] = val; red[2 * w + 1] = (double)idx; }
      sync();
      val = red[0]; idx = (int)red[1];
      for (int ww = 1; ww < W; ++ww) {
        const double v2 = red[2 * ww];
        const int i2 = (int)red[2 * ww + 1];
        if (i2 >= 0 && (idx < 0 || v2 > val || (v2 == val && i2 < idx))) { val = v2; idx = i2; }
      }
      sync();
    }
    return idx;
  }
};

// thermo: thread <-> species
template <int W>
__device__ __forceinline__ void kr_grp_thermo(const KrNetDev& n, const KrGrpLayout& L, double* c, const KrGrp<W>& G,
                                              double T, double invT, double lnT) {
  for (int s = G.gl; s < n.S; s += 32 * W) {
    double g, u, ch;
    kr_thermo_species(n.nasa + 14 * s, n.T_mid[s], T, invT, lnT, g, u, ch);
    c[L.oTH + s] = g; c[L.oTH + n.S + s] = u; c[L.oTH + 2 * n.S + s] = ch;
  }
}

// reaction pass: thread <-> reaction.  Writes KF/KR (when computeK), Q (= q_r), DQT (= dq_r/dT), QH/MT for
// third-body reactions; returns this thread's partial sums of (q_ext/k_B) q_r and (q_ext/k_B) dq_r/dT.
template <bool ENERGY, int W>
__device__ __forceinline__ void kr_grp_reactions(const KrNetDev& n, const KrGrpLayout& L, double* c, const KrGrp<W>& G,
                                                 double Ncal, double invT, double lnT, double aux0,
                                                 const double* __restrict__ aux, long long cell, long long n_cells,
                                                 bool computeK, double& heat_sum, double& heat_dT) {
  const int S = n.S;
  heat_sum = 0.0; heat_dT = 0.0;
  for (int r = G.gl; r < n.R; r += 32 * W) {
    const int fl = n.flags[r];
    double kf, kr, dlf = 0.0, dlr = 0.0;
    if (computeK) {
      double ax = aux0;
      if ((fl & KR_DF_AUX) && n.auxi[r] > 0) ax = aux[(long long)n.auxi[r] * n_cells + cell];
      kr_rate_constants(n, r, fl, invT, lnT, ax, [&](int s) { return c[L.oTH + s]; },
                        [&](int s) { return c[L.oTH + S + s]; }, kf, kr, dlf, dlr);
      c[L.oKF + r] = kf; c[L.oKR + r] = kr;
    } else {
      kf = c[L.oKF + r]; kr = c[L.oKR + r];
    }
    double Pf = 1.0, Pr = 1.0;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const int s = n.sp[6 * r + k];
      if (s >= 0) {
        const double p = kr_ipow(Ncal * c[L.oU + s], n.nu[6 * r + k]);
        if (k < 3) Pf *= p; else Pr *= p;
      }
    }
    double Mtb = 1.0;
    const double qhat = kf * Pf - kr * Pr;
    if (fl & KR_DF_TB) {
      Mtb = 0.0;
      for (int s = 0; s < S; ++s) Mtb += n.tb_eff[r * S + s] * (Ncal * c[L.oU + s]);
      c[L.oQH + r] = qhat; c[L.oMT + r] = Mtb;
    }
    const double q = Mtb * qhat;
    c[L.oQ + r] = q;
    const double qk = n.any_qext ? n.qk[r] : 0.0;
    heat_sum += qk * q;
    if (ENERGY) {
      const double dqdT = Mtb * (kf * dlf * Pf - kr * dlr * Pr);
      c[L.oDQT + r] = dqdT;
      heat_dT += qk * dqdT;
    }
  }
}

// f rows (and the T column of J when wantJ): thread <-> species row, gather in reaction order
template <bool ENERGY, int W>
__device__ __forceinline__ void kr_grp_rows(const KrNetDev& n, const KrGrpLayout& L, double* c, const KrGrp<W>& G,
                                            double Ncal, bool wantJ) {
  for (int s = G.gl; s < n.S; s += 32 * W) {
    double ys = 0.0, jt = 0.0;
    for (int p = n.row_ptr[s]; p < n.row_ptr[s + 1]; ++p) {
      const int ent = n.row_ent[p];
      const int r = ent >> 8;
      const double dnu = (double)((ent & 255) - 128);
      ys += dnu * c[L.oQ + r];
      if (ENERGY) jt += dnu * c[L.oDQT + r];
    }
    c[L.oF + s] = ys / Ncal;
    if (ENERGY && wantJ) c[L.oM + s * n.ld + n.S] = jt / Ncal;
  }
}

// Jacobian columns (eq. 19): thread <-> column m.  Cval = sum_s y_s chat_s (energy equation only).
template <bool ENERGY, int W>
__device__ __forceinline__ void kr_grp_columns(const KrNetDev& n, const KrGrpLayout& L, double* c, const KrGrp<W>& G,
                                               double Ncal, double T, double Cval) {
  const int S = n.S, ld = n.ld;
  for (int m = G.gl; m < S; m += 32 * W) {
    for (int i = 0; i < n.N; ++i) c[L.oM + i * ld + m] = 0.0;
    double heat_dn = 0.0;
    const double nm = Ncal * c[L.oU + m];
    for (int p = n.col_ptr[m]; p < n.col_ptr[m + 1]; ++p) {
      const int ent = n.col_ent[p];
      const int r = ent >> 4, slot = ent & 15;
      const int fl = n.flags[r];
      double d;
      if (slot < 6) {
        const int base = (slot < 3) ? 0 : 3;
        double others = 1.0;
#pragma unroll
        for (int kk = 0; kk < 3; ++kk) {
          const int idx = base + kk;
          const int s2 = n.sp[6 * r + idx];
          if (idx != slot && s2 >= 0) others *= kr_ipow(Ncal * c[L.oU + s2], n.nu[6 * r + idx]);
        }
        const int e = n.nu[6 * r + slot];
        const double kk2 = (slot < 3) ? c[L.oKF + r] : -c[L.oKR + r];
        const double Mtb = (fl & KR_DF_TB) ? c[L.oMT + r] : 1.0;
        d = Mtb * (kk2 * (double)e * kr_ipow(nm, e - 1) * others);
      } else {
        d = n.tb_eff[r * S + m] * c[L.oQH + r];
      }
#pragma unroll
      for (int i = 0; i < 6; ++i) {
        const int s = n.sp[6 * r + i];
        if (s >= 0) c[L.oM + s * ld + m] += ((i < 3) ? -(double)n.nu[6 * r + i] : (double)n.nu[6 * r + i]) * d;
      }
      if (ENERGY && n.any_qext) heat_dn += n.qk[r] * d;
    }
    if (ENERGY) {
      double acc = 0.0;
      for (int s = 0; s < S; ++s) acc += c[L.oTH + S + s] * c[L.oM + s * ld + m];
      c[L.oM + S * ld + m] = (heat_dn - T * acc) / Cval;
    }
  }
}

// Full evaluation of f (and J) at U for the group.  Assumes thermo / KF / KR valid as the flags say.
template <bool ENERGY, int W>
__device__ __forceinline__ void kr_grp_eval(const KrNetDev& n, const KrGrpLayout& L, double* c, const KrGrp<W>& G,
                                            double Ncal, double T, double aux0, const double* __restrict__ aux,
                                            long long cell, long long n_cells, bool computeK, bool wantJ) {
  const int S = n.S;
  const double invT = 1.0 / T, lnT = (ENERGY || computeK) ? log(T) : 0.0;
  double red[3];
  kr_grp_reactions<ENERGY, W>(n, L, c, G, Ncal, invT, lnT, aux0, aux, cell, n_cells, computeK, red[0], red[1]);
  red[2] = 0.0;
  if (ENERGY)
    for (int s = G.gl; s < S; s += 32 * W) red[2] += c[L.oU + s] * c[L.oTH + 2 * S + s];
  if (ENERGY) G.sum(red);
  G.sync();
  const double heat_sum = red[0], heat_dT = red[1], Cval = red[2];
  kr_grp_rows<ENERGY, W>(n, L, c, G, Ncal, wantJ);
  if (wantJ) kr_grp_columns<ENERGY, W>(n, L, c, G, Ncal, T, Cval);
  G.sync();
  if (ENERGY) {
    double r2[3] = {0.0, 0.0, 0.0};
    for (int s = G.gl; s < S; s += 32 * W) {
      const double fs = c[L.oF + s], uh = c[L.oTH + S + s];
      r2[0] += uh * fs;
      r2[1] += c[L.oTH + 2 * S + s] * fs;
      if (wantJ) r2[2] += uh * c[L.oM + s * n.ld + S];
    }
    G.sum(r2);
    if (G.gl == 0) {
      c[L.oF + S] = (heat_sum / Ncal - T * r2[0]) / Cval;
      if (wantJ) c[L.oM + S * n.ld + S] = (heat_dT / Ncal - T * r2[2] - r2[1]) / Cval;
    }
    G.sync();
  }
}

// Step 7 for the group: rows <-> threads; B carried along; solution left in V.  Uniform return value.
template <int W>
__device__ __forceinline__ bool kr_grp_lu_solve(const KrGrpLayout& L, double* c, const KrGrp<W>& G, int N, int ld) {
  const int GT = 32 * W;
  double* M = c + L.oM;
  double* B = c + L.oB;
  double* V = c + L.oV;
  for (int j = 0; j < N; ++j) {
    double best = -1.0;
    int bi = -1;
    for (int i = G.gl; i < N; i += GT)
      if (i >= j) {
        const double t = fabs(M[i * ld + j]) / V[i];
        if (t > best) { best = t; bi = i; }
      }
    int imax = G.argmax(best, bi);
    if (imax < 0) imax = j;                       // every candidate was NaN: the pivot test below fails
    if (imax != j) {
      for (int k = j + G.gl; k < N; k += GT) {
        const double x = M[imax * ld + k]; M[imax * ld + k] = M[j * ld + k]; M[j * ld + k] = x;
      }
      if (G.gl == 0) {
        double x = V[imax]; V[imax] = V[j]; V[j] = x;
        x = B[imax]; B[imax] = B[j]; B[j] = x;
      }
      G.sync();
    }
    const double piv = M[j * ld + j];
    if (!(fabs(piv) >= 1e-300)) return false;
    const double bj = B[j];
    for (int i = G.gl; i < N; i += GT)
      if (i > j) {
        const double l = M[i * ld + j] / piv;
        for (int k = j + 1; k < N; ++k) M[i * ld + k] -= l * M[j * ld + k];
        B[i] -= l * bj;
      }
    G.sync();
  }
  for (int i = N - 1; i >= 0; --i) {               // back substitution, column oriented; solution -> V
    const double x = B[i] / M[i * ld + i];
    for (int r = G.gl; r < i; r += GT) B[r] -= M[r * ld + i] * x;
    if (G.gl == (i % GT)) V[i] = x;
    G.sync();
  }
  return true;
}

template <bool ENERGY, int W>
__global__ void __launch_bounds__(256) kr_grp_kernel(const KrNetDev n, const KrOptsDev o, const KrStepArgs a) {
  extern __shared__ double kr_sm[];
  const int S = n.S, N = n.N, K = o.max_newton, ld = n.ld;
  const int GT = 32 * W;
  const KrGrpLayout L = kr_grp_layout(N, S, n.R, ld, n.energy, n.any_tb, W);
  KrGrp<W> G;
  G.g = threadIdx.x / GT; G.gl = threadIdx.x % GT;
  double* c = kr_sm + (size_t)G.g * L.total;
  G.red = c + L.oRED;
  volatile long long* cellslot = (volatile long long*)(c + L.oRED + 8 * W);

  unsigned long long c_acc = 0, c_rej = 0, c_newton = 0, c_rate = 0, c_failed = 0;   // counted by thread 0 of the group

  for (;;) {
    if (G.gl == 0) *cellslot = (long long)atomicAdd(a.counter, 1ull);
    G.sync();
    const long long cell = *cellslot;
    G.sync();
    if (cell >= a.n_cells) break;

    // ---- step 1 -------------------------------------------------------------------------------
    int st = 0;
    double Tc = a.T[cell];
    if (Tc < n.T_lo) { Tc = n.T_lo; st |= KR_DST_T_CLAMPED; }
    if (Tc > n.T_hi) { Tc = n.T_hi; st |= KR_DST_T_CLAMPED; }
    const double Ncal = a.rho[cell] / KR_M_U;
    const double T_iso = Tc;
    const double aux0 = (n.n_aux > 0) ? a.aux[cell] : 0.0;
    for (int s = G.gl; s < S; s += GT) { const double x = a.y[cell * S + s]; c[L.oUN + s] = x; c[L.oU + s] = x; }
    if (ENERGY && G.gl == 0) { c[L.oUN + S] = Tc; c[L.oU + S] = Tc; }
    G.sync();
    double t = 0.0, h = a.dt;
    int n_acc = 0, n_rej = 0;
    {
      const double invT = 1.0 / Tc, lnT = log(Tc);
      bool haveK = false;
      if (!ENERGY) {
        if (n.any_rev) { kr_grp_thermo<W>(n, L, c, G, Tc, invT, lnT); G.sync(); }
        if (o.h0_mode != 1) {        // rate constants only (the h0 evaluation below would compute them as well)
          double hs, hd;
          kr_grp_reactions<ENERGY, W>(n, L, c, G, Ncal, invT, lnT, aux0, a.aux, cell, a.n_cells, true, hs, hd);
          G.sync();
        }
        c_rate++;
        haveK = false;
      }
      if (o.h0_mode == 1) {
        if (ENERGY) { kr_grp_thermo<W>(n, L, c, G, Tc, invT, lnT); G.sync(); c_rate++; }
        kr_grp_eval<ENERGY, W>(n, L, c, G, Ncal, Tc, aux0, a.aux, cell, a.n_cells, !haveK, false);
        double big = 0.0;
        for (int s = G.gl; s < S; s += GT) {
          const double x = fabs(c[L.oF + s]) / (fabs(c[L.oUN + s]) + o.y_floor);
          big = (x > big) ? x : big;
        }
        big = G.max(big);
        if (big > 0.0 && kr_finite(big)) h = fmin(a.dt, o.eta / big);
      }
    }
    const double h_floor = o.h_min_rel * fmin(h, a.dt);

    // ---- sub-step loop (steps 6-8) ----------------------------------------------------------------
    bool failed = false;
    for (;;) {
      const double rem = a.dt - t;
      bool last = false;
      if (h >= rem) { h = rem; last = true; }
      if (h < h_floor || n_acc + n_rej > o.max_substeps) { failed = true; break; }
      for (int i = G.gl; i < N; i += GT) c[L.oU + i] = c[L.oUN + i];
      G.sync();
      double e = __longlong_as_double(0x7ff0000000000000LL), e_prev = 0.0;
      int it = K + 1;
      bool ran = true;
      for (int k = 1; k <= K; ++k) {
        const double T = ENERGY ? c[L.oU + S] : T_iso;
        if (ENERGY) { kr_grp_thermo<W>(n, L, c, G, T, 1.0 / T, log(T)); G.sync(); c_rate++; }
        kr_grp_eval<ENERGY, W>(n, L, c, G, Ncal, T, aux0, a.aux, cell, a.n_cells, ENERGY, true);
        c_newton++;
        // G = u - u_n - h f (negated into B), M = I - h J, row scales v_i
        bool rows_ok = true;
        for (int i = G.gl; i < N; i += GT) {
          c[L.oB + i] = -(c[L.oU + i] - c[L.oUN + i] - h * c[L.oF + i]);
          double big = 0.0;
          for (int j = 0; j < N; ++j) {
            const double x = ((i == j) ? 1.0 : 0.0) - h * c[L.oM + i * ld + j];
            c[L.oM + i * ld + j] = x;
            big = fmax(big, fabs(x));
          }
          c[L.oV + i] = big;
          if (!(big > 0.0)) rows_ok = false;
        }
        rows_ok = G.all(rows_ok);
        G.sync();
        if (!rows_ok || !kr_grp_lu_solve<W>(L, c, G, N, ld)) { ran = false; break; }
        bool fin = true;
        double en = 0.0;
        for (int i = G.gl; i < N; i += GT) {
          const double dl = c[L.oV + i];
          const double x = c[L.oU + i] + dl;
          c[L.oU + i] = x;
          fin = fin && kr_finite(x);
          const double w = fabs(dl) / (o.rtol * fabs(x) + ((i < S) ? o.atol_y : o.atol_T));
          en = (w > en) ? w : en;
        }
        fin = G.all(fin);
        G.sync();
        if (!fin) { ran = false; break; }
        e = G.max(en);
        if (it == K + 1 && e <= 1.0) it = k;
        if (!o.fixed_newton) {
          if (e <= 1.0) break;
          if (k >= 2 && e > o.bail_ratio * e_prev) { ran = false; break; }
        }
        e_prev = e;
      }
      // step 8
      bool ok = ran && (e <= 1.0);
      if (ok) {
        double miny = __longlong_as_double(0x7ff0000000000000LL);
        for (int s = G.gl; s < S; s += GT) miny = fmin(miny, c[L.oU + s]);
        miny = G.min(miny);
        if (!(miny >= -o.neg_tol)) ok = false;
      }
      if (ok && ENERGY) {
        const double Tn = c[L.oU + S];
        if (!(Tn >= n.T_lo && Tn <= n.T_hi)) ok = false;
      }
      if (ok && kr_finite(o.chg_max)) {
        double chg = 0.0;
        for (int i = G.gl; i < N; i += GT) {
          const double den = (i < S) ? (fabs(c[L.oUN + i]) + o.chg_floor) : c[L.oUN + i];
          chg = fmax(chg, fabs(c[L.oU + i] - c[L.oUN + i]) / den);
        }
        chg = G.max(chg);
        if (!(chg <= o.chg_max)) ok = false;
      }
      if (ok) {
        n_acc++;
        for (int i = G.gl; i < N; i += GT) c[L.oUN + i] = c[L.oU + i];
        G.sync();
        if (last) break;
        t = t + h;
        if (it <= o.it_fast) h = h * o.grow_fast;
        else if (it <= o.it_mid) h = h * o.grow_mid;
      } else {
        n_rej++;
        st |= KR_DST_REJECTED;
        h = h * o.shrink;
        G.sync();
      }
    }
    c_acc += n_acc; c_rej += n_rej;
    if (failed) {                                               // R13: revert
      if (a.fail_list) { if (G.gl == 0) a.fail_list[atomicAdd(a.fail_count, 1ull)] = cell; }   // second attempt
      else { c_failed++; if (a.status && G.gl == 0) a.status[cell] = st | KR_DST_FAILED; }
      G.sync();
      continue;
    }
    // ---- step 9: finalise (stages 1-3, kr_post.cuh; serial in thread 0: O(E S) once per cell) + layout-out ------------------
    if (o.finalize && G.gl == 0) {
      st |= kr_postprocess(kr_post_lists(n), o.cons_tol, [&](int s) { return a.y[cell * n.S + s]; }, [&](int s) -> double& { return c[L.oUN + s]; });
      if (a.status) a.status[cell] = st;
    } else if (G.gl == 0 && a.status) {
      a.status[cell] = st;
    }
    G.sync();
    for (int s = G.gl; s < S; s += GT) a.y[cell * S + s] = c[L.oUN + s];
    if (ENERGY && G.gl == 0) a.T[cell] = c[L.oUN + S];
    G.sync();
  }
  if (G.gl == 0) {
    atomicAdd(a.stats + 0, c_acc); atomicAdd(a.stats + 1, c_rej); atomicAdd(a.stats + 2, c_newton);
    atomicAdd(a.stats + 3, c_newton); atomicAdd(a.stats + 4, c_rate); atomicAdd(a.stats + 5, c_failed);
  }
}
