// kr_wpc.cuh -- warp-per-cell solve kernel with the per-cell matrix in REGISTERS (13 <= N <= 64 in fp64; any
// N <= 64 in mixed precision).  Compiled at kr_network_create (NVRTC, sm_100a) with the sizes of the network
// as macros, so every register tile is exactly as large as the network needs:
//   KRW_N KRW_S KRW_R KRW_E KRW_ENERGY KRW_ANY_REV KRW_ANY_TB KRW_ANY_QEXT KRW_NAUX    the network
//   KRW_W      warps per cell (1 or 2)         KRW_TR  row groups inside a warp (4, 8 or 16; TC = 32 / TR)
//   KRW_RB     rows per thread (TR RB >= N)    KRW_CB  columns per thread (TC W CB >= N + 1)
//   KRW_MIXED  0: fp64 throughout   1: fp32 matrix + elimination, fp64 residuals, iterative refinement (R15)
//   KRW_CPB    cells per block                 KRW_MIN_BLOCKS  launch bound
//
// Work split of one Newton iteration (DESIGN.md steps 2-7) inside the group of 32 W threads that owns a cell:
//   thermo            : thread <-> species
//   rate constants, q : thread <-> reaction
//   Jacobian          : thread <-> ENTRY J[s][m]: every entry is the sum of host-built terms dnu_rs dq_r/dn_m, each a
//                       multiply chain over the cell's shared-memory block; the terms reach each thread as one
//                       coalesced stream (entries dealt longest first): no atomics, no read-modify-write of shared
//                       memory, fixed order (replaces PAPER.md:232), eq. 19 / eq. 20
//   elimination       : the matrix [I - hJ | -G] is spread over the threads as a TR x (TC W) grid of RB x CB
//                       REGISTER tiles (rows blocked, columns cyclic).  Column k: scaled-pivot search among the
//                       not yet used rows as a warp-wide integer maximum of pivot keys (REDUX), raw column, pivot
//                       value and pivot row published through shared memory, rank-1 update of every tile -- RB x CB
//                       independent FMAs per thread and step against RB + CB shared-memory loads.  Rows are never
//                       exchanged (implicit pivoting: a used row is marked); the update is applied to the used
//                       rows as well (Gauss-Jordan form of Algorithm 1's elimination), which
//                       removes the serial back substitution: after N columns row p_k holds x_k * pivot_k.
//   mixed precision   : J is assembled in fp32, rows are scaled to unit max-norm, the elimination runs in fp32 and
//                       its column vectors are kept (N^2 floats in the space J occupied); the linear residual
//                       r = -G - (I - hJ) d is formed in fp64 WITHOUT a stored fp64 matrix (J d is the analytic
//                       directional derivative, one pass over the reactions) and the correction is obtained by
//                       replaying the kept multipliers on r -- refinement until the correction is far below the
//                       Newton tolerance.
// Controller scalars are replicated in every thread and evolve identically.  Persistent: a group that finishes a
// cell pulls the next one from the global counter (a8).
#pragma once
#include "kr_tables.h"
#include "kr_math.cuh"
#include "kr_post.cuh"

#ifndef KRW_REF_MAX
#define KRW_REF_MAX 5          // most refinement passes per Newton iteration (mixed mode)
#endif

namespace krw {

constexpr int N = KRW_N, S = KRW_S, R = KRW_R, E = KRW_E;
constexpr int W = KRW_W, GT = 32 * KRW_W;
constexpr int TR = KRW_TR, TC = 32 / KRW_TR, RB = KRW_RB, CB = KRW_CB;
constexpr int NCG = TC * W;                 // column groups; column c belongs to group c % NCG, local index c / NCG
constexpr int LD = (N + 1) | 1;             // leading dimension of J in shared memory (elements)
constexpr int LTS = TR * RB + TR;           // stride of one multiplier vector (one pad element per row group)
constexpr bool ENERGY = KRW_ENERGY != 0, MIXED = KRW_MIXED != 0;
static_assert(TR * RB >= N, "row tiles do not cover N");
static_assert(NCG * CB >= N + 1, "column tiles do not cover N + 1");
static_assert(W == 1 || W == 2, "one or two warps per cell");

#if KRW_MIXED
typedef float MT;
#else
typedef double MT;
#endif

// ---- shared memory of one cell (byte offsets, all 8-byte aligned) ------------------------------------------------
constexpr int a8(int x) { return (x + 7) & ~7; }
constexpr int MAT_ELEMS = N * ((MIXED && LTS > LD) ? LTS : LD);   // J, later (mixed) the N multiplier vectors
constexpr int oU = 0;                                   // double[N]  iterate u^{k-1}
constexpr int oUN = oU + 8 * N;                         // double[N]  last accepted state
constexpr int oF = oUN + 8 * N;                         // double[N]  f(u)
constexpr int oB = oF + 8 * N;                          // double[N]  -G
constexpr int oX = oB + 8 * N;                          // double[N]  Newton update delta
constexpr int oRS = oX + 8 * N;                         // double[N]  residual of the linear system (mixed)
constexpr int oVI = oRS + 8 * N;                        // double[N]  1 / row scale
constexpr int oNN = oVI + 8 * N;                        // double[S+1] number densities n_s = Ncal y_s, then the constant 1
constexpr int oTH = oNN + 8 * (S + 1);                  // double[3S] ghat, uhat, chat
constexpr int oKF = oTH + 8 * 3 * S;                    // double[R]
constexpr int oKR = oKF + 8 * R;                        // double[R]
constexpr int oQ = oKR + 8 * R;                         // double[R]  q_r, later dq_r (mixed refinement)
constexpr int oDQT = oQ + 8 * R;                        // double[R]  dq_r/dT (energy)
constexpr int oQH = oDQT + (ENERGY ? 8 * R : 0);        // double[R]  k_f P' - k_r P'' (third body)
constexpr int oMT = oQH + (KRW_ANY_TB ? 8 * R : 0);     // double[R]  M_r
constexpr int oRED = oMT + (KRW_ANY_TB ? 8 * R : 0);    // double[8 W + 4] reduction scratch, cell slot, scalars
constexpr int oRP = oRED + 8 * (8 * W + 4);             // MT[N]      reciprocal pivots
constexpr int oUR = a8(oRP + int(sizeof(MT)) * N);      // MT[NCG CB] pivot row
constexpr int oLK = a8(oUR + int(sizeof(MT)) * NCG * CB);   // MT[2 LTS] multipliers of the current column (fp64 mode)
constexpr int oKOF = a8(oLK + int(sizeof(MT)) * 2 * LTS);   // int[TR RB] column in which row i was the pivot row
constexpr int oPOF = a8(oKOF + 4 * TR * RB);            // int[N]     pivot row of column k
constexpr int oPIV = a8(oPOF + 4 * N);                  // int[2]     pivot row of the current column (double buffered)
constexpr int oPVS = a8(oPIV + 8);                      // MT[2]      pivot value of the current column (double buffered)
constexpr int oMAT = a8(oPVS + 2 * int(sizeof(MT)));    // MT[MAT_ELEMS]
constexpr int CELL_BYTES = a8(oMAT + int(sizeof(MT)) * MAT_ELEMS);

#ifdef KRW_CELL_BYTES
static_assert(CELL_BYTES == KRW_CELL_BYTES, "host and device disagree on the shared-memory layout");
static_assert(oNN == 8 * KRW_I_NN && oKF == 8 * KRW_I_KF && oKR == 8 * KRW_I_KR, "host and device disagree on the vector offsets");
static_assert(!KRW_ANY_TB || (oQH == 8 * KRW_I_QH && oMT == 8 * KRW_I_MT), "host and device disagree on the third-body offsets");
#endif

struct Cell {
  char* base;
  __device__ __forceinline__ double* d(int off) const { return reinterpret_cast<double*>(base + off); }
  __device__ __forceinline__ MT* m(int off) const { return reinterpret_cast<MT*>(base + off); }
  __device__ __forceinline__ int* i(int off) const { return reinterpret_cast<int*>(base + off); }
};

// ---- the group of 32 W threads -----------------------------------------------------------------------------------
struct Grp {
  double* red;   // [8 W + 4]
  int g, gl;     // group index in the block, thread index in the group
  __device__ __forceinline__ void sync() const {
    if (W == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(g + 1), "r"(32 * W) : "memory");
  }
  template <int NV>
  __device__ __forceinline__ void sum(double (&x)[NV]) const {     // fixed order: butterfly, then warps in index order
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
  __device__ __forceinline__ double max(double x) const {          // NaN-dropping, the oracle's "if (x > m) m = x"
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
};

__device__ __forceinline__ bool finite(double x) { return fabs(x) <= 1.79769313486231570e308; }
__device__ __forceinline__ MT mt_rcp(MT x) {
#if KRW_MIXED
  return __frcp_rn(x);
#else
  return krs_rcp(x);
#endif
}

// ---- steps 2-3: thermo, thread <-> species (R7) --------------------------------------------------
__device__ __forceinline__ void thermo(const KrNetDev& n, const Cell& c, const Grp& G, double T, double invT, double lnT) {
  double* TH = c.d(oTH);
  const double T2 = T * T, T3 = T2 * T, T4 = T3 * T;
  for (int s = G.gl; s < S; s += GT) {
    const double* a = n.nasa + 14 * s + ((T <= n.T_mid[s]) ? 0 : 7);
    const double a0 = a[0], a1 = a[1], a2 = a[2], a3 = a[3], a4 = a[4], a5 = a[5], a6 = a[6];
    const double cp = a0 + a1 * T + a2 * T2 + a3 * T3 + a4 * T4;
    const double h = a0 + a1 * T * 0.5 + a2 * T2 * (1.0 / 3.0) + a3 * T3 * 0.25 + a4 * T4 * 0.2 + a5 * invT;
    const double sR = a0 * lnT + a1 * T + a2 * T2 * 0.5 + a3 * T3 * (1.0 / 3.0) + a4 * T4 * 0.25 + a6;
    TH[s] = h - sR; TH[S + s] = h - 1.0; TH[2 * S + s] = cp - 1.0;
  }
}

// ---- steps 3-4: thread <-> reaction.  Rate constants (eq. 16 with R4, detailed balance R5, unary R16/R17) when
// computeK, then q_r, dq_r/dT, and the third-body factors.  Number densities come from NN (filled by eval), the
// mass-action products from the host-built factor lists (powers expanded, the constant 1 for unused factors).
// Returns partial sums of (q_ext/k_B) q and (q_ext/k_B) dq/dT.
__device__ __forceinline__ void reactions(const KrNetDev& n, const Cell& c, const Grp& G, double invT, double lnT,
                                          double aux0, const double* __restrict__ aux, long long cell, long long n_cells,
                                          bool computeK, double& heat_sum, double& heat_dT) {
  double *NN = c.d(oNN), *TH = c.d(oTH), *KF = c.d(oKF), *KR = c.d(oKR), *Q = c.d(oQ);
  heat_sum = 0.0; heat_dT = 0.0;
  for (int r = G.gl; r < R; r += GT) {
    // every table value of the reaction is requested up front: independent loads, one exposed latency instead of a chain
    const int fl = __ldg(n.flags + r);
    const int2* fp = reinterpret_cast<const int2*>(n.fac + 6 * r);
    const int2 f01 = __ldg(fp), f23 = __ldg(fp + 1), f45 = __ldg(fp + 2);
    const double A_r = __ldg(n.A + r);
    const double qk = KRW_ANY_QEXT ? __ldg(n.qk + r) : 0.0;
    double beta = 0.0, Ea = 0.0, c0 = 0.0;
    int dn_tot = 0;
    int4 tg0 = make_int4(0, 0, 0, 0), tg1 = make_int4(0, 0, 0, 0);
    if (computeK) {
      beta = __ldg(n.beta + r); Ea = __ldg(n.Ea + r); c0 = __ldg(n.c0 + r);
      if (KRW_ANY_REV) {
        dn_tot = __ldg(n.dnu_tot + r);
        const int4* tp = reinterpret_cast<const int4*>(n.tgt + 8 * r);
        tg0 = __ldg(tp); tg1 = __ldg(tp + 1);
      }
    }
    double kf, kr = 0.0, dlf = 0.0, dlr = 0.0;
    if (computeK) {
      if (fl & KR_DF_CONST) kf = A_r;
      else if (fl & KR_DF_AUX) {
        const int ai = n.auxi[r];
        kf = A_r * (ai > 0 ? aux[(long long)ai * n_cells + cell] : aux0);
      } else {
        const double lnkf = c0 + beta * lnT - Ea * invT;
        kf = krs_exp(lnkf);
        dlf = (beta + Ea * invT) * invT;
        if (KRW_ANY_REV && (fl & KR_DF_REV)) {
          double sg = 0.0, su = 0.0;
          const int tg[8] = {tg0.x, tg0.y, tg0.z, tg0.w, tg1.x, tg1.y, tg1.z, tg1.w};
#pragma unroll
          for (int t = 0; t < 7; ++t)
            if (t < tg[0]) {
              const int e = tg[1 + t];
              const double cf = (double)((e >> 8) - 128);
              sg += cf * TH[e & 255];
              su += cf * TH[S + (e & 255)];
            }
          const double lnKc = -sg + (double)dn_tot * (n.ln_p0_kB - lnT);
          kr = krs_exp(lnkf - lnKc);
          dlr = dlf - su * invT;
        }
      }
      KF[r] = kf; KR[r] = kr;
    } else {
      kf = KF[r]; kr = KR[r];
    }
    const double Pf = NN[f01.x] * NN[f01.y] * NN[f23.x];
    const double Pr = NN[f23.y] * NN[f45.x] * NN[f45.y];
    double Mtb = 1.0;
    const double qhat = kf * Pf - kr * Pr;
    if (KRW_ANY_TB && (fl & KR_DF_TB)) {
      Mtb = 0.0;
      for (int s = 0; s < S; ++s) Mtb += n.tb_eff[r * S + s] * NN[s];
      c.d(oQH)[r] = qhat; c.d(oMT)[r] = Mtb;
    }
    const double q = Mtb * qhat;
    Q[r] = q;
    heat_sum += qk * q;
    if (ENERGY) {
      const double dqdT = Mtb * (kf * dlf * Pf - kr * dlr * Pr);
      c.d(oDQT)[r] = dqdT;
      heat_dT += qk * dqdT;
    }
  }
}

// ---- f rows (and the T column of J when wantJ): thread <-> species row, gather in reaction order (eq. 15, eq. 20)
__device__ __forceinline__ void rows(const KrNetDev& n, const Cell& c, const Grp& G, double invN, bool wantJ) {
  double *Q = c.d(oQ), *F = c.d(oF);
  MT* J = c.m(oMAT);
  for (int s = G.gl; s < S; s += GT) {
    double ys = 0.0, jt = 0.0;
    const int p1 = n.row_ptr[s + 1];
#pragma unroll 4
    for (int p = n.row_ptr[s]; p < p1; ++p) {
      const int ent = __ldg(n.row_ent + p);
      const int r = ent >> 8;
      const double dnu = (double)((ent & 255) - 128);
      ys += dnu * Q[r];
      if (ENERGY) jt += dnu * c.d(oDQT)[r];
    }
    F[s] = ys * invN;
    if (ENERGY && wantJ) J[s * LD + S] = (MT)(jt * invN);
  }
}

// ---- Jacobian (eq. 19), thread <-> ENTRY: J[s][m] = sum of its host-built terms dnu_rs dq_r/dn_m, each one multiply
// chain over the cell's shared-memory block; entries are dealt to the threads longest first, so the threads of a
// group finish together (column lists are very uneven: an abundant reactant sits in a third of the reactions).
// No read-modify-write of shared memory, no atomics, fixed order (replaces PAPER.md:232).  J was zeroed by eval().
__device__ __forceinline__ void entries(const KrNetDev& n, const Cell& c, const Grp& G) {
  const double* D = c.d(0);
  MT* J = c.m(oMAT);
  // {coef lo, coef hi, g0 | g1 << 16, g2 | g3 << 16}: one coalesced 16-byte load per thread and step, no dependent loads
  const uint4* terms = reinterpret_cast<const uint4*>(n.estream[W - 1]) + G.gl;
  const int* meta = n.emeta[W - 1] + G.gl;
  const int len = n.elen[W - 1];
  double acc = 0.0;
#pragma unroll 4
  for (int i = 0; i < len; ++i) {
    const uint4 t = __ldg(terms + i * GT);
    const int dst = __ldg(meta + i * GT);
    const double coef = __hiloint2double((int)t.y, (int)t.x);
    acc += coef * D[t.z & 0xffffu] * D[t.z >> 16] * D[t.w & 0xffffu] * D[t.w >> 16];
    if (dst >= 0) { J[dst] = (MT)acc; acc = 0.0; }
  }
}

// ---- T row of J (eq. 20 with the dropped dC/dy term, DESIGN.md step 5): thread <-> column m; row S holds the raw heat sum
__device__ __forceinline__ void trow(const Cell& c, const Grp& G, double T, double invC) {
  double* TH = c.d(oTH);
  MT* J = c.m(oMAT);
  for (int m = G.gl; m < S; m += GT) {
    double acc = 0.0;
    for (int s = 0; s < S; ++s) acc += TH[S + s] * (double)J[s * LD + m];
    J[S * LD + m] = (MT)(((double)J[S * LD + m] - T * acc) * invC);
  }
}

// ---- full evaluation of f (and J) at U.  Thermo / KF / KR valid as the flags say.  Leaves 1/C and sum_s chat_s f_s
// in the scalar slots (used by the matrix-free product of the mixed mode).
__device__ __forceinline__ void eval(const KrNetDev& n, const Cell& c, const Grp& G, double Ncal, double T, double aux0,
                                  const double* __restrict__ aux, long long cell, long long n_cells, bool computeK,
                                  bool wantJ) {
  const double invT = krs_rcp(T), lnT = (ENERGY || computeK) ? log(T) : 0.0;
  const double invN = krs_rcp(Ncal);
  double *U = c.d(oU), *TH = c.d(oTH), *F = c.d(oF), *NN = c.d(oNN);
  for (int s = G.gl; s <= S; s += GT) NN[s] = (s < S) ? Ncal * U[s] : 1.0;
  if (wantJ) {
    MT* Jz = c.m(oMAT);
    for (int i = G.gl; i < N * LD; i += GT) Jz[i] = (MT)0;
  }
  G.sync();
  double red[3];
  reactions(n, c, G, invT, lnT, aux0, aux, cell, n_cells, computeK, red[0], red[1]);
  red[2] = 0.0;
  if (ENERGY) {
    for (int s = G.gl; s < S; s += GT) red[2] += U[s] * TH[2 * S + s];
    G.sum(red);
  }
  G.sync();
  const double heat_sum = red[0], heat_dT = red[1];
  const double invC = ENERGY ? krs_rcp(red[2]) : 1.0;
  rows(n, c, G, invN, wantJ);
  if (wantJ) entries(n, c, G);
  G.sync();
  if (ENERGY && wantJ) { trow(c, G, T, invC); G.sync(); }
  if (ENERGY) {
    MT* J = c.m(oMAT);
    double r2[3] = {0.0, 0.0, 0.0};
    for (int s = G.gl; s < S; s += GT) {
      const double fs = F[s], uh = TH[S + s];
      r2[0] += uh * fs;
      r2[1] += TH[2 * S + s] * fs;
      if (wantJ) r2[2] += uh * (double)J[s * LD + S];
    }
    G.sum(r2);
    if (G.gl == 0) {
      F[S] = (heat_sum * invN - T * r2[0]) * invC;
      if (wantJ) J[S * LD + S] = (MT)((heat_dT * invN - T * r2[2] - r2[1]) * invC);
      G.red[8 * W + 1] = invC; G.red[8 * W + 2] = r2[1];
    }
    G.sync();
  }
}

#if KRW_MIXED
// ---- mixed mode: RS = B - (I - hJ) X in fp64 without a stored fp64 matrix.  J X is the analytic directional
// derivative of f along X with exactly the terms of DESIGN.md step 5: per reaction
//   dq_r = sum_terms (dq_r/dn_m) Ncal X_m  (the terms of the Jacobian program, grouped by reaction) + (dq_r/dT) X_T,
// then (J X)_s = (1/Ncal) sum_r dnu_rs dq_r and (J X)_T = [ (1/Ncal) sum_r (q_ext/k_B) dq_r - T sum_s uhat_s (J X)_s
// - (sum_s chat_s f_s) X_T ] / C.
__device__ __forceinline__ void residual(const KrNetDev& n, const Cell& c, const Grp& G, double Ncal, double T, double h) {
  const double* D = c.d(0);
  double *TH = c.d(oTH), *DQ = c.d(oQ), *X = c.d(oX), *B = c.d(oB), *RS = c.d(oRS);
  const double invN = krs_rcp(Ncal);
  const double dT = ENERGY ? X[S] : 0.0;
  double red[2] = {0.0, 0.0};
  for (int r = G.gl; r < R; r += GT) {
    double dq = 0.0;
    const int p1 = n.rprog_ptr[r + 1];
    for (int p = n.rprog_ptr[r]; p < p1; ++p) {
      const KrDEnt t = n.rprog[p];
      dq += t.coef * D[t.g0] * D[t.g1] * D[t.g2] * D[t.g3] * (Ncal * X[t.m]);
    }
    if (ENERGY) dq += c.d(oDQT)[r] * dT;
    DQ[r] = dq;
    if (ENERGY && KRW_ANY_QEXT) red[0] += n.qk[r] * dq;
  }
  G.sync();
  for (int s = G.gl; s < S; s += GT) {
    double js = 0.0;
    const int p1 = n.row_ptr[s + 1];
    for (int p = n.row_ptr[s]; p < p1; ++p) {
      const int ent = n.row_ent[p];
      js += (double)((ent & 255) - 128) * DQ[ent >> 8];
    }
    js *= invN;
    RS[s] = B[s] - (X[s] - h * js);
    if (ENERGY) red[1] += TH[S + s] * js;
  }
  if (ENERGY) {
    G.sum(red);
    if (G.gl == 0) {
      const double invC = G.red[8 * W + 1], scf = G.red[8 * W + 2];
      const double jT = (red[0] * invN - T * red[1] - scf * dT) * invC;
      RS[S] = B[S] - (dT - h * jT);
    }
  }
  G.sync();
}
#endif

// ---- step 7: elimination of [I - hJ | -G] in register tiles ------------------------------------------------------
struct Lane {
  int lane, wq, tr, tc, cg;
  __device__ __forceinline__ explicit Lane(int gl) : lane(gl & 31), wq(gl >> 5), tr((gl & 31) / TC), tc((gl & 31) % TC),
                                                     cg((gl >> 5) * TC + (gl & 31) % TC) {}
};
__device__ __forceinline__ int lidx(int row) { return row + row / RB; }     // padded index into a column vector

// executed by EVERY lane of the warp (the row index I is warp-uniform); only the stores are predicated on holding
// the row, so the warp never splits here
template <int I>
__device__ __forceinline__ void publish_row(const MT (&a)[RB][CB], MT (&sc)[RB], int kb, MT* UR, int cg, bool holds) {
#pragma unroll
  for (int j = 0; j < CB; ++j)
    if (j >= kb) { if (holds) UR[j * NCG + cg] = a[I][j]; }
  sc[I] = holds ? (MT)-1 : sc[I];            // the row is used: never a pivot candidate again
}

#define KRW_PUB_CASE(I) \
  case I: if constexpr (I < RB) publish_row<(I < RB ? I : 0)>(a, sc, kb, UR, L.cg, holds); break;

// Pivot keys: the bits of |a| / scale with the row index in the 6 low bits, so that an integer maximum gives the scaled
// pivot of Algorithm 1 and its tie rule (smallest row).  Candidates closer than 2^-46 (fp64) / 2^-17 (fp32) relative
// count as tied; used rows carry a negative scale and lose against every candidate.

// Pass A (thread <-> row): B = -(U - UN - h F), row scales of I - hJ.  Pass B: tiles.  Then N elimination columns.
// On success X holds the solution of (I - hJ) X = B; in mixed mode the column vectors, reciprocal pivots and the row
// order stay in shared memory for replay().  Uniform return value (false: zero row, non-finite entry or no pivot).
__device__ __forceinline__ bool eliminate(const Cell& c, const Grp& G, double h) {
  const Lane L(G.gl);
  double *U = c.d(oU), *UN = c.d(oUN), *F = c.d(oF), *B = c.d(oB), *VI = c.d(oVI), *X = c.d(oX);
  MT* J = c.m(oMAT);
  const MT hm = (MT)h;
  // Tiles of [I - hJ | -G] straight from J; the row scales (max-norm of each row, Algorithm 1's implicit scaling) are
  // reduced from the tiles themselves: shuffles across the column groups of a warp, shared memory between two warps.
  MT a[RB][CB];
  MT sc[RB];                                  // > 0: 1 / row scale of a candidate row;  < 0: used or padding row
  MT big[RB];
  bool fin = true;
  constexpr int cgN = N % NCG;                // the column group that holds the right-hand side
#pragma unroll
  for (int i = 0; i < RB; ++i) {
    const int row = L.tr * RB + i;
    const bool rin = row < N;
    big[i] = (MT)0;
#pragma unroll
    for (int j = 0; j < CB; ++j) {
      const int col = j * NCG + L.cg;
      MT x = (MT)0;
      if (rin && col < N) {
        x = ((row == col) ? (MT)1 : (MT)0) - hm * J[row * LD + col];
        const MT ax = fabs(x);
        big[i] = (ax > big[i]) ? ax : big[i];
        fin = fin && (ax <= (MT)(MIXED ? 3.0e38 : 1.7e308));      // false for inf and NaN
      } else if (rin && col == N) {
        const double bb = -(U[row] - UN[row] - h * F[row]);
        B[row] = bb;
        x = (MT)bb;
      }
      a[i][j] = x;
    }
  }
#pragma unroll
  for (int off = 1; off < TC; off <<= 1) {
#pragma unroll
    for (int i = 0; i < RB; ++i) {
      const MT y = __shfl_xor_sync(0xffffffffu, big[i], off);
      big[i] = (y > big[i]) ? y : big[i];
    }
  }
  if (W > 1) {                                // warp 0 leaves its partial maxima in RS, warp 1 in X (both free here)
    double* part = (L.wq == 0) ? c.d(oRS) : X;
    if (L.tc == 0) {
#pragma unroll
      for (int i = 0; i < RB; ++i)
        if (L.tr * RB + i < N) part[L.tr * RB + i] = (double)big[i];
    }
    G.sync();
#pragma unroll
    for (int i = 0; i < RB; ++i)
      if (L.tr * RB + i < N) {
        const MT y0 = (MT)c.d(oRS)[L.tr * RB + i], y1 = (MT)X[L.tr * RB + i];
        big[i] = (y0 > y1) ? y0 : y1;
      }
  }
  bool rows_ok = fin;
#pragma unroll
  for (int i = 0; i < RB; ++i) {
    const int row = L.tr * RB + i;
    const bool rin = row < N;
    const bool ok = big[i] > (MT)(MIXED ? 1e-30 : 1e-300);
    rows_ok = rows_ok && (ok || !rin);
    const double vi = (rin && ok) ? krs_rcp((double)big[i]) : 0.0;
    sc[i] = rin ? (MIXED ? (MT)1 : (MT)vi) : (MT)-1;
    if (rin && L.cg == 0) VI[row] = vi;
    if (MIXED) {
#pragma unroll
      for (int j = 0; j < CB; ++j) a[i][j] *= (MT)vi;
    }
  }
  rows_ok = G.all(rows_ok);
  G.sync();                                   // J is dead from here on: the mixed mode reuses its space
  if (!rows_ok) return false;

  MT* UR = c.m(oUR);
  MT* RP = c.m(oRP);
  MT* PVS = c.m(oPVS);
  int* PIV = c.i(oPIV);
  int* KOF = c.i(oKOF);
  int* POF = c.i(oPOF);
  bool fail = false;                          // uniform; no early exit from the column loop (keeps the warp converged)
#pragma unroll
  for (int kb = 0; kb < CB; ++kb) {
    for (int kc = 0; kc < NCG; ++kc) {
      const int k = kb * NCG + kc;
      if (k >= N) break;
      MT* Lk = MIXED ? (c.m(oMAT) + k * LTS) : (c.m(oLK) + (k & 1) * LTS);
      int p;
      if (W == 1 || L.wq == kc / TC) {        // the warp that holds column k
        const bool mine = (L.tc == kc % TC);
        // scaled pivot search (Algorithm 1): the warp-wide integer maximum (REDUX) of the candidates' keys.  fp64: the
        // high words first, then among the rows that share the largest high word the low words with the row index in
        // the 6 low bits -- together the 64-bit lexicographic maximum, exact to 2^-46, ties -> smallest row.
        const int rowbase = L.tr * RB;
#if KRW_MIXED
        int key = -2147483647 - 1;
#pragma unroll
        for (int i = 0; i < RB; ++i) {
          const MT v = a[i][kb];
          if (mine) Lk[rowbase + i + L.tr] = v;                      // column k as it stands (the multipliers x pivot)
          const int ki = (__float_as_int(fabsf(v) * sc[i]) | 63) - (rowbase + i);
          key = (ki > key) ? ki : key;
        }
        key = __reduce_max_sync(0xffffffffu, mine ? key : (-2147483647 - 1));
        p = (key >= 0) ? (63 - (key & 63)) : -1;
#else
        int hi[RB], hmax = -2147483647 - 1;
        unsigned lo[RB];
#pragma unroll
        for (int i = 0; i < RB; ++i) {
          const MT v = a[i][kb];
          if (mine) Lk[rowbase + i + L.tr] = v;                      // column k as it stands (the multipliers x pivot)
          const double t = fabs(v) * sc[i];
          hi[i] = __double2hiint(t); lo[i] = (unsigned)__double2loint(t);
          hmax = (hi[i] > hmax) ? hi[i] : hmax;
        }
        const int H = __reduce_max_sync(0xffffffffu, mine ? hmax : (-2147483647 - 1));
        unsigned lk = 0u;
#pragma unroll
        for (int i = 0; i < RB; ++i) {
          const unsigned ki = (lo[i] | 63u) - (unsigned)(rowbase + i);
          lk = (mine && hi[i] == H && ki > lk) ? ki : lk;
        }
        const unsigned Lw = __reduce_max_sync(0xffffffffu, lk);
        p = (H >= 0) ? (63 - (int)(Lw & 63u)) : -1;
#endif
        if (mine && p >= 0 && p / RB == L.tr) {                     // the lane that holds a[p][k]
          const int ix = p + L.tr;
          PVS[k & 1] = Lk[ix];
          Lk[ix] = (MT)0;                                            // row p itself is not updated
          if (W > 1) PIV[k & 1] = p;
        }
        if (W > 1 && p < 0 && L.lane == 0) PIV[k & 1] = -1;
      }
      if (W > 1) { G.sync(); p = PIV[k & 1]; }
      fail = fail || (p < 0);
      if (G.gl == 0) POF[k] = p;
      const int trp = (p >= 0) ? p / RB : 0, ip = (p >= 0) ? p - trp * RB : -1;
      {                                       // the lanes that hold row p publish it and retire it
        const bool holds = (L.tr == trp);
        switch (ip) {
          KRW_PUB_CASE(0) KRW_PUB_CASE(1) KRW_PUB_CASE(2) KRW_PUB_CASE(3) KRW_PUB_CASE(4) KRW_PUB_CASE(5) KRW_PUB_CASE(6)
          KRW_PUB_CASE(7) KRW_PUB_CASE(8) KRW_PUB_CASE(9) KRW_PUB_CASE(10) KRW_PUB_CASE(11) KRW_PUB_CASE(12)
          KRW_PUB_CASE(13) KRW_PUB_CASE(14) KRW_PUB_CASE(15) KRW_PUB_CASE(16) KRW_PUB_CASE(17) KRW_PUB_CASE(18)
          KRW_PUB_CASE(19) KRW_PUB_CASE(20) KRW_PUB_CASE(21)
          default: break;
        }
      }
      __syncwarp();
      const MT pv = PVS[k & 1];
      const bool pok = (fabs(pv) >= (MT)(MIXED ? 1e-30 : 1e-300)) && (fabs(pv) <= (MT)(MIXED ? 3.0e38 : 1.7e308));
      fail = fail || !pok;
      const MT rp = mt_rcp(pok ? pv : (MT)1);
      if (L.cg == 0 && L.tr == 0) RP[k] = rp;
      MT l[RB], u[CB];
#pragma unroll
      for (int i = 0; i < RB; ++i) l[i] = Lk[L.tr * RB + i + L.tr] * rp;
#pragma unroll
      for (int j = 0; j < CB; ++j)
        if (j >= kb) u[j] = UR[j * NCG + L.cg];
      if (L.cg <= kc) u[kb] = (MT)0;          // columns <= k of this block are finished
#pragma unroll
      for (int j = 0; j < CB; ++j)
        if (j >= kb) {
#pragma unroll
          for (int i = 0; i < RB; ++i) a[i][j] = fma(-l[i], u[j], a[i][j]);
        }
    }
  }
  G.sync();
  if (fail) return false;
  for (int k = G.gl; k < N; k += GT) KOF[POF[k]] = k;      // the column in which each row was the pivot row
  G.sync();
  constexpr int jN = N / NCG;                 // the right-hand-side column
  if (L.cg == cgN) {
#pragma unroll
    for (int i = 0; i < RB; ++i) {
      const int row = L.tr * RB + i;
      if (row < N) { const int k = KOF[row]; X[k] = (double)a[i][jN] * (double)RP[k]; }
    }
  }
  G.sync();
  return true;
}
#undef KRW_PUB_CASE

#if KRW_MIXED
// ---- mixed mode: correction d = (I - hJ)^-1 RS from the kept multipliers (2 N^2 fp32 flops), X += d.
// Each warp replays all rows (lane <-> rows lane, lane + 32): no traffic between warps.  Returns the weighted
// max-norms of the correction and of the corrected update, in units of the Newton tolerance (step 6's e_k).
__device__ __forceinline__ void replay(const Cell& c, const Grp& G, const KrOptsDev& o, double& wD, double& wX) {
  constexpr int NRL = (N + 31) / 32;
  const int lane = G.gl & 31;
  double *RS = c.d(oRS), *VI = c.d(oVI), *X = c.d(oX), *U = c.d(oU);
  const MT* LT = c.m(oMAT);
  const MT* RP = c.m(oRP);
  const int *POF = c.i(oPOF), *KOF = c.i(oKOF);
  float r[NRL];
#pragma unroll
  for (int q = 0; q < NRL; ++q) {
    const int row = lane + 32 * q;
    r[q] = (row < N) ? (float)(RS[row] * VI[row]) : 0.0f;
  }
  for (int k = 0; k < N; ++k) {
    const int p = POF[k];
    float mine = r[0];
#pragma unroll
    for (int q = 1; q < NRL; ++q) mine = ((p >> 5) == q) ? r[q] : mine;
    const float rp = __shfl_sync(0xffffffffu, mine, p & 31) * RP[k];   // r_p / pivot_k
#pragma unroll
    for (int q = 0; q < NRL; ++q) {
      const int row = lane + 32 * q;
      if (row < N) r[q] = fmaf(-LT[k * LTS + lidx(row)], rp, r[q]);       // column k (zero at row p) times r_p / pivot_k
    }
  }
  double xn[NRL];
  int kk[NRL];
  double wd = 0.0, wx = 0.0;
#pragma unroll
  for (int q = 0; q < NRL; ++q) {
    const int row = lane + 32 * q;
    kk[q] = -1; xn[q] = 0.0;
    if (row < N) {
      const int k = KOF[row];
      const double d = (double)(r[q] * RP[k]);
      const double x = X[k] + d;
      const double wgt = o.rtol * fabs(U[k] + x) + ((k < S) ? o.atol_y : o.atol_T);
      const double a = fabs(d) / wgt, b = fabs(x) / wgt;
      wd = (a > wd || !(a == a)) ? a : wd;      // NaN sticks
      wx = (b > wx) ? b : wx;
      kk[q] = k; xn[q] = x;
    }
  }
  for (int off = 16; off > 0; off >>= 1) {
    const double y = __shfl_xor_sync(0xffffffffu, wd, off); wd = (y > wd || !(y == y)) ? y : wd;
    const double z = __shfl_xor_sync(0xffffffffu, wx, off); wx = (z > wx) ? z : wx;
  }
  if (W > 1) G.sync();                         // every warp has read X
  if (G.gl < 32) {
#pragma unroll
    for (int q = 0; q < NRL; ++q)
      if (kk[q] >= 0) X[kk[q]] = xn[q];
  }
  G.sync();
  wD = wd; wX = wx;
}
#endif

}  // namespace krw

extern "C" __global__ void __launch_bounds__(32 * KRW_W * KRW_CPB, KRW_MIN_BLOCKS)
kr_wpc_kernel(const KrNetDev n, const KrOptsDev o, const KrStepArgs a) {
  using namespace krw;
  extern __shared__ __align__(16) char kr_sm_raw[];
  const int K = o.max_newton;
  Grp G;
  Cell c;
#if KRW_CPB == 1
  G.g = 0; G.gl = threadIdx.x;                // one cell per block: every shared-memory offset is a compile-time constant
  c.base = kr_sm_raw;
#else
  G.g = threadIdx.x / GT; G.gl = threadIdx.x % GT;
  c.base = kr_sm_raw + (size_t)G.g * CELL_BYTES;
#endif
  G.red = c.d(oRED);
  volatile long long* cellslot = (volatile long long*)(c.d(oRED) + 8 * W);
  double *U = c.d(oU), *UN = c.d(oUN), *F = c.d(oF), *X = c.d(oX);

  unsigned long long c_acc = 0, c_rej = 0, c_newton = 0, c_rate = 0, c_failed = 0, c_ref = 0;   // thread 0 of the group
  unsigned long long c_disc = 0;        // Newton iterations of fp32 attempts that were handed to the fp64 kernel (not algorithmic work)

  for (;;) {
    if (G.gl == 0) {
      long long idx = (long long)atomicAdd(a.counter, 1ull);
      if (a.list) idx = (idx < (long long)*a.list_count) ? a.list[idx] : a.n_cells;
      *cellslot = idx;
    }
    G.sync();
    const long long cell = *cellslot;
    G.sync();
    if (cell >= a.n_cells) break;

    // ---- step 1: layout-in, clamp, first sub-step -------------------------------------------------
    const unsigned long long s_newton = c_newton, s_rate = c_rate, s_ref = c_ref;     // counters at the start of this cell
    int st = a.list ? a.list_flag : 0;
    double Tc = a.T[cell];
    if (Tc < n.T_lo) { Tc = n.T_lo; st |= KR_DST_T_CLAMPED; }
    if (Tc > n.T_hi) { Tc = n.T_hi; st |= KR_DST_T_CLAMPED; }
    const double Ncal = a.rho[cell] * (1.0 / KR_M_U);
    const double T_iso = Tc;
    const double aux0 = (KRW_NAUX > 0) ? a.aux[cell] : 0.0;
    for (int s = G.gl; s < S; s += GT) { const double x = a.y[cell * S + s]; UN[s] = x; U[s] = x; }
    if (ENERGY && G.gl == 0) { UN[S] = Tc; U[S] = Tc; }
    G.sync();
    double t = 0.0, h = a.dt, h_floor = o.h_min_rel * a.dt;
    int n_acc = 0, n_rej = 0;
    // The first pass of a cell through the evaluation below is its preliminary evaluation: rate constants of an
    // isothermal cell, f(u_in) for the first sub-step (step 1, h0_mode 1).  One call site keeps the kernel small.
    bool prelim = (o.h0_mode == 1) || !ENERGY || (a.cost_out != nullptr);
    if (!prelim) { h = h * o.h0_scale; h_floor = o.h_min_rel * fmin(h, a.dt); }

    // ---- sub-step loop (steps 6-8) -------------------------------------------------------------------------------
    bool failed = false, handoff = false;
    for (;;) {
      bool last = false;
      if (!prelim) {
        const double rem = a.dt - t;
        if (h >= rem) { h = rem; last = true; }
        if (h < h_floor || n_acc + n_rej > o.max_substeps) { failed = true; break; }
        for (int i = G.gl; i < N; i += GT) U[i] = UN[i];
        G.sync();
      }
      double e = __longlong_as_double(0x7ff0000000000000LL), e_prev = 0.0;
      int it = K + 1;
      bool ran = true, was_prelim = false;
      for (int k = 1; k <= K; ++k) {
        const double T = ENERGY ? U[S] : T_iso;
        if (ENERGY || (prelim && KRW_ANY_REV)) { thermo(n, c, G, T, krs_rcp(T), log(T)); G.sync(); }
        if ((ENERGY || prelim) && !a.cost_out) c_rate++;
        eval(n, c, G, Ncal, T, aux0, a.aux, cell, a.n_cells, ENERGY || prelim, !prelim);
        if (prelim) {
          if (o.h0_mode == 1 || a.cost_out) {
            double big = 0.0;
            for (int s = G.gl; s < S; s += GT) {
              const double x = fabs(F[s]) / (fabs(UN[s]) + o.y_floor);
              big = (x > big) ? x : big;
            }
            big = G.max(big);
            if (big > 0.0 && finite(big)) h = fmin(a.dt, o.eta / big);
          }
          h = h * o.h0_scale;
          h_floor = o.h_min_rel * fmin(h, a.dt);
          prelim = false; was_prelim = true;
          break;
        }
        c_newton++;
        if (!eliminate(c, G, h)) { ran = false; if (MIXED) handoff = a.retry_list != nullptr; break; }
#if KRW_MIXED
        {                                        // iterative refinement on the fp64 residual of the linear system
          bool done = false;
          double wprev = __longlong_as_double(0x7ff0000000000000LL);
          for (int ref = 0; ref < KRW_REF_MAX; ++ref) {
            residual(n, c, G, Ncal, T, h);
            double wD, wX;
            replay(c, G, o, wD, wX);
            c_ref++;
            if (!(wD == wD) || !finite(wD)) break;
            if (wD <= 1e-4 || wD <= 1e-9 * wX) { done = true; break; }
            if (wD > 0.25 * wprev) break;          // not contracting: fp32 does not resolve this matrix
            wprev = wD;
          }
          if (!done) { handoff = a.retry_list != nullptr; ran = false; break; }
        }
#endif
        bool fin = true;
        double en = 0.0;
        for (int i = G.gl; i < N; i += GT) {
          const double dl = X[i];
          const double x = U[i] + dl;
          U[i] = x;
          fin = fin && finite(x);
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
      if (handoff) break;
      if (was_prelim) {
        if (a.cost_out) { handoff = true; break; }   // cost pass: the key is the first sub-step
        continue;
      }
      // step 8: accept / reject
      bool ok = ran && (e <= 1.0);
      if (ok) {
        double miny = __longlong_as_double(0x7ff0000000000000LL);
        for (int s = G.gl; s < S; s += GT) miny = fmin(miny, U[s]);
        miny = G.min(miny);
        if (!(miny >= -o.neg_tol)) ok = false;
      }
      if (ok && ENERGY) {
        const double Tn = U[S];
        if (!(Tn >= n.T_lo && Tn <= n.T_hi)) ok = false;
      }
      if (ok && finite(o.chg_max)) {
        double chg = 0.0;
        for (int i = G.gl; i < N; i += GT) {
          const double den = (i < S) ? (fabs(UN[i]) + o.chg_floor) : UN[i];
          chg = fmax(chg, fabs(U[i] - UN[i]) / den);
        }
        chg = G.max(chg);
        if (!(chg <= o.chg_max)) ok = false;
      }
      if (ok) {
        n_acc++;
        for (int i = G.gl; i < N; i += GT) UN[i] = U[i];
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
    if (handoff && a.cost_out) {
      if (G.gl == 0) a.cost_out[cell] = (float)h;
      G.sync();
      continue;
    }
    if (handoff) {            // the caller's buffers were never written: the fp64 kernel redoes this cell from its input
      c_disc += c_newton - s_newton;                              // the abandoned attempt is not counted as work of the step
      c_newton = s_newton; c_rate = s_rate; c_ref = s_ref;
      if (G.gl == 0) a.retry_list[atomicAdd(a.retry_count, 1ull)] = cell;
      G.sync();
      continue;
    }
    c_acc += n_acc; c_rej += n_rej;
    if (failed) {                                                 // R13: revert (the caller's buffers were never written)
      if (a.fail_list) { if (G.gl == 0) a.fail_list[atomicAdd(a.fail_count, 1ull)] = cell; }   // second attempt
      else { c_failed++; if (a.status && G.gl == 0) a.status[cell] = st | KR_DST_FAILED; }
      G.sync();
      continue;
    }
    // ---- step 9: finalise (PAPER.md:212-216 stages 1-3, kr_post.cuh; serial in thread 0, once per cell) + layout-out ----
    if (o.finalize && G.gl == 0) {
      st |= kr_postprocess(kr_post_lists(n), o.cons_tol, [&](int s) { return a.y[cell * S + s]; }, [&](int s) -> double& { return UN[s]; });
      if (a.status) a.status[cell] = st;
    } else if (G.gl == 0 && a.status) {
      a.status[cell] = st;
    }
    G.sync();
    for (int s = G.gl; s < S; s += GT) a.y[cell * S + s] = UN[s];
    if (ENERGY && G.gl == 0) a.T[cell] = UN[S];
    G.sync();
  }
  if (G.gl == 0) {
    atomicAdd(a.stats + 0, c_acc); atomicAdd(a.stats + 1, c_rej); atomicAdd(a.stats + 2, c_newton);
    atomicAdd(a.stats + 3, c_newton); atomicAdd(a.stats + 4, c_rate); atomicAdd(a.stats + 5, c_failed);
    if (c_ref) atomicAdd(a.stats + 6, c_ref);
    if (c_disc) atomicAdd(a.stats + 13, c_disc);
  }
}
