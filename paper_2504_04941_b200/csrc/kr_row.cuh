// kr_row.cuh -- warp-per-cell solve kernel with ONE MATRIX ROW PER LANE (2 <= N <= 64, fp64).  Compiled at
// kr_network_create (NVRTC, sm_100a) with the sizes of the network as macros:
//   KRR_N KRR_S KRR_R KRR_E KRR_ENERGY KRR_ANY_REV KRR_ANY_TB KRR_ANY_QEXT KRR_NAUX    the network
//   KRR_W          warps per cell: 1 (N <= 34) or 2 (N <= 64)
//   KRR_MIN_BLOCKS launch bound; KRR_CELL_BYTES shared memory of one cell (checked against the layout below)
//
// Work split of one Newton iteration (DESIGN.md steps 2-7) inside the group of 32 W threads that owns a cell:
//   thermo            : thread <-> species
//   rate constants, q : thread <-> reaction
//   Jacobian          : thread <-> ENTRY J[s][m], host-built term streams, no atomics (replaces PAPER.md:232), eq. 19 / 20
//   elimination       : thread i holds ROW i of the augmented system in registers (N + 1 doubles); rows beyond 32 W
//                       (at most two: N = 33, 34 on one warp) are held spread over the lanes, element j in lane j % 32.
//                       Column k of Algorithm 1: every lane forms the scaled candidate of its row
//                       from ONE register, the warp-wide integer maximum of the candidates' bit patterns (REDUX) names the
//                       pivot row, the lane that holds it writes its row to shared memory once, every lane reads it
//                       back as a broadcast and applies the rank-1 update to its own row: N - k independent FMAs per
//                       lane against (N - k) / 2 broadcast 16-byte loads, one warp-level sync per column, no shuffles,
//                       no dynamic register indexing (the column loop is rolled and the row shifts by one register per
//                       column, see struct Elim; a used row is marked, and the update is applied to used rows as well --
//                       the Gauss-Jordan form -- so that after N columns row p_k holds x_k * pivot_k in its first
//                       register and no substitution pass is needed).  The system that is
//                       eliminated is step 6's (I - hJ) delta = -G multiplied through by -1/h, (J - I/h) delta = G/h:
//                       same pivots under implicit row scaling, same solution, and the rows of J load into registers
//                       as they are.
// Controller scalars are replicated in every thread and evolve identically.  Persistent: a group that finishes a
// cell pulls the next one from the global counter (a8).
#pragma once
#include "kr_tables.h"
#include "kr_math.cuh"
#include "kr_post.cuh"

namespace krr {

constexpr int N = KRR_N, S = KRR_S, R = KRR_R, E = KRR_E;
constexpr int W = KRR_W, GT = 32 * KRR_W;
constexpr bool ENERGY = KRR_ENERGY != 0;
constexpr int NR = (N < GT) ? N : GT;       // rows held one per thread (thread i <-> row i)
constexpr int XR = N - NR;                  // rows held spread over the lanes of the (single) warp
constexpr int NC = N + 1;                   // columns of the augmented system: N matrix columns + the right-hand side
constexpr int NC2 = (NC + 1) / 2;           // ... in pairs (16-byte shared-memory accesses)
constexpr int XQ = (NC + 31) / 32;          // elements of a spread row per lane
constexpr int LDJ = NC + ((2 - NC % 4) + 4) % 4;   // row stride of J: >= N + 1 and = 2 mod 4, so that the 16-byte row loads of
                                                   // 8 consecutive lanes fall into 8 different bank groups
static_assert(W == 1 || W == 2, "one or two warps per cell");
static_assert(XR >= 0 && XR <= 2 && (XR == 0 || W == 1), "at most two spread rows, on one warp only");
static_assert(N <= 64, "the pivot key keeps the row index in 6 bits");
static_assert(LDJ % 4 == 2 && LDJ >= NC, "row stride");

// ---- shared memory of one cell (byte offsets; everything is a double unless noted) ----------------------------------
constexpr int a16(int x) { return (x + 15) & ~15; }
constexpr int oU = 0;                                   // [N]  iterate u^{k-1}
constexpr int oUN = oU + 8 * N;                         // [N]  last accepted state
constexpr int oX = oUN + 8 * N;                         // [N]  Newton update delta
constexpr int oNN = oX + 8 * N;                         // [S+1] number densities n_s = Ncal y_s, then the constant 1
constexpr int oTH = oNN + 8 * (S + 1);                  // [3S] ghat, uhat, chat
constexpr int oKF = oTH + 8 * 3 * S;                    // [R]
constexpr int oKR = oKF + 8 * R;                        // [R]
constexpr int oQ = oKR + (KRR_ANY_REV ? 8 * R : 0);     // [R]  q_r (KR exists only when some reaction is reversible)
constexpr int oDQT = oQ + 8 * R;                        // [R]  dq_r/dT (energy)
constexpr int oQH = oDQT + (ENERGY ? 8 * R : 0);        // [R]  k_f P' - k_r P'' (third body)
constexpr int oMT = oQH + (KRR_ANY_TB ? 8 * R : 0);     // [R]  M_r
constexpr int oRED = oMT + (KRR_ANY_TB ? 8 * R : 0);    // [8 W + 4] reduction scratch, cell slot, scalars
constexpr int oPK = oRED + 8 * (8 * W + 4);             // [W][12] per-warp parking slots of the controller state + [6] counters
constexpr int oKEY = oPK + 8 * (12 * W + 6);            // Key[2][W] best pivot keys of the two warps (double buffered; W = 2 only)
#ifndef KRR_RU
#define KRR_RU 3
#endif
constexpr int RU = KRR_RU;                              // reactions in flight per thread (reactions())
#ifndef KRR_SB
#define KRR_SB 4      // measured (full size): 8 -> 4 steps per batch c3 -2.9 %, c4 -3.2 %; 2: c4 +9 %
#endif
constexpr int SB = KRR_SB;                              // steps per batch of the term streams (the host pads to it)
constexpr int NSLOT = KRR_NSLOT;                        // partial sums of the row program (host-built chunks)
constexpr int oPART = a16(oKEY + 4 * 2 * W * 2);        // [NSLOT] partial f sums, then (energy) [NSLOT] partial T-column sums
constexpr int oUR = a16(oPART + 8 * NSLOT * (ENERGY ? 2 : 1));   // [2][W][2 (NC2 + 1)] published pivot-row candidates + reciprocal (double buffered)
constexpr int oJ = a16(oUR + 8 * 2 * W * 2 * (NC2 + 1));      // [N][LDJ] J; column N holds f (the right-hand side is built from it)
constexpr int CELL_BYTES = a16(oJ + 8 * N * LDJ);

#ifdef KRR_CELL_BYTES
static_assert(CELL_BYTES == KRR_CELL_BYTES, "host and device disagree on the shared-memory layout");
static_assert(oNN == 8 * KRR_I_NN && oKF == 8 * KRR_I_KF && (!KRR_ANY_REV || oKR == 8 * KRR_I_KR), "host and device disagree on the vector offsets");
static_assert(!KRR_ANY_TB || (oQH == 8 * KRR_I_QH && oMT == 8 * KRR_I_MT), "host and device disagree on the third-body offsets");
static_assert(LDJ == KRR_LDJ, "host and device disagree on the row stride of J");
#endif

// shared-memory accesses of the term streams by 32-bit shared-window address: the base is converted once per evaluation (the
// compiler otherwise rebuilds it from a special register in front of every access with a data-dependent offset)
__device__ __forceinline__ double lds(unsigned a) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v; }
__device__ __forceinline__ void sts(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v)); }

struct Cell {
  char* base;
  unsigned sb;                     // the same address in the shared window (set by eval)
  __device__ __forceinline__ double* d(int off) const { return reinterpret_cast<double*>(base + off); }
  __device__ __forceinline__ int* i(int off) const { return reinterpret_cast<int*>(base + off); }
  __device__ __forceinline__ double& F(int row) const { return d(oJ)[row * LDJ + N]; }
};

// ---- the group of 32 W threads -----------------------------------------------------------------------------------
// maximum of non-negative doubles (or NaN, which wins and sticks) over a warp: two integer REDUX on the bit pattern
__device__ __forceinline__ double warp_max_nonneg(double x) {
  const int hi = __double2hiint(x);
  const unsigned lo = (unsigned)__double2loint(x);
  const int H = __reduce_max_sync(0xffffffffu, hi);
  const unsigned L = __reduce_max_sync(0xffffffffu, (hi == H) ? lo : 0u);
  return __hiloint2double(H, (int)L);
}

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
  // maximum of non-negative values; a NaN operand gives NaN (every caller treats NaN as "not acceptable")
  __device__ __forceinline__ double max(double x) const {
    x = warp_max_nonneg(x);
    if (W > 1) {
      const int w = gl >> 5;
      if ((gl & 31) == 0) red[w] = x;
      sync();
      double m = red[0];
      for (int ww = 1; ww < W; ++ww) { const double y = red[ww]; m = (y > m || !(y == y)) ? y : m; }
      x = m;
      sync();
    }
    return x;
  }
  __device__ __forceinline__ double min_signed(double x) const {   // plain minimum, NaN-dropping
    for (int off = 16; off > 0; off >>= 1) { const double y = __shfl_xor_sync(0xffffffffu, x, off); x = (y < x) ? y : x; }
    if (W > 1) {
      const int w = gl >> 5;
      if ((gl & 31) == 0) red[w] = x;
      sync();
      double m = red[0];
      for (int ww = 1; ww < W; ++ww) { const double y = red[ww]; m = (y < m) ? y : m; }
      x = m;
      sync();
    }
    return x;
  }
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
  // RU reactions per thread are in flight at a time, stage by stage and without branches on the kind of the reaction
  // (the kinds are selected at the end of a stage): the exponentials and the table loads of different reactions are
  // independent chains, and a thread that took them one reaction after the other waited for each in turn.
  for (int r0 = G.gl; r0 < R; r0 += GT * RU) {
    int fl[RU], rr[RU];
    bool on[RU];
    int2 f01[RU], f23[RU], f45[RU];
    double A_r[RU], qk[RU], kf[RU], kr[RU], dlf[RU], dlr[RU];
    // ---- stage 1: every table value of the reactions is requested up front ----
#pragma unroll
    for (int u = 0; u < RU; ++u) {
      const int r = r0 + u * GT;
      on[u] = r < R; rr[u] = on[u] ? r : (R - 1);
      fl[u] = __ldg(n.flags + rr[u]);
      const int2* fp = reinterpret_cast<const int2*>(n.fac + 6 * rr[u]);
      f01[u] = __ldg(fp); f23[u] = __ldg(fp + 1); f45[u] = __ldg(fp + 2);
      A_r[u] = __ldg(n.A + rr[u]);
      qk[u] = KRR_ANY_QEXT ? __ldg(n.qk + rr[u]) : 0.0;
      kr[u] = 0.0; dlf[u] = 0.0; dlr[u] = 0.0;
    }
    if (computeK) {
      double beta[RU], Ea[RU], c0[RU], auxv[RU];
      int dn_tot[RU];
      int4 tg0[RU], tg1[RU];
#pragma unroll
      for (int u = 0; u < RU; ++u) {
        beta[u] = __ldg(n.beta + rr[u]); Ea[u] = __ldg(n.Ea + rr[u]); c0[u] = __ldg(n.c0 + rr[u]);
        dn_tot[u] = 0; tg0[u] = make_int4(0, 0, 0, 0); tg1[u] = make_int4(0, 0, 0, 0);
        if (KRR_ANY_REV) {
          dn_tot[u] = __ldg(n.dnu_tot + rr[u]);
          const int4* tp = reinterpret_cast<const int4*>(n.tgt + 8 * rr[u]);
          tg0[u] = __ldg(tp); tg1[u] = __ldg(tp + 1);
        }
        auxv[u] = aux0;
        if (KRR_NAUX > 0 && (fl[u] & KR_DF_AUX)) {
          const int ai = n.auxi[rr[u]];
          if (ai > 0) auxv[u] = aux[(long long)ai * n_cells + cell];
        }
      }
      // ---- stage 2: Arrhenius form for every reaction (eq. 16 with R4), detailed balance (R5) where reversible ----
      double lnkf[RU], kfa[RU];
#pragma unroll
      for (int u = 0; u < RU; ++u) lnkf[u] = c0[u] + beta[u] * lnT - Ea[u] * invT;
#pragma unroll
      for (int u = 0; u < RU; ++u) kfa[u] = krs_exp(lnkf[u]);
      if (KRR_ANY_REV) {
        double sg[RU], su[RU], kra[RU];
#pragma unroll
        for (int u = 0; u < RU; ++u) {
          sg[u] = 0.0; su[u] = 0.0;
          const int tg[8] = {tg0[u].x, tg0[u].y, tg0[u].z, tg0[u].w, tg1[u].x, tg1[u].y, tg1[u].z, tg1[u].w};
#pragma unroll
          for (int t = 0; t < 7; ++t)
            if (t < tg[0]) {
              const int e = tg[1 + t];
              const double cf = (double)((e >> 8) - 128);
              sg[u] += cf * TH[e & 255];
              su[u] += cf * TH[S + (e & 255)];
            }
        }
#pragma unroll
        for (int u = 0; u < RU; ++u) {
          const double lnKc = -sg[u] + (double)dn_tot[u] * (n.ln_p0_kB - lnT);
          kra[u] = krs_exp(lnkf[u] - lnKc);
        }
#pragma unroll
        for (int u = 0; u < RU; ++u) {
          const bool arr = !(fl[u] & (KR_DF_CONST | KR_DF_AUX)), rev = arr && (fl[u] & KR_DF_REV);
          const double d = arr ? (beta[u] + Ea[u] * invT) * invT : 0.0;
          kr[u] = rev ? kra[u] : 0.0;
          dlr[u] = rev ? d - su[u] * invT : 0.0;
        }
      }
#pragma unroll
      for (int u = 0; u < RU; ++u) {
        const bool arr = !(fl[u] & (KR_DF_CONST | KR_DF_AUX));
        dlf[u] = arr ? (beta[u] + Ea[u] * invT) * invT : 0.0;
        kf[u] = (fl[u] & KR_DF_CONST) ? A_r[u] : ((fl[u] & KR_DF_AUX) ? A_r[u] * auxv[u] : kfa[u]);
      }
    } else {
#pragma unroll
      for (int u = 0; u < RU; ++u) {
        kf[u] = KF[rr[u]];
        if (KRR_ANY_REV) kr[u] = KR[rr[u]];
      }
    }
    // ---- stage 3: mass-action products, q_r, dq_r/dT (loads of all reactions first, then the stores) ----
    double Pf[RU], Pr[RU], Mtb[RU];
#pragma unroll
    for (int u = 0; u < RU; ++u) {
      Pf[u] = NN[f01[u].x] * NN[f01[u].y] * NN[f23[u].x];
      Pr[u] = NN[f23[u].y] * NN[f45[u].x] * NN[f45[u].y];
      Mtb[u] = 1.0;
      if (KRR_ANY_TB && (fl[u] & KR_DF_TB)) {
        Mtb[u] = 0.0;
        for (int s = 0; s < S; ++s) Mtb[u] += n.tb_eff[rr[u] * S + s] * NN[s];
      }
    }
#pragma unroll
    for (int u = 0; u < RU; ++u) {
      if (!on[u]) continue;
      const int r = rr[u];
      if (computeK) { KF[r] = kf[u]; if (KRR_ANY_REV) KR[r] = kr[u]; }
      const double qhat = kf[u] * Pf[u] - kr[u] * Pr[u];
      if (KRR_ANY_TB && (fl[u] & KR_DF_TB)) { c.d(oQH)[r] = qhat; c.d(oMT)[r] = Mtb[u]; }
      const double q = Mtb[u] * qhat;
      Q[r] = q;
      heat_sum += qk[u] * q;
      if (ENERGY) {
        const double dqdT = Mtb[u] * (kf[u] * dlf[u] * Pf[u] - kr[u] * dlr[u] * Pr[u]);
        c.d(oDQT)[r] = dqdT;
        heat_dT += qk[u] * dqdT;
      }
    }
  }
}

// ---- f rows (column N of J) and the T column of J (eq. 15, eq. 20), in two passes.  Pass 1, thread <-> CHUNK of a species'
// (reaction, dnu) list: the lists are cut into chunks of equal length on the host and dealt to the threads, so that the
// row of an abundant species (three times the average length) does not hold up the group; the chunks reach each thread
// as ONE coalesced stream of 8-byte words.  Pass 2, thread <-> species: the few partial sums of a species, in chunk
// order (a fixed order: results do not depend on which thread summed what).
__device__ __forceinline__ void row_partials(const KrNetDev& n, const Cell& c, const Grp& G) {
  const unsigned sQ = c.sb + oQ, sD = c.sb + oDQT, sP = c.sb + oPART;
  const uint2* rs = n.rstream[W - 1] + G.gl;
  const int nb = n.rlen[W - 1] / SB;           // batches of SB steps (the host pads to it)
  // A batch requests all of its operands before its first sum, and the stream words of the next batch before that: the
  // stores of the partial sums close a batch, not a step, and the latency of the stream (L2) hides under the batch in
  // front of it.
  double af = 0.0, at = 0.0;
  uint2 ta[SB], tb[SB];
  auto load = [&](uint2 (&t)[SB], int b) {
#pragma unroll
    for (int q = 0; q < SB; ++q) t[q] = __ldg(rs + (b * SB + q) * GT);
  };
  auto work = [&](const uint2 (&t)[SB]) {
    double qv[SB], dv[SB];
#pragma unroll
    for (int q = 0; q < SB; ++q) {
      const unsigned r8 = (t[q].x & 0xffffu) * 8u;
      qv[q] = lds(sQ + r8);
      dv[q] = ENERGY ? lds(sD + r8) : 0.0;
    }
#pragma unroll
    for (int q = 0; q < SB; ++q) {
      const double dnu = (double)((int)(t[q].x >> 16) - 128);
      af = fma(dnu, qv[q], af);
      if (ENERGY) at = fma(dnu, dv[q], at);
      if ((int)t[q].y >= 0) {
        sts(sP + 8u * t[q].y, af); af = 0.0;
        if (ENERGY) { sts(sP + 8u * (NSLOT + t[q].y), at); at = 0.0; }
      }
    }
  };
  load(ta, 0);
  for (int b = 0; b < nb; b += 2) {
    if (b + 1 < nb) load(tb, b + 1);
    work(ta);
    if (b + 1 >= nb) break;
    if (b + 2 < nb) load(ta, b + 2);
    work(tb);
  }
}
__device__ __forceinline__ void row_combine(const KrNetDev& n, const Cell& c, const Grp& G, double invN, bool wantJ) {
  const double* PART = c.d(oPART);
  double* J = c.d(oJ);
  const int* sp = n.rslot_ptr[W - 1];
  for (int s = G.gl; s < S; s += GT) {
    double ys = 0.0, jt = 0.0;
    const int p1 = sp[s + 1];
    for (int p = sp[s]; p < p1; ++p) { ys += PART[p]; if (ENERGY) jt += PART[NSLOT + p]; }
    J[s * LDJ + N] = ys * invN;
    if (ENERGY && wantJ) J[s * LDJ + S] = jt * invN;
  }
}

// ---- Jacobian (eq. 19), thread <-> ENTRY: J[s][m] = sum of its host-built terms dnu_rs dq_r/dn_m, each one multiply
// chain over the cell's shared-memory block; entries are dealt to the threads longest first, so the threads of a
// group finish together.  No read-modify-write of shared memory, no atomics, fixed order (replaces PAPER.md:232).
// Entries that are structurally zero are never written: J is zeroed once per block.
__device__ __forceinline__ void entries(const KrNetDev& n, const Cell& c, const Grp& G) {
  // {coef lo, coef hi, g0 | g1 << 16, g2 | g3 << 16}: one coalesced 16-byte load per thread and step, no dependent loads.
  // Batches of SB steps as in row_partials.
  const uint4* terms = reinterpret_cast<const uint4*>(n.estream[W - 1]) + G.gl;
  const int nb = n.elen[W - 1] / SB;
  const unsigned sb = c.sb, sJ = c.sb + oJ;
  double acc = 0.0;
#if KRR_COMPACT_TERMS
  // compact form: {coef, byte offset of factor 0 | factor 1 << 16, destination entry (0xffff: none)}
  uint4 ta[SB], tb[SB];
  auto load = [&](uint4 (&t)[SB], int b) {
#pragma unroll
    for (int q = 0; q < SB; ++q) t[q] = __ldg(terms + (b * SB + q) * GT);
  };
  auto work = [&](const uint4 (&t)[SB]) {
    double p[SB], f1[SB];
#pragma unroll
    for (int q = 0; q < SB; ++q) {
      p[q] = lds(sb + (t[q].z & 0xffffu));
      f1[q] = lds(sb + (t[q].z >> 16));
    }
#pragma unroll
    for (int q = 0; q < SB; ++q) p[q] *= __hiloint2double((int)t[q].y, (int)t[q].x);
#pragma unroll
    for (int q = 0; q < SB; ++q) {
      acc = fma(p[q], f1[q], acc);
      const unsigned dst = t[q].w & 0xffffu;
      if (dst != 0xffffu) { sts(sJ + 8u * dst, acc); acc = 0.0; }
    }
  };
  load(ta, 0);
  for (int b = 0; b < nb; b += 2) {
    if (b + 1 < nb) load(tb, b + 1);
    work(ta);
    if (b + 1 >= nb) break;
    if (b + 2 < nb) load(ta, b + 2);
    work(tb);
  }
#else
  const int* meta = n.emeta[W - 1] + G.gl;
  const int len = nb * SB;
#pragma unroll 4
  for (int i = 0; i < len; ++i) {
    const uint4 t = __ldg(terms + i * GT);
    const int dst = __ldg(meta + i * GT);
    const double coef = __hiloint2double((int)t.y, (int)t.x);
    acc += coef * lds(sb + 8u * (t.z & 0xffffu)) * lds(sb + 8u * (t.z >> 16)) * lds(sb + 8u * (t.w & 0xffffu)) * lds(sb + 8u * (t.w >> 16));
    if (dst >= 0) { sts(sJ + 8u * dst, acc); acc = 0.0; }
  }
#endif
}

// ---- T row of J (eq. 20 with the dropped dC/dy term, DESIGN.md step 5): thread <-> column m; row S holds the raw heat sum
__device__ __forceinline__ void trow(const Cell& c, const Grp& G, double T, double invC) {
  double *TH = c.d(oTH), *J = c.d(oJ);
  for (int m = G.gl; m < S; m += GT) {
    double acc = 0.0;
    for (int s = 0; s < S; ++s) acc += TH[S + s] * J[s * LDJ + m];
    J[S * LDJ + m] = (J[S * LDJ + m] - T * acc) * invC;
  }
}

// ---- full evaluation of f (and J) at U.  Thermo / KF / KR valid as the flags say.
__device__ __forceinline__ void eval(const KrNetDev& n, const Cell& c_in, const Grp& G, double Ncal, double T, double aux0,
                                  const double* __restrict__ aux, long long cell, long long n_cells, bool computeK,
                                  bool wantJ) {
  Cell c = c_in;
  {                                  // the shared-window address of the cell, opaque to the compiler: converted once per
    const unsigned sb0 = (unsigned)__cvta_generic_to_shared(c_in.base);     // evaluation and held in a register while it runs
    asm volatile("mov.u32 %0, %1;" : "=r"(c.sb) : "r"(sb0));
  }
  const double invT = krs_rcp(T), lnT = (ENERGY || computeK) ? log(T) : 0.0;
  const double invN = krs_rcp(Ncal);
  double *U = c.d(oU), *TH = c.d(oTH), *NN = c.d(oNN), *J = c.d(oJ);
  for (int s = G.gl; s <= S; s += GT) NN[s] = (s < S) ? Ncal * U[s] : 1.0;
  if (ENERGY && wantJ)
    for (int m = G.gl; m < S; m += GT) J[S * LDJ + m] = 0.0;       // the raw heat row is accumulated by entries()
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
  row_partials(n, c, G);
  if (wantJ) entries(n, c, G);
  G.sync();
  row_combine(n, c, G, invN, wantJ);
  if (ENERGY && wantJ) trow(c, G, T, invC);
  G.sync();
  if (ENERGY) {
    double r2[3] = {0.0, 0.0, 0.0};
    for (int s = G.gl; s < S; s += GT) {
      const double fs = J[s * LDJ + N], uh = TH[S + s];
      r2[0] += uh * fs;
      r2[1] += TH[2 * S + s] * fs;
      if (wantJ) r2[2] += uh * J[s * LDJ + S];
    }
    G.sum(r2);
    if (G.gl == 0) {
      J[S * LDJ + N] = (heat_sum * invN - T * r2[0]) * invC;
      if (wantJ) J[S * LDJ + S] = (heat_dT * invN - T * r2[2] - r2[1]) * invC;
    }
    G.sync();
  }
}

// ---- step 7: elimination, one matrix row per lane ------------------------------------------------------------------
// Pivot key of a row: the bit pattern of |a| / scale with the row index folded into its 6 low bits (63 - row), so that a
// warp-wide integer maximum (REDUX on the high words, then on the low words of the rows that share the largest high
// word) names the pivot row: Algorithm 1's scaled pivot, candidates closer than 2^-46 relative counting as tied, ties to
// the smallest row (reading R14' of DESIGN.md).  A used row carries a negative scale: its key is negative and loses
// against every candidate.
// (32-bit keys -- one REDUX -- were measured at +5 % throughput, but candidates within 2^-14 then tie, and on config 4 that
// changed the accept / reject path of cells whose decisions have wide margins: not built.)
typedef long long Key;
__device__ __forceinline__ Key key_of(double v, double sc, int row) {
  return (__double_as_longlong(fabs(v) * sc) | 63LL) - (long long)row;
}

// The elimination state of one thread.  The column loop is a ROLLED loop: on this chip a kernel whose hot path is more
// than ~32 KB of straight-line code is bound by instruction fetch (measured with a microbenchmark: 1.5 instructions per
// clock and SM with 8-12 warps at different places of 64 KB+ of code, against 3 when the code fits the instruction
// caches), and an unrolled column loop is 60 KB (N = 33) to 140 KB (N = 64).  Register indices stay static because the
// row SHIFTS: the update of column k writes entry j of the row into the register of entry j - 1, so that entry 0 is
// always the column being eliminated and the right-hand side the last live entry, and the pivot row is published (and
// read back) in the same shifted layout.  The row shrinks by one entry per column; the loop is cut into SEG segments,
// each compiled for the width the row has at its start (entries beyond the right-hand side are dead: neither published
// nor updated).
//
// The loop is software-pipelined: as soon as the update of column k has produced the entries of column k + 1 the search
// for pivot k + 1 is started, and the two reductions of the search are issued BETWEEN the chunks of the remaining update
// (a warp issues in order: a reduction that waits for the one in front of it would hold up everything behind it), with
// the pivot-row reads of a chunk requested one chunk ahead.  The lane that wins publishes its row with its reciprocal.
constexpr int XRD = XR > 0 ? XR : 1;
constexpr int URS = NC2 + 1;                  // one published row: NC2 pairs + {reciprocal of its column-k entry, its key}
#ifndef KRR_SEG
#define KRR_SEG (KRR_N >= 64 ? 16 : 8)      // measured on N = 64: 16 segments -2.5 % (less dead width per column), 4: +6 %; N = 33: 4 +2 %, 11 +21 %
#endif
constexpr int SEG = (N >= 4 * KRR_SEG) ? KRR_SEG : 1;
constexpr int seg_lo(int i) { return (int)((long long)i * N / SEG); }
#ifndef KRR_UCH
#define KRR_UCH (KRR_W == 1 ? 2 : 4)      // measured (full size): two warps 6 -> 4 pairs per chunk -3 %; one warp 6 -> 2 with 12 instead of 8 cells per SM -2.3 % on top of -4 % from the batches; 8: +2.5 %
#endif
#ifndef KRR_EARLY_PUB
#define KRR_EARLY_PUB 1
#endif
constexpr int UCH = KRR_UCH;                  // pairs of the pivot row per chunk (two chunks in flight)

struct Elim {
  double2 a[NC2];                             // the lane's row of [J - I/h | G/h], shifted: a[0].x is the entry of the current column
  double xr[XRD][XQ];                         // spread rows (not shifted): element j of spread row e in lane j % 32, slot j / 32
  double sc, xsc[XRD];                        // > 0: 1 / scale of a candidate row; < 0: used (or no row)
  double xk[XRD];                             // the spread rows' entries of the column being searched
  double myrp, xrp[XRD];                      // reciprocal pivot of the column in which the row was the pivot row ...
  int mycol, xcol[XRD];                       // ... and that column
  Key kw;                                     // the warp's best key for the column being searched
  Key kwin;                                   // two warps: the better of the two warps' keys ...
  int wwin;                                   // ... and the warp that holds it (it alone publishes its row)
  volatile Key* KX;                           // two warps: the key exchange slots
  int khi, kH;                                // search in flight: high word of this lane's key, the warp's largest high word
  unsigned klo;
  double rk;                                  // speculative reciprocal of this lane's candidate
  int gl, lane, wq;
  double2* URb;
  const Grp* G;

  // candidate search for column kk on the rows as they stand (entry 0 of the shifted row), first half: this lane's key, the
  // warp-wide maximum of the high words (REDUX), and the speculative reciprocal of this lane's candidate (only the
  // winner's is used)
  __device__ __forceinline__ void pick_a(int kk) {
    const double ak = a[0].x;
    Key key = key_of(ak, sc, gl);
#pragma unroll
    for (int e = 0; e < XR; ++e) {             // element kk of a spread row sits in lane kk % 32, which enters it in the
      double v = xr[e][0];                     // search beside its own row (no shuffle in front of the reduction); every
#pragma unroll                                 // lane gets the value for the multiplier of the next update
      for (int q = 1; q < XQ; ++q) v = ((kk >> 5) == q) ? xr[e][q] : v;
      const Key kx = key_of(v, xsc[e], NR + e);
      key = (lane == (kk & 31) && kx > key) ? kx : key;
      xk[e] = __shfl_sync(0xffffffffu, v, kk & 31);
    }
    khi = (int)(key >> 32); klo = (unsigned)key;
    kH = __reduce_max_sync(0xffffffffu, khi);
    rk = krs_rcp(ak);
  }
  // second half: the maximum of the low words among the rows that share the largest high word
  __device__ __forceinline__ void pick_b() {
    const unsigned L = __reduce_max_sync(0xffffffffu, (khi == kH) ? klo : 0u);
    kw = ((long long)kH << 32) | (long long)L;
  }
  // two warps per cell: the warps exchange their best keys for column kk (8 bytes each, one named barrier of its own) so
  // that only the warp that holds the pivot row publishes it.  (Both warps used to publish their candidate -- N / 2 16-byte
  // stores from one lane each -- and the profile showed the single-lane stores throttled by the shared-memory pipe: 17 % of
  // all stall samples of config 4, half of them for rows nobody reads.)
  __device__ __forceinline__ void exchange(int kk) {
    if (W > 1) {
      volatile Key* kx = KX + (kk & 1) * W;
      if (lane == 0) kx[wq] = kw;
      asm volatile("bar.sync 2, %0;" ::"r"(32 * W) : "memory");
      const Key ko = kx[1 - wq];
      const Key k0 = (wq == 0) ? kw : ko, k1 = (wq == 0) ? ko : kw;
      const bool second = k1 > k0;                         // keys carry the row: they are never equal unless both are -1
      wwin = second ? 1 : 0;
      kwin = second ? k1 : k0;
    }
  }
  // publication of the warp's winner for column kk: its row (WD entries from the current column on, every earlier update
  // applied), the reciprocal of its current-column entry and the key
  template <int WD, int FROM = 0>
  __device__ __forceinline__ void publish(int kk) {
    if (W > 1 && wwin != wq) return;
    const int pw = (kw >= 0) ? (63 - (int)(kw & 63)) : -1;
    double2* URw = URb + ((kk & 1) * W + wq) * URS;
    if (gl == pw) {
#pragma unroll
      for (int j = FROM; j < (WD + 1) / 2; ++j) URw[j] = a[j];
      URw[NC2] = make_double2(rk, __longlong_as_double((long long)kw));
    }
#pragma unroll
    for (int e = 0; e < XR; ++e)
      if (pw == NR + e) {
#pragma unroll
        for (int q = 0; q < XQ; ++q) {
          const int c = lane + 32 * q;         // absolute column; published at its distance from the current column
          if (c >= kk && c < NC) reinterpret_cast<double*>(URw)[c - kk] = xr[e][q];
        }
        if (lane == 0) URw[NC2] = make_double2(krs_rcp(xk[e]), __longlong_as_double((long long)kw));
      }
    if (W > 1 && pw < 0 && lane == 0) URw[NC2] = make_double2(0.0, __longlong_as_double(-1LL));   // no candidate in this warp
  }

  // Early publication: the pivot row of the NEXT column is named while the update of this column has hardly begun, so the
  // lane that holds it stores every chunk of its row as soon as the chunk is updated instead of all of it behind the update
  // (N / 2 back-to-back 16-byte stores from one lane fill the queue of the shared-memory pipe -- mio throttle was 17 % of
  // the stall samples of config 4 -- and the rest of the group waits for the last of them).  Pairs lo .. hi of the row as it
  // will stand for the next column; fin is the last pair an update chunk completes.
  template <int WDN>
  __device__ __forceinline__ void pub_pairs(double2* URn, bool pubme, int lo, int hi, int fin) {
#pragma unroll
    for (int q = 0; q < UCH; ++q) {
      const int pp = lo + q;
      if (pp <= hi && pp <= fin && pp < (WDN + 1) / 2) { if (pubme) URn[pp] = a[pp]; }
    }
  }

  // update of the pairs j0 .. j0 + UCH - 1 of the shifted row from the chunk u: entries 2j, 2j + 1 -> 2j - 1, 2j
  template <int WD>
  __device__ __forceinline__ void apply(int j0, double l, const double2 (&u)[UCH]) {
    constexpr int NP = (WD + 1) / 2;
#pragma unroll
    for (int q = 0; q < UCH; ++q) {
      const int j = j0 + q;
      if (j < NP) {
        a[j - 1].y = fma(l, u[q].x, a[j].x);
        if (2 * j + 1 < WD) a[j].x = fma(l, u[q].y, a[j].y);
      }
    }
  }
  template <int WD>
  __device__ __forceinline__ void fetch(int j0, const double2* URw, double2 (&u)[UCH]) {
    constexpr int NP = (WD + 1) / 2;
#pragma unroll
    for (int q = 0; q < UCH; ++q)
      if (j0 + q < NP) u[q] = URw[j0 + q];
  }

  // column k of a segment whose rows have WD live entries at its start (entry 0: column k, ..., the right-hand side last)
  template <int WD>
  __device__ __forceinline__ void column(int k) {
    constexpr int NP = (WD + 1) / 2;                         // pairs of the row; pair 0 holds the current column
    // ---- the pivot row of column k: the warp's candidate, or the better of the two warps' candidates -------------------
    Key kbest = kw;
    const double2* URw = URb + ((k & 1) * W + wq) * URS;
    double2 tail;
    if (W > 1) {
      G->sync();
      kbest = kwin;
      URw = URb + ((k & 1) * W + wwin) * URS;
      tail = URw[NC2];
    } else {
      __syncwarp();
      tail = URw[NC2];
    }
    // ---- broadcast reads of the pivot row: pair 0 and the first chunk at once, every further chunk one chunk ahead ------
    const double2 u0 = URw[0];
    double2 ua[UCH], ub[UCH];
    fetch<WD>(1, URw, ua);
    const int p = (kbest >= 0) ? (63 - (int)(kbest & 63)) : -1;
    const double rp = tail.x;
    const bool mine = (gl == p);
    const double l = mine ? 0.0 : -(a[0].x * rp);            // the pivot row itself is not updated
    if (mine) { sc = -1.0; mycol = k; myrp = rp; }
    double xl[XRD];
#pragma unroll
    for (int e = 0; e < XR; ++e) {
      const bool xmine = (p == NR + e);
      xl[e] = xmine ? 0.0 : -(xk[e] * rp);
      if (xmine) { xsc[e] = -1.0; xcol[e] = k; xrp[e] = rp; }
    }
    // column k + 1 first: its entries feed the next search
    a[0].x = fma(l, u0.y, a[0].y);
#pragma unroll
    for (int e = 0; e < XR; ++e)
#pragma unroll
      for (int q = 0; q < XQ; ++q) {
        const int c = lane + 32 * q;
        if (c > k && c < NC) xr[e][q] = fma(xl[e], reinterpret_cast<const double*>(URw)[c - k], xr[e][q]);
      }
    // the search for pivot k + 1 is issued in front of the rest of update k, its second reduction behind the first chunk
    const bool more = k + 1 < N;
    if (more) pick_a(k + 1);
    if (NP <= 1 && more) { pick_b(); exchange(k + 1); }
    constexpr int FIN = NP - 2;                              // new pair p is complete once the chunk with old pair p + 1 is applied
    bool pubme = false;
    double2* URn = URb + (((k + 1) & 1) * W + wq) * URS;
#pragma unroll
    for (int j0 = 1; j0 < NP; j0 += 2 * UCH) {
      fetch<WD>(j0 + UCH, URw, ub);
      apply<WD>(j0, l, ua);
      if (j0 == 1 && more) {
        pick_b(); exchange(k + 1);
        pubme = (KRR_EARLY_PUB != 0) && (kw >= 0) && (gl == 63 - (int)(kw & 63)) && (W == 1 || wwin == wq);
      }
      if (KRR_EARLY_PUB && more) pub_pairs<WD - 1>(URn, pubme, j0 == 1 ? 0 : j0 - 1, j0 + UCH - 2, FIN);
      fetch<WD>(j0 + 2 * UCH, URw, ua);
      apply<WD>(j0 + UCH, l, ub);
      if (KRR_EARLY_PUB && more) pub_pairs<WD - 1>(URn, pubme, j0 + UCH - 1, j0 + 2 * UCH - 2, FIN);
    }
    if (more) publish<WD - 1, (KRR_EARLY_PUB && FIN >= 0) ? FIN + 1 : 0>(k + 1);
  }

  template <int SI>
  __device__ __forceinline__ void segment() {
    constexpr int k0 = seg_lo(SI), k1 = seg_lo(SI + 1);
#pragma unroll 1
    for (int k = k0; k < k1; ++k) column<NC - k0>(k);
    if constexpr (SI + 1 < SEG) segment<SI + 1>();
  }
};

// On success X holds the solution delta of (I - hJ) delta = -(U - UN - h f).  Uniform return value (false: zero row,
// non-finite entry, no pivot or a pivot below 1e-300 in the units of I - hJ).
__device__ __forceinline__ bool eliminate(const Cell& c, const Grp& G, double h) {
  Elim E;
  E.gl = G.gl; E.lane = G.gl & 31; E.wq = G.gl >> 5; E.G = &G;
  const int gl = E.gl, lane = E.lane;
  double *U = c.d(oU), *UN = c.d(oUN), *X = c.d(oX), *J = c.d(oJ);
  const double invh = krs_rcp(h);
  const bool rin = gl < NR;
  {
    const double2* Jr = reinterpret_cast<const double2*>(J + (rin ? gl : 0) * LDJ);
    double d0 = 0.0;
    if (rin) { d0 = J[gl * LDJ + gl]; J[gl * LDJ + gl] = d0 - invh; J[gl * LDJ + N] = (U[gl] - UN[gl]) * invh - J[gl * LDJ + N]; }
    if (XR > 0) {                             // spread rows: the diagonal and the right-hand side by the lane that holds them
#pragma unroll
      for (int e = 0; e < XR; ++e) {
        const int row = NR + e;
        if (lane == (row & 31)) J[row * LDJ + row] -= invh;
        if (lane == (N & 31)) J[row * LDJ + N] = (U[row] - UN[row]) * invh - J[row * LDJ + N];
      }
    }
    __syncwarp();
#pragma unroll
    for (int j = 0; j < NC2; ++j) E.a[j] = rin ? Jr[j] : make_double2(0.0, 0.0);
    if (rin) J[gl * LDJ + gl] = d0;           // J keeps its entries (structural zeros are never rewritten)
#pragma unroll
    for (int e = 0; e < XR; ++e)
#pragma unroll
      for (int q = 0; q < XQ; ++q) {
        const int j = lane + 32 * q;
        E.xr[e][q] = (j < NC) ? J[(NR + e) * LDJ + j] : 0.0;
      }
  }
  // row scales (max-norm of the matrix part, Algorithm 1's implicit scaling)
  double big = 0.0;
#pragma unroll
  for (int j = 0; j < NC2; ++j) {
    if (2 * j < N) { const double ax = fabs(E.a[j].x); big = (ax > big || !(ax == ax)) ? ax : big; }
    if (2 * j + 1 < N) { const double ay = fabs(E.a[j].y); big = (ay > big || !(ay == ay)) ? ay : big; }
  }
  bool rows_ok = !rin || (big > 0.0 && big <= 1.7e308);
  E.sc = (rin && big > 0.0) ? krs_rcp(big) : -1.0;
#pragma unroll
  for (int e = 0; e < XR; ++e) {
    double m = 0.0;
#pragma unroll
    for (int q = 0; q < XQ; ++q)
      if (lane + 32 * q < N) { const double ax = fabs(E.xr[e][q]); m = (ax > m || !(ax == ax)) ? ax : m; }
    m = warp_max_nonneg(m);
    rows_ok = rows_ok && (m > 0.0) && (m <= 1.7e308);
    E.xsc[e] = (m > 0.0) ? krs_rcp(m) : -1.0;
  }
  rows_ok = G.all(rows_ok);
  if (!rows_ok) return false;

  E.URb = reinterpret_cast<double2*>(c.d(oUR));
  E.KX = reinterpret_cast<volatile Key*>(c.base + oKEY);
  E.kwin = -1; E.wwin = 0;
  E.mycol = -1; E.myrp = 0.0; E.kw = -1; E.rk = 0.0; E.khi = 0; E.kH = 0; E.klo = 0u;
#pragma unroll
  for (int e = 0; e < XRD; ++e) { E.xcol[e] = -1; E.xrp[e] = 0.0; E.xk[e] = 0.0; if (e >= XR) E.xsc[e] = -1.0; }

  E.pick_a(0);
  E.pick_b();
  E.exchange(0);
  E.template publish<NC>(0);
  E.template segment<0>();

  // every row must have been a pivot row, with |pivot| >= 1e-300 in the units of I - hJ (|pivot'| >= 1e-300 / h here) and finite
  const double rmax = 1e300 * h;
  bool ok = !rin || (E.mycol >= 0 && fabs(E.myrp) <= rmax && fabs(E.myrp) > 0.0);
#pragma unroll
  for (int e = 0; e < XR; ++e) ok = ok && (E.xcol[e] >= 0 && fabs(E.xrp[e]) <= rmax && fabs(E.xrp[e]) > 0.0);
  ok = G.all(ok);
  if (!ok) return false;
  // row p_k now holds x_k * pivot_k in its right-hand-side slot
  if (rin) X[E.mycol] = E.a[0].x * E.myrp;         // N shifts have brought the right-hand side to entry 0
#pragma unroll
  for (int e = 0; e < XR; ++e)
    if (lane == (N & 31)) X[E.xcol[e]] = E.xr[e][N >> 5] * E.xrp[e];
  G.sync();
  return true;
}

}  // namespace krr

extern "C" __global__ void __launch_bounds__(32 * KRR_W, KRR_MIN_BLOCKS)
kr_row_kernel(const KrNetDev n, const KrOptsDev o, const KrStepArgs a) {
  using namespace krr;
  extern __shared__ __align__(16) char kr_sm_raw[];
  const int K = o.max_newton;
  Grp G;
  Cell c;
  G.g = 0; G.gl = threadIdx.x;                // one cell per block: every shared-memory offset is a compile-time constant
  c.base = kr_sm_raw;
  c.sb = 0;
  G.red = c.d(oRED);
  volatile long long* cellslot = (volatile long long*)(c.d(oRED) + 8 * W);
  double *U = c.d(oU), *UN = c.d(oUN), *X = c.d(oX);

  for (int i = G.gl; i < N * LDJ; i += GT) c.d(oJ)[i] = 0.0;    // structural zeros of J: written once, never touched again
  G.sync();

  // The solver's counters (thread 0) and, across every elimination, the controller state of the cell live in shared
  // memory: the elimination needs the register file for the row and for two chunks of the pivot row in flight.
  volatile unsigned long long* CNT = reinterpret_cast<volatile unsigned long long*>(c.d(oPK) + 12 * W);   // acc rej newton rate failed
  volatile double* PK = c.d(oPK) + 12 * (G.gl >> 5);
  if (G.gl == 0)
    for (int i = 0; i < 6; ++i) CNT[i] = 0ull;

  for (;;) {
    if (G.gl == 0) {
      long long idx = (long long)atomicAdd(a.counter, 1ull);
      if (a.list) idx = (idx < (long long)*a.list_count) ? a.list[idx] : a.n_cells;
      *cellslot = idx;
    }
    G.sync();
    long long cell = *cellslot;
    G.sync();
    if (cell >= a.n_cells) break;

    // ---- step 1: layout-in, clamp, first sub-step -------------------------------------------------
    int st = a.list ? a.list_flag : 0;
    double Tc = a.T[cell];
    if (Tc < n.T_lo) { Tc = n.T_lo; st |= KR_DST_T_CLAMPED; }
    if (Tc > n.T_hi) { Tc = n.T_hi; st |= KR_DST_T_CLAMPED; }
    double Ncal = a.rho[cell] * (1.0 / KR_M_U);
    double T_iso = Tc;
    double aux0 = (KRR_NAUX > 0) ? a.aux[cell] : 0.0;
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
    bool failed = false, costed = false;
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
        if (ENERGY || (prelim && KRR_ANY_REV)) { thermo(n, c, G, T, krs_rcp(T), log(T)); G.sync(); }
        if ((ENERGY || prelim) && !a.cost_out && G.gl == 0) CNT[3] = CNT[3] + 1ull;
        eval(n, c, G, Ncal, T, aux0, a.aux, cell, a.n_cells, ENERGY || prelim, !prelim);
        if (prelim) {
          if (o.h0_mode == 1 || a.cost_out) {
            double big = 0.0;
            for (int s = G.gl; s < S; s += GT) {
              const double x = fabs(c.F(s)) / (fabs(UN[s]) + o.y_floor);
              big = (x > big) ? x : big;        // NaN-dropping, as the oracle's "if (x > big)"
            }
            for (int off = 16; off > 0; off >>= 1) { const double y = __shfl_xor_sync(0xffffffffu, big, off); big = (y > big) ? y : big; }
            if (W > 1) {
              if ((G.gl & 31) == 0) G.red[G.gl >> 5] = big;
              G.sync();
              big = (G.red[1] > G.red[0]) ? G.red[1] : G.red[0];
              G.sync();
            }
            if (big > 0.0 && finite(big)) h = fmin(a.dt, o.eta / big);
          }
          h = h * o.h0_scale;
          h_floor = o.h_min_rel * fmin(h, a.dt);
          prelim = false; was_prelim = true;
          break;
        }
        if (G.gl == 0) CNT[2] = CNT[2] + 1ull;
        // park the controller state (every lane of a warp writes the same values to the warp's slots and reads them back)
        PK[0] = t; PK[1] = h_floor; PK[2] = e_prev; PK[3] = Ncal; PK[4] = T_iso; PK[5] = aux0;
        PK[6] = __longlong_as_double(cell);
        PK[7] = __hiloint2double(st, n_acc); PK[8] = __hiloint2double(n_rej, it); PK[9] = __hiloint2double(k, last ? 1 : 0);
        const bool solved = eliminate(c, G, h);
        t = PK[0]; h_floor = PK[1]; e_prev = PK[2]; Ncal = PK[3]; T_iso = PK[4]; aux0 = PK[5];
        cell = __double_as_longlong(PK[6]);
        { const double w7 = PK[7], w8 = PK[8], w9 = PK[9];
          st = __double2hiint(w7); n_acc = __double2loint(w7); n_rej = __double2hiint(w8); it = __double2loint(w8);
          k = __double2hiint(w9); last = __double2loint(w9) != 0; }
        if (!solved) { ran = false; break; }
        bool fin = true;
        double en = 0.0;
        for (int i = G.gl; i < N; i += GT) {
          const double dl = X[i];
          const double x = U[i] + dl;
          U[i] = x;
          fin = fin && finite(x);
          const double w = fabs(dl) / (o.rtol * fabs(x) + ((i < S) ? o.atol_y : o.atol_T));
          en = (w > en || !(w == w)) ? w : en;
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
      if (was_prelim) {
        if (a.cost_out) { costed = true; break; }   // cost pass: the key is the first sub-step
        continue;
      }
      // step 8: accept / reject
      bool ok = ran && (e <= 1.0);
      if (ok) {
        double miny = __longlong_as_double(0x7ff0000000000000LL);
        for (int s = G.gl; s < S; s += GT) miny = fmin(miny, U[s]);
        miny = G.min_signed(miny);
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
    if (costed) {
      if (G.gl == 0) a.cost_out[cell] = (float)h;
      G.sync();
      continue;
    }
    if (G.gl == 0) { CNT[0] = CNT[0] + (unsigned long long)n_acc; CNT[1] = CNT[1] + (unsigned long long)n_rej; }
    if (failed) {                                                 // R13: revert (the caller's buffers were never written)
      if (a.fail_list) { if (G.gl == 0) a.fail_list[atomicAdd(a.fail_count, 1ull)] = cell; }   // second attempt
      else if (G.gl == 0) { CNT[4] = CNT[4] + 1ull; if (a.status) a.status[cell] = st | KR_DST_FAILED; }
      G.sync();
      continue;
    }
    // ---- step 9: finalise (PAPER.md:212-216 stages 1-3, kr_post.cuh; serial in thread 0, once per cell) + layout-out ----
    if (o.finalize && G.gl == 0) {
      st |= kr_postprocess<E>(kr_post_lists(n), o.cons_tol, [&](int s) { return a.y[cell * S + s]; }, [&](int s) -> double& { return UN[s]; });
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
    atomicAdd(a.stats + 0, CNT[0]); atomicAdd(a.stats + 1, CNT[1]); atomicAdd(a.stats + 2, CNT[2]);
    atomicAdd(a.stats + 3, CNT[2]); atomicAdd(a.stats + 4, CNT[3]); atomicAdd(a.stats + 5, CNT[4]);
  }
}
