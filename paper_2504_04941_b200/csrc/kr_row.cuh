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
//                       no dynamic register indexing (the column loop is unrolled, rows never move: a used row is
//                       marked, and the update is applied to used rows as well -- the Gauss-Jordan form -- so that after
//                       N columns row p_k holds x_k * pivot_k and no substitution pass is needed).  The system that is
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
constexpr int oKEY = oRED + 8 * (8 * W + 4);            // int[2][W][2] pivot keys of the two warps (double buffered)
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

struct Cell {
  char* base;
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
  for (int r = G.gl; r < R; r += GT) {
    // every table value of the reaction is requested up front: independent loads, one exposed latency instead of a chain
    const int fl = __ldg(n.flags + r);
    const int2* fp = reinterpret_cast<const int2*>(n.fac + 6 * r);
    const int2 f01 = __ldg(fp), f23 = __ldg(fp + 1), f45 = __ldg(fp + 2);
    const double A_r = __ldg(n.A + r);
    const double qk = KRR_ANY_QEXT ? __ldg(n.qk + r) : 0.0;
    double beta = 0.0, Ea = 0.0, c0 = 0.0;
    int dn_tot = 0;
    int4 tg0 = make_int4(0, 0, 0, 0), tg1 = make_int4(0, 0, 0, 0);
    if (computeK) {
      beta = __ldg(n.beta + r); Ea = __ldg(n.Ea + r); c0 = __ldg(n.c0 + r);
      if (KRR_ANY_REV) {
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
        if (KRR_ANY_REV && (fl & KR_DF_REV)) {
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
      KF[r] = kf;
      if (KRR_ANY_REV) KR[r] = kr;
    } else {
      kf = KF[r];
      if (KRR_ANY_REV) kr = KR[r];
    }
    const double Pf = NN[f01.x] * NN[f01.y] * NN[f23.x];
    const double Pr = NN[f23.y] * NN[f45.x] * NN[f45.y];
    double Mtb = 1.0;
    const double qhat = kf * Pf - kr * Pr;
    if (KRR_ANY_TB && (fl & KR_DF_TB)) {
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

// ---- f rows (column N of J) and the T column of J (eq. 15, eq. 20), in two passes.  Pass 1, thread <-> CHUNK of a species'
// (reaction, dnu) list: the lists are cut into chunks of equal length on the host and dealt to the threads, so that the
// row of an abundant species (three times the average length) does not hold up the group; the chunks reach each thread
// as ONE coalesced stream of 8-byte words.  Pass 2, thread <-> species: the few partial sums of a species, in chunk
// order (a fixed order: results do not depend on which thread summed what).
__device__ __forceinline__ void row_partials(const KrNetDev& n, const Cell& c, const Grp& G) {
  const double *Q = c.d(oQ), *DQT = c.d(oDQT);
  double* PART = c.d(oPART);
  const uint2* rs = n.rstream[W - 1] + G.gl;
  const int len = n.rlen[W - 1];
  double af = 0.0, at = 0.0;
#pragma unroll 4
  for (int i = 0; i < len; ++i) {
    const uint2 t = __ldg(rs + i * GT);
    const int r = (int)(t.x & 0xffffu);
    const double dnu = (double)((int)(t.x >> 16) - 128);
    af += dnu * Q[r];
    if (ENERGY) at += dnu * DQT[r];
    if ((int)t.y >= 0) {
      PART[t.y] = af; af = 0.0;
      if (ENERGY) { PART[NSLOT + t.y] = at; at = 0.0; }
    }
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
  const double* D = c.d(0);
  double* J = c.d(oJ);
  // {coef lo, coef hi, g0 | g1 << 16, g2 | g3 << 16}: one coalesced 16-byte load per thread and step, no dependent loads
  const uint4* terms = reinterpret_cast<const uint4*>(n.estream[W - 1]) + G.gl;
  const int* meta = n.emeta[W - 1] + G.gl;
  const int len = n.elen[W - 1];
  double acc = 0.0;
#if KRR_COMPACT_TERMS
  // compact form: {coef, byte offset of factor 0 | factor 1 << 16, destination entry (0xffff: none)}
  (void)D; (void)meta;
  const char* base = c.base;
#pragma unroll 8
  for (int i = 0; i < len; ++i) {
    const uint4 t = __ldg(terms + i * GT);
    const double coef = __hiloint2double((int)t.y, (int)t.x);
    const double f0 = *reinterpret_cast<const double*>(base + (t.z & 0xffffu));
    const double f1 = *reinterpret_cast<const double*>(base + (t.z >> 16));
    acc = fma(coef * f0, f1, acc);
    const unsigned dst = t.w & 0xffffu;
    if (dst != 0xffffu) { J[dst] = acc; acc = 0.0; }
  }
#else
#pragma unroll 4
  for (int i = 0; i < len; ++i) {
    const uint4 t = __ldg(terms + i * GT);
    const int dst = __ldg(meta + i * GT);
    const double coef = __hiloint2double((int)t.y, (int)t.x);
    acc += coef * D[t.z & 0xffffu] * D[t.z >> 16] * D[t.w & 0xffffu] * D[t.w >> 16];
    if (dst >= 0) { J[dst] = acc; acc = 0.0; }
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
__device__ __forceinline__ void eval(const KrNetDev& n, const Cell& c, const Grp& G, double Ncal, double T, double aux0,
                                  const double* __restrict__ aux, long long cell, long long n_cells, bool computeK,
                                  bool wantJ) {
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
#ifndef KRR_KEY64
#define KRR_KEY64 1      // 0: 32-bit keys, one REDUX (measured: +5 % throughput, but candidates within 2^-14 tie, and on config 4
#endif                   // that changed the accept / reject path of cells whose decisions have wide margins) -- kept for experiments only
#if KRR_KEY64
// the whole bit pattern of |a| / scale with the row in the 6 low bits (ties to 2^-46), two REDUX
typedef long long Key;
__device__ __forceinline__ Key key_of(double v, double sc, int row) {
  return (__double_as_longlong(fabs(v) * sc) | 63LL) - (long long)row;
}
__device__ __forceinline__ Key warp_max_key(Key k) {
  const int hi = (int)(k >> 32);
  const unsigned lo = (unsigned)k;
  const int H = __reduce_max_sync(0xffffffffu, hi);
  const unsigned L = __reduce_max_sync(0xffffffffu, (hi == H) ? lo : 0u);
  return ((long long)H << 32) | (long long)L;
}
#else
typedef int Key;
__device__ __forceinline__ Key key_of(double v, double sc, int row) {
  return (__double2hiint(fabs(v) * sc) | 63) - row;
}
__device__ __forceinline__ Key warp_max_key(Key k) { return __reduce_max_sync(0xffffffffu, k); }
#endif

// The elimination state of one thread; the column loop is a compile-time recursion (run<K>), so that every register
// index is static whatever N is.
//
// The column loop is software-pipelined: as soon as the update of column k has produced the entries of column k + 1 the
// search for pivot k + 1 is started (candidate keys, REDUX, a speculative reciprocal of every candidate), and the
// remaining FMAs of update k are issued behind it, so that the latency of the search hides under the update.  The lane
// that wins publishes its row together with its reciprocal.
constexpr int XRD = XR > 0 ? XR : 1;
constexpr int URS = NC2 + 1;                  // one published row: NC2 pairs + {reciprocal of its column-k entry, its key}

struct Elim {
  double2 a[NC2];                             // the lane's row of [J - I/h | G/h]
  double xr[XRD][XQ];                         // spread rows: element j of spread row e in lane j % 32, slot j / 32
  double sc, xsc[XRD];                        // > 0: 1 / scale of a candidate row; < 0: used (or no row)
  double xk[XRD];                             // the spread rows' entries of the column being searched
  double myrp, xrp[XRD];                      // reciprocal pivot of the column in which the row was the pivot row ...
  int mycol, xcol[XRD];                       // ... and that column
  Key kw;                                     // the warp's best key for the column being searched
  double rk;                                  // speculative reciprocal of this lane's candidate
  int gl, lane, wq;
  double2* URb;
  const Grp* G;

  __device__ __forceinline__ double col(int k) const { return (k & 1) ? a[k >> 1].y : a[k >> 1].x; }

  // candidate search for column KK on the rows as they stand: the warp's best key (REDUX), and the speculative
  // reciprocal of this lane's candidate (overlaps the reduction; only the winner's is used)
  template <int KK>
  __device__ __forceinline__ void pick() {
    const double ak = col(KK);
    Key key = key_of(ak, sc, gl);
#pragma unroll
    for (int e = 0; e < XR; ++e) {             // element KK of a spread row sits in lane KK % 32: every lane gets it
      xk[e] = __shfl_sync(0xffffffffu, xr[e][KK >> 5], KK & 31);
      const Key kx = key_of(xk[e], xsc[e], NR + e);
      key = (kx > key) ? kx : key;
    }
    kw = warp_max_key(key);
    rk = krs_rcp(ak);
  }
  // publication of the warp's winner: its row from column KK on (every earlier update applied), the reciprocal of its
  // column-KK entry and the key
  template <int KK>
  __device__ __forceinline__ void publish() {
    constexpr int buf = KK & 1;
    const int pw = (kw >= 0) ? (63 - (int)(kw & 63)) : -1;
    double2* URw = URb + (buf * W + wq) * URS;
    if (gl == pw) {
#pragma unroll
      for (int j = KK >> 1; j < NC2; ++j) URw[j] = a[j];
      URw[NC2] = make_double2(rk, __longlong_as_double((long long)kw));
    }
#pragma unroll
    for (int e = 0; e < XR; ++e)
      if (pw == NR + e) {
#pragma unroll
        for (int q = 0; q < XQ; ++q)
          if (lane + 32 * q < NC) reinterpret_cast<double*>(URw)[lane + 32 * q] = xr[e][q];
        if (lane == 0) URw[NC2] = make_double2(krs_rcp(xk[e]), __longlong_as_double((long long)kw));
      }
    if (W > 1 && pw < 0 && lane == 0) URw[NC2] = make_double2(0.0, __longlong_as_double(-1LL));   // no candidate in this warp
  }

  template <int K>
  __device__ __forceinline__ void column() {
    constexpr int buf = K & 1, K2 = K >> 1;
    // ---- the pivot row of column K: the warp's candidate, or the better of the two warps' candidates -------------------
    Key kbest = kw;
    const double2* URw = URb + (buf * W + wq) * URS;
    double2 tail;
    if (W > 1) {
      G->sync();
      const double2 t0 = URb[(buf * W + 0) * URS + NC2], t1 = URb[(buf * W + 1) * URS + NC2];
      const Key k0 = (Key)__double_as_longlong(t0.y), k1 = (Key)__double_as_longlong(t1.y);
      const bool second = k1 > k0;                           // keys carry the row: they are never equal unless both are -1
      kbest = second ? k1 : k0;
      tail = second ? t1 : t0;
      URw = URb + (buf * W + (second ? 1 : 0)) * URS;
    } else {
      __syncwarp();
      tail = URw[NC2];
    }
    const int p = (kbest >= 0) ? (63 - (int)(kbest & 63)) : -1;
    // ---- broadcast read of the pivot row and its reciprocal, rank-1 update of the lane's row -----------------------------
    const double rp = tail.x;
    const bool mine = (gl == p);
    const double l = mine ? 0.0 : -(col(K) * rp);          // the pivot row itself is not updated
    if (mine) { sc = -1.0; mycol = K; myrp = rp; }
    double xl[XRD];
#pragma unroll
    for (int e = 0; e < XR; ++e) {
      const bool xmine = (p == NR + e);
      xl[e] = xmine ? 0.0 : -(xk[e] * rp);
      if (xmine) { xsc[e] = -1.0; xcol[e] = K; xrp[e] = rp; }
    }
    // column K + 1 first: its entries feed the next search
    constexpr int J1 = (K & 1) ? K2 + 1 : K2;              // the pair that holds column K + 1
    const double2 u1 = URw[J1];
    if (K & 1) a[J1].x = fma(l, u1.x, a[J1].x);
    else a[J1].y = fma(l, u1.y, a[J1].y);
#pragma unroll
    for (int e = 0; e < XR; ++e)
#pragma unroll
      for (int q = 0; q < XQ; ++q) {
        const int j = lane + 32 * q;
        if (j > K && j < NC) xr[e][q] = fma(xl[e], reinterpret_cast<const double*>(URw)[j], xr[e][q]);
      }
    // the search for pivot K + 1 is issued in front of the rest of update K; its winner publishes its row behind it
    if constexpr (K + 1 < N) pick<K + 1>();
    if (K & 1) a[J1].y = fma(l, u1.y, a[J1].y);
#pragma unroll
    for (int j = J1 + 1; j < NC2; ++j) {
      const double2 u = URw[j];
      a[j].x = fma(l, u.x, a[j].x); a[j].y = fma(l, u.y, a[j].y);
    }
    if constexpr (K + 1 < N) publish<K + 1>();
  }

  template <int K>
  __device__ __forceinline__ void run() {
    column<K>();
    if constexpr (K + 1 < N) run<K + 1>();
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
  E.mycol = -1; E.myrp = 0.0; E.kw = -1; E.rk = 0.0;
#pragma unroll
  for (int e = 0; e < XRD; ++e) { E.xcol[e] = -1; E.xrp[e] = 0.0; E.xk[e] = 0.0; if (e >= XR) E.xsc[e] = -1.0; }

  E.template pick<0>();
  E.template publish<0>();
  E.template run<0>();

  // every row must have been a pivot row, with |pivot| >= 1e-300 in the units of I - hJ (|pivot'| >= 1e-300 / h here) and finite
  const double rmax = 1e300 * h;
  bool ok = !rin || (E.mycol >= 0 && fabs(E.myrp) <= rmax && fabs(E.myrp) > 0.0);
#pragma unroll
  for (int e = 0; e < XR; ++e) ok = ok && (E.xcol[e] >= 0 && fabs(E.xrp[e]) <= rmax && fabs(E.xrp[e]) > 0.0);
  ok = G.all(ok);
  if (!ok) return false;
  // row p_k now holds x_k * pivot_k in its right-hand-side slot
  if (rin) X[E.mycol] = E.col(N) * E.myrp;
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
  G.red = c.d(oRED);
  volatile long long* cellslot = (volatile long long*)(c.d(oRED) + 8 * W);
  double *U = c.d(oU), *UN = c.d(oUN), *X = c.d(oX);

  for (int i = G.gl; i < N * LDJ; i += GT) c.d(oJ)[i] = 0.0;    // structural zeros of J: written once, never touched again
  G.sync();

  unsigned long long c_acc = 0, c_rej = 0, c_newton = 0, c_rate = 0, c_failed = 0;   // thread 0 of the group

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
    int st = a.list ? a.list_flag : 0;
    double Tc = a.T[cell];
    if (Tc < n.T_lo) { Tc = n.T_lo; st |= KR_DST_T_CLAMPED; }
    if (Tc > n.T_hi) { Tc = n.T_hi; st |= KR_DST_T_CLAMPED; }
    const double Ncal = a.rho[cell] * (1.0 / KR_M_U);
    const double T_iso = Tc;
    const double aux0 = (KRR_NAUX > 0) ? a.aux[cell] : 0.0;
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
        if ((ENERGY || prelim) && !a.cost_out) c_rate++;
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
        c_newton++;
        if (!eliminate(c, G, h)) { ran = false; break; }
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
    c_acc += n_acc; c_rej += n_rej;
    if (failed) {                                                 // R13: revert (the caller's buffers were never written)
      if (a.fail_list) { if (G.gl == 0) a.fail_list[atomicAdd(a.fail_count, 1ull)] = cell; }   // second attempt
      else { c_failed++; if (a.status && G.gl == 0) a.status[cell] = st | KR_DST_FAILED; }
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
    atomicAdd(a.stats + 0, c_acc); atomicAdd(a.stats + 1, c_rej); atomicAdd(a.stats + 2, c_newton);
    atomicAdd(a.stats + 3, c_newton); atomicAdd(a.stats + 4, c_rate); atomicAdd(a.stats + 5, c_failed);
  }
}
