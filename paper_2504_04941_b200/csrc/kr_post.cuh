// kr_post.cuh -- the end-of-step repair of a cell's abundances (DESIGN.md step 9), run by ONE thread per
// cell, once per cell, from every solve kernel.  Written against host-built gather lists (kr_lib.cu, build_post_lists):
//
//   sp list   species s -> its non-zero conservation rows          entry = (row << 8) | (N_{row,s} + 128)
//   res list  row nu    -> the species made of row nu only          entry = (species << 8) | (N_{nu,s} + 128)
//   cmp list  row nu    -> the neutral compounds that hold nu and   entry = (species << 8) | (N_{nu,s} + 128)
//                          whose other rows all have a res list
//
// One pass over the species does the clamping of PAPER.md:214 and gathers, per row, the three sums the repair of
// PAPER.md:215 needs: the initial-minus-final total, the part of it the clamping brought, and the scale of the row.
// One pass over the rows then moves the compensation into the most abundant species of the row's res list, and a last
// pass refills reservoirs that went negative from the cmp lists, most abundant compound first.  Which of
// the two compensations a row gets (reading R12 of DESIGN.md): the full initial-minus-final difference when it exceeds
// cons_tol x scale -- a real violation -- and otherwise only what the clamping brought, so that rounding-level drift of the
// solver never lands in a trace species.
#pragma once
#include "kr_tables.h"

#define KR_MAX_ROWS 16

struct KrPostLists {
  int E, S;
  const int *sp_ptr, *sp_ent;      // [S + 1], entries
  const int *res_ptr, *res_ent;    // [E + 1], entries
  const int *cmp_ptr, *cmp_ent;    // [E + 1], entries
  const int* signed_row;           // [E] 1: the row has negative entries (a charge row): never refilled from compounds
};

__device__ __forceinline__ int kr_pk_index(int e) { return e >> 8; }
__device__ __forceinline__ double kr_pk_coef(int e) { return (double)((e & 255) - 128); }

// most abundant member of a packed list [lo, hi); first one wins a tie; -1 when the list is empty.  `positive`: only
// members with y > 0 qualify.  *ent receives the packed entry of the winner.
template <class Y>
__device__ __forceinline__ int kr_post_argmax(const int* list, int lo, int hi, Y& y, bool positive, int* ent) {
  int best = -1;
  double top = 0.0;
  for (int i = lo; i < hi; ++i) {
    const int e = list[i];
    const double v = y(kr_pk_index(e));
    if (positive && !(v > 0.0)) continue;
    if (best < 0 || v > top) { best = kr_pk_index(e); top = v; *ent = e; }
  }
  return best;
}

// yin(s): abundance of species s at the start of the step (read-only); y(s): reference to its final abundance.
// MAXR: an upper bound of the number of conservation rows known at compile time (the network-specialised kernels pass E).
template <int MAXR = KR_MAX_ROWS, class Yin, class Y>
__device__ inline int kr_postprocess(const KrPostLists& L, double cons_tol, Yin yin, Y y) {
  double full[MAXR], clamp[MAXR], scale[MAXR];
  int home[MAXR];                        // packed res entry of the species that took the row's compensation, or -1
  int bits = 0;
  for (int nu = 0; nu < L.E; ++nu) { full[nu] = 0.0; clamp[nu] = 0.0; scale[nu] = 0.0; home[nu] = -1; }

  // species pass: PAPER.md:214 (negatives to zero) and the row sums of PAPER.md:215
  for (int s = 0; s < L.S; ++s) {
    const double before = yin(s);
    double now = y(s);
    const bool neg = now < 0.0;
    const double cut = neg ? now : 0.0;
    if (neg) { now = 0.0; y(s) = 0.0; bits |= KR_DST_CLAMPED_NEG; }
    const double moved = before - now, mag = fabs(before);
    for (int i = L.sp_ptr[s]; i < L.sp_ptr[s + 1]; ++i) {
      const int e = L.sp_ent[i], nu = kr_pk_index(e);
      const double c = kr_pk_coef(e);
      full[nu] += c * moved;
      scale[nu] += fabs(c) * mag;
      if (neg) clamp[nu] += c * cut;
    }
  }

  // row pass: compensation into the row's most abundant single-row species
  for (int nu = 0; nu < L.E; ++nu) {
    const double give = (fabs(full[nu]) > cons_tol * scale[nu]) ? full[nu] : clamp[nu];
    if (give == 0.0) continue;
    int ent = 0;
    const int r = kr_post_argmax(L.res_ent, L.res_ptr[nu], L.res_ptr[nu + 1], y, false, &ent);
    if (r < 0) { bits |= KR_DST_NO_RESERVOIR; continue; }
    home[nu] = ent;
    y(r) = y(r) + give / kr_pk_coef(ent);
  }

  // refill pass: an element row whose reservoir is negative takes atoms from compounds, largest first
  for (int nu = 0; nu < L.E; ++nu) {
    if (home[nu] < 0 || L.signed_row[nu]) continue;
    const int r = kr_pk_index(home[nu]);
    const double per_r = kr_pk_coef(home[nu]);
    if (!(y(r) < 0.0) || !(per_r > 0.0)) continue;
    double missing = -y(r) * per_r;                     // atoms of row nu still owed
    for (int round = 0; round < L.S && missing > 0.0; ++round) {
      int ent = 0;
      const int c = kr_post_argmax(L.cmp_ent, L.cmp_ptr[nu], L.cmp_ptr[nu + 1], y, true, &ent);
      if (c < 0) break;
      const double per_c = kr_pk_coef(ent), have = y(c);
      double take = missing / per_c;
      const bool exhausts = !(take < have);
      if (exhausts) take = have;
      y(c) = exhausts ? 0.0 : have - take;
      for (int i = L.sp_ptr[c]; i < L.sp_ptr[c + 1]; ++i) {          // the compound's atoms go home row by row
        const int e = L.sp_ent[i], mu = kr_pk_index(e);
        if (mu == nu) continue;
        if (home[mu] < 0) {
          int em = 0;
          kr_post_argmax(L.res_ent, L.res_ptr[mu], L.res_ptr[mu + 1], y, false, &em);
          home[mu] = em;                                             // never empty: the cmp list was filtered for it
        }
        const int rm = kr_pk_index(home[mu]);
        y(rm) = y(rm) + kr_pk_coef(e) * take / kr_pk_coef(home[mu]);
      }
      y(r) = y(r) + per_c * take / per_r;
      missing = exhausts ? missing - per_c * take : 0.0;
      bits |= KR_DST_STAGE3;
    }
    if (!(missing > 0.0)) y(r) = 0.0;                   // paid in full: exactly empty, not a rounding residue
  }
  for (int nu = 0; nu < L.E; ++nu)
    if (home[nu] >= 0 && y(kr_pk_index(home[nu])) < 0.0) bits |= KR_DST_NEEDS_STAGE3;
  return bits;
}

// the view of the table-driven kernels
__device__ __forceinline__ KrPostLists kr_post_lists(const KrNetDev& n) {
  return KrPostLists{n.E, n.S, n.post_sp_ptr, n.post_sp_ent, n.post_res_ptr, n.post_res_ent, n.post_cmp_ptr, n.post_cmp_ent,
                     n.signed_row};
}
