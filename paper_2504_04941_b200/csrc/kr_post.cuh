// kr_post.cuh -- step 9 of DESIGN.md: post-processing of a cell's final abundances, stages 1-3 of PAPER.md:212-216,
// shared by every solve kernel (one thread per cell runs it, once per cell).
//   Stage 1: negatives -> 0.
//   Stage 2 (reading R12): what stage 1 added to conservation row nu, -sum_s N_{nu,s} min(y_s, 0), is taken
//     back from that row's reservoir: the species with only row nu non-zero that has the largest abundance.
//   Stage 3 (reading R23): for every unsigned row whose reservoir went negative, in row order, the most
//     abundant neutral compound (>= 2 non-zero rows, none of them signed) that contains the element is disintegrated
//     just enough -- z = min(y_c, need / N_{nu,c}) -- its atoms go to the reservoirs of their rows; repeated with the next
//     most abundant compound until the need is met (the reservoir ends at exactly 0) or none is left (NEEDS_STAGE3).
// `Tab` gives the network (E, S, comp(nu, s), resv(nu, s), compound(s), signed_row(nu)); `un(s)` is a reference to the
// abundance of species s.  Returns the status bits set.  Every row total is unchanged by construction.
#pragma once
#include "kr_tables.h"

#define KR_MAX_ROWS 16

template <class Tab, class Acc>
__device__ inline int kr_postprocess(const Tab& tb, Acc un) {
  const int E = tb.E(), S = tb.S();
  int st = 0;
  double removed[KR_MAX_ROWS];
  int res_of[KR_MAX_ROWS];
  bool any = false;
  for (int nu = 0; nu < E; ++nu) {
    double rem = 0.0;
    for (int s = 0; s < S; ++s) {
      const double x = un(s);
      if (x < 0.0) rem += (double)tb.comp(nu, s) * x;
    }
    removed[nu] = rem; res_of[nu] = -1;
  }
  for (int s = 0; s < S; ++s)
    if (un(s) < 0.0) { un(s) = 0.0; st |= KR_DST_CLAMPED_NEG; any = true; }
  if (!any) return st;
  auto reservoir = [&](int nu) {
    int res = -1;
    double best = 0.0;
    for (int s = 0; s < S; ++s) {
      if (!tb.resv(nu, s)) continue;
      const double x = un(s);
      if (res < 0 || x > best) { res = s; best = x; }
    }
    return res;
  };
  bool need3 = false;
  for (int nu = 0; nu < E; ++nu) {
    if (removed[nu] == 0.0) continue;
    const int res = reservoir(nu);
    if (res < 0) { st |= KR_DST_NO_RESERVOIR; continue; }
    res_of[nu] = res;
    const double x = un(res) + removed[nu] / (double)tb.comp(nu, res);
    un(res) = x;
    if (x < 0.0) need3 = true;
  }
  if (!need3) return st;
  for (int nu = 0; nu < E; ++nu) {                                   // stage 3
    const int res = res_of[nu];
    if (res < 0 || !(un(res) < 0.0)) continue;
    const double nres = (double)tb.comp(nu, res);
    if (tb.signed_row(nu) || !(nres > 0.0)) { st |= KR_DST_NEEDS_STAGE3; continue; }
    double need = -un(res) * nres;
    for (int iter = 0; iter < S && need > 0.0; ++iter) {
      int c = -1;
      double best = 0.0;
      for (int s = 0; s < S; ++s) {
        if (!tb.compound(s) || tb.comp(nu, s) <= 0 || !(un(s) > 0.0)) continue;
        bool placeable = true;                     // every other row of the compound needs a reservoir for its atoms
        for (int mu = 0; mu < E && placeable; ++mu)
          if (mu != nu && tb.comp(mu, s) != 0 && res_of[mu] < 0 && reservoir(mu) < 0) placeable = false;
        if (!placeable) continue;
        const double x = un(s);
        if (c < 0 || x > best) { c = s; best = x; }
      }
      if (c < 0) break;
      const double nc = (double)tb.comp(nu, c);
      double z = need / nc;
      const bool all = !(z < un(c));
      if (all) z = un(c);
      un(c) = all ? 0.0 : un(c) - z;
      for (int mu = 0; mu < E; ++mu) {
        const int nm = tb.comp(mu, c);
        if (nm == 0 || mu == nu) continue;
        if (res_of[mu] < 0) res_of[mu] = reservoir(mu);
        const int rm = res_of[mu];
        un(rm) = un(rm) + (double)nm * z / (double)tb.comp(mu, rm);
      }
      un(res) = un(res) + nc * z / nres;
      need = all ? need - nc * z : 0.0;
    }
    if (need > 0.0) st |= KR_DST_NEEDS_STAGE3;
    else { un(res) = 0.0; st |= KR_DST_STAGE3; }   // "just sufficiently": the reservoir ends at exactly zero
  }
  return st;
}

// the table-driven kernels' view of the network
struct KrPostTab {
  const KrNetDev& n;
  __device__ __forceinline__ int E() const { return n.E; }
  __device__ __forceinline__ int S() const { return n.S; }
  __device__ __forceinline__ int comp(int nu, int s) const { return n.comp[nu * n.S + s]; }
  __device__ __forceinline__ int resv(int nu, int s) const { return n.resv[nu * n.S + s]; }
  __device__ __forceinline__ int compound(int s) const { return n.compound[s]; }
  __device__ __forceinline__ int signed_row(int nu) const { return n.signed_row[nu]; }
};
