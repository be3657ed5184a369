// kr_device.cuh -- device helpers shared by the thread-per-cell and group-per-cell kernels:
// thermo polynomials (reading R7), rate constants (eq. 16 with R4;
// detailed balance R5; unary R16/R17), small integer powers.  fp64 throughout.
#pragma once
#include "kr_tables.h"

__device__ __forceinline__ double kr_ipow(double x, int e) {
  // e in 0..3 (reaction order <= 3 per side, R20)
  double p = 1.0;
  if (e >= 1) p = x;
  if (e >= 2) p *= x;
  if (e >= 3) p *= x;
  return p;
}

__device__ __forceinline__ double kr_exp_clamped(double lnk) {   // R18: clamp at +690, underflow allowed
  return exp(lnk > KR_EXP_CLAMP ? KR_EXP_CLAMP : lnk);
}

// Thermo of one species at T (step 2 of DESIGN.md "Algorithm"):
//   cp/R = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4
//   h/RT = a1 + a2 T/2 + a3 T^2/3 + a4 T^3/4 + a5 T^4/5 + a6/T
//   s/R  = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7
//   ghat = h/RT - s/R, uhat = h/RT - 1, chat = cp/R - 1
__device__ __forceinline__ void kr_thermo_species(const double* __restrict__ nasa14, double T_mid, double T, double invT,
                                                  double lnT, double& ghat, double& uhat, double& chat) {
  const double* a = (T <= T_mid) ? nasa14 : nasa14 + 7;
  const double a0 = a[0], a1 = a[1], a2 = a[2], a3 = a[3], a4 = a[4], a5 = a[5], a6 = a[6];
  const double T2 = T * T, T3 = T2 * T, T4 = T3 * T;
  const double cp = a0 + a1 * T + a2 * T2 + a3 * T3 + a4 * T4;
  const double h = a0 + a1 * T * 0.5 + a2 * T2 * (1.0 / 3.0) + a3 * T3 * 0.25 + a4 * T4 * 0.2 + a5 * invT;
  const double s = a0 * lnT + a1 * T + a2 * T2 * 0.5 + a3 * T3 * (1.0 / 3.0) + a4 * T4 * 0.25 + a6;
  ghat = h - s;
  uhat = h - 1.0;
  chat = cp - 1.0;
}

// Rate constants of reaction r at T (step 3).  GH(s) / UH(s) return ghat_s / uhat_s of the cell.
//   ln k_f = ln A + beta (ln T - ln T_ref) - Ea/T ; ln K_c = -sum dnu_s ghat_s + dnu ln(p0 / k_B T)
//   ln k_r = ln k_f - ln K_c ; d ln k_f/dT = (beta + Ea/T)/T ; d ln k_r/dT = d ln k_f/dT - (sum dnu_s uhat_s)/T
template <class GH, class UH>
__device__ __forceinline__ void kr_rate_constants(const KrNetDev& n, int r, int fl, double invT, double lnT,
                                                  double aux_val, GH gh, UH uh, double& kf, double& kr, double& dlnkf,
                                                  double& dlnkr) {
  kr = 0.0; dlnkf = 0.0; dlnkr = 0.0;
  if (fl & KR_DF_CONST) { kf = n.A[r]; return; }
  if (fl & KR_DF_AUX) { kf = n.A[r] * aux_val; return; }
  const double beta = n.beta[r], Ea = n.Ea[r];
  const double lnkf = n.c0[r] + beta * lnT - Ea * invT;
  kf = kr_exp_clamped(lnkf);
  dlnkf = (beta + Ea * invT) * invT;
  if (fl & KR_DF_REV) {
    double sum_g = 0.0, sum_u = 0.0;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const int s = n.sp[6 * r + k];
      if (s >= 0) {
        const double c = (k < 3) ? -(double)n.nu[6 * r + k] : (double)n.nu[6 * r + k];
        sum_g += c * gh(s);
        sum_u += c * uh(s);
      }
    }
    const double lnKc = -sum_g + (double)n.dnu_tot[r] * (n.ln_p0_kB - lnT);
    kr = kr_exp_clamped(lnkf - lnKc);
    dlnkr = dlnkf - sum_u * invT;
  }
}

__device__ __forceinline__ bool kr_finite(double x) { return fabs(x) <= 1.79769313486231570e308; }  // false for NaN/inf
