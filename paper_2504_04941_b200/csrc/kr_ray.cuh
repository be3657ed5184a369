// kr_ray.cuh -- ray tracing on a uniform Cartesian mesh and the photo-reaction rate coefficients it feeds to the chemistry
// step (section 3: eqs. 23-24 cell walk, eq. 29 depletion of the ray, eqs. 30-31 rate coefficient of every
// absorbing species from every ray and energy bin).  One thread per ray: the walk is a serial chain per ray (each cell's
// depletion feeds the next cell), rays are independent.  A cell crossed by several rays receives their contributions
// through FP64 atomic adds (the sum over j in eq. 31); with one ray per cell (plane-parallel rays along a mesh axis)
// every cell has a single writer.  Cross sections travel in the parameter block (constant bank).
#pragma once
#include "kr_math.cuh"

#define KR_RAY_MAX_ABS 8
#define KR_RAY_MAX_BINS 16

struct KrRayArgs {
  int nx, ny, nz, n_abs, n_bins;
  long long n_rays, n_cells;
  double h[3], lo[3];
  const double* origins;      // [n_rays * 3]
  const double* dirs;         // [n_rays * 3]
  const double* L_in;         // [n_rays * n_bins]
  const double* n_dens;       // [n_abs * n_cells], cell = (ix * ny + iy) * nz + iz
  double* k_out;              // [n_abs * n_cells], zeroed before the launch
  double* L_out;              // [n_rays * n_bins] or null
  double* path;               // [n_rays] or null
  double sigma[KR_RAY_MAX_ABS * KR_RAY_MAX_BINS];   // [n_abs][n_bins]
};

// exp(x) and expm1(x) for x <= 0 from ONE reduction and ONE polynomial (eqs. 28-30 need both in every cell and energy bin:
// the attenuation exp(-tau) and, reading R30, (1 - exp(-tau)) / tau as -expm1(-tau) / tau).  x = n ln 2 + r, |r| <= ln 2 / 2;
// p = expm1(r) as r times a degree-12 Taylor polynomial; exp = 2^n + 2^n p, expm1 = (2^n - 1) + 2^n p, both one FMA on exact
// operands: <= 1.8e-16 / 2.8e-16 relative against long-double exp / expm1 on 3e7 arguments in [-700, -1e-12].  Below -708
// the pair is (0, -1) (the attenuated photon count there is < 1e-307 of the incoming one).
__device__ __forceinline__ void kr_exp_pair(double x, double& e, double& m) {
  const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);
  const int n = __double2loint(t);
  const double fn = t - 6755399441055744.0;
  double r = fma(fn, -6.93147180369123816490e-01, x);
  r = fma(fn, -1.90821492927058770002e-10, r);
  double p = 1.0 / 6227020800.0;
  p = fma(p, r, 1.0 / 479001600.0);
  p = fma(p, r, 1.0 / 39916800.0);
  p = fma(p, r, 1.0 / 3628800.0);
  p = fma(p, r, 1.0 / 362880.0);
  p = fma(p, r, 1.0 / 40320.0);
  p = fma(p, r, 1.0 / 5040.0);
  p = fma(p, r, 1.0 / 720.0);
  p = fma(p, r, 1.0 / 120.0);
  p = fma(p, r, 1.0 / 24.0);
  p = fma(p, r, 1.0 / 6.0);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = p * r;
  const double s = __hiloint2double((1023 + n) << 20, 0);      // 2^n, -1022 <= n <= 0
  const bool tiny = x < -708.0;
  e = tiny ? 0.0 : fma(s, p, s);
  m = tiny ? -1.0 : fma(s, p, s - 1.0);
}

// NA, NB > 0: the numbers of absorbers and energy bins are compile-time constants (every per-cell array is then a set of
// registers; with run-time bounds they are local-memory arrays); 0: run-time bounds up to the maxima.
template <int NA, int NB>
__global__ void __launch_bounds__(128) kr_raytrace_kernel(const KrRayArgs a) {
  constexpr int MA = NA > 0 ? NA : KR_RAY_MAX_ABS, MB = NB > 0 ? NB : KR_RAY_MAX_BINS;
  const int n_abs = NA > 0 ? NA : a.n_abs, n_bins = NB > 0 ? NB : a.n_bins;
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= a.n_rays) return;
  const int n[3] = {a.nx, a.ny, a.nz};
  double d[3] = {a.dirs[3 * j], a.dirs[3 * j + 1], a.dirs[3 * j + 2]};
  const double o[3] = {a.origins[3 * j], a.origins[3 * j + 1], a.origins[3 * j + 2]};
  const double norm = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2])));
  double L[MB];
#pragma unroll
  for (int b = 0; b < MB; ++b) L[b] = (b < n_bins) ? a.L_in[j * n_bins + b] : 0.0;
  double total = 0.0;
  // entry into the mesh: slab method
  double t0 = 0.0, t1 = __longlong_as_double(0x7ff0000000000000LL);
  bool hit = true;
  double hi[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    d[c] = d[c] / norm;
    hi[c] = __dadd_rn(a.lo[c], __dmul_rn((double)n[c], a.h[c]));
    if (d[c] == 0.0) { hit = hit && !(o[c] < a.lo[c] || o[c] > hi[c]); continue; }
    double ta = (a.lo[c] - o[c]) / d[c], tb = (hi[c] - o[c]) / d[c];
    if (ta > tb) { const double s = ta; ta = tb; tb = s; }
    t0 = fmax(t0, ta); t1 = fmin(t1, tb);
  }
  hit = hit && (t0 <= t1);
  if (hit) {
    double x[3];
    int idx[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      x[c] = __dadd_rn(o[c], __dmul_rn(t0, d[c]));
      const double q = (x[c] - a.lo[c]) / a.h[c];
      int i = (int)floor(q);
      if (q == (double)i && d[c] < 0.0) i -= 1;          // on a face: the cell on the side of the direction
      idx[c] = min(max(i, 0), n[c] - 1);
    }
    const double inv_dV = 1.0 / (a.h[0] * a.h[1] * a.h[2]);
    const int limit = a.nx + a.ny + a.nz + 3;
    // the absorber densities of a cell are requested as soon as the walk knows the cell -- at the end of the step before --
    // so that their latency hides under eq. 24 of the step that uses them
    double nd[MA];
    auto request = [&]() {
      const bool in = !(idx[0] < 0 || idx[0] >= n[0] || idx[1] < 0 || idx[1] >= n[1] || idx[2] < 0 || idx[2] >= n[2]);
      const long long cn = in ? ((long long)idx[0] * a.ny + idx[1]) * a.nz + idx[2] : 0;
#pragma unroll
      for (int i = 0; i < MA; ++i) nd[i] = (in && i < n_abs) ? __ldg(a.n_dens + (long long)i * a.n_cells + cn) : 0.0;
    };
    request();
    for (int step = 0; step < limit; ++step) {
      if (idx[0] < 0 || idx[0] >= n[0] || idx[1] < 0 || idx[1] >= n[1] || idx[2] < 0 || idx[2] >= n[2]) break;
      // eq. 24: 0 = x_d dl + (x_in - x_int) for the three surfaces on the side of the direction
      double dls[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        // (a component of +-1 -- a ray along a mesh axis -- divides exactly: the product is the same number without the
        // FP64 divide, which is a ~25-instruction routine on this chip)
        if (d[c] > 0.0) { const double df = __dadd_rn(a.lo[c], __dmul_rn((double)(idx[c] + 1), a.h[c])) - x[c]; dls[c] = (d[c] == 1.0) ? df : df / d[c]; }
        else if (d[c] < 0.0) { const double df = __dadd_rn(a.lo[c], __dmul_rn((double)idx[c], a.h[c])) - x[c]; dls[c] = (d[c] == -1.0) ? -df : df / d[c]; }
        else dls[c] = __longlong_as_double(0x7ff0000000000000LL);
      }
      const double dl = fmax(fmin(fmin(dls[0], dls[1]), dls[2]), 0.0);        // the smallest positive solution
      const long long cell = ((long long)idx[0] * a.ny + idx[1]) * a.nz + idx[2];
      total += dl;
      // eqs. 29-31 in this cell
      double add[MA];
#pragma unroll
      for (int i = 0; i < MA; ++i) add[i] = 0.0;
#pragma unroll
      for (int b = 0; b < MB; ++b)
        if (b < n_bins) {
          double tau = 0.0;
#pragma unroll
          for (int i = 0; i < MA; ++i)
            if (i < n_abs) tau += nd[i] * a.sigma[i * n_bins + b] * dl;
          double e, m;
          kr_exp_pair(-tau, e, m);
          // (1 - exp(-tau)) / tau of eqs. 28 and 30 (reading R30); the reciprocal by krs_rcp (1 ulp, 5 instructions) for normal tau
          const double f = (tau == 0.0) ? 1.0 : ((tau > 1e-290) ? -m * krs_rcp(tau) : -m / tau);
#pragma unroll
          for (int i = 0; i < MA; ++i)                             // in this order: deep inside an absorber L sigma is subnormal
            if (i < n_abs) add[i] += L[b] * a.sigma[i * n_bins + b] * dl * inv_dV * f;
          L[b] *= e;
        }
#pragma unroll
      for (int i = 0; i < MA; ++i)
        if (i < n_abs && add[i] != 0.0) atomicAdd(a.k_out + (long long)i * a.n_cells + cell, add[i]);
      // leave through every surface reached at dl (edges and corners: several at once)
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        if (dls[c] <= dl) {
          idx[c] += (d[c] > 0.0) ? 1 : -1;
          x[c] = __dadd_rn(a.lo[c], __dmul_rn((double)(idx[c] + ((d[c] > 0.0) ? 0 : 1)), a.h[c]));    // exactly on the surface
        } else {
          x[c] = __dadd_rn(x[c], __dmul_rn(dl, d[c]));
        }
      }
      request();
    }
  }
  if (a.L_out) {
#pragma unroll
    for (int b = 0; b < MB; ++b)
      if (b < n_bins) a.L_out[j * n_bins + b] = L[b];
  }
  if (a.path) a.path[j] = total;
}
