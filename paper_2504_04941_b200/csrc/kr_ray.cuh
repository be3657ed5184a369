// kr_ray.cuh -- ray tracing on a uniform Cartesian mesh and the photo-reaction rate coefficients it feeds to the chemistry
// step (section 3: eqs. 23-24 cell walk, eq. 29 depletion of the ray, eqs. 30-31 rate coefficient of every
// absorbing species from every ray and energy bin).  One thread per ray: the walk is a serial chain per ray (each cell's
// depletion feeds the next cell), rays are independent.  A cell crossed by several rays receives their contributions
// through FP64 atomic adds (the sum over j in eq. 31); with one ray per cell (plane-parallel rays along a mesh axis)
// every cell has a single writer.  Cross sections travel in the parameter block (constant bank).
#pragma once

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

// (1 - exp(-tau)) / tau of eqs. 28 and 30 (reading R30)
__device__ __forceinline__ double kr_thin_factor(double tau) { return (tau == 0.0) ? 1.0 : -expm1(-tau) / tau; }

__global__ void __launch_bounds__(128) kr_raytrace_kernel(const KrRayArgs a) {
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= a.n_rays) return;
  const int n[3] = {a.nx, a.ny, a.nz};
  double d[3] = {a.dirs[3 * j], a.dirs[3 * j + 1], a.dirs[3 * j + 2]};
  const double o[3] = {a.origins[3 * j], a.origins[3 * j + 1], a.origins[3 * j + 2]};
  const double norm = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2])));
  double L[KR_RAY_MAX_BINS];
  for (int b = 0; b < a.n_bins; ++b) L[b] = a.L_in[j * a.n_bins + b];
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
    for (int step = 0; step < limit; ++step) {
      if (idx[0] < 0 || idx[0] >= n[0] || idx[1] < 0 || idx[1] >= n[1] || idx[2] < 0 || idx[2] >= n[2]) break;
      // eq. 24: 0 = x_d dl + (x_in - x_int) for the three surfaces on the side of the direction
      double dls[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        if (d[c] > 0.0) dls[c] = (__dadd_rn(a.lo[c], __dmul_rn((double)(idx[c] + 1), a.h[c])) - x[c]) / d[c];
        else if (d[c] < 0.0) dls[c] = (__dadd_rn(a.lo[c], __dmul_rn((double)idx[c], a.h[c])) - x[c]) / d[c];
        else dls[c] = __longlong_as_double(0x7ff0000000000000LL);
      }
      const double dl = fmax(fmin(fmin(dls[0], dls[1]), dls[2]), 0.0);        // the smallest positive solution
      const long long cell = ((long long)idx[0] * a.ny + idx[1]) * a.nz + idx[2];
      total += dl;
      // eqs. 29-31 in this cell
      double nd[KR_RAY_MAX_ABS];
      for (int i = 0; i < a.n_abs; ++i) nd[i] = a.n_dens[(long long)i * a.n_cells + cell];
      double add[KR_RAY_MAX_ABS];
      for (int i = 0; i < a.n_abs; ++i) add[i] = 0.0;
      for (int b = 0; b < a.n_bins; ++b) {
        double tau = 0.0;
        for (int i = 0; i < a.n_abs; ++i) tau += nd[i] * a.sigma[i * a.n_bins + b] * dl;
        const double f = kr_thin_factor(tau);
        for (int i = 0; i < a.n_abs; ++i) add[i] += L[b] * a.sigma[i * a.n_bins + b] * dl * inv_dV * f;
        L[b] *= exp(-tau);
      }
      for (int i = 0; i < a.n_abs; ++i)
        if (add[i] != 0.0) atomicAdd(a.k_out + (long long)i * a.n_cells + cell, add[i]);
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
    }
  }
  if (a.L_out) for (int b = 0; b < a.n_bins; ++b) a.L_out[j * a.n_bins + b] = L[b];
  if (a.path) a.path[j] = total;
}
