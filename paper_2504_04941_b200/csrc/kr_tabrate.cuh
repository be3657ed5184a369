// kr_tabrate.cuh -- tabulated reaction rates (rate type 3 of section 2.3): "multi-dimensional tables are
// reduced to one-dimensional in T per cell, assuming fixed total mass density and elemental abundances during
// thermochemical steps", then interpolated at the cell's temperature.  Readings R32 / R33 of DESIGN.md: tables in
// (ln rho, ln T) on uniform nodes, piecewise linear in the logarithms, end values outside the table.  One thread per cell
// and launch: the cell's density fixes the two density nodes and their weights ONCE (the reduction: of the 1-D table in T
// that belongs to the cell only the two nodes that bracket its temperature are ever formed), every table is then
// evaluated with four loads from the (L1 / L2 resident) table.  HBM traffic: 16 B in, 8 B per table out, per cell.
#pragma once

struct KrTabArgs {
  long long n_cells;
  int n_tab, n_rho, n_T;
  double ln_rho0, d_ln_rho, ln_T0, d_ln_T;
  const double* ln_k;       // [n_tab][n_rho][n_T]
  const double* rho;        // [n_cells]
  const double* T;          // [n_cells]
  double* k_out;            // [n_tab][n_cells]
};

// fractional position on a uniform grid of n nodes: the interval index (0 .. n - 2) and the weight of its upper node
__device__ __forceinline__ void kr_tab_locate(double lx, double x0, double dx, int n, int& i, double& f) {
  double x = (lx - x0) / dx;
  x = fmin(fmax(x, 0.0), (double)(n - 1));
  i = min((int)floor(x), n - 2);
  f = x - (double)i;
}

__global__ void __launch_bounds__(256) kr_table_rates_kernel(const KrTabArgs a) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < a.n_cells; c += stride) {
    int i = 0, j = 0;
    double fr = 0.0, ft = 0.0;
    if (a.n_rho > 1) kr_tab_locate(log(a.rho[c]), a.ln_rho0, a.d_ln_rho, a.n_rho, i, fr);
    if (a.n_T > 1) kr_tab_locate(log(a.T[c]), a.ln_T0, a.d_ln_T, a.n_T, j, ft);
    for (int t = 0; t < a.n_tab; ++t) {
      const double* tab = a.ln_k + ((size_t)t * a.n_rho + i) * a.n_T + j;
      double lo = tab[0], hi = (a.n_T > 1) ? tab[1] : 0.0;
      if (a.n_rho > 1) {                                  // the cell's 1-D table at the two bracketing T nodes
        lo = (1.0 - fr) * lo + fr * tab[a.n_T];
        if (a.n_T > 1) hi = (1.0 - fr) * hi + fr * tab[a.n_T + 1];
      }
      const double lnk = (a.n_T > 1) ? (1.0 - ft) * lo + ft * hi : lo;
      a.k_out[(size_t)t * a.n_cells + c] = exp(lnk);
    }
  }
}
