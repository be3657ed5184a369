// kr_tabrate.cuh -- tabulated reaction rates (rate type 3 of section 2.3): "multi-dimensional tables are
// reduced to one-dimensional in T per cell, assuming fixed total mass density and elemental abundances during
// thermochemical steps", then interpolated at the cell's temperature.  Readings R32 / R33 of DESIGN.md: tables in
// (ln rho, ln T) on uniform nodes, piecewise linear in the logarithms, end values outside the table.  One thread per cell
// and launch: the cell's density fixes the two density nodes and their weights ONCE (the reduction: of the 1-D table in T
// that belongs to the cell only the two nodes that bracket its temperature are ever formed), every table is then
// evaluated with four loads from the (L1 / L2 resident) table.  HBM traffic: 16 B in, 8 B per table out, per cell.
#pragma once
#include "kr_math.cuh"

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
__device__ __forceinline__ void kr_tab_locate(double lx, double x0, double inv_dx, int n, int& i, double& f) {
  double x = (lx - x0) * inv_dx;
  x = fmin(fmax(x, 0.0), (double)(n - 1));
  i = min((int)floor(x), n - 2);
  f = x - (double)i;
}

// STAGED: the tables fit shared memory (<= 200 KiB) and every block copies them there first (one coalesced pass over an L2
// resident array): the node loads are gathers at the cells' temperatures -- 32 different sectors per warp and load -- and
// the L1's tag rate, not arithmetic or HBM, bound the kernel while they went to global memory (measured: a leaner exp and
// batched loads changed nothing); shared memory serves a gather of 8-byte words at bank speed.
template <bool STAGED>
__global__ void __launch_bounds__(STAGED ? 1024 : 256) kr_table_rates_kernel(const KrTabArgs a) {
  extern __shared__ __align__(16) double kr_tab_sm[];
  const double* table = a.ln_k;
  if (STAGED) {
    const int n = a.n_tab * a.n_rho * a.n_T;
    for (int q = threadIdx.x; q < n; q += blockDim.x) kr_tab_sm[q] = __ldg(a.ln_k + q);
    __syncthreads();
    table = kr_tab_sm;
  }
  const long long stride = (long long)gridDim.x * blockDim.x;
  // FP64 divides and libm's exp are long DFMA strings on this chip and this kernel should stay HBM bound: the two spacings are
  // inverted once (krs_rcp, 1 ulp), exp is the lean krs_exp_core (1 ulp) inside its range and libm's outside
  const double inv_d_rho = (a.n_rho > 1) ? krs_rcp(a.d_ln_rho) : 0.0, inv_d_T = (a.n_T > 1) ? krs_rcp(a.d_ln_T) : 0.0;
  for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < a.n_cells; c += stride) {
    int i = 0, j = 0;
    double fr = 0.0, ft = 0.0;
    if (a.n_rho > 1) kr_tab_locate(log(a.rho[c]), a.ln_rho0, inv_d_rho, a.n_rho, i, fr);
    if (a.n_T > 1) kr_tab_locate(log(a.T[c]), a.ln_T0, inv_d_T, a.n_T, j, ft);
    // tables in batches of TB: the (independent, L1 / L2 resident) node loads of a batch are requested before the first
    // of them is used, and the TB exponentials run as independent chains (one table at a time left the thread waiting for
    // a cache latency and a dependent exp chain per table)
    constexpr int TB = 3;
    for (int t0 = 0; t0 < a.n_tab; t0 += TB) {
      double lo[TB], hi[TB], lo2[TB], hi2[TB];
#pragma unroll
      for (int q = 0; q < TB; ++q) {
        const int t = min(t0 + q, a.n_tab - 1);
        const double* tab = table + ((size_t)t * a.n_rho + i) * a.n_T + j;
        lo[q] = tab[0]; hi[q] = (a.n_T > 1) ? tab[1] : 0.0;
        lo2[q] = 0.0; hi2[q] = 0.0;
        if (a.n_rho > 1) { lo2[q] = tab[a.n_T]; if (a.n_T > 1) hi2[q] = tab[a.n_T + 1]; }
      }
      double k[TB];
#pragma unroll
      for (int q = 0; q < TB; ++q) {
        double l = lo[q], h = hi[q];
        if (a.n_rho > 1) {                                // the cell's 1-D table at the two bracketing T nodes
          l = (1.0 - fr) * l + fr * lo2[q];
          if (a.n_T > 1) h = (1.0 - fr) * h + fr * hi2[q];
        }
        const double lnk = (a.n_T > 1) ? (1.0 - ft) * l + ft * h : l;
        k[q] = (lnk > -700.0 && lnk < 690.0) ? krs_exp_core(lnk) : exp(lnk);
      }
#pragma unroll
      for (int q = 0; q < TB; ++q)
        if (t0 + q < a.n_tab) a.k_out[(size_t)(t0 + q) * a.n_cells + c] = k[q];
    }
  }
}
