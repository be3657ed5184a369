// kr_recon.cuh -- stoichiometry-compatible reconstruction and conservative advection of the species field on a uniform
// 1-D grid (section 2.1: eq. 1 species flux, eq. 6 donor cell, eqs. 9-12 piecewise-linear states with the
// modified van Leer limiter, eq. 13 projection of the corrections onto the stoichiometric space, eq. 14 upwind choice;
// step (3) of the Godunov scheme of PAPER.md:40).  One forward-Euler stage, optionally blended with an earlier state
// (U_out = wa U0 + wb (U - lambda dF)), so that the caller can run SSP Runge-Kutta schemes.
//
// HBM-bound by design: every cell's S abundances are read once and written once.  A block owns a tile of consecutive
// cells: the tile plus two halo cells on each side is staged in shared memory with coalesced loads (the field is
// cell-major, so a tile is one contiguous range), the limited half-differences of tile + 1 halo are formed there
// (thread <-> (cell, species)), projected with the S x S matrix P held in shared memory (S FMAs per value, all operands
// on chip), and the update of the tile is written back coalesced.  No atomics, fixed summation order.
#pragma once
#include "kr_math.cuh"

#define KR_RECON_DONOR 0
#define KR_RECON_PLM 1
#define KR_RECON_PLM_PROJECTED 2

struct KrAdvectArgs {
  long long n_cells;
  int S, T;                 // species, cells per tile
  int scheme, periodic;
  double lambda, dx;        // dt / dx, dx
  double wa, wb;
  const double* y;          // [n_cells * S] cell-major
  const double* rho;        // [n_cells]
  const double* flux;       // periodic: [n_cells], flux[i] = mass flux through face i - 1/2; else [n_cells + 1]
  const double* y0;         // blend state or null
  const double* rho0;
  const double* P;          // [S * S] row-major, device
  double* y_out;
  double* rho_out;
};

// Limited half-difference of eq. 10 on a uniform grid: with the forward and backward differences dp = y_{i+1} - y_i and
// dm = y_i - y_{i-1}, the modified van Leer slope (eq. 12, reading R25: c_f = c_b = 2, the harmonic mean 2ab/(a+b) of the
// difference quotients a = dp / dx, b = dm / dx) times dx / 2 is dp dm / (dp + dm): dx cancels, one reciprocal per value.
// (FP64 divides are DFMA sequences on this chip and this kernel must stay HBM-bound: krs_rcp is 1 ulp in 5 instructions.)
__device__ __forceinline__ double kr_limited_half_difference(double dp, double dm) {
  const double prod = dp * dm;
  const double sum = dp + dm;
  return (prod > 0.0) ? prod * krs_rcp(sum) : 0.0;
}

__device__ __forceinline__ long long kr_wrap(long long c, long long n, int periodic) {
  if (periodic) { c %= n; return c < 0 ? c + n : c; }
  return c < 0 ? 0 : (c >= n ? n - 1 : c);
}

// thread <-> (cell, species) without a division per element: element i = cl * S + s advances by the block size
struct KrElemWalk {
  int cl, s, dq, dr, S;
  __device__ __forceinline__ KrElemWalk(int tid, int nthr, int S_) : cl(tid / S_), s(tid % S_), dq(nthr / S_), dr(nthr % S_), S(S_) {}
  __device__ __forceinline__ void next() { cl += dq; s += dr; if (s >= S) { s -= S; ++cl; } }
};

__global__ void __launch_bounds__(128) kr_advect_kernel(const KrAdvectArgs a) {
  extern __shared__ double kr_rs[];
  const int S = a.S, T = a.T, LDP = S | 1;
  double* sP = kr_rs;                          // [S][LDP]
  double* sy = sP + S * LDP;                   // [T + 4][S]   cells c0 - 2 .. c0 + T + 1
  double* sg = sy + (T + 4) * S;               // [T + 2][S]   limited half-differences of cells c0 - 1 .. c0 + T
  double* sd = sg + (T + 2) * S;               // [T + 2][S]   ... projected
  double* sr = sd + (T + 2) * S;               // [T][4]       per cell: rho, left flux, right flux, 1 / rho_out
  const long long c0 = (long long)blockIdx.x * T;
  const int nt = (int)min((long long)T, a.n_cells - c0);
  const int tid = threadIdx.x, nthr = blockDim.x;

  if (a.scheme == KR_RECON_PLM_PROJECTED)
    for (int i = tid; i < S * S; i += nthr) sP[(i / S) * LDP + (i % S)] = a.P[i];
  // stage the tile + halo (coalesced: consecutive threads read consecutive doubles; the interior is one contiguous range)
  {
    const long long e0 = (c0 - 2) * S, n_el = a.n_cells * S;
    const int tot = (nt + 4) * S;
    if (c0 >= 2 && c0 + nt + 2 <= a.n_cells) {
      for (int i = tid; i < tot; i += nthr) sy[i] = a.y[e0 + i];
    } else {
      for (KrElemWalk w(tid, nthr, S); w.cl < nt + 4; w.next())
        sy[w.cl * S + w.s] = a.y[kr_wrap(c0 - 2 + w.cl, a.n_cells, a.periodic) * S + w.s];
    }
    (void)n_el;
  }
  // per-cell scalars: density, the two face fluxes, the reciprocal of the new density (one per cell, not one per value)
  for (int cl = tid; cl < nt; cl += nthr) {
    const long long c = c0 + cl;
    const double fl = a.flux[c];
    const double fr = a.periodic ? a.flux[(c + 1 == a.n_cells) ? 0 : c + 1] : a.flux[c + 1];
    const double rho = a.rho[c];
    double rn = rho - a.lambda * (fr - fl);
    if (a.y0) rn = a.wa * a.rho0[c] + a.wb * rn;
    sr[4 * cl] = rho; sr[4 * cl + 1] = fl; sr[4 * cl + 2] = fr; sr[4 * cl + 3] = krs_rcp(rn);
    if (a.rho_out) a.rho_out[c] = rn;
  }
  __syncthreads();
  // limited half-differences of cells c0 - 1 .. c0 + nt (eqs. 10-12); open ends: the halo rows hold copies of the end cell
  // (zero-gradient ghost cells), whose own difference is then 0
  if (a.scheme != KR_RECON_DONOR) {
    const int tot = (nt + 2) * S;
    for (int i = tid; i < tot; i += nthr) {                    // element i of sg <-> element i + S of sy
      const double yc = sy[i + S];
      sg[i] = kr_limited_half_difference(sy[i + 2 * S] - yc, yc - sy[i]);
    }
    __syncthreads();
    if (a.scheme == KR_RECON_PLM_PROJECTED) {                  // eq. 13: d^s <- sum_r P^s_r d^r
      for (KrElemWalk w(tid, nthr, S); w.cl < nt + 2; w.next()) {
        const double* g = sg + w.cl * S;
        const double* p = sP + w.s * LDP;
        double acc = 0.0;
        for (int r = 0; r < S; ++r) acc += p[r] * g[r];
        sd[w.cl * S + w.s] = acc;
      }
    } else {
      for (int i = tid; i < tot; i += nthr) sd[i] = sg[i];
    }
  } else {
    for (int i = tid; i < (nt + 2) * S; i += nthr) sd[i] = 0.0;
  }
  __syncthreads();
  // conservative update of the tile (eq. 1, eq. 14, step 3 of PAPER.md:40)
  for (KrElemWalk w(tid, nthr, S); w.cl < nt; w.next()) {
    const int i = w.cl * S + w.s;                              // cell c0 + cl: sy row cl + 2, sd row cl + 1
    const double rho = sr[4 * w.cl], fl = sr[4 * w.cl + 1], fr = sr[4 * w.cl + 2], rinv = sr[4 * w.cl + 3];
    const double yc = sy[i + 2 * S], dc = sd[i + S];
    const double yl = (fl > 0.0) ? sy[i + S] + sd[i] : yc - dc;
    const double yr = (fr > 0.0) ? yc + dc : sy[i + 3 * S] - sd[i + 2 * S];
    double un = rho * yc - a.lambda * (yr * fr - yl * fl);
    const long long e = (c0 + w.cl) * S + w.s;
    if (a.y0) un = a.wa * a.rho0[c0 + w.cl] * a.y0[e] + a.wb * un;
    a.y_out[e] = un * rinv;
  }
}


// ---- the same stage for S <= KR_RECON_SMAX species, S a compile-time constant: thread <-> CELL --------------------------
// The generic kernel above spends ~300 instructions per value on index arithmetic, shared-memory operands and loop
// control, which makes it issue-bound at a quarter of the HBM rate.  Here a thread keeps the S values of its cell in
// registers, every loop over species is unrolled, and P travels in the kernel's parameter block: parameters live in the
// constant bank, so each of the S^2 products of eq. 13 is ONE DFMA with a constant-bank operand -- no load, no index.
#define KR_RECON_SMAX 16

template <bool V> struct KrBool { static constexpr bool value = V; };

template <int S>
struct KrAdvectArgsP {
  KrAdvectArgs a;
  double P[S * S];
};

__device__ __forceinline__ void kr_cp_async8(double* smem_dst, const double* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void kr_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void kr_cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void kr_cp_async16(double* smem_dst, const double* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}

// Persistent blocks walk the tiles with a stride of gridDim.x; the abundances of the NEXT tile are already on their way
// into the second staging buffer (cp.async, 16 bytes per request where the field allows) while the current tile is
// limited, projected and updated, so that the HBM reads overlap the arithmetic instead of alternating with it.
// A block of T threads owns T - 2 cells: the update of a tile needs the corrections of its cells and of one halo cell on
// each side, T values, so thread t forms the correction of cell c0 - 1 + t -- one pass for every thread (with T cells per
// tile the two halo corrections cost the whole first warp a second pass, and the block waited for it at the barrier).
// Two block barriers per tile: the tile has landed / the corrections are written.  The results are staged per WARP (a
// warp's 32 cells are one contiguous range of the output) and written out coalesced behind a warp-level sync.
template <int S>
struct KrAdvectTile { static constexpr int T = (S <= 10) ? 128 : 64; static constexpr int TO = T - 2; };   // < 48 KiB of static shared memory

template <int S>
__global__ void __launch_bounds__(KrAdvectTile<S>::T) kr_advect_cell_kernel(const KrAdvectArgsP<S> ap) {
  constexpr int T = KrAdvectTile<S>::T, TO = KrAdvectTile<S>::TO, LDY = S | 1;   // padded row: conflict-free 64-bit accesses
  const KrAdvectArgs& a = ap.a;
  __shared__ __align__(16) double sybuf[2][(T + 2) * LDY];   // cells c0 - 2 .. c0 + TO + 1, double buffered
  __shared__ __align__(16) double sd[T * LDY];               // corrections of cells c0 - 1 .. c0 + TO
  __shared__ __align__(16) double so[T * LDY];               // results of the tile, rows of a warp written and read by that warp only
  const int tid = threadIdx.x, lane = tid & 31, w0 = tid & ~31;
  const long long n_tiles = (a.n_cells + TO - 1) / TO;

  auto stage = [&](long long tile, double* sy) {      // asynchronous, coalesced copy of tile + halo into sy
    const long long c0 = tile * TO;
    const int nt = (int)min((long long)TO, a.n_cells - c0);
    if (c0 >= 2 && c0 + nt + 2 <= a.n_cells) {
      const double* src = a.y + (c0 - 2) * S;
      const int cnt = (nt + 4) * S;
      if (LDY == S) {
        if ((reinterpret_cast<unsigned long long>(src) & 15ull) == 0ull) {      // c0 is even: true whenever a.y is 16-byte aligned
          for (int i = tid; i < cnt / 2; i += T) kr_cp_async16(sy + 2 * i, src + 2 * i);
          if ((cnt & 1) && tid == 0) kr_cp_async8(sy + cnt - 1, src + cnt - 1);
        } else {
          for (int i = tid; i < cnt; i += T) kr_cp_async8(sy + i, src + i);
        }
      } else {
        for (int i = tid; i < cnt; i += T) kr_cp_async8(sy + (i / S) * LDY + (i % S), src + i);
      }
    } else {
      for (int i = tid; i < (nt + 4) * S; i += T) {
        const int cl = i / S, s = i % S;
        kr_cp_async8(sy + cl * LDY + s, a.y + kr_wrap(c0 - 2 + cl, a.n_cells, a.periodic) * S + s);
      }
    }
    kr_cp_async_commit();
  };

  int buf = 0;
  if ((long long)blockIdx.x < n_tiles) stage(blockIdx.x, sybuf[0]);
  for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, buf ^= 1) {
    const double* sy = sybuf[buf];
    const long long c0 = tile * TO;
    const int nt = (int)min((long long)TO, a.n_cells - c0);
    kr_cp_async_wait_all();
    __syncthreads();                                  // the tile is in sy; everybody is done with the other buffer and with sd
    if (tile + gridDim.x < n_tiles) stage(tile + gridDim.x, sybuf[buf ^ 1]);
    // the cell's scalars are requested now, so that their latency hides under the corrections
    const int cl = tid;                               // thread <-> cell c0 + cl of the update, correction of cell c0 - 1 + cl
    double fl = 0.0, fr = 0.0, rho = 1.0, r0 = 0.0;
    if (cl < nt) {
      const long long c = c0 + cl;
      fl = a.flux[c];
      fr = a.periodic ? a.flux[(c + 1 == a.n_cells) ? 0 : c + 1] : a.flux[c + 1];
      rho = a.rho[c];
      if (a.y0) r0 = a.rho0[c];
    }
    // corrections of cells c0 - 1 .. c0 + nt: limited half-differences (eqs. 10-12), projected (eq. 13)
    if (cl < nt + 2) {
      double g[S];
      if (a.scheme == KR_RECON_DONOR) {
#pragma unroll
        for (int s = 0; s < S; ++s) g[s] = 0.0;
      } else {
#pragma unroll
        for (int s = 0; s < S; ++s) {
          const double yc = sy[(cl + 1) * LDY + s];
          g[s] = kr_limited_half_difference(sy[(cl + 2) * LDY + s] - yc, yc - sy[cl * LDY + s]);
        }
      }
      if (a.scheme == KR_RECON_PLM_PROJECTED) {
#pragma unroll
        for (int s = 0; s < S; ++s) {
          double acc = 0.0;
#pragma unroll
          for (int r = 0; r < S; ++r) acc += ap.P[s * S + r] * g[r];
          sd[cl * LDY + s] = acc;
        }
      } else {
#pragma unroll
        for (int s = 0; s < S; ++s) sd[cl * LDY + s] = g[s];
      }
    }
    __syncthreads();
    // conservative update of the tile (eq. 1, eq. 14, step 3 of PAPER.md:40); results staged per warp for a coalesced write
    if (cl < nt) {
      const long long c = c0 + cl;
      double rn = rho - a.lambda * (fr - fl);
      if (a.y0) rn = a.wa * r0 + a.wb * rn;
      const double rinv = krs_rcp(rn);
      if (a.rho_out) a.rho_out[c] = rn;
      const bool lup = fl > 0.0, rup = fr > 0.0;
      // eq. 14: the upwind side of each face.  One code path per pair of directions, so that only the operands of the
      // sides that are used are read from shared memory (2 to 6 loads per species; the flow direction is coherent over
      // long stretches of cells, so the lanes of a warp mostly agree)
      auto update = [&](auto LUP, auto RUP) {
#pragma unroll
        for (int s = 0; s < S; ++s) {
          const double yc = sy[(cl + 2) * LDY + s], dc = sd[(cl + 1) * LDY + s];
          double yl, yr;
          if constexpr (decltype(LUP)::value) yl = sy[(cl + 1) * LDY + s] + sd[cl * LDY + s]; else yl = yc - dc;
          if constexpr (decltype(RUP)::value) yr = yc + dc; else yr = sy[(cl + 3) * LDY + s] - sd[(cl + 2) * LDY + s];
          double un = rho * yc - a.lambda * (yr * fr - yl * fl);
          if (a.y0) un = a.wa * r0 * a.y0[c * S + s] + a.wb * un;
          so[cl * LDY + s] = un * rinv;
        }
      };
      if (lup) { if (rup) update(KrBool<true>{}, KrBool<true>{}); else update(KrBool<true>{}, KrBool<false>{}); }
      else { if (rup) update(KrBool<false>{}, KrBool<true>{}); else update(KrBool<false>{}, KrBool<false>{}); }
    }
    __syncwarp();
    {                                                 // the warp's cells c0 + w0 .. : one contiguous range of y_out
      const int nw = min(32, nt - w0);                // may be <= 0
      double* dst = a.y_out + (c0 + w0) * S;
      const double* src = so + w0 * LDY;
      if (LDY == S) {
        if ((reinterpret_cast<unsigned long long>(dst) & 15ull) == 0ull) {
          const int cnt = nw * S;
          for (int i = lane; i < cnt / 2; i += 32) reinterpret_cast<double2*>(dst)[i] = reinterpret_cast<const double2*>(src)[i];
          if ((cnt & 1) && lane == 0) dst[cnt - 1] = src[cnt - 1];
        } else {
          for (int i = lane; i < nw * S; i += 32) dst[i] = src[i];
        }
      } else {
        for (int i = lane; i < nw * S; i += 32) dst[i] = src[(i / S) * LDY + (i % S)];
      }
    }
    __syncwarp();                                     // the warp's rows of so are free again
  }
}

template <int S>
inline cudaError_t kr_advect_cell_launch(const KrAdvectArgs& a, const double* P_host, cudaStream_t st) {
  KrAdvectArgsP<S> ap;
  ap.a = a;
  for (int i = 0; i < S * S; ++i) ap.P[i] = P_host[i];
  static int n_sm = 0;
  if (n_sm == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  }
  int per_sm = 0;
  constexpr int T = KrAdvectTile<S>::T, TO = KrAdvectTile<S>::TO;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kr_advect_cell_kernel<S>, T, 0);
  const long long n_tiles = (a.n_cells + TO - 1) / TO;
  const unsigned grid = unsigned(std::min<long long>(n_tiles, (long long)std::max(1, per_sm) * std::max(1, n_sm)));
  kr_advect_cell_kernel<S><<<grid, T, 0, st>>>(ap);
  return cudaGetLastError();
}
