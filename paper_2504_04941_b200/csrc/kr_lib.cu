// kr_lib.cu -- host side of libkratos_chem.so: the C ABI of include/kratos_chem.h.
// Network validation and table construction (host), device upload, mapping choice, kernel launches,
// statistics, the host-buffer (end-to-end) variant, the layout kernels and the FP64 peak microbenchmark.
// No CPU fallback: every compute entry point fails with KR_ECUDA when there is no CUDA device.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

#include "../../include/kratos_chem.h"
#include "kr_grp.cuh"
#include "kr_tpc.cuh"

namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}

#define KR_CUDA(call)                                                                              \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) return fail(KR_ECUDA, "%s failed: %s", #call, cudaGetErrorString(e_));  \
  } while (0)

template <class T>
size_t push(std::vector<unsigned char>& blob, const std::vector<T>& v) {
  size_t off = (blob.size() + 15) & ~size_t(15);
  blob.resize(off + std::max<size_t>(v.size(), 1) * sizeof(T));
  if (!v.empty()) std::memcpy(blob.data() + off, v.data(), v.size() * sizeof(T));
  return off;
}

}  // namespace

struct kr_network {
  int E = 0, S = 0, R = 0, N = 0, energy = 0, n_aux = 0;
  KrNetDev dev{};
  kr_solver_opts opts{};
  void* blob = nullptr;            // device tables
  unsigned long long* ws = nullptr;  // device: [0] work counter, [1..6] statistics
  cudaStream_t stream = nullptr;
  int mapping = KR_MAP_THREAD, tpc = 32, smem = 0, cells_per_block = 1, block = 64, grid_cap = 0, n_sm = 0;
  int last_launches = 0;
  // host-variant staging
  double *s_rho = nullptr, *s_T = nullptr, *s_y = nullptr, *s_aux = nullptr;
  int32_t* s_status = nullptr;
  int64_t s_cells = 0;
  int s_naux = 0;
};

namespace {

KrOptsDev to_dev(const kr_solver_opts& o) {
  KrOptsDev d;
  d.max_newton = o.max_newton; d.fixed_newton = o.fixed_newton; d.h0_mode = o.h0_mode; d.it_fast = o.it_fast;
  d.it_mid = o.it_mid; d.max_substeps = o.max_substeps; d.finalize = o.finalize;
  d.rtol = o.rtol; d.atol_y = o.atol_y; d.atol_T = o.atol_T; d.neg_tol = o.neg_tol; d.eta = o.eta; d.y_floor = o.y_floor;
  d.shrink = o.shrink; d.grow_fast = o.grow_fast; d.grow_mid = o.grow_mid; d.chg_floor = o.chg_floor; d.chg_max = o.chg_max;
  d.h_min_rel = o.h_min_rel; d.bail_ratio = o.bail_ratio;
  return d;
}

template <class K>
int max_blocks_per_sm(K kernel, int block, size_t smem) {
  int nb = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, block, smem) != cudaSuccess) { cudaGetLastError(); nb = 0; }
  return nb;
}

// pick block shape, shared memory and grid cap for the current mapping; returns KR_OK or an error
int configure(kr_network* n) {
  const int N = n->N, S = n->S, R = n->R;
  const size_t smem_max = 227 * 1024;
  if (n->mapping == KR_MAP_THREAD) {
    if (N > KR_TPC_MAX_N) return fail(KR_EUNSUPPORTED, "thread-per-cell mapping supports N <= %d (N = %d)", KR_TPC_MAX_N, N);
    const size_t per_lane = size_t(kr_tpc_doubles_per_lane(N, S, R, n->energy)) * sizeof(double);
    int bd = KR_TPC_BD;
    while (bd > 32 && per_lane * bd > smem_max) bd /= 2;
    if (per_lane * bd > smem_max) return fail(KR_EUNSUPPORTED, "thread-per-cell state (%zu B per lane) does not fit shared memory", per_lane);
    n->block = bd; n->tpc = 1; n->cells_per_block = bd; n->smem = int(per_lane * bd);
    int nb;
    if (n->energy) {
      KR_CUDA(cudaFuncSetAttribute(kr_tpc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, n->smem));
      nb = max_blocks_per_sm(kr_tpc_kernel<true>, bd, n->smem);
    } else {
      KR_CUDA(cudaFuncSetAttribute(kr_tpc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, n->smem));
      nb = max_blocks_per_sm(kr_tpc_kernel<false>, bd, n->smem);
    }
    if (nb < 1) return fail(KR_ECUDA, "thread-per-cell kernel cannot be resident (smem %d B)", n->smem);
    n->grid_cap = nb * n->n_sm;
    return KR_OK;
  }
  int W = n->tpc / 32;
  if (W != 1 && W != 2 && W != 4 && W != 8) return fail(KR_EINVAL, "threads_per_cell must be 32, 64, 128 or 256");
  const KrGrpLayout L = kr_grp_layout(N, S, R, n->dev.ld, n->energy, n->dev.any_tb, W);
  const size_t per_cell = size_t(L.total) * sizeof(double);
  if (per_cell > smem_max) return fail(KR_EUNSUPPORTED, "per-cell state (%zu B) does not fit shared memory (N = %d)", per_cell, N);
  int cpb = std::max(1, std::min(128 / (32 * W), int((64 * 1024) / per_cell)));
  cpb = std::min(cpb, 15);
  n->cells_per_block = cpb; n->block = 32 * W * cpb; n->smem = int(per_cell * cpb);
  int nb = 0;
#define KR_GRP_CFG(EN, WW)                                                                                         \
  do {                                                                                                             \
    KR_CUDA(cudaFuncSetAttribute(kr_grp_kernel<EN, WW>, cudaFuncAttributeMaxDynamicSharedMemorySize, n->smem));    \
    nb = max_blocks_per_sm(kr_grp_kernel<EN, WW>, n->block, n->smem);                                              \
  } while (0)
  if (n->energy) { if (W == 1) KR_GRP_CFG(true, 1); else if (W == 2) KR_GRP_CFG(true, 2); else if (W == 4) KR_GRP_CFG(true, 4); else KR_GRP_CFG(true, 8); }
  else { if (W == 1) KR_GRP_CFG(false, 1); else if (W == 2) KR_GRP_CFG(false, 2); else if (W == 4) KR_GRP_CFG(false, 4); else KR_GRP_CFG(false, 8); }
#undef KR_GRP_CFG
  if (nb < 1) return fail(KR_ECUDA, "group kernel cannot be resident (smem %d B, block %d)", n->smem, n->block);
  n->grid_cap = nb * n->n_sm;
  return KR_OK;
}

void auto_mapping(kr_network* n) {
  // thread-per-cell for N <= 12, one warp per cell up to N = 64, a CTA slice above.
  if (n->N <= 12) { n->mapping = KR_MAP_THREAD; n->tpc = 1; }
  else if (n->N <= 64) { n->mapping = KR_MAP_WARP; n->tpc = 32; }
  else { n->mapping = KR_MAP_CTA; n->tpc = (n->N <= 128) ? 64 : 128; }
}

int launch_step(kr_network* n, int64_t n_cells, const double* rho, double* T, double* y, double dt, int mode,
                const double* aux, int32_t* status, cudaStream_t st) {
  if (mode != KR_FP64) return fail(KR_EUNSUPPORTED, "precision_mode %d is not built yet", mode);
  KrStepArgs a;
  a.n_cells = n_cells; a.rho = rho; a.T = T; a.y = y; a.aux = aux; a.status = status; a.dt = dt;
  a.counter = n->ws; a.stats = n->ws + 1;
  KR_CUDA(cudaMemsetAsync(n->ws, 0, 8 * sizeof(unsigned long long), st));
  n->last_launches = 0;
  if (n_cells == 0) return KR_OK;
  const KrOptsDev od = to_dev(n->opts);
  const int64_t blocks_needed = (n_cells + n->cells_per_block - 1) / n->cells_per_block;
  const int grid = int(std::min<int64_t>(blocks_needed, n->grid_cap));
  if (n->mapping == KR_MAP_THREAD) {
    if (n->energy) kr_tpc_kernel<true><<<grid, n->block, n->smem, st>>>(n->dev, od, a);
    else kr_tpc_kernel<false><<<grid, n->block, n->smem, st>>>(n->dev, od, a);
  } else {
    const int W = n->tpc / 32;
#define KR_GRP_GO(EN, WW) kr_grp_kernel<EN, WW><<<grid, n->block, n->smem, st>>>(n->dev, od, a)
    if (n->energy) { if (W == 1) KR_GRP_GO(true, 1); else if (W == 2) KR_GRP_GO(true, 2); else if (W == 4) KR_GRP_GO(true, 4); else KR_GRP_GO(true, 8); }
    else { if (W == 1) KR_GRP_GO(false, 1); else if (W == 2) KR_GRP_GO(false, 2); else if (W == 4) KR_GRP_GO(false, 4); else KR_GRP_GO(false, 8); }
#undef KR_GRP_GO
  }
  n->last_launches = 1;
  KR_CUDA(cudaGetLastError());
  return KR_OK;
}

int fetch_stats(kr_network* n, kr_step_stats* stats, cudaStream_t st) {
  unsigned long long h[8];
  KR_CUDA(cudaMemcpyAsync(h, n->ws, sizeof h, cudaMemcpyDeviceToHost, st));
  KR_CUDA(cudaStreamSynchronize(st));
  stats->n_substeps = (int64_t)h[1]; stats->n_rejected = (int64_t)h[2]; stats->n_newton = (int64_t)h[3];
  stats->n_lu = (int64_t)h[4]; stats->n_rate_evals = (int64_t)h[5]; stats->n_failed = (int64_t)h[6];
  return KR_OK;
}

// ---- layout kernels: cell-major <-> species-SoA through a padded shared tile --------------------------
__global__ void kr_cell_to_soa_kernel(const double* __restrict__ yc, double* __restrict__ ys, long long n_cells, int S) {
  extern __shared__ double tile[];                       // [256][S | 1]
  const int ldt = S | 1;
  const long long c0 = (long long)blockIdx.x * blockDim.x;
  const long long nloc = min((long long)blockDim.x, n_cells - c0);
  for (long long i = threadIdx.x; i < nloc * S; i += blockDim.x) tile[(i / S) * ldt + (i % S)] = yc[c0 * S + i];
  __syncthreads();
  if (threadIdx.x < nloc)
    for (int s = 0; s < S; ++s) ys[(long long)s * n_cells + c0 + threadIdx.x] = tile[threadIdx.x * ldt + s];
}

__global__ void kr_soa_to_cell_kernel(const double* __restrict__ ys, double* __restrict__ yc, long long n_cells, int S) {
  extern __shared__ double tile[];
  const int ldt = S | 1;
  const long long c0 = (long long)blockIdx.x * blockDim.x;
  const long long nloc = min((long long)blockDim.x, n_cells - c0);
  if (threadIdx.x < nloc)
    for (int s = 0; s < S; ++s) tile[threadIdx.x * ldt + s] = ys[(long long)s * n_cells + c0 + threadIdx.x];
  __syncthreads();
  for (long long i = threadIdx.x; i < nloc * S; i += blockDim.x) yc[c0 * S + i] = tile[(i / S) * ldt + (i % S)];
}

// ---- FP64 peak: 8 independent DFMA chains per thread ---------------------------------------------------
__global__ void kr_dfma_kernel(double* out, int n_iter, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < n_iter; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

}  // namespace

extern "C" {

const char* kr_last_error(void) { return g_err.c_str(); }
const char* kr_version(void) { return "kratos-chem-b200 0.1 (sm_100a)"; }

void kr_default_opts(kr_solver_opts* o) {
  if (!o) return;
  o->max_newton = 8; o->fixed_newton = 0; o->h0_mode = 1;
  o->rtol = 1e-8; o->atol_y = 1e-20; o->atol_T = 1e-8; o->neg_tol = 1e-12; o->eta = 0.1; o->y_floor = 1e-12;
  o->shrink = 0.25; o->grow_fast = 8.0; o->grow_mid = 2.0; o->chg_floor = 1e-12;
  o->chg_max = std::numeric_limits<double>::infinity();
  o->it_fast = 3; o->it_mid = 5; o->max_substeps = 4096; o->finalize = 1; o->h_min_rel = 1e-12; o->bail_ratio = 10.0;
}

int kr_network_create(const kr_network_desc* d, kr_network** out) {
  if (!d || !out) return fail(KR_EINVAL, "null argument");
  *out = nullptr;
  const int E = d->n_elem, S = d->n_species, R = d->n_reac;
  if (E <= 0 || S <= 0 || R < 0) return fail(KR_EINVAL, "bad sizes E=%d S=%d R=%d", E, S, R);
  if (!d->elem_mass || !d->composition || !d->nasa_lo || !d->nasa_hi || !d->T_mid) return fail(KR_EINVAL, "null table");
  if (R > 0 && (!d->reac_idx || !d->reac_nu || !d->prod_idx || !d->prod_nu || !d->A || !d->beta || !d->Ea_over_k || !d->flags))
    return fail(KR_EINVAL, "null reaction table");
  if (!(d->T_lo > 0) || !(d->T_hi >= d->T_lo)) return fail(KR_EINVAL, "bad temperature range");
  if (R >= (1 << 23)) return fail(KR_EUNSUPPORTED, "too many reactions");

  std::vector<int> sp(6 * size_t(R), -1), nu(6 * size_t(R), 0), flags(R), auxi(R, -1), dnu_tot(R, 0);
  std::vector<double> c0(R), A(R), beta(R), Ea(R), qk(R, 0.0), tb;
  int n_aux = 0, any_rev = 0, any_tb = 0, any_qext = 0;
  for (int r = 0; r < R; ++r) {
    int order_r = 0, order_p = 0;
    std::vector<long> tot(E, 0);
    for (int k = 0; k < 3; ++k) {
      const int ia = d->reac_idx[3 * r + k], ib = d->prod_idx[3 * r + k];
      if (ia >= S || ib >= S) return fail(KR_ENETWORK, "reaction %d: species index out of range", r);
      if (ia >= 0) {
        const int c = d->reac_nu[3 * r + k];
        if (c <= 0) return fail(KR_ENETWORK, "reaction %d: reactant coefficient must be >= 1", r);
        sp[6 * r + k] = ia; nu[6 * r + k] = c; order_r += c; dnu_tot[r] -= c;
        for (int e = 0; e < E; ++e) tot[e] -= long(d->composition[size_t(e) * S + ia]) * c;
      }
      if (ib >= 0) {
        const int c = d->prod_nu[3 * r + k];
        if (c <= 0) return fail(KR_ENETWORK, "reaction %d: product coefficient must be >= 1", r);
        sp[6 * r + 3 + k] = ib; nu[6 * r + 3 + k] = c; order_p += c; dnu_tot[r] += c;
        for (int e = 0; e < E; ++e) tot[e] += long(d->composition[size_t(e) * S + ib]) * c;
      }
    }
    if (order_r < 1 || order_r > 3 || order_p > 3) return fail(KR_ENETWORK, "reaction %d: order must be 1..3 per side (R20)", r);
    for (int e = 0; e < E; ++e)
      if (tot[e] != 0) return fail(KR_ENETWORK, "reaction %d does not conserve row %d of the composition matrix", r, e);
    const int fl = d->flags[r];
    flags[r] = fl;
    if ((fl & (KR_F_CONST_UNARY | KR_F_AUX_UNARY)) && (fl & (KR_F_REVERSIBLE | KR_F_THIRD_BODY)))
      return fail(KR_ENETWORK, "reaction %d: unary rate types cannot be reversible or third-body", r);
    if (fl & KR_F_AUX_UNARY) {
      const int ai = d->aux_index ? d->aux_index[r] : -1;
      if (ai < 0) return fail(KR_ENETWORK, "reaction %d: aux-scaled rate without aux_index", r);
      auxi[r] = ai; n_aux = std::max(n_aux, ai + 1);
    }
    A[r] = d->A[r]; beta[r] = d->beta[r]; Ea[r] = d->Ea_over_k[r];
    if (!(fl & (KR_F_CONST_UNARY | KR_F_AUX_UNARY))) {
      if (!(A[r] > 0)) return fail(KR_ENETWORK, "reaction %d: Arrhenius A must be positive", r);
      c0[r] = std::log(A[r]) - beta[r] * std::log(KR_T_REF);
    } else c0[r] = 0.0;
    if (fl & KR_F_REVERSIBLE) any_rev = 1;
    if (fl & KR_F_THIRD_BODY) any_tb = 1;
    if (d->q_ext) { qk[r] = d->q_ext[r] / KR_K_B; if (qk[r] != 0.0) any_qext = 1; }
  }
  if (any_tb) {
    tb.assign(size_t(R) * S, 1.0);
    if (d->tb_eff) tb.assign(d->tb_eff, d->tb_eff + size_t(R) * S);
  }
  const int energy = d->energy_equation ? 1 : 0;
  const int N = S + energy;

  // gather lists of the group kernels: row list (species <- reactions) and column list (derivative owner)
  std::vector<int> row_ptr(S + 1, 0), col_ptr(S + 1, 0), row_ent, col_ent;
  {
    std::vector<std::vector<int>> rows(S), cols(S);
    for (int r = 0; r < R; ++r) {
      for (int k = 0; k < 6; ++k) {
        const int s = sp[6 * r + k];
        if (s < 0) continue;
        const int dn = (k < 3) ? -nu[6 * r + k] : nu[6 * r + k];
        rows[s].push_back((r << 8) | (dn + 128));
        // a derivative exists for reactants always and for products when there is a reverse rate
        if (k < 3 || (flags[r] & KR_F_REVERSIBLE)) cols[s].push_back((r << 4) | k);
      }
      if (flags[r] & KR_F_THIRD_BODY)
        for (int m = 0; m < S; ++m) cols[m].push_back((r << 4) | 15);
    }
    for (int s = 0; s < S; ++s) {
      row_ptr[s + 1] = row_ptr[s] + int(rows[s].size());
      col_ptr[s + 1] = col_ptr[s] + int(cols[s].size());
      row_ent.insert(row_ent.end(), rows[s].begin(), rows[s].end());
      col_ent.insert(col_ent.end(), cols[s].begin(), cols[s].end());
    }
  }
  std::vector<double> nasa(size_t(S) * 14), T_mid(d->T_mid, d->T_mid + S);
  for (int s = 0; s < S; ++s) {
    std::memcpy(&nasa[14 * s], d->nasa_lo + 7 * s, 7 * sizeof(double));
    std::memcpy(&nasa[14 * s + 7], d->nasa_hi + 7 * s, 7 * sizeof(double));
  }
  std::vector<int> comp(d->composition, d->composition + size_t(E) * S), resv(size_t(E) * S, 0);
  for (int e = 0; e < E; ++e)
    for (int s = 0; s < S; ++s) {
      bool only = comp[size_t(e) * S + s] != 0;
      for (int m = 0; m < E && only; ++m)
        if (m != e && comp[size_t(m) * S + s] != 0) only = false;
      resv[size_t(e) * S + s] = only ? 1 : 0;
    }

  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) {
    cudaGetLastError();
    return fail(KR_ECUDA, "no CUDA device: this library has no CPU path");
  }
  kr_network* n = new kr_network;
  n->E = E; n->S = S; n->R = R; n->N = N; n->energy = energy; n->n_aux = n_aux;
  kr_default_opts(&n->opts);
  int devid = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&devid) != cudaSuccess || cudaGetDeviceProperties(&prop, devid) != cudaSuccess) {
    delete n;
    return fail(KR_ECUDA, "cannot query the CUDA device: %s", cudaGetErrorString(cudaGetLastError()));
  }
  n->n_sm = prop.multiProcessorCount;

  std::vector<unsigned char> blob;
  const size_t o_sp = push(blob, sp), o_nu = push(blob, nu), o_fl = push(blob, flags), o_ax = push(blob, auxi),
               o_dn = push(blob, dnu_tot), o_c0 = push(blob, c0), o_A = push(blob, A), o_be = push(blob, beta),
               o_Ea = push(blob, Ea), o_qk = push(blob, qk), o_tb = push(blob, tb), o_na = push(blob, nasa),
               o_tm = push(blob, T_mid), o_cp = push(blob, comp), o_rs = push(blob, resv), o_rp = push(blob, row_ptr),
               o_re = push(blob, row_ent), o_cpn = push(blob, col_ptr), o_ce = push(blob, col_ent);
  cudaError_t ce = cudaMalloc(&n->blob, blob.size());
  if (ce == cudaSuccess) ce = cudaMemcpy(n->blob, blob.data(), blob.size(), cudaMemcpyHostToDevice);
  if (ce == cudaSuccess) ce = cudaMalloc((void**)&n->ws, 8 * sizeof(unsigned long long));
  if (ce != cudaSuccess) {
    const int rc = fail(KR_ECUDA, "device allocation failed: %s", cudaGetErrorString(ce));
    kr_network_destroy(n);
    return rc;
  }
  const unsigned char* b = static_cast<const unsigned char*>(n->blob);
  KrNetDev& D = n->dev;
  D.E = E; D.S = S; D.R = R; D.N = N; D.energy = energy; D.n_aux = n_aux; D.any_rev = any_rev; D.any_tb = any_tb;
  D.any_qext = any_qext; D.ld = (N + 1) | 1;
  D.T_lo = d->T_lo; D.T_hi = d->T_hi; D.ln_p0_kB = std::log(KR_P0 / KR_K_B);
  D.sp = (const int*)(b + o_sp); D.nu = (const int*)(b + o_nu); D.flags = (const int*)(b + o_fl);
  D.auxi = (const int*)(b + o_ax); D.dnu_tot = (const int*)(b + o_dn); D.c0 = (const double*)(b + o_c0);
  D.A = (const double*)(b + o_A); D.beta = (const double*)(b + o_be); D.Ea = (const double*)(b + o_Ea);
  D.qk = (const double*)(b + o_qk); D.tb_eff = (const double*)(b + o_tb); D.nasa = (const double*)(b + o_na);
  D.T_mid = (const double*)(b + o_tm); D.comp = (const int*)(b + o_cp); D.resv = (const int*)(b + o_rs);
  D.row_ptr = (const int*)(b + o_rp); D.row_ent = (const int*)(b + o_re); D.col_ptr = (const int*)(b + o_cpn);
  D.col_ent = (const int*)(b + o_ce);

  auto_mapping(n);
  const int rc = configure(n);
  if (rc != KR_OK) { kr_network_destroy(n); return rc; }
  *out = n;
  return KR_OK;
}

void kr_network_destroy(kr_network* n) {
  if (!n) return;
  if (n->blob) cudaFree(n->blob);
  if (n->ws) cudaFree(n->ws);
  if (n->s_rho) cudaFree(n->s_rho);
  if (n->s_T) cudaFree(n->s_T);
  if (n->s_y) cudaFree(n->s_y);
  if (n->s_aux) cudaFree(n->s_aux);
  if (n->s_status) cudaFree(n->s_status);
  delete n;
}

int kr_network_set_options(kr_network* n, const kr_solver_opts* o) {
  if (!n || !o) return fail(KR_EINVAL, "null argument");
  if (o->max_newton < 1 || o->max_newton > 1000 || !(o->rtol > 0) || !(o->shrink > 0 && o->shrink < 1) || o->max_substeps < 1 ||
      !(o->atol_y >= 0) || !(o->atol_T >= 0) || !(o->grow_fast >= 1) || !(o->grow_mid >= 1) || !(o->h_min_rel >= 0))
    return fail(KR_EINVAL, "solver options out of range");
  n->opts = *o;
  return KR_OK;
}

int kr_network_get_options(const kr_network* n, kr_solver_opts* o) {
  if (!n || !o) return fail(KR_EINVAL, "null argument");
  *o = n->opts;
  return KR_OK;
}

int kr_set_stream(kr_network* n, void* s) {
  if (!n) return fail(KR_EINVAL, "null network");
  n->stream = static_cast<cudaStream_t>(s);
  return KR_OK;
}

int kr_network_set_mapping(kr_network* n, int32_t mapping, int32_t threads_per_cell) {
  if (!n) return fail(KR_EINVAL, "null network");
  const int old_m = n->mapping, old_t = n->tpc;
  if (mapping == KR_MAP_AUTO) auto_mapping(n);
  else if (mapping == KR_MAP_THREAD) { n->mapping = KR_MAP_THREAD; n->tpc = 1; }
  else if (mapping == KR_MAP_WARP) { n->mapping = KR_MAP_WARP; n->tpc = 32; }
  else if (mapping == KR_MAP_CTA) { n->mapping = KR_MAP_CTA; n->tpc = threads_per_cell > 0 ? threads_per_cell : 64; }
  else return fail(KR_EINVAL, "unknown mapping %d", mapping);
  const int rc = configure(n);
  if (rc != KR_OK) { n->mapping = old_m; n->tpc = old_t; configure(n); g_err = "mapping rejected: " + g_err; }
  return rc;
}

int kr_network_info(const kr_network* n, int32_t* n_unknowns, int32_t* mapping, int32_t* threads_per_cell, int32_t* smem_bytes) {
  if (!n) return fail(KR_EINVAL, "null network");
  if (n_unknowns) *n_unknowns = n->N;
  if (mapping) *mapping = n->mapping;
  if (threads_per_cell) *threads_per_cell = n->tpc;
  if (smem_bytes) *smem_bytes = n->smem;
  return KR_OK;
}

int kr_thermochem_step_ex(kr_network* n, int64_t n_cells, const double* rho, double* T, double* y, double dt, int mode,
                          const double* aux, int32_t n_aux, int32_t* status, kr_step_stats* stats, void* stream) {
  if (!n) return fail(KR_EINVAL, "null network");
  if (n_cells < 0 || !(dt > 0)) return fail(KR_EINVAL, "n_cells must be >= 0 and dt > 0");
  if (n_cells > 0 && (!rho || !T || !y)) return fail(KR_EINVAL, "null state pointer");
  if (mode != KR_FP64 && mode != KR_MIXED) return fail(KR_EINVAL, "precision_mode must be KR_FP64 or KR_MIXED");
  if (n->n_aux > n_aux || (n->n_aux > 0 && n_cells > 0 && !aux)) return fail(KR_EINVAL, "network needs %d aux rows", n->n_aux);
  cudaStream_t st = stream ? static_cast<cudaStream_t>(stream) : n->stream;
  const int rc = launch_step(n, n_cells, rho, T, y, dt, mode, aux, status, st);
  if (rc != KR_OK) return rc;
  if (stats) return fetch_stats(n, stats, st);
  return KR_OK;
}

int kr_thermochem_step(kr_network* n, int64_t n_cells, const double* rho, double* T, double* y, double dt, int mode) {
  return kr_thermochem_step_ex(n, n_cells, rho, T, y, dt, mode, nullptr, 0, nullptr, nullptr, nullptr);
}

int kr_thermochem_step_host(kr_network* n, int64_t n_cells, const double* rho, double* T, double* y, double dt, int mode,
                            const double* aux, int32_t n_aux, int32_t* status, kr_step_stats* stats) {
  if (!n) return fail(KR_EINVAL, "null network");
  if (n_cells < 0) return fail(KR_EINVAL, "n_cells must be >= 0");
  if (n_cells > 0 && (!rho || !T || !y)) return fail(KR_EINVAL, "null state pointer");
  if (n_aux < 0 || (n_aux > 0 && !aux)) return fail(KR_EINVAL, "bad aux");
  if (n_cells > n->s_cells || n_aux > n->s_naux) {
    cudaFree(n->s_rho); cudaFree(n->s_T); cudaFree(n->s_y); cudaFree(n->s_aux); cudaFree(n->s_status);
    n->s_rho = n->s_T = n->s_y = n->s_aux = nullptr; n->s_status = nullptr; n->s_cells = 0; n->s_naux = 0;
    const size_t c = size_t(std::max<int64_t>(n_cells, 1));
    KR_CUDA(cudaMalloc((void**)&n->s_rho, c * sizeof(double)));
    KR_CUDA(cudaMalloc((void**)&n->s_T, c * sizeof(double)));
    KR_CUDA(cudaMalloc((void**)&n->s_y, c * n->S * sizeof(double)));
    KR_CUDA(cudaMalloc((void**)&n->s_aux, c * std::max(n_aux, 1) * sizeof(double)));
    KR_CUDA(cudaMalloc((void**)&n->s_status, c * sizeof(int32_t)));
    n->s_cells = n_cells; n->s_naux = n_aux;
  }
  cudaStream_t st = n->stream;
  const size_t c = size_t(n_cells);
  KR_CUDA(cudaMemcpyAsync(n->s_rho, rho, c * sizeof(double), cudaMemcpyHostToDevice, st));
  KR_CUDA(cudaMemcpyAsync(n->s_T, T, c * sizeof(double), cudaMemcpyHostToDevice, st));
  KR_CUDA(cudaMemcpyAsync(n->s_y, y, c * n->S * sizeof(double), cudaMemcpyHostToDevice, st));
  if (n_aux > 0) KR_CUDA(cudaMemcpyAsync(n->s_aux, aux, c * n_aux * sizeof(double), cudaMemcpyHostToDevice, st));
  const int rc = kr_thermochem_step_ex(n, n_cells, n->s_rho, n->s_T, n->s_y, dt, mode, n_aux > 0 ? n->s_aux : nullptr, n_aux,
                                       n->s_status, nullptr, st);
  if (rc != KR_OK) return rc;
  if (n->energy) KR_CUDA(cudaMemcpyAsync(T, n->s_T, c * sizeof(double), cudaMemcpyDeviceToHost, st));
  KR_CUDA(cudaMemcpyAsync(y, n->s_y, c * n->S * sizeof(double), cudaMemcpyDeviceToHost, st));
  if (status) KR_CUDA(cudaMemcpyAsync(status, n->s_status, c * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (stats) return fetch_stats(n, stats, st);
  KR_CUDA(cudaStreamSynchronize(st));
  return KR_OK;
}

int kr_last_launch_count(const kr_network* n) { return n ? n->last_launches : 0; }

int kr_layout_cell_to_soa(const double* yc, double* ys, int64_t n_cells, int32_t S, void* stream) {
  if (n_cells < 0 || S <= 0 || (n_cells > 0 && (!yc || !ys))) return fail(KR_EINVAL, "bad layout arguments");
  if (n_cells == 0) return KR_OK;
  const int bd = 256;
  const size_t smem = size_t(bd) * (S | 1) * sizeof(double);
  if (smem > 200 * 1024) return fail(KR_EUNSUPPORTED, "S too large for the layout tile");
  KR_CUDA(cudaFuncSetAttribute(kr_cell_to_soa_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)));
  kr_cell_to_soa_kernel<<<unsigned((n_cells + bd - 1) / bd), bd, smem, static_cast<cudaStream_t>(stream)>>>(yc, ys, n_cells, S);
  KR_CUDA(cudaGetLastError());
  return KR_OK;
}

int kr_layout_soa_to_cell(const double* ys, double* yc, int64_t n_cells, int32_t S, void* stream) {
  if (n_cells < 0 || S <= 0 || (n_cells > 0 && (!yc || !ys))) return fail(KR_EINVAL, "bad layout arguments");
  if (n_cells == 0) return KR_OK;
  const int bd = 256;
  const size_t smem = size_t(bd) * (S | 1) * sizeof(double);
  if (smem > 200 * 1024) return fail(KR_EUNSUPPORTED, "S too large for the layout tile");
  KR_CUDA(cudaFuncSetAttribute(kr_soa_to_cell_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)));
  kr_soa_to_cell_kernel<<<unsigned((n_cells + bd - 1) / bd), bd, smem, static_cast<cudaStream_t>(stream)>>>(ys, yc, n_cells, S);
  KR_CUDA(cudaGetLastError());
  return KR_OK;
}

int kr_measure_fp64_peak(int32_t n_iter, double* tflops) {
  if (n_iter <= 0 || !tflops) return fail(KR_EINVAL, "bad arguments");
  int devid = 0;
  cudaDeviceProp prop;
  KR_CUDA(cudaGetDevice(&devid));
  KR_CUDA(cudaGetDeviceProperties(&prop, devid));
  const int bd = 256, grid = prop.multiProcessorCount * 8;
  double* out = nullptr;
  KR_CUDA(cudaMalloc((void**)&out, size_t(bd) * grid * sizeof(double)));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  kr_dfma_kernel<<<grid, bd>>>(out, n_iter / 8 + 1, 0.999999, 1e-9);       // warm-up
  double best_ms = 1e30;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0);
    kr_dfma_kernel<<<grid, bd>>>(out, n_iter, 0.999999, 1e-9);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    best_ms = std::min(best_ms, double(ms));
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(out);
  KR_CUDA(cudaGetLastError());
  const double flops = 2.0 * 64.0 * double(n_iter) * bd * grid;
  *tflops = flops / (best_ms * 1e-3) / 1e12;
  return KR_OK;
}

}  // extern "C"
