/* kratos_chem.h -- C ABI of the B200-native per-cell implicit thermochemistry step.
 *
 * What the library computes (arxiv 2504.04941, "PAPER.md"):
 *   the per-cell ODE system  dn^i/dt = sum A^i_jk n^j n^k + sum B^i_j n^j,  d(eps)/dt = Gamma - Lambda
 *   (eq. 15) with modified-Arrhenius two-body rates (eq. 16),
 *   per-cell unary (photo / cosmic-ray) rates (eq. 17), the analytic Jacobian of
 *   abundances plus temperature (eqs. 18-20), integrated by an implicit
 *   ("semi-implicit") scheme with adaptive sub-steps, each
 *   Newton iteration solving one small dense system by LU with implicit-scaled row pivoting
 *   (Algorithm 1), followed by the post-processing repair stages 1-3 and the
 *   retry / revert policy.  Readings of everything the paper leaves open are
 *   listed in DESIGN.md ("Readings R1-R22").
 *
 * Conventions
 *   - All functions return int: KR_OK (0) or a negative KR_E* code; kr_last_error() gives a
 *     thread-local message for the last failing call on the calling thread.
 *   - "host" / "device" is stated for every pointer.  The library never frees or reallocates a
 *     caller buffer.  It owns its network tables and a small device workspace (work counter,
 *     statistics), created in kr_network_create and released in kr_network_destroy.
 *   - State variable: y_s = n_s m_u / rho (dimensionless; R10), cell-major y[n_cells*S].
 *   - CGS units: rho g cm^-3, T K, dt s, A cm^3 s^-1 (two-body) or s^-1 (unary), Ea_over_k K,
 *     q_ext erg.
 *   - Every step of the path runs in CUDA kernels for sm_100a.  There is no CPU fallback: without a
 *     CUDA device every compute call fails with KR_ECUDA.
 */
#ifndef KRATOS_CHEM_H
#define KRATOS_CHEM_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { KR_OK = 0, KR_EINVAL = -1, KR_ENETWORK = -2, KR_ECUDA = -3, KR_EUNSUPPORTED = -4 };

/* reaction flag bits (kr_network_desc.flags) */
enum { KR_F_REVERSIBLE = 1,   /* reverse rate from detailed balance, k_r = k_f / K_c(T) (R5) */
       KR_F_THIRD_BODY = 2,   /* both directions multiplied by M = sum_s eff_s n_s (R6)      */
       KR_F_CONST_UNARY = 4,  /* k = A, no temperature dependence (cosmic ray; R17)          */
       KR_F_AUX_UNARY = 8 };  /* k = A * aux[aux_index][cell] (photo rate, eq. 17; R16)      */

/* per-cell status bits (status[] of kr_thermochem_step_ex) */
enum { KR_ST_REJECTED_ONCE = 1,    /* at least one sub-step was rejected and retried */
       KR_ST_CLAMPED_NEG = 2,      /* post-processing stage 1 zeroed a negative abundance */
       KR_ST_FP64_FALLBACK = 4,    /* mixed precision: fp32 could not resolve a linear system of this cell; it was redone in fp64 */
       KR_ST_FAILED_REVERTED = 8,  /* controller gave up; the cell's T and y are left as given (R13) */
       KR_ST_T_CLAMPED = 16,       /* input T was outside [T_lo, T_hi] and was clamped */
       KR_ST_NO_RESERVOIR = 32,    /* stage 2: a conservation row has no single-element species */
       KR_ST_NEEDS_STAGE3 = 64,    /* stage 2 drove a reservoir negative and stage 3 found no neutral compound to disintegrate */
       KR_ST_STAGE3 = 128,         /* stage 3 disintegrated compound species to refill a reservoir */
       KR_ST_RETRIED = 256 };      /* the first attempt failed; the result (or the revert) is the second attempt's */

/* precision_mode */
enum { KR_FP64 = 0,    /* everything in fp64 */
       KR_MIXED = 1 }; /* fp32 Jacobian + elimination on the row-scaled system, fp64 residuals, iterative refinement (R15); a cell
                        * whose refinement does not contract is redone in fp64 (two launches).  Built for N <= 64. */

/* per-cell mapping (kr_network_set_mapping); KR_MAP_AUTO picks from N by measurement */
enum { KR_MAP_AUTO = 0,
       KR_MAP_THREAD = 1,        /* one lane per cell; kernel SPECIALISED to the network at create time (NVRTC) */
       KR_MAP_WARP = 2,          /* one warp per cell: matrix in register tiles, kernel compiled for the network's sizes (NVRTC) */
       KR_MAP_CTA = 3,           /* 64..256 threads per cell: register tiles on 64 threads (N <= 64), else matrix in shared memory */
       KR_MAP_THREAD_TABLE = 4,  /* one lane per cell, table driven (no run-time compilation) */
       KR_MAP_GROUP_TABLE = 5 }; /* 32..256 threads per cell, matrix in shared memory, table driven (no run-time compilation) */

typedef struct kr_network kr_network; /* opaque; owns host + device tables and the workspace */

/* Network description.  All pointers are HOST pointers, read during kr_network_create only. */
typedef struct {
  int32_t n_elem, n_species, n_reac; /* E conservation rows (elements, optional charge row), S, R */
  const double *elem_mass;           /* [E] amu (0 on a charge row) */
  const int32_t *composition;        /* [E*S] row-major N_{nu,s}; signed on a charge row */
  const int32_t *reac_idx, *reac_nu; /* [R*3] reactant species index (-1 = unused) and coefficient >= 1 */
  const int32_t *prod_idx, *prod_nu; /* [R*3] products, same packing; a species appears once per side */
  const double *A, *beta, *Ea_over_k; /* [R] k_f = A (T/300K)^beta exp(-Ea_over_k/T) (eq. 16, R4) */
  const int32_t *flags;              /* [R] KR_F_* bits */
  const int32_t *aux_index;          /* [R] row of aux[] for KR_F_AUX_UNARY reactions, else -1; may be NULL */
  const double *tb_eff;              /* [R*S] third-body efficiencies, or NULL (all 1) */
  const double *q_ext;               /* [R] erg deposited per forward event, or NULL (0) */
  const double *nasa_lo, *nasa_hi;   /* [S*7] a1..a7 for T <= T_mid[s] / T > T_mid[s] (R7) */
  const double *T_mid;               /* [S] */
  double T_lo, T_hi;                 /* clamp / validity range (R19) */
  int32_t energy_equation;           /* 0: isothermal, N = S;  1: T is an unknown, N = S + 1 (eq. 18) */
} kr_network_desc;

/* Solver options; kr_default_opts() fills the defaults of DESIGN.md "Algorithm" (h0_mode = 1). */
typedef struct {
  int32_t max_newton;   /* K: Newton iterations per sub-step (>= 1) */
  int32_t fixed_newton; /* 1: always K iterations (parity runs); 0: stop at the first e_k <= 1, bail out on divergence */
  int32_t h0_mode;      /* 0: first sub-step h = dt; 1: h = min(dt, eta / max_s |ydot_s|/(|y_s|+y_floor)) */
  double rtol, atol_y, atol_T; /* Newton convergence: e = max_i |delta_i| / (rtol |u_i| + atol_i) <= 1 */
  double neg_tol;       /* reject a sub-step whose smallest abundance is < -neg_tol */
  double eta, y_floor;  /* first-sub-step rule (h0_mode 1) */
  double shrink;        /* h <- h * shrink after a rejection (0 < shrink < 1) */
  double grow_fast, grow_mid; /* h <- h * grow_fast if it <= it_fast, * grow_mid if it <= it_mid */
  double chg_floor, chg_max;  /* optional accuracy limiter; off when chg_max = +inf */
  int32_t it_fast, it_mid, max_substeps;
  int32_t finalize;     /* 1: run post-processing stages 1-3; 0: skip */
  double h_min_rel;     /* fail when h < h_min_rel * (first sub-step size) */
  double bail_ratio;    /* early-exit mode: abort the sub-step when e_k > bail_ratio * e_{k-1}, k >= 2 */
  int32_t retry;        /* 1: a cell whose first attempt fails is redone from its input with tightened control before it is
                         * reverted (R24): one more launch (fp64) on the listed cells.  Default 0. */
  double retry_h0;      /* factor on the first sub-step of the second attempt (default 0.01) */
  double cons_tol;      /* post-processing stage 2: a conservation row whose initial-minus-final total exceeds
                         * cons_tol * sum_s |N_nu,s| |y_in,s| is compensated in full through its reservoir species; below it only
                         * what stage 1 clamped is compensated (default 1e-13; reading R12) */
} kr_solver_opts;

/* Work counters of one call, summed over cells. */
typedef struct {
  int64_t n_substeps; /* accepted sub-steps */
  int64_t n_rejected; /* rejected sub-steps */
  int64_t n_newton;   /* Newton iterations = Jacobian assemblies */
  int64_t n_lu;       /* LU factorisations (+ substitutions) */
  int64_t n_rate_evals; /* evaluations of the rate-constant set (thermo + Arrhenius + K_c) */
  int64_t n_failed;   /* cells reverted */
} kr_step_stats;

/* Build a network.  desc and everything it points to are host memory, copied; the call validates
 * indices, reaction order <= 3 per side (R20) and element conservation N . dnu_r = 0 of every
 * reaction against the composition matrix -> KR_ENETWORK when violated, builds
 * the device tables (reaction records, Jacobian gather lists) and picks the per-cell mapping.
 * Needs a CUDA device (current device of the calling thread) -> KR_ECUDA without one. */
int kr_network_create(const kr_network_desc *desc, kr_network **out);
void kr_network_destroy(kr_network *net);

void kr_default_opts(kr_solver_opts *opts);                      /* host pointer, filled */
int kr_network_set_options(kr_network *net, const kr_solver_opts *opts); /* host pointer, copied; KR_EINVAL on nonsense */
int kr_network_get_options(const kr_network *net, kr_solver_opts *opts);
/* Stream used by kr_thermochem_step (a cudaStream_t passed as void*; NULL = legacy default stream). */
int kr_set_stream(kr_network *net, void *cuda_stream);
/* Override the mapping picked from N: mapping = KR_MAP_*, threads_per_cell = 0 (auto) or a multiple
 * of 32 for KR_MAP_WARP (32) / KR_MAP_CTA (64..256).  KR_EUNSUPPORTED when N does not fit it. */
int kr_network_set_mapping(kr_network *net, int32_t mapping, int32_t threads_per_cell);
/* Test and study hooks (the defaults are what the library measures best): stiffest_first -1 = automatic (a cost pass and a
 * sort before warp-per-cell launches of several waves), 0 = always index order, 1 = as automatic; host_chunks 0 = automatic,
 * 1..8 = that many chunks in kr_thermochem_step_host.  Results do not depend on either (cells are independent). */
int kr_network_set_tuning(kr_network *net, int32_t stiffest_first, int32_t host_chunks);
/* Query: N (unknowns per cell), mapping in use, threads per cell, dynamic shared memory per block. */
int kr_network_info(const kr_network *net, int32_t *n_unknowns, int32_t *mapping, int32_t *threads_per_cell,
                    int32_t *smem_bytes);

/* One implicit chemistry step of size dt for n_cells independent cells (DESIGN.md steps 1-9).
 *   rho  [n_cells]    DEVICE, read-only (fixed during the step)
 *   T    [n_cells]    DEVICE, in/out when the energy equation is on, read-only otherwise
 *   y    [n_cells*S]  DEVICE, cell-major, in/out
 *   precision_mode    KR_FP64 or KR_MIXED, anything else -> KR_EINVAL
 * Runs asynchronously on the stream set by kr_set_stream; returns after the launches are queued.
 * A cell whose controller fails is left untouched (reverted); that is not a call failure.
 * A network with KR_F_AUX_UNARY reactions needs kr_thermochem_step_ex (KR_EINVAL here). */
int kr_thermochem_step(kr_network *net, int64_t n_cells, const double *rho, double *T, double *y, double dt,
                       int precision_mode);

/* Same, plus per-cell auxiliary rates, status and statistics.
 *   aux    [n_aux*n_cells] DEVICE, row a = values of auxiliary field a (photo rate, shielding), or NULL
 *   status [n_cells]       DEVICE int32, KR_ST_* bits per cell, or NULL
 *   stats                  HOST, or NULL; non-NULL forces one stream synchronisation before returning
 *   cuda_stream            stream for this call (void* cudaStream_t; NULL = the stream of kr_set_stream) */
int kr_thermochem_step_ex(kr_network *net, int64_t n_cells, const double *rho, double *T, double *y, double dt,
                          int precision_mode, const double *aux, int32_t n_aux, int32_t *status,
                          kr_step_stats *stats, void *cuda_stream);

/* Host-buffer convenience used for the end-to-end measurement: same arguments as kr_thermochem_step_ex
 * but rho, T, y, aux, status are HOST pointers; the call stages them through device buffers cached on
 * the handle (host->device copies, the step, device->host copies of T, y, status) and synchronises.  Batches of
 * 2^19 cells or more without stats are cut into 4 chunks and pipelined (copy-in, step, copy-out on separate
 * streams) once an unchunked call on the handle has shown the copies to exceed 30 % of the step; results are identical
 * to the unchunked call.  Host buffers should be pinned for the copies to overlap. */
int kr_thermochem_step_host(kr_network *net, int64_t n_cells, const double *rho, double *T, double *y, double dt,
                            int precision_mode, const double *aux, int32_t n_aux, int32_t *status,
                            kr_step_stats *stats);

/* ---- Allocation-free variant of the step (callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it).  Same operation, same kernels and same results as kr_thermochem_step_ex in KR_FP64 for the
 * networks the specialised thread-per-cell kernel serves (N <= 12 unknowns, default mapping: BASELINE configs 0, 1, 2;
 * KR_EUNSUPPORTED otherwise, and when opts.retry != 0).  Its scratch -- 16 work / statistics counters and, for isothermal
 * networks, the [2R + 1][n_cells] doubles the preliminary kernel hands to the solve kernel -- is a file-scope static device
 * array of kr_static_scratch_bytes() = 16 MiB, which every GPU that loads the library holds until the process exits.
 *   kr_static_setup(net)   once per device, with that device current, OUTSIDE any capture: resolves the device address of the
 *                          array (cudaGetSymbolAddress) and runs the kernels once on zero cells; synchronises the handle's stream.
 *   kr_static_max_cells    largest n_cells one call takes for this network: (16 MiB - 256 B) / (8 (2R + 1)) for isothermal
 *                          networks (config 2, R = 9: 110 374 cells), INT64_MAX for networks with an energy equation.
 *   kr_thermochem_step_static  arguments as kr_thermochem_step_ex (DEVICE pointers, in place, asynchronous on cuda_stream unless
 *                          stats is non-NULL).  Calls no cudaMalloc, cudaFree or allocating library routine.  KR_EINVAL with a
 *                          message naming the limit when n_cells needs more scratch than the array holds, or when
 *                          kr_static_setup has not run on the current device.
 * Every call on a device shares the one array, which keeps the last call's contents: the call clears the counters itself (the
 * workspace is written before it is read), and two calls that overlap on the GPU (different streams, or different handles
 * on the same device) RACE on it -- serialise them.  kr_last_mixed_stats and the retry procedure do not apply. */
int64_t kr_static_scratch_bytes(void);
int kr_static_setup(kr_network *net);
int kr_static_max_cells(const kr_network *net, int64_t *max_cells);
int kr_thermochem_step_static(kr_network *net, int64_t n_cells, const double *rho, double *T, double *y, double dt,
                              const double *aux, int32_t n_aux, int32_t *status, kr_step_stats *stats, void *cuda_stream);

/* One-line description of the kernel the current mapping launches (registers, blocks per SM ...), host buffer. */
int kr_network_kernel_desc(const kr_network *net, char *buf, int64_t cap);
/* The generated translation unit (struct KrNet of constexpr tables) the specialised kernel is compiled against;
 * host only, needs no GPU.  Returns the length, or a negative KR_E* code; buf may be NULL to query the length. */
int kr_network_spec_source(const kr_network_desc *desc, char *buf, int64_t cap);

/* Compile (NVRTC, sm_100a; needs no GPU) the specialised kernel of a network without loading it: the build-time
 * check of the run-time compiled path.  *cubin_bytes (host) receives the cubin size, log (host, may be NULL) the
 * compiler log.  KR_ECUDA when NVRTC is unavailable or the compilation fails. */
int kr_network_spec_compile(const kr_network_desc *desc, int64_t *cubin_bytes, char *log, int64_t log_cap);

/* Build-time check of the register-tile kernel (csrc/kr_wpc.cuh) for a network: compile it with NVRTC for sm_100a without
 * loading it (needs no GPU).  precision_mode KR_FP64 / KR_MIXED, warps_per_cell 1 or 2.  *cubin_bytes (host) receives the
 * cubin size, log (host, may be NULL) the compiler log, cubin (host, may be NULL) up to cubin_cap bytes of the image. */
int kr_network_wpc_compile(const kr_network_desc *desc, int precision_mode, int32_t warps_per_cell, int64_t *cubin_bytes,
                           char *log, int64_t log_cap, void *cubin, int64_t cubin_cap);

/* Build-time check of the row-per-lane kernel (csrc/kr_row.cuh: fp64, one matrix row per lane, N <= 34 on one warp, N <= 64 on
 * two): compile it with NVRTC for sm_100a without loading it (needs no GPU).  Arguments as kr_network_wpc_compile. */
int kr_network_row_compile(const kr_network_desc *desc, int32_t warps_per_cell, int64_t *cubin_bytes, char *log, int64_t log_cap,
                           void *cubin, int64_t cubin_cap);

/* Mixed precision only, counters of the last step call summed over cells: refinement passes (fp64 residual + fp32
 * replay), cells whose fp32 factorisation could not be refined and that were redone by the fp64 kernel (status bit
 * KR_ST_FP64_FALLBACK), and the Newton iterations of those abandoned fp32 attempts (they are NOT part of kr_step_stats:
 * the statistics count the work of the attempt that produced the result).  Synchronises the stream of the last step
 * call.  HOST pointers, each may be NULL. */
int kr_last_mixed_stats(kr_network *net, int64_t *n_refine, int64_t *n_fp64_cells, int64_t *n_discarded_newton);

/* Number of kernel launches the last step call on this handle queued (for bench.py's gpu_launches). */
int kr_last_launch_count(const kr_network *net);

/* Layout boundary on its own (DESIGN.md a1/a9): cell-major y[n_cells*S] <-> species-SoA ys[S][n_cells],
 * DEVICE pointers, coalesced both ways through shared-memory tiles.  Exposed for hydro codes that keep
 * species-SoA fields; kr_thermochem_step does its own transposition inside the solve kernels. */
int kr_layout_cell_to_soa(const double *y_cell, double *y_soa, int64_t n_cells, int32_t S, void *cuda_stream);
int kr_layout_soa_to_cell(const double *y_soa, double *y_cell, int64_t n_cells, int32_t S, void *cuda_stream);

/* Accuracy probe of the two lean FP64 primitives the specialised kernels use instead of the library divide and exp
 * (csrc/kr_math.cuh): rcp[i] = 1/x[i] (x normal), ex[i] = exp(min(x[i], 690)).  DEVICE pointers, n elements. */
int kr_math_probe(const double *x, double *rcp, double *ex, int64_t n, void *cuda_stream);

/* FP64 FMA peak microbenchmark (independent DFMA chains on every SM).  Returns
 * the achieved TFLOP/s in *tflops (host) measured with CUDA events over n_iter inner iterations. */
int kr_measure_fp64_peak(int32_t n_iter, double *tflops);

/* ---- Species reconstruction and advection (section 2.1, eqs. 1-14) -------------------------
 * The step that precedes the chemistry step in the paper's cycle: the abundances y (the chemistry step's variable, y = n m_u / rho
 * = m_u x of eq. 1) are advected with the mass fluxes of the hydrodynamics, F^s = y_{i-1/2} F^rho (eq. 1), the interface state
 * being the upwind cell's (eq. 6, donor cell), its piecewise-linear extrapolation with the modified van Leer limiter (eqs. 9-12),
 * or that extrapolation with the correction projected onto the stoichiometric space, P = V V^T from the SVD of the
 * element-species matrix (eqs. 7, 8, 13), which keeps every element total of the interface state equal to the upwind cell's. */
typedef struct kr_recon kr_recon;
enum { KR_RECON_SCHEME_DONOR = 0, KR_RECON_SCHEME_PLM = 1, KR_RECON_SCHEME_PLM_PROJECTED = 2 };
/* composition: HOST [n_elem * n_species] row-major N_{nu,s}.  Builds P on the host (one-sided Jacobi SVD) and
 * uploads it when a CUDA device is present (without one the handle only serves kr_recon_projector). */
int kr_recon_create(int32_t n_elem, int32_t n_species, const int32_t *composition, kr_recon **out);
void kr_recon_destroy(kr_recon *r);
/* P: HOST [n_species * n_species] row-major, filled; rank (HOST, may be NULL) receives the rank of the composition matrix. */
int kr_recon_projector(const kr_recon *r, double *P, int32_t *rank);
/* One forward-Euler stage of the conservative update on a uniform 1-D grid (step (3) of PAPER.md:40), DEVICE pointers:
 *   y [n_cells * S] cell-major, rho [n_cells], mass_flux: periodic != 0 -> [n_cells], mass_flux[i] = F^rho through the LEFT face
 *   of cell i (the right face of the last cell is the left face of the first); periodic == 0 -> [n_cells + 1], zero-gradient
 *   ghost cells at both ends.  rho_out = wa rho0 + wb (rho - dt_over_dx dF^rho), (rho y)_out likewise, y_out = (rho y)_out /
 *   rho_out; y0 / rho0 NULL -> plain stage (wa, wb ignored as 0, 1).  y_out [n_cells * S] must not alias y; rho_out [n_cells] may
 *   be NULL.  scheme = KR_RECON_SCHEME_*.  Asynchronous on cuda_stream.  KR_EINVAL on bad arguments, KR_ECUDA without a device. */
int kr_advect_species_1d(kr_recon *r, int64_t n_cells, const double *y, const double *rho, const double *mass_flux,
                         double dt_over_dx, double dx, int32_t scheme, int32_t periodic, double wa, double wb,
                         const double *y0, const double *rho0, double *y_out, double *rho_out, void *cuda_stream);

/* ---- Ray tracing on a uniform Cartesian mesh and the photo-reaction rates it feeds (section 3) ----
 * Every ray is walked cell by cell (eqs. 23-24: the exit point is the smallest positive delta-l among the cell's surfaces); in each
 * cell, for every energy bin k, tau_jk = sum_i n_i sigma_ik dl_j, every absorbing species i receives the rate coefficient
 * L_jk sigma_ik dl_j / dV * (1 - exp(-tau_jk)) / tau_jk (eqs. 30-31) and the ray goes on with L_jk exp(-tau_jk) (eq. 29).  The
 * result k_out[i] is the per-cell unary rate field the chemistry step takes as an aux row (KR_F_AUX_UNARY, eq. 17).
 *   nx, ny, nz; spacing, lower: HOST [3] cell sizes and coordinates of the mesh's lower corner (lower NULL -> 0), cm
 *   origins, directions [n_rays * 3] DEVICE (a ray that starts outside the mesh enters through the first face it meets; one that
 *   misses leaves its photons untouched); L_in [n_rays * n_bins] DEVICE photons per second per ray and bin
 *   sigma: HOST [n_abs * n_bins] cm^2; n_dens: DEVICE [n_abs * n_cells] cm^-3, cell = (ix * ny + iy) * nz + iz
 *   k_out: DEVICE [n_abs * n_cells] s^-1, overwritten (zeroed, then accumulated over rays and bins: FP64 atomic adds, so cells
 *   crossed by several rays are summed in an order that may differ between calls at rounding level)
 *   L_out [n_rays * n_bins], path [n_rays] (total length inside the mesh): DEVICE, may be NULL.
 * At most 8 absorbing species and 16 bins (KR_EUNSUPPORTED beyond).  Asynchronous on cuda_stream. */
int kr_raytrace_cartesian(int32_t nx, int32_t ny, int32_t nz, const double *spacing, const double *lower, int64_t n_rays,
                          const double *origins, const double *directions, int32_t n_bins, const double *L_in, int32_t n_abs,
                          const double *sigma, const double *n_dens, double *k_out, double *L_out, double *path,
                          void *cuda_stream);

/* ---- Tabulated reaction rates (rate type 3: "precomputed tables are read in ... multi-
 * dimensional tables are reduced to one-dimensional in T per cell, assuming fixed total mass density and elemental abundances
 * during thermochemical steps") ----
 * n_tab tables of ln k on nodes uniform in ln rho (n_rho nodes from ln_rho0, spacing d_ln_rho; n_rho = 1: no density
 * dependence) and in ln T (n_T nodes from ln_T0, spacing d_ln_T).  For every cell the table is reduced along rho at the cell's
 * density and the resulting 1-D table is interpolated at the cell's temperature; both steps are piecewise linear in the
 * logarithms, end values outside the table (readings R32 / R33 of DESIGN.md).  The result is the per-cell rate coefficient the
 * chemistry step takes as an aux row (KR_F_AUX_UNARY with A = 1: any mass-action order): k_out row t may point straight into
 * the aux array of kr_thermochem_step_ex.  The rates are those at the cell's T at the START of the step: exact for an
 * isothermal network; for a network with an energy equation they are frozen over the step (not re-interpolated in the
 * Newton loop).
 *   ln_k  DEVICE [n_tab * n_rho * n_T], table t, density node i, temperature node j at (t * n_rho + i) * n_T + j
 *   rho, T  DEVICE [n_cells] (g cm^-3, K);  k_out  DEVICE [n_tab * n_cells], overwritten
 * Asynchronous on cuda_stream.  KR_EINVAL on bad sizes / spacings / null pointers, KR_ECUDA without a device. */
int kr_table_rates(int32_t n_tab, int32_t n_rho, int32_t n_T, double ln_rho0, double d_ln_rho, double ln_T0, double d_ln_T,
                   const double *ln_k, int64_t n_cells, const double *rho, const double *T, double *k_out, void *cuda_stream);

const char *kr_last_error(void);
const char *kr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* KRATOS_CHEM_H */
