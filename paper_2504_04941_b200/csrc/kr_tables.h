// kr_tables.h -- plain-data views of a network and of the solver options as the kernels see them.
// Internal to the CUDA path (never included by oracle/).  All pointers are DEVICE pointers.
#pragma once

// physical constants, CGS
#define KR_K_B 1.380649e-16
#define KR_M_U 1.66053906660e-24
#define KR_P0 1.01325e6
#define KR_T_REF 300.0
#define KR_EXP_CLAMP 690.0

// One multiplicative term of the analytic Jacobian (eq. 19) as the register-tile kernel evaluates it:
//   d = coef * D[g0] * D[g1] * D[g2] * D[g3],   D = the cell's shared-memory block viewed as doubles
// (g0: k_f / k_r / qhat of reaction r; g1, g2: number densities of the remaining factors or the constant 1; g3: the
// third-body factor M_r or 1).  d = dq_r / dn_m.  Built on the host (kr_lib.cu, build_programs).
struct KrDEnt {
  int g0, g1, g2, g3;
  double coef;
  int r, m;
};

// One term of one Jacobian ENTRY (kr_wpc.cuh assembles J entry by entry): J[dst] = sum_terms coef * D[g0] D[g1] D[g2] D[g3].
struct KrETerm {
  double coef;                     // dnu_rs * (+-exponent | third-body efficiency) [* q_ext/k_B on the heat row]
  unsigned short g0, g1, g2, g3;   // as in KrDEnt
};

static_assert(sizeof(KrETerm) == 16, "KrETerm is read as one 16-byte word");

struct KrNetDev {
  int E, S, R, N;        // conservation rows, species, reactions, unknowns (S or S+1)
  int energy;            // 1: T is the last unknown
  int n_aux;             // aux rows the network needs
  int any_rev;           // some reaction is reversible (thermo needed for K_c)
  int any_tb, any_qext;  // third-body / external heat present
  int ld;                // leading dimension of the per-cell matrix in the group kernels (odd, >= N+1)
  double T_lo, T_hi;
  double ln_p0_kB;       // ln(p0 / k_B)
  // reaction records
  const int* sp;         // [R*6] species of slot k: 0..2 reactants, 3..5 products, -1 = unused
  const int* nu;         // [R*6] stoichiometric coefficient of the slot (0 when unused)
  const int* flags;      // [R]
  const int* auxi;       // [R]
  const int* dnu_tot;    // [R] sum products nu - sum reactants nu
  const double* c0;      // [R] ln A - beta ln T_ref
  const double* A;       // [R]
  const double* beta;    // [R]
  const double* Ea;      // [R]
  const double* qk;      // [R] q_ext / k_B
  const double* tb_eff;  // [R*S] (valid when any_tb)
  // thermo
  const double* nasa;    // [S*14]: 7 low-range then 7 high-range coefficients
  const double* T_mid;   // [S]
  // conservation rows
  const int* signed_row; // [E] 1: the row has negative entries (a charge row)
  // gather lists of the end-of-step repair (kr_post.cuh; packed (index << 8) | (coefficient + 128))
  const int* post_sp_ptr;   // [S+1] species s -> its non-zero rows
  const int* post_sp_ent;
  const int* post_res_ptr;  // [E+1] row nu -> species made of row nu only (the reservoir candidates)
  const int* post_res_ent;
  const int* post_cmp_ptr;  // [E+1] row nu -> neutral compounds holding nu whose other rows all have a reservoir candidate (R23)
  const int* post_cmp_ent;
  // gather lists of the group (warp / CTA per cell) kernels
  const int* row_ptr;    // [S+1]  row list of species s: entries row_ptr[s]..row_ptr[s+1]
  const int* row_ent;    // packed (reaction << 8) | (dnu + 128)
  const int* col_ptr;    // [S+1]  column list of species m
  const int* col_ent;    // packed (reaction << 4) | slot, slot 0..5 = participant slot, 15 = third-body only
  // programs of the register-tile kernel (kr_wpc.cuh); null when N > 64
  const KrDEnt* rprog;   // the derivative terms grouped by reaction r: rprog_ptr[r] .. rprog_ptr[r+1] (mixed-mode residual)
  const int* rprog_ptr;  // [R+1]
  const int* fac;        // [R*6] mass-action factors with powers expanded: 3 forward, 3 reverse species, S = the constant 1
  const int* tgt;        // [R*8] [0] = number of rows the reaction feeds, then (row | (dnu + 128) << 8) with the net dnu
  int n_entries;         // structurally non-zero entries of J[0..S-1][0..S-1] plus the raw heat row (row S)
  // the entry terms as one coalesced stream per thread of a group of 32 (index 0) or 64 (index 1) threads: step i of thread
  // t reads estream[i * GT + t]; emeta holds row * LD + column (LD = (N + 1) | 1) at the last term of an entry, else -1;
  // entries are dealt to the threads longest first, padded with zero terms to elen steps
  const KrETerm* estream[2];
  const int* emeta[2];
  int elen[2];
  // row program of kr_row.cuh: step i of thread t reads rstream[i * GT + t] = {reaction | (dnu + 128) << 16, slot or -1};
  // the partial sums of species s are the slots rslot_ptr[s] .. rslot_ptr[s + 1]
  const uint2* rstream[2];
  const int* rslot_ptr[2];
  int rlen[2];
};

struct KrOptsDev {
  int max_newton, fixed_newton, h0_mode, it_fast, it_mid, max_substeps, finalize;
  double rtol, atol_y, atol_T, neg_tol, eta, y_floor, shrink, grow_fast, grow_mid, chg_floor, chg_max;
  double h_min_rel, bail_ratio;
  double h0_scale;       // factor on the first sub-step (1; retry_h0 in the second attempt of the retry procedure)
  double cons_tol;       // end-of-step repair: rows drifting by more than cons_tol x scale are compensated in full
};

struct KrStepArgs {
  long long n_cells;
  const double* rho;
  double* T;
  double* y;
  const double* aux;
  int* status;
  double dt;
  unsigned long long* counter;   // work queue head
  unsigned long long* stats;     // [6] device counters (+ [6]: refinement passes of the mixed mode)
  // mixed precision: cells whose fp32 factorisation cannot be refined are appended to retry_list and redone in fp64
  long long* retry_list;               // [n_cells] or null
  unsigned long long* retry_count;     // number of entries appended
  const long long* list;               // null: cells 0..n_cells-1; else the cells to process, in this order ...
  const unsigned long long* list_count;  // ... and how many of them (device memory)
  int list_flag;                       // status bits set on every cell of the list (KR_DST_FP64_FALLBACK for the retry pass)
  // cost pass (stiffest-first scheduling): when non-null the kernel only evaluates f(u_in) and writes the first sub-step
  // it would take, min(dt, eta / max_s |ydot_s| / (|y_s| + y_floor)), as the cell's key
  float* cost_out;                     // [n_cells] or null
  // isothermal networks, specialised thread-per-cell kernel: rate constants and first sub-step of every cell, written by
  // kr_spec_prelim_kernel as [2R + 1][n_cells] (k_f rows, k_r rows, h0), read by the solve kernel when it loads a cell
  double* prelim;
  // retry procedure (R24): when non-null, a cell whose controller gives up is appended here (and left
  // untouched, unflagged, uncounted) for the second attempt instead of being reverted
  long long* fail_list;
  unsigned long long* fail_count;
};

// status bits (mirror of include/kratos_chem.h, kept numeric so that device code needs no host header)
#define KR_DST_REJECTED 1
#define KR_DST_CLAMPED_NEG 2
#define KR_DST_FP64_FALLBACK 4
#define KR_DST_FAILED 8
#define KR_DST_T_CLAMPED 16
#define KR_DST_NO_RESERVOIR 32
#define KR_DST_NEEDS_STAGE3 64
#define KR_DST_STAGE3 128
#define KR_DST_RETRIED 256

#define KR_DF_REV 1
#define KR_DF_TB 2
#define KR_DF_CONST 4
#define KR_DF_AUX 8
