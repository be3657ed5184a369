/* kr_oracle.h -- C interface of the CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, single-threaded restatement of the per-cell implicit thermochemistry
 * step of arxiv 2504.04941 (section 2.2, eqs. 15-20; section 2.2.3; Algorithm 1),
 * following SURVEY.md 8(c) / DESIGN.md "Algorithm" step by step.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 * It shares NO source, header, table or helper with paper_2504_04941_b200/csrc (the CUDA
 * path); the descriptor structs below are re-declared here on purpose.
 *
 * All pointers are HOST pointers.  Functions return 0 on success, <0 on error.
 */
#ifndef KR_ORACLE_H
#define KR_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct kr_oracle_network kr_oracle_network;

typedef struct {
  int32_t n_elem, n_species, n_reac;
  const double *elem_mass;                 /* [E] */
  const int32_t *composition;              /* [E*S] row-major N_{nu,s} */
  const int32_t *reac_idx, *reac_nu;       /* [R*3] reactants, -1 = unused */
  const int32_t *prod_idx, *prod_nu;       /* [R*3] products */
  const double *A, *beta, *Ea_over_k;      /* [R]  k = A (T/300K)^beta exp(-Ea_over_k/T) (eq. 16, R4) */
  const int32_t *flags;                    /* [R]  1 reversible, 2 third-body, 4 const unary, 8 aux unary */
  const int32_t *aux_index;                /* [R] */
  const double *tb_eff;                    /* [R*S] or NULL */
  const double *q_ext;                     /* [R] erg per forward event, or NULL */
  const double *nasa_lo, *nasa_hi;         /* [S*7] */
  const double *T_mid;                     /* [S] */
  double T_lo, T_hi;
  int32_t energy_equation;
} kr_oracle_desc;

typedef struct {
  int32_t max_newton, fixed_newton, h0_mode;
  double rtol, atol_y, atol_T, neg_tol, eta, y_floor, shrink, grow_fast, grow_mid, chg_floor, chg_max;
  int32_t it_fast, it_mid, max_substeps, finalize;
  double h_min_rel;                        /* fail when h < h_min_rel * (first sub-step size) */
  double bail_ratio;                       /* early-exit mode: abort the sub-step when e_k > bail_ratio * e_{k-1}, k >= 2 */
  int32_t retry;                           /* 1: a failed cell is tried once more with tightened control (R24) */
  double retry_h0;                         /* factor on the first sub-step of the second attempt */
  double cons_tol;                         /* stage 2: a row whose initial-minus-final total exceeds cons_tol * sum|N||y_in| is compensated in full */
} kr_oracle_opts;

typedef struct { int64_t n_substeps, n_rejected, n_newton, n_lu, n_rate_evals, n_failed; } kr_oracle_stats;

int  kr_oracle_network_create(const kr_oracle_desc*, kr_oracle_network** out);
void kr_oracle_network_destroy(kr_oracle_network*);
int  kr_oracle_set_options(kr_oracle_network*, const kr_oracle_opts*);

/* The step, double arithmetic.  y is [n_cells*S] cell-major, in/out;
 * T in/out when the energy equation is on; aux is [n_aux*n_cells] or NULL; status [n_cells] or
 * NULL; stats or NULL; margins [n_cells] or NULL receives the smallest relative margin of any
 * controller decision taken for the cell; n_threads >= 1 splits the cells into disjoint
 * contiguous ranges (std::thread), each range running the same single-threaded code. */
int kr_oracle_thermochem_step_ex(kr_oracle_network*, int64_t n_cells, const double* rho, double* T, double* y,
                                 double dt, const double* aux, int32_t n_aux, int32_t* status,
                                 kr_oracle_stats* stats, double* margins, int32_t n_threads);
/* Same step with one more diagnostic per cell: amps [n_cells] or NULL receives the largest cancellation any Newton
 * update of the cell went through, max over iterations and unknowns of |delta_i| / (|u_i + delta_i| + 1e-20 for an
 * abundance): a value of 10^a says that a digits of the update cancelled, i.e. that rounding differences inside the
 * linear solve were amplified by 10^a in the iterate (a Newton iteration started far from the solution; DESIGN.md
 * section 3 uses it to tell which cells fp64 determines to 1e-9).  Diagnostic only: it does not enter the algorithm. */
int kr_oracle_thermochem_step_diag(kr_oracle_network*, int64_t n_cells, const double* rho, double* T, double* y,
                                   double dt, const double* aux, int32_t n_aux, int32_t* status,
                                   kr_oracle_stats* stats, double* margins, double* amps, int32_t n_threads);
/* Same algorithm carried in long double (the "witness"); results rounded to double. */
int kr_oracle_witness_step_ex(kr_oracle_network*, int64_t n_cells, const double* rho, double* T, double* y,
                              double dt, const double* aux, int32_t n_aux, int32_t* status,
                              kr_oracle_stats* stats, int32_t n_threads);

/* ---- pieces exposed so that the pins can reach each step on its own ---- */
/* step 3: rate constants of one cell; kf, kr [R] */
int kr_oracle_rate_constants(kr_oracle_network*, double T, const double* aux_cell, double* kf, double* kr);
/* steps 2-4: f = (ydot[, Tdot]) of one cell; f [N] */
int kr_oracle_eval_rhs(kr_oracle_network*, double rho, double T, const double* y, const double* aux_cell, double* f);
/* same with complex arguments (complex-step derivative, pin P6) */
int kr_oracle_eval_rhs_complex(kr_oracle_network*, double rho, double T_re, double T_im, const double* y_re,
                               const double* y_im, const double* aux_cell, double* f_re, double* f_im);
/* step 5: analytic Jacobian, row-major [N*N] */
int kr_oracle_eval_jacobian(kr_oracle_network*, double rho, double T, const double* y, const double* aux_cell, double* J);
/* step 7: LU with implicit-scaled row pivoting + substitution; M [n*n] row-major is overwritten by the
 * factors, perm [n] receives p_j, x [n] the solution of M x = b.  Returns -1 when singular. */
int kr_oracle_lu_solve(int32_t n, double* M, const double* b, double* x, int32_t* perm);
/* step 6: one backward-Euler sub-step of size h from u_n = (y[, T]); u_out [N];
 * e_out = last e_k, it_out = first k with e_k <= 1 (K+1 if none); returns 0, or 1 when the
 * sub-step aborted (LU failure / non-finite / bail-out). */
/* Post-processing stages 1-3 applied to one final state y[S] in place, given the initial state
 * y_in[S] of the step (NULL: the final state itself, i.e. only what stage 1 clamps is compensated); *status receives the bits set. */
int kr_oracle_finalize(kr_oracle_network*, const double* y_in, double* y, int32_t* status);

int kr_oracle_be_substep(kr_oracle_network*, double rho, double T, const double* y, const double* aux_cell,
                         double h, double* u_out, double* e_out, int32_t* it_out);

#ifdef __cplusplus
}
#endif
#endif
