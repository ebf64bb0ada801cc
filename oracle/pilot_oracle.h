/*
 * pilot_oracle.h — plain, slow, double-precision CPU ORACLE of the PiLoT v2 hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT. Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code and no header with the product (include/, paper_2606_31098_b200/csrc):
 * the data interface is restated in pilot_oracle_types.h, with every "_dev" pointer
 * holding a HOST pointer here.
 *
 * It follows the paper's algorithm step by step (arxiv/paper_2606_31098, PAPER.md):
 *   Eq.(1)-(2) photo residual / robust cost
 *   Eq.(3) gravity residual
 *   Eq.(4)-(6) range point / height residual
 *   Eq.(7) total cost
 *   Eq.(8) damped normal equation
 *   Eq.(9) SE(3) update
 *   supp Eq.(5)(6) prior fusion
 * with the readings A1-A19 of DESIGN.md §3 where the paper is silent.
 *
 * Parity pins: every function below is pinned by tests/test_oracle_pins.py
 * (closed forms, finite differences, brute force, library routines, invariances).
 * UNPINNED (stated in DESIGN.md §3): the paper's alpha_range/alpha_grav
 * gradient-magnitude auto-scaling heuristic has no formula and is
 * not implemented; the constants of the authors' LM schedule are not in the paper.
 */
#ifndef PILOT_ORACLE_H
#define PILOT_ORACLE_H

#include "pilot_oracle_types.h"

#ifdef __cplusplus
extern "C" {
#endif

/* flags returned by pilot_oracle_eval */
#define PILOT_ORACLE_FEW_VALID  2u
#define PILOT_ORACLE_RANGE_SKIP 8u

/* rho(x), rho'(x) of Eq.(2)/(7) on x = squared (weighted) residual norm; scale<=0 or L2 => rho=x. */
void pilot_oracle_loss(int loss, double x, double scale, double* rho, double* drho);

/* exp of Eq.(9): xi = (rho; phi). E = exp([phi]x) (row-major 3x3), V = left Jacobian. */
void pilot_oracle_se3_exp(const double xi[6], double E[9], double V[9]);

/* Eq.(9) on T_cw=[R_cw | -R_cw C]:  R' = E R_cw,  C' = C - R_cw^T E^T V rho. */
void pilot_oracle_retract(const double R_cw[9], const double C[3], const double xi[6],
                          double R_out[9], double C_out[3]);

/* Cholesky solve A x = b for a 6x6 row-major SPD A. Returns 1 on success, 0 if not PD / non-finite. */
int pilot_oracle_chol_solve6(const double A[36], const double b[6], double x[6]);

/* Bilinear DSM sample D^r(x,y) (Eq.6) and its exact gradient (per metre). Returns 1 if in bounds. */
int pilot_oracle_dsm_sample(const pilot_refine_inputs* in, double x, double y,
                            double* z, double* dzdx, double* dzdy);

/*
 * One photo term of Eq.(1) at pose (R_cw, C): projection, visibility, bilinear sample.
 * Outputs (any may be NULL): uv[2]; f, gx, gy, r (each `channels[level]` doubles);
 * Juv[12] = d(u,v)/d(rho,phi) row-major 2x6; w = w_ref * w_query. Returns 1 if visible.
 */
int pilot_oracle_photo_point(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                             const pilot_refine_params* p, int level,
                             const double R_cw[9], const double C[3], int j,
                             double uv[2], double* f, double* gx, double* gy, double* r,
                             double Juv[12], double* w);

/* Gravity residual r = R_cw gamma^W - gamma^imu (Eq.3) and its 3x6 Jacobian (row-major). */
void pilot_oracle_gravity(const pilot_refine_inputs* in, const double R_cw[9],
                          double r[3], double J[18]);

/*
 * Range residual (Eq.5-6 for HEIGHT; predicted-minus-measured range for MARCH) and its 1x6
 * Jacobian; d_hit (MARCH only, may be NULL). Returns 1 if evaluated, 0 if skipped.
 */
int pilot_oracle_range(const pilot_refine_inputs* in, const pilot_refine_params* p,
                       const double R_cw[9], const double C[3],
                       double* r, double J[6], double* d_hit);

/*
 * EVAL: total system at pose (R_cw, C) on `level`: H (36, row-major, undamped), g (6),
 * cost (Eq.7; +inf if n_valid < min_valid), n_valid, g_abs = sum_j || omega_j Juv_j^T b_j ||_2
 * (+ prior terms' norms), flags (PILOT_ORACLE_*). Any output may be NULL.
 * `which`: bit0 photo, bit1 gravity, bit2 range (7 = everything enabled in p).
 */
void pilot_oracle_eval(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                       const pilot_refine_params* p, int level, int which,
                       const double R_cw[9], const double C[3],
                       double H[36], double g[6], double* cost, int* n_valid,
                       double* g_abs, unsigned* flags);

/* Per-hypothesis extra outputs of the oracle run (host arrays, any may be NULL). */
typedef struct {
  double* poses;        /* [H][12] refined [R_wc | C] in double */
  double* cost;         /* [H] */
  double* last_step;    /* [H] ||dxi|| of the last ACCEPTED step at the last level (inf if none) */
  double* iter_gabs;    /* [sum(iters)][H] g_abs of each recorded system */
  double* iter_poses;   /* [sum(iters)][H][12] pose [R_wc | C] at which each recorded system was built */
} pilot_oracle_extra;

/*
 * The full refinement, same contract as pilot_refine_run but with HOST pointers everywhere,
 * float outputs rounded from double. hyp_begin/hyp_step select hypotheses hyp_begin,
 * hyp_begin+hyp_step, ... (others untouched). n_threads > 1 uses OpenMP over hypotheses if
 * compiled with -fopenmp. Returns PILOT_OK or PILOT_ERR_ARG / PILOT_ERR_UNSUPPORTED.
 */
int pilot_oracle_run(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                     const pilot_refine_params* p, const pilot_refine_outputs* out,
                     const pilot_oracle_extra* extra,
                     int hyp_begin, int hyp_step, int n_threads);

/* Number of threads an n_threads request would actually use (1 without OpenMP). */
int pilot_oracle_threads(int n_threads);

#ifdef __cplusplus
}
#endif
#endif
