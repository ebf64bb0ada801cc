/*
 * pilot_oracle_types.h — the oracle's OWN statement of the data interface: constants, enums and the four POD structs
 * (configuration, inputs, LM parameters, outputs) of SURVEY.md 8(b). The oracle includes nothing from the product
 * (include/, paper_2606_31098_b200/csrc/): these declarations are restated here, with every "_dev" pointer holding a HOST
 * pointer, and tests/test_abi.py checks that they still describe the same bytes as include/pilot_refine.h.
 * TEST INFRASTRUCTURE, like everything under oracle/. No arithmetic lives here.
 */
#ifndef PILOT_ORACLE_TYPES_H
#define PILOT_ORACLE_TYPES_H

#include <stddef.h>

#define PILOT_MAX_LEVELS 4

/* return codes of every entry point */
#define PILOT_OK               0
#define PILOT_ERR_ARG         (-1)  /* NULL / out-of-range argument                          */
#define PILOT_ERR_WORKSPACE   (-2)  /* caller-provided workspace too small                   */
#define PILOT_ERR_UNSUPPORTED (-3)  /* shape not supported (C*sizeof not pow2 multiple of 16 B, a level map of 4 GiB or more, over capacity) */
#define PILOT_ERR_CUDA        (-4)  /* a CUDA runtime call failed                            */

/* per-hypothesis status bits (outputs.status_dev) */
#define PILOT_STATUS_NONFINITE   1u /* sticky: a NaN total cost was seen (a non-finite STEP counts as a failed factorisation: bit 4) */
#define PILOT_STATUS_FEW_VALID   2u /* the final accepted state has n_valid < min_valid (its cost is +inf) */
#define PILOT_STATUS_CHOL_FAIL   4u /* sticky: Cholesky failed with lambda already at lambda_max */
#define PILOT_STATUS_RANGE_SKIP  8u /* the final accepted state's range prior was skipped (ray leaves the DSM / no hit) */

typedef struct pilot_refine_handle pilot_refine_handle; /* opaque */

typedef enum { PILOT_F32 = 0, PILOT_BF16 = 1, PILOT_F16 = 2 } pilot_dtype;
typedef enum { PILOT_LOSS_L2 = 0, PILOT_LOSS_HUBER = 1, PILOT_LOSS_CAUCHY = 2 } pilot_loss;
typedef enum { PILOT_RANGE_OFF = 0, PILOT_RANGE_HEIGHT = 1, PILOT_RANGE_MARCH = 2 } pilot_range_mode;
typedef enum { PILOT_LM_ADAPTIVE = 0, PILOT_LM_FIXED = 1 } pilot_lm_mode;
typedef enum { PILOT_DAMP_IDENTITY = 0, PILOT_DAMP_DIAG = 1 } pilot_damp_mode;
typedef enum { PILOT_GRAD_BILINEAR_EXACT = 0, PILOT_GRAD_CENTRAL_SAMPLED = 1 } pilot_grad_mode;

/* Capacity / static shape, fixed at create(). */
typedef struct {
  int device;                          /* CUDA ordinal */
  int n_levels;                        /* 1..PILOT_MAX_LEVELS; level 0 = coarsest, processed first */
  int width[PILOT_MAX_LEVELS];         /* query feature map size per level (pixels) */
  int height[PILOT_MAX_LEVELS];
  int channels[PILOT_MAX_LEVELS];      /* C per level; C*sizeof(elem)/16 must be a power of two in [1,32] */
  pilot_dtype feat_dtype;              /* element type of query maps AND reference features */
  int max_hypotheses;                  /* capacity H */
  int max_points;                      /* capacity N (per level) */
  int max_total_iters;                 /* capacity sum(iters) */
  void*  workspace_dev;                /* optional caller scratch (device); NULL => create() cudaMallocs it once */
  size_t workspace_bytes;
} pilot_refine_config;

/* Per-run inputs. Host scalars are read before run() returns. */
typedef struct {
  int n_hypotheses;                                  /* H <= max_hypotheses */
  int n_points[PILOT_MAX_LEVELS];                    /* N_l <= max_points */
  const void*  query_feat_dev[PILOT_MAX_LEVELS];     /* [height][width][channels], C innermost, base 16-B aligned (Eq.1 f^q_l) */
  const float* query_conf_dev[PILOT_MAX_LEVELS];     /* [height][width] query confidence w^q_l, or NULL (=1) */
  float        intrinsics[PILOT_MAX_LEVELS][4];      /* fx, fy, cx, cy of K_l (Eq.1); pixel (x,y) sits at continuous (x,y) */
  const float* points_dev[PILOT_MAX_LEVELS];         /* [n_points][4] = geo-anchor P_j x,y,z (world, metres), w_ref>=0 (supp Eq.3) */
  const void*  ref_feat_dev[PILOT_MAX_LEVELS];       /* [n_points][channels] reference descriptors f^r_l(p_j) (Eq.1) */
  const float* init_poses_dev;                       /* [H][12] row-major 3x4 [R_wc | C]: camera-to-world, the paper's T~_m */
  float gravity_world[3], gravity_imu[3];            /* unit vectors gamma^W, gamma^imu of Eq.(3) */
  float range_ray_cam[3], range_meas;                /* unit centre ray v (Eq.4), d^range in metres (Eq.5) */
  const float* dsm_dev; int dsm_width, dsm_height;   /* [dsm_height][dsm_width] fp32 heights D^r; may be NULL if range off */
  float dsm_origin_x, dsm_origin_y, dsm_gsd;         /* world x,y of sample (0,0); metres per sample; x = ox + ix*gsd, y = oy + iy*gsd */
} pilot_refine_inputs;

/* LM parameters. */
typedef struct {
  int iters[PILOT_MAX_LEVELS];                       /* K_l solves per level (2/3/4) */
  pilot_loss loss; float loss_scale;                 /* rho of Eq.(2); scale delta acts on sqrt(w*||r||^2) */
  pilot_lm_mode lm_mode; pilot_damp_mode damp_mode;  /* Eq.(8) uses lambda*I = DAMP_IDENTITY */
  float lambda_init, lambda_up, lambda_down, lambda_min, lambda_max;
  pilot_grad_mode grad_mode;                         /* "local feature-gradient estimation" PAPER.md:485 */
  float z_near; int min_valid;                       /* visibility: Z > z_near; n_valid < min_valid => cost = +inf */
  float w_gravity, gravity_scale;                    /* lambda_imu of Eq.(7) (0 = off); robust scale (0 => L2) */
  pilot_range_mode range_mode; float w_range, range_scale; /* lambda_range of Eq.(7); robust scale in metres (0 => L2) */
  int march_steps, bisect_steps; float march_tfar_scale;   /* RANGE_MARCH: 64, 8, 2.0 */
} pilot_refine_params;

/* Outputs: device pointers, any may be NULL to skip. */
typedef struct {
  float*    poses_dev;          /* [H][12] refined [R_wc | C] */
  float*    cost_dev;           /* [H] total cost (Eq.7) of the final accepted state at the last level */
  int*      n_valid_dev;        /* [H] valid points of that state */
  unsigned* status_dev;         /* [H] PILOT_STATUS_* bitmask */
  float*    iter_hessian_dev;   /* [sum(iters)][H][36] H_total (supp Eq.5), undamped, row-major symmetric, order (rho, phi) */
  float*    iter_gradient_dev;  /* [sum(iters)][H][6]  g_total (supp Eq.6) */
  float*    iter_cost_dev;      /* [sum(iters)][H]     total cost at the pose where that system was built */
  float*    iter_lambda_dev;    /* [sum(iters)][H]     lambda used in that solve */
} pilot_refine_outputs;

#endif /* PILOT_ORACLE_TYPES_H */
