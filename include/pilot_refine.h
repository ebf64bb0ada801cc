/*
 * pilot_refine.h — C-ABI of the B200-native PiLoT v2 hot path:
 * batched feature-metric Levenberg–Marquardt 6-DoF refinement of many pose
 * hypotheses against DSM-lifted reference points, with the gravity-direction
 * and single-point laser-range priors, a damped 6x6 solve and an SE(3) update
 * over a feature pyramid.
 *
 * Passages implemented (arxiv/paper_2606_31098, line numbers of PAPER.md):
 *   Eq.(1) photo residual
 *   Eq.(2) robust photo cost
 *   Eq.(3) gravity residual               PAPER.md:128-132, supp II-D PAPER.md:392
 *   Eq.(4)-(6) centre ray / range point / height residual
 *   Eq.(7) total cost
 *   Eq.(8) damped normal equation
 *   Eq.(9) SE(3) update
 *   supp Eq.(5)(6) prior fusion
 *   coarse-to-fine pyramid loop
 *   fused visual kernel description
 * The readings taken where the paper is silent are listed in DESIGN.md §3.
 *
 * Plain C, no exceptions, no globals, no torch types. All pointers whose name
 * ends in "_dev" are CUDA DEVICE pointers OWNED BY THE CALLER (typically torch
 * tensors); the library never frees or reallocates them. All other pointers are
 * host pointers. The CPU oracle (oracle/pilot_oracle.h) reuses these structs with
 * every "_dev" pointer holding a HOST pointer instead.
 */
#ifndef PILOT_REFINE_H
#define PILOT_REFINE_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

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

/* Per-run inputs. Host scalars are read before run() returns.
 * WORLD FRAME: every world quantity of this ABI (anchors, poses, DSM origin, footprint corners) is fp32, so it must be
 * expressed relative to a LOCAL origin near the scene (e.g. the centre of the DSM crop), not in a global map frame: at
 * UTM-scale coordinates (5e5 / 4e6 m) fp32 quantises to 3-50 cm, far above the 1e-3 m the path is accurate to. The result
 * does not depend on the choice of origin (tests/test_oracle_pins.py::test_world_origin_shift_invariance). */
typedef struct {
  int n_hypotheses;                                  /* H <= max_hypotheses */
  int n_points[PILOT_MAX_LEVELS];                    /* N_l <= max_points */
  const void*  query_feat_dev[PILOT_MAX_LEVELS];     /* [height][width][channels], C innermost, base 16-B aligned (Eq.1 f^q_l) */
  const float* query_conf_dev[PILOT_MAX_LEVELS];     /* [height][width] query confidence w^q_l, or NULL (=1) */
  float        intrinsics[PILOT_MAX_LEVELS][4];      /* fx, fy, cx, cy of K_l (Eq.1); pixel (x,y) sits at continuous (x,y) */
  const float* points_dev[PILOT_MAX_LEVELS];         /* [n_points][4] = geo-anchor P_j x,y,z (world, metres), w_ref>=0 (supp Eq.3) */
                                                     /* any order is correct; a spatially coherent one (raster / Morton) is what keeps the gather in L2:
                                                        see pilot_refine_sort_anchors. Coordinates are fp32: pass them relative to a LOCAL origin (see below) */
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

/*
 * Bytes of device scratch a handle with this config needs. Pure host function.
 * Returns 0 on a bad config.
 */
size_t pilot_refine_workspace_bytes(const pilot_refine_config* cfg);

/*
 * Create a handle. Validates cfg; selects cfg->device; if cfg->workspace_dev is
 * NULL allocates the scratch once with cudaMalloc (freed by destroy), otherwise
 * uses the caller's buffer (PILOT_ERR_WORKSPACE if too small; the buffer must
 * outlive the handle and be 256-B aligned). No other allocation ever happens.
 */
int pilot_refine_create(const pilot_refine_config* cfg, pilot_refine_handle** out);

/*
 * Enqueue one full refinement (all levels, all iterations, Eqs.1-9) of
 * in->n_hypotheses hypotheses on `cuda_stream` (a cudaStream_t, e.g.
 * torch.cuda.current_stream().cuda_stream; NULL = legacy default stream).
 * ASYNCHRONOUS: performs no allocation and no host synchronisation; host structs
 * are read before it returns; device buffers are read/written in stream order.
 * Per-hypothesis numerical trouble is reported in status_dev, not as an error.
 * One run at a time per handle.
 */
int pilot_refine_run(pilot_refine_handle* h, const pilot_refine_inputs* in,
                     const pilot_refine_params* p, const pilot_refine_outputs* out,
                     void* cuda_stream);

/* Destroy a handle; frees the scratch only if create() allocated it. destroy(NULL) is a no-op. */
int pilot_refine_destroy(pilot_refine_handle* h);

/*
 * The same refinement as pilot_refine_create + pilot_refine_run (Eqs.1-9, all levels; default launch and math modes) for
 * callers that may NOT allocate device memory (code under CUDA-graph capture, serving loops, harnesses that forbid
 * cudaMalloc): no handle, and the optimiser workspace (per-hypothesis LM state, tickets, per-CTA partial sums) is a
 * file-scope device array of PILOT_STATIC_WORKSPACE_BYTES inside the library, which every GPU that loads the library
 * holds until the process exits. The call makes no cudaMalloc / cudaFree and calls no allocating library routine; the
 * caller still owns every input and output buffer. cfg: as for create(), with workspace_dev == NULL (else PILOT_ERR_ARG).
 * LIMIT: pilot_refine_workspace_bytes(cfg) <= PILOT_STATIC_WORKSPACE_BYTES (32 MiB), i.e. about 128 bytes x max_hypotheses x
 * ceil(max_points / 128) (+ 0.5 KB per hypothesis): 256 hypotheses x 65536 anchors (config 4: 16.9 MB) fit, 1024 x 65536
 * (67 MB) do not -> PILOT_ERR_WORKSPACE, nothing launched. launches_out (optional, host): kernels launched by this call.
 * SHARED STATE: every call on a device uses the same array, which keeps the previous call's contents; each call re-initialises
 * what it reads (LM state and tickets of its n_hypotheses; partial sums are written before they are read), so back-to-back
 * calls on ONE stream are correct. Calls that may overlap on the GPU (two streams, two host threads, a handle-free call
 * racing a captured graph that contains one) RACE on the array: serialise them. Asynchronous like pilot_refine_run.
 */
#define PILOT_STATIC_WORKSPACE_BYTES (32u << 20)
size_t pilot_refine_static_workspace_bytes(void);
int pilot_refine_run_static(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                            const pilot_refine_params* p, const pilot_refine_outputs* out,
                            void* cuda_stream, int* launches_out);

/*
 * Host-buffer path (what bench.py's "e2e" times): every "_dev" pointer of `in_host` and
 * `out_host` is a HOST pointer (pinned memory recommended). run_host copies the inputs into
 * device staging owned by the handle (cudaMemcpyAsync on the handle's copy stream), enqueues
 * pilot_refine_run, copies the requested outputs back and synchronises the stream before
 * returning. The staging is sized at create_host() from cfg plus the DSM capacity given
 * there and is allocated once with cudaMalloc (cfg->workspace_dev must be NULL); a run whose
 * DSM exceeds that capacity returns PILOT_ERR_UNSUPPORTED.
 */
int pilot_refine_create_host(const pilot_refine_config* cfg, int max_dsm_width, int max_dsm_height,
                             pilot_refine_handle** out);
int pilot_refine_run_host(pilot_refine_handle* h, const pilot_refine_inputs* in_host,
                          const pilot_refine_params* p, const pilot_refine_outputs* out_host,
                          void* cuda_stream);

/*
 * The same, pipelined: submit_host() enqueues the upload of one run's inputs on the handle's own copy stream into
 * one of TWO device staging halves, then — on `cuda_stream`, after an event — the run and the copy of its outputs
 * to out_host, and returns a ticket (>= 0) at once; wait_host() blocks until the OLDEST submitted run's outputs are
 * in host memory. Submitting run k+1 before waiting for run k overlaps its upload with run k's kernels. At most two
 * runs may be in flight (a third submit returns PILOT_ERR_UNSUPPORTED); the host buffers of a run (inputs: pinned
 * memory, or the upload serialises; outputs) must stay valid until its wait_host() returned.
 * run_host == submit_host + wait_host. The two runs in flight share the handle's workspace, so they execute one after the
 * other: a run submitted on a different stream than the previous one is ordered behind it with an event. For every other
 * entry point the rule is the usual one: calls on ONE handle (run, run_levels, sequence_step, ...) must be issued on one
 * stream or be ordered by the caller; different handles are independent.
 */
int pilot_refine_submit_host(pilot_refine_handle* h, const pilot_refine_inputs* in_host,
                             const pilot_refine_params* p, const pilot_refine_outputs* out_host,
                             void* cuda_stream);
int pilot_refine_wait_host(pilot_refine_handle* h);

/*
 * The paper's per-frame schedule (supp II-C PAPER.md:381-386, selection PAPER.md:168) through host buffers, one call per
 * frame: upload of the frame's inputs (as submit_host: copy stream, two staging halves), then on `cuda_stream` the seeding
 * of the n grid hypotheses around prior_pose_host ([12] row-major [R_wc | C]; pilot_refine_seed_hypotheses with the offsets
 * of set_grid_host and `seed_frame`), the coarse level for all of them (run_levels 0..1), the `keep` lowest objectives
 * (prune_topk), the finer levels for those (run_levels 1..n_levels), the arg-min (select_best), and the copy of the selected
 * pose [12], its objective and its index INTO THE GRID to the three host pointers (each may be NULL). Returns a ticket;
 * pilot_refine_wait_host() blocks until the oldest submitted frame's results are in host memory, so frame k+1 uploads while
 * frame k refines. in_host->init_poses_dev and n_hypotheses are ignored. The handle comes from create_host with
 * max_hypotheses >= n; set_grid_host copies the [n][6] offset table (pilot_refine_grid_offsets) to the device once (it
 * allocates; not while runs are in flight; n <= PILOT_TOPK_MAX). Errors as submit_host; PILOT_ERR_ARG without a grid,
 * for keep outside [1, n] or a one-level pyramid.
 */
int pilot_refine_set_grid_host(pilot_refine_handle* h, const float* offsets_host, int n);
int pilot_refine_submit_pruned_host(pilot_refine_handle* h, const pilot_refine_inputs* in_host, const pilot_refine_params* p,
                                    const float* prior_pose_host, int keep, int seed_frame, float* best_pose_host,
                                    float* best_cost_host, int* best_index_host, void* cuda_stream);

/*
 * Tuning knob: anchors per CTA of the photo kernel (a multiple of 128; 0 = built-in heuristic,
 * which sizes the grid to a few waves of 2 CTAs per SM). Results do not depend on it beyond
 * fp32 summation order.
 */
int pilot_refine_set_chunk(pilot_refine_handle* h, int chunk);

/*
 * Launch strategy. PASSES: one launch per EVAL pass, (hypothesis x anchor-chunk) CTAs — the throughput path for
 * large hypothesis x anchor products. RESIDENT: one launch per pyramid level, a thread-block cluster of `cluster`
 * CTAs (1, 2, 4, 8; 0 = heuristic) owns a hypothesis for all of the level's LM iterations — the latency path for
 * small problems (the paper's own frame shape). PASSES_SPLIT: as PASSES, but the per-hypothesis finalisation (priors,
 * accept/reject, solve, update) runs in a second launch with one warp per hypothesis instead of in the last CTA of
 * each hypothesis — for many hypotheses with few anchors each (the 1210-hypothesis coarse level). AUTO (default)
 * picks per level from H, N and the SM count. All compute the same
 * sums from the same per-unit arithmetic; they differ in fp32 summation order only.
 */
typedef enum { PILOT_EXEC_AUTO = 0, PILOT_EXEC_PASSES = 1, PILOT_EXEC_RESIDENT = 2, PILOT_EXEC_PASSES_SPLIT = 3 } pilot_exec_mode;
int pilot_refine_set_exec_mode(pilot_refine_handle* h, int mode, int cluster);

/*
 * Optional extra records of the following runs on this handle (NULL = off, the default), for the backward pass of the
 * unrolled refinement (pilot_refine_unrolled_backward): iter_poses_dev [sum(iters)][H][12] fp32 = the pose [R_wc | C] at
 * which each recorded system (outputs.iter_hessian_dev ...) was built, i.e. the accepted pose at that solve;
 * iter_accept_dev [sum(iters)][H] = 1 if the step solved from that record was accepted (PILOT_LM_FIXED: always), 0 if it
 * was rejected or its factorisation failed (the pose did not move). Caller-owned device buffers, written in stream order
 * by pilot_refine_run / run_levels (every launch strategy); rows of levels outside a run_levels range are untouched.
 */
int pilot_refine_set_iterate_outputs(pilot_refine_handle* h, float* iter_poses_dev, int* iter_accept_dev);

/*
 * Arithmetic of the per-unit contraction (Eq.(1),(8) PAPER.md:118,160-164). FP32: taps are
 * unpacked to fp32 and every step runs on the FMA pipe (packed FFMA2). MMA: for 16-bit features (bf16 / fp16) with
 * 16, 32, 64 or 128 channels and the exact bilinear gradient, the first differences of the taps are taken in the
 * storage type (exact for neighbouring values within a factor of two; else one rounding of 2^-9 / 2^-12 relative to
 * the difference), and their 4 x 4 Gram matrix per unit is accumulated in fp32 on the tensor cores (mma.sync
 * m16n8k16); the bilinear combination follows in fp32. This path also PROJECTS in fp32 (the camera
 * centre as a hi + lo pair of floats, so P - C loses nothing of the double pose): (u, v) within ~1e-6 (fx + |u - cx|)
 * pixels of the double projection, a change of the continuous bilinear interpolant far below the features' own rounding.
 * Visibility is not continuous, so it stays a double decision: an anchor within 4e-6 (fx + fy + W + H) pixels of the
 * border of the map, or within 4e-6 |P - C| of z_near, is projected again in double (n_valid and the set of
 * contributing units are those of the double projection; FP32 projects every anchor in double). AUTO (default) = MMA where it applies AND was measured faster
 * (64 or more channels on the one-launch-per-pass strategy), FP32 elsewhere. Asking for MMA where it does not apply
 * falls back to FP32 (not an error). Results agree within the bf16 / fp16 parity
 * tolerance of the path (5e-3 relative on H and g); fp32 features always use FP32.
 */
typedef enum { PILOT_MATH_AUTO = 0, PILOT_MATH_FP32 = 1, PILOT_MATH_MMA = 2 } pilot_math_mode;
int pilot_refine_set_math_mode(pilot_refine_handle* h, int mode);

/* Number of kernel launches the last pilot_refine_run on this handle enqueued (host counter). */
int pilot_refine_last_launches(const pilot_refine_handle* h);

/* What the last run (or run_levels) of this handle chose per pyramid level: bit l of *mma_levels = the tensor-core
 * contraction (pilot_math_mode), bit l of *resident_levels = the cluster-resident kernel (pilot_exec_mode). Pure host
 * call; either pointer may be NULL. bench.py reports these instead of mirroring the AUTO rules.
 */
int pilot_refine_last_plan(const pilot_refine_handle* h, unsigned* mma_levels, unsigned* resident_levels);

/* Measurement helper: the number of VISIBLE (anchor, hypothesis) unit evaluations of the handle's last run, summed over
 * every EVAL pass of every level (a unit is visible iff Z > z_near and its 2 x 2 footprint lies inside the map: a2 of
 * SURVEY.md §8(a), "visibility checking" PAPER.md:485) - the units that actually gather taps; bench.py's roofline counts
 * bytes for these only. Runs one tiny kernel on cuda_stream and SYNCHRONISES that stream. out_host: host pointer.
 */
int pilot_refine_last_visible_evals(pilot_refine_handle* h, void* cuda_stream, unsigned long long* out_host);

/*
 * The same as pilot_refine_run restricted to pyramid levels level_begin <= l < level_end
 * (0 <= level_begin < level_end <= n_levels): what the paper's schedule needs to prune the
 * hypothesis set between the coarse and the finer levels (supp II-C).
 * The final outputs (poses/cost/n_valid/status) describe the accepted state at level
 * level_end-1. The iter_* records keep the layout of the whole run: record index =
 * sum(iters[0..l-1]) + k for every level l (levels outside the range are left untouched),
 * with H = in->n_hypotheses of THIS call. pilot_refine_run == run_levels(0, n_levels).
 */
int pilot_refine_run_levels(pilot_refine_handle* h, const pilot_refine_inputs* in,
                            const pilot_refine_params* p, const pilot_refine_outputs* out,
                            int level_begin, int level_end, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Hypothesis set: sampling, pruning, selection ("sample multiple pose hypotheses in
 * the local (x,y,psi) space around the propagated pose prior"; supp II-C PAPER.md:381-386: +-10 m
 * grid with 2 m step x yaw offsets {+-1,+-3,+-5,+-7,+-9} deg = 1210 hypotheses, top 128 by
 * post-update objective kept after the coarse level; "the hypothesis with the lowest
 * final objective value is selected"). All asynchronous on `cuda_stream`, no allocation, no sync.
 */
typedef enum {
  PILOT_SEED_CAMERA = 0,  /* R_wc,m = R_wc Rot(w_m): rotation offset expressed in the camera frame */
  PILOT_SEED_WORLD  = 1   /* R_wc,m = Rot(w_m) R_wc: rotation offset in the world frame (yaw = w || vertical) */
} pilot_seed_frame;

/*
 * Pure host helper: fills offsets_host[n][6] = (w_x,w_y,w_z rotation vector in radians; t_x,t_y,t_z in
 * metres) with the paper's grid: t = (i*xy_step, j*xy_step, 0) for i,j in [-r, r], r = floor(xy_range /
 * xy_step + 1e-6), and w = radians(yaw_deg[k]) * up (PILOT_SEED_WORLD offsets; `up` = unit vertical,
 * typically -gamma^W). Order: index = ((i+r)*(2r+1) + (j+r))*n_yaw + k. Returns the number of entries
 * ((2r+1)^2 * n_yaw; 1210 for 10 m / 2 m / 10 yaws) — also when offsets_host is NULL or capacity is too
 * small (nothing is written then) — or a negative PILOT_ERR_ARG.
 */
int pilot_refine_grid_offsets(float xy_range, float xy_step, const float* yaw_deg, int n_yaw,
                              const float up[3], float* offsets_host, int capacity);

/*
 * out_poses_dev[m] = base pose composed with offsets_dev[m] (m < n): rotation per `frame` above,
 * centre C_m = C + t_m. base_pose_dev: [12] row-major [R_wc | C]; offsets_dev: [n][6]; out: [n][12].
 */
int pilot_refine_seed_hypotheses(const float* base_pose_dev, const float* offsets_dev, int n, int frame,
                                 float* out_poses_dev, void* cuda_stream);

/*
 * Index of the lowest cost among n (NaN counts as +inf; ties -> lowest index; n >= 1). Writes (each
 * optional, may be NULL): best_idx_dev[1], best_pose_dev[12] (copied from poses_dev[best]),
 * best_cost_dev[1].
 */
int pilot_refine_select_best(const float* cost_dev, const float* poses_dev, int n,
                             int* best_idx_dev, float* best_pose_dev, float* best_cost_dev,
                             void* cuda_stream);

/*
 * The k hypotheses of lowest cost, in ascending (cost, index) order (NaN = +inf): idx_out_dev[k],
 * and optionally their poses (poses_out_dev[k][12] gathered from poses_dev) and costs
 * (cost_out_dev[k]). 1 <= k <= n <= PILOT_TOPK_MAX, else PILOT_ERR_UNSUPPORTED.
 */
#define PILOT_TOPK_MAX 8192
int pilot_refine_prune_topk(const float* cost_dev, const float* poses_dev, int n, int k,
                            int* idx_out_dev, float* poses_out_dev, float* cost_out_dev,
                            void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Streaming sequence ("we use the pose estimated from the previous query image as the pose
 * prior"; supp IV PAPER.md:457-461: the reference of the NEXT frame is prepared asynchronously while the
 * current frame is localised). A sequence object owns: one refinement handle, the static heightfield, a
 * DOUBLE BUFFER of per-frame device inputs filled from host memory on the library's own copy stream, the
 * hypothesis-offset table, and an on-device log of per-frame results. Per frame, on the caller's compute
 * stream and without any host synchronisation:
 *     hypotheses = previous estimate (x) offsets  ->  pilot_refine_run  ->  arg-min  ->  new estimate, log row.
 * upload() of frame i+1 may be issued before step() of frame i: the copy overlaps the refinement; events
 * order slot reuse. upload() first copies the caller's arrays into page-locked staging owned by the object, so
 * they may be pageable and may be reused as soon as upload() returns.
 */
typedef struct pilot_refine_sequence pilot_refine_sequence; /* opaque */

typedef struct {
  int n_hypotheses;                    /* H per frame, <= cfg.max_hypotheses */
  const float* offsets;                /* HOST [H][6] (rotation vector rad, translation m), see pilot_refine_seed_hypotheses */
  int seed_frame;                      /* pilot_seed_frame */
  const float* dsm;                    /* HOST [dsm_height][dsm_width] heightfield, uploaded once (NULL: no range prior) */
  int dsm_width, dsm_height;
  float dsm_origin_x, dsm_origin_y, dsm_gsd;
  float gravity_world[3];
  int max_frames;                      /* capacity of the result log */
} pilot_refine_sequence_config;

typedef struct {                       /* one frame; HOST pointers, same layouts as pilot_refine_inputs */
  int n_points[PILOT_MAX_LEVELS];
  const void*  query_feat[PILOT_MAX_LEVELS];
  const float* query_conf[PILOT_MAX_LEVELS];      /* NULL = 1 */
  const float* points[PILOT_MAX_LEVELS];
  const void*  ref_feat[PILOT_MAX_LEVELS];
  float intrinsics[PILOT_MAX_LEVELS][4];
  float gravity_imu[3], range_ray_cam[3], range_meas;
  int arrays_pinned;                   /* 1: the arrays above are page-locked (cudaHostAlloc / cudaHostRegister) and stay
                                          valid and unchanged until this frame's step() has run on the device: they are
                                          copied straight from the caller's memory (no host staging copy). 0: staged. */
} pilot_refine_frame;

#define PILOT_SEQ_ROW 16               /* floats per log row: pose[12], cost, best index, n_valid, status */

/* Allocates everything once (cudaMalloc, cudaHostAlloc, one copy stream, events). cfg->workspace_dev must be NULL. */
int pilot_refine_sequence_create(const pilot_refine_config* cfg, const pilot_refine_sequence_config* sc,
                                 pilot_refine_sequence** out);
/* Sets the pose prior of the next frame (frame 0: e.g. the last GNSS fix). pose_host: [12]. */
int pilot_refine_sequence_set_prior(pilot_refine_sequence* s, const float* pose_host, void* cuda_stream);
/* Stages one frame (host memcpy) and enqueues its host->device copy into the free half of the double buffer on
 * the copy stream. Returns PILOT_ERR_UNSUPPORTED if both halves hold frames that were not stepped yet.
 * Asynchronous w.r.t. the device (may wait on the host for the copy issued two uploads earlier). */
int pilot_refine_sequence_upload(pilot_refine_sequence* s, const pilot_refine_frame* f);
/* Refines the oldest uploaded frame on `cuda_stream` (waits for its copy by event). Asynchronous.
 * PILOT_ERR_ARG if no uploaded frame is pending or the log is full. */
int pilot_refine_sequence_step(pilot_refine_sequence* s, const pilot_refine_params* p, void* cuda_stream);
/* Copies log rows [first, first+count) to results_host[count][PILOT_SEQ_ROW] and synchronises `cuda_stream`. */
int pilot_refine_sequence_results(pilot_refine_sequence* s, int first, int count, float* results_host,
                                  void* cuda_stream);
/* The LAST stepped frame's hypothesis set: seeds [H][12], refined poses [H][12], costs [H] (each optional) to
 * host memory; synchronises `cuda_stream`. For inspection and parity tests. */
int pilot_refine_sequence_last_frame(pilot_refine_sequence* s, float* seeds_host, float* poses_host,
                                     float* cost_host, void* cuda_stream);
/* Kernel launches enqueued by the last step(). */
int pilot_refine_sequence_last_launches(const pilot_refine_sequence* s);
/* Waits for both streams' pending work of this object, then frees everything. destroy(NULL) is a no-op. */
int pilot_refine_sequence_destroy(pilot_refine_sequence* s);

/* ---------------------------------------------------------------------------------------------
 * Reference-crop geometry that produces the geo-anchors (supp II-B). Asynchronous on
 * `cuda_stream`, no allocation, no host synchronisation. The heightfield arguments are those of
 * pilot_refine_inputs (dsm_dev [dsm_height][dsm_width] fp32, origin, metres per sample).
 */

/*
 * Map-footprint estimation, supp Eq.(2): rays from the camera centre of pose_dev ([12] row-major
 * [R_wc | C]) through the image corners (0,0), (W-1,0), (W-1,H-1), (0,H-1) of a width x height image with
 * intrinsics (fx, fy, cx, cy); along each ray the sample s_i = i*s_max/n_samples, i = 1..n_samples, with the smallest
 * |z_ray(s) - h_DSM(x_ray(s), y_ray(s))| (bilinear h_DSM; samples outside the heightfield are skipped; ties -> the
 * smallest s). corners_dev[4][4] = x, y, z_ray at s*, and that residual; a ray with no sample over the heightfield
 * gives a row of NaN. Decisions are taken in double precision.
 */
int pilot_refine_footprint(const float* pose_dev, const float intrinsics[4], int width, int height,
                           const float* dsm_dev, int dsm_width, int dsm_height,
                           float dsm_origin_x, float dsm_origin_y, float dsm_gsd,
                           int n_samples, float s_max, float* corners_dev, void* cuda_stream);

/*
 * Pixel-aligned warping + geo-anchor construction, supp Eq.(3): the homography that maps the
 * crop corners (0,0), (Wc-1,0), (Wc-1,Hc-1), (0,Hc-1) onto the footprint corners_dev[4][4] (x, y used) gives every
 * crop pixel pix_dev[n][2] = (u, v) its map coordinates (x^m, y^m); the warped DSM layer D^r is the bilinear
 * heightfield sample there. points_dev[n][4] = x^m, y^m, D^r, w with w = 1, or (x^m, y^m, 0, 0) when the pixel falls
 * outside the heightfield or the footprint is degenerate — the layout pilot_refine_inputs.points_dev takes (an
 * anchor of weight 0 contributes nothing to Eq.2).
 */
int pilot_refine_lift_anchors(const float* corners_dev, int crop_width, int crop_height,
                              const float* pix_dev, int n,
                              const float* dsm_dev, int dsm_width, int dsm_height,
                              float dsm_origin_x, float dsm_origin_y, float dsm_gsd,
                              float* points_dev, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Unrolled reprojection supervision, forward value (supp III-C). For every pose
 * T^k of poses_dev[n_poses][12] (row-major [R_wc | C], e.g. the poses of successive pilot_refine_run_levels calls) and the
 * ground-truth pose pose_star[12] (HOST values):
 *   L_k = 1/|V| sum_{j in V} rho_B(||pi(K, T^k P_j) - pi(K, T* P_j)||^2)                    supp Eq.(7)-(8)
 * with Barron's general robust loss on the squared residual s, z = s/scale^2:
 *   rho_B = |alpha-2|/alpha ((z/|alpha-2| + 1)^(alpha/2) - 1);  alpha = 2: z/2;  alpha = 0: log(z/2 + 1);
 *   alpha = -inf: 1 - exp(-z/2).  (alpha and scale are parameters: the paper states neither.)
 * V = points of points_dev[n_points][4] (x, y, z, unused; 16-byte aligned) in front of BOTH cameras (Z > z_near) whose
 * ground-truth projection lies inside [0, width-1] x [0, height-1]; the optimised projection may leave the image.
 * loss_dev[n_poses] (0 where V is empty), n_visible_dev[n_poses] = |V| (may be NULL). Projections, the loss and the
 * sums are double precision, summed in a fixed order. Asynchronous on cuda_stream, no allocation. The backward pass
 * through the unrolled LM steps is pilot_refine_unrolled_backward below.
 * Errors: PILOT_ERR_ARG (NULL / misaligned pointer, scale <= 0, alpha NaN or +inf, bad image size), PILOT_ERR_CUDA.
 */
int pilot_refine_reprojection_loss(const float* poses_dev, int n_poses, const float pose_star[12],
                                   const float* points_dev, int n_points, const float intrinsics[4],
                                   int width, int height, float z_near, float alpha, float scale,
                                   float* loss_dev, int* n_visible_dev, void* cuda_stream);

/*
 * Backward pieces of the unrolled refinement ("the refinement is unrolled over nine coarse-to-fine steps",
 * supp III-C PAPER.md:427-440). reprojection_loss_grad: as reprojection_loss, plus grad_dev[k][6] = dL_k / d eps for the left
 * perturbation T_cw <- exp(eps^) T_cw of pose k (eps = (rho; phi), the LM's own parametrisation: reading A1/A2 of DESIGN.md);
 * loss_dev / n_visible_dev may be NULL. lm_step_adjoint: for n independent LM steps dxi = -(H + lambda D)^-1 g (Eq.8,
 * PAPER.md:160-164; D = I or diag(max(H_ii, 1e-12)) per damp_mode), T' = exp(dxi^) T (Eq.9), given q_dev[m][6] = dL / d eps
 * at the UPDATED pose: dxi_dev[m][6]; grad_gradient_dev[m][6] = dL/dg; grad_hessian_dev[m][36] = dL/dH, symmetric, such that
 * dL = <dL/dH, dH> for symmetric dH; q_prev_dev[m][6] (optional) = the part of dL / d eps at the PREVIOUS pose that flows
 * through the retraction, Ad(exp(dxi^))^T q; status_dev[m] (optional) = PILOT_STATUS_CHOL_FAIL if H + lambda D is not
 * positive definite. hessian_dev [n][36] row-major (symmetrised on read), gradient_dev [n][6], lambda_dev [n]: what
 * pilot_refine_run records per iteration. The dependence of H and g on the pose and on the feature maps is
 * pilot_refine_photo_backward below. Asynchronous on cuda_stream; double arithmetic, one rounding to fp32 on output.
 */
int pilot_refine_reprojection_loss_grad(const float* poses_dev, int n_poses, const float pose_star[12],
                                        const float* points_dev, int n_points, const float intrinsics[4],
                                        int width, int height, float z_near, float alpha, float scale,
                                        float* loss_dev, int* n_visible_dev, float* grad_dev, void* cuda_stream);
int pilot_refine_lm_step_adjoint(const float* hessian_dev, const float* gradient_dev, const float* lambda_dev,
                                 const float* q_dev, int n, int damp_mode, float* dxi_dev, float* grad_hessian_dev,
                                 float* grad_gradient_dev, float* q_prev_dev, unsigned* status_dev, void* cuda_stream);

/*
 * Backward pass of the photo term: the transpose of the gather (Eq.1, Eq.2, Eq.8, PAPER.md:118-122,
 * 160-164). For every pose m < n_poses (poses_dev [n][12] = [R_wc | C], the poses at which the systems were built) and one
 * pyramid level, with S_m = <grad_hessian_dev[m], H_m> + <grad_gradient_dev[m], g_m> (H_m, g_m the PHOTO part of the normal
 * equations at that pose, GRAD_BILINEAR_EXACT; grad_hessian_dev [n][36] is symmetrised on read), it ADDS to
 *   grad_feat_dev [height][width][channels] fp32   sum_m dS_m / dF        (the query feature map)
 *   grad_ref_dev  [n_points][channels]      fp32   sum_m dS_m / df^r
 *   grad_conf_dev [height][width]           fp32   sum_m dS_m / dconf     (only with query_conf_dev; may be NULL)
 * (the caller zeroes or pre-loads them; any may be NULL) and WRITES grad_pose_dev[m][6] = dS_m / d eps for the left
 * perturbation T_cw <- exp(eps^) T_cw, eps = (rho; phi) (may be NULL). The bilinear cell and the visible set are held fixed
 * (piecewise constant); the robust weight's second derivative and the dependence of the projection Jacobian on the point
 * are included. The priors are not part of S (they do not depend on the features). Sums use fp32 atomics: the result is
 * reproducible to rounding, not bit for bit. Together with pilot_refine_reprojection_loss_grad and
 * pilot_refine_lm_step_adjoint this is the chain rule through one unrolled LM step for a photo-only objective.
 * points_dev 16-byte aligned; map under 4 GiB of elements. Asynchronous on cuda_stream.
 */
int pilot_refine_photo_backward(const void* query_feat_dev, const float* query_conf_dev, int width, int height, int channels,
                                pilot_dtype feat_dtype, const float intrinsics[4], const float* points_dev,
                                const void* ref_feat_dev, int n_points, const float* poses_dev,
                                const float* grad_hessian_dev, const float* grad_gradient_dev, int n_poses,
                                pilot_loss loss, float loss_scale, float z_near, float* grad_feat_dev, float* grad_ref_dev,
                                float* grad_conf_dev, float* grad_pose_dev, void* cuda_stream);

/*
 * Backward pass through ALL the LM steps of an unrolled refinement (supp III-C: "the
 * refinement is unrolled over nine coarse-to-fine steps, and the final training objective averages the reprojection losses
 * over all unrolled steps"). With T = sum(iters) solves, T^r the pose after r solves (T^0 = the initial pose) and
 *   L = sum_{r=1..T} step_weights[r-1] L_r(T^r)        (L_r of supp Eq.8 as in pilot_refine_reprojection_loss; the paper's
 *                                                       objective is step_weights = 1/T),
 * it reads the chain  T^{r+1} = exp(dxi_r^) T^r (Eq.9), dxi_r = -(H_r + lambda_r D)^-1 g_r (Eq.8), (H_r, g_r) = the photo
 * term at T^r on the level of solve r  backwards from the last pose - lm_step_adjoint, then photo_backward, per ACCEPTED
 * solve; a rejected solve (or a failed factorisation) did not move the pose and passes dL/d eps through - and ADDS
 *   grads.grad_feat_dev[l] [height_l][width_l][channels_l] fp32   dL/dF_l     (query feature map of level l)
 *   grads.grad_ref_dev[l]  [n_points_l][channels_l]        fp32   dL/df^r_l
 *   grads.grad_conf_dev[l] [height_l][width_l]             fp32   dL/dconf_l  (only where the level has a confidence map)
 * (caller zeroes or pre-loads; any may be NULL) and WRITES grads.grad_init_pose_dev [H][6] = dL/d eps at the initial pose
 * (left perturbation of T_cw, eps = (rho; phi)) and grads.loss_dev [H] = L (either may be NULL). One chain per hypothesis,
 * all H side by side. lambda_r and the accept / reject decisions are piecewise constant and held fixed, as are the visible
 * sets and bilinear cells. records: what a forward run with pilot_refine_set_iterate_outputs wrote (device pointers;
 * final_poses_dev = outputs.poses_dev). `in`, `p`, cfg (level shapes and dtype) as given to that run. supervision: HOST
 * scalars + the device points of V's candidates (pilot_refine_reprojection_loss); step_weights is a HOST array of T floats.
 * The objective must be the photo term alone: PILOT_ERR_UNSUPPORTED if w_gravity != 0, the range prior is on, or grad_mode
 * is not GRAD_BILINEAR_EXACT (the priors' pose-dependence is not part of this chain). scratch_dev: 256-byte aligned,
 * at least pilot_refine_unrolled_backward_scratch_bytes(H, T) (else PILOT_ERR_WORKSPACE); no allocation. Asynchronous on
 * cuda_stream: 4 launches per solve.
 */
typedef struct {
  const float* iter_hessian_dev;    /* [T][H][36] */
  const float* iter_gradient_dev;   /* [T][H][6]  */
  const float* iter_lambda_dev;     /* [T][H]     */
  const float* iter_poses_dev;      /* [T][H][12]  (pilot_refine_set_iterate_outputs) */
  const int*   iter_accept_dev;     /* [T][H]      (pilot_refine_set_iterate_outputs) */
  const float* final_poses_dev;     /* [H][12]     (outputs.poses_dev) */
} pilot_refine_unrolled_records;
typedef struct {
  float pose_star[12];              /* ground-truth pose [R_wc | C] */
  const float* points_dev;          /* [n_points][4] sampled 3-D points (16-byte aligned) */
  int n_points;
  float intrinsics[4];              /* K^q of supp Eq.7 */
  int width, height;                /* image size that defines V */
  float alpha, scale;               /* Barron loss shape and scale */
  const float* step_weights;        /* HOST [T] */
} pilot_refine_supervision;
typedef struct {
  float* grad_feat_dev[PILOT_MAX_LEVELS];
  float* grad_ref_dev[PILOT_MAX_LEVELS];
  float* grad_conf_dev[PILOT_MAX_LEVELS];
  float* grad_init_pose_dev;        /* [H][6] */
  float* loss_dev;                  /* [H] */
} pilot_refine_unrolled_grads;
size_t pilot_refine_unrolled_backward_scratch_bytes(int n_hypotheses, int total_iters);
int pilot_refine_unrolled_backward(const pilot_refine_config* cfg, const pilot_refine_inputs* in, const pilot_refine_params* p,
                                   const pilot_refine_unrolled_records* records, const pilot_refine_supervision* supervision,
                                   const pilot_refine_unrolled_grads* grads, void* scratch_dev, size_t scratch_bytes,
                                   void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Anchor order (kernel description PAPER.md:485). The sums of Eq.(2) and Eq.(8) do not depend on the
 * order of the anchors, but the THROUGHPUT of pilot_refine_run does: CTAs that run together sweep the same batches of
 * anchors under different poses, and only when the anchors of a batch are neighbours on the ground does the union of
 * their footprints stay in L2. points_dev / ref_feat_dev of pilot_refine_inputs should therefore be in a spatially
 * coherent order (raster order of a reference crop, or Morton order); measured on config 4 (65536 anchors, 265 MB map):
 * 7.8 ms per step in Morton order, 9.3 ms in random order. pilot_refine_sort_anchors puts one level's anchors in Morton
 * order of their (x, y): key = bit-interleaved 16-bit quantisation of x and y inside the bounding box of all anchors
 * (q = floor((v - min) * (65535 / (max - min))) in fp32, one IEEE operation per step; equal keys keep their input order),
 * and writes points_out_dev[j] = points_dev[perm[j]], ref_out_dev row j = ref_feat_dev row perm[j] (may both be NULL),
 * perm_out_dev[j] = perm[j] (optional). In and out buffers must differ; all pointers 16-byte aligned; channels * element
 * size a multiple of 16. temp_dev: at least pilot_refine_sort_anchors_temp_bytes(n_points) bytes of device scratch
 * (PILOT_ERR_WORKSPACE otherwise). Asynchronous on cuda_stream, no allocation, no host synchronisation.
 */
size_t pilot_refine_sort_anchors_temp_bytes(int n_points);
int pilot_refine_sort_anchors(const float* points_dev, const void* ref_feat_dev, int n_points, int channels, pilot_dtype dtype,
                              float* points_out_dev, void* ref_out_dev, int* perm_out_dev, void* temp_dev, size_t temp_bytes,
                              void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Measurement helper: random-gather bandwidth of this GPU with the photo kernel's access
 * shape — aligned reads of vec_bytes (16..512, power of two; vec_bytes/16 lanes x 16-byte ld.global.nc) at
 * hashed positions of a buffer of buffer_bytes (e.g. 16 MiB = L2-resident, 1 GiB = HBM). Allocates and frees
 * its own buffer, times `launches` launches with CUDA events on the default stream and SYNCHRONISES; writes
 * the best GB/s. Not part of the refinement path.
 */
int pilot_refine_probe_gather(int device, size_t buffer_bytes, int vec_bytes, int launches, double* gbps_out);

/* The same for the access shape of one (anchor, hypothesis) unit of the tensor-core gather (kernel description PAPER.md:485,
 * "descriptor interpolation"): a warp reads rounds of 8 random units, each 2 x 2 pixels of px_bytes (64 or
 * 128: 32 or 64 bf16 channels) - the two x-adjacent pixels contiguous, the two map rows 1920 pixels apart - plus one
 * reference row of px_bytes, from a buffer of buffer_bytes (16 MiB = L2-resident: the denominator of bench.py's binding
 * roofline; 4 GiB = HBM). variant 0: the product's shape, four lanes per unit with one px_bytes/4-byte ld.global.nc each
 * per vector (LDG.256 at 128 bytes), 6, 8 and 12 resident CTAs of 4 warps per SM, the best taken. variant 1: the same bytes
 * staged through shared memory with cp.async.bulk (three bulk copies per unit issued by lanes 0-7, mbarrier completion,
 * three rounds in flight per warp) and read back with LDS.128 - north_star's "staged via TMA or shared memory" variant,
 * kept as a measurement so that the choice is a number (profiles/r2_staged_vs_ldg.md). Writes the best GB/s of TAP bytes
 * (4 * px_bytes per unit; the reference row is moved as well and not counted, as in SURVEY.md §8(d)'s 4*C*s per unit).
 * Allocates and frees its own buffer, times `launches` launches with CUDA events on the default stream and SYNCHRONISES.
 * PILOT_ERR_ARG for other px_bytes / variants or a buffer under 65536 pixels. Not part of the refinement path.
 */
int pilot_refine_probe_unit_gather(int device, size_t buffer_bytes, int px_bytes, int variant, int launches, double* gbps_out);

#ifdef __cplusplus
}
#endif
#endif /* PILOT_REFINE_H */
