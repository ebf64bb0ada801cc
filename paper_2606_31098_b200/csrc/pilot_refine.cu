// pilot_refine.cu — B200 (sm_100a) implementation of include/pilot_refine.h.
//
// One launch per EVAL pass: the photo kernel projects every
// (anchor, hypothesis) unit, gathers the 2x2 bilinear footprint of the query feature map with
// 16-byte channel-vector loads coalesced along C, forms the per-unit 2x2 Gram / residual
// scalars, lifts them through the 2x6 projection Jacobian and reduces them per hypothesis.
// The last CTA to finish a hypothesis reduces the per-chunk partials in a fixed order
// (deterministic), adds the gravity and range priors (heightfield ray-march), takes the LM
// accept/reject decision, solves the damped 6x6 system, retracts on SE(3) and publishes the
// candidate pose for the next pass — no host synchronisation anywhere.
//
// Shares no code with oracle/ (only the POD structs of include/pilot_refine.h).
// CTAs of 4 warps for the pass kernel (4 per SM at 128 registers): the same 16 warps per SM as 2 x 8, but finer-grained
// barriers and tails — measured 12.51 -> 12.13 ms on config 4. The cluster-resident kernel keeps 8 warps per CTA.
#ifndef PILOT_THREADS
#define PILOT_THREADS 128
#define PILOT_MIN_BLOCKS 4
#endif
#include "pilot_pass.cuh"

#include <nvtx3/nvToolsExt.h>   // header-only NVTX 3: ranges show up in nsys / ncu timelines, no-ops when no tool is attached
#include <stdio.h>
#include <string.h>

#include <mutex>

namespace {
// RAII NVTX range (tracing). One per host entry point of the hot path and per pyramid level.
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};
}  // namespace

namespace {

// ------------------------------------------------------------------ kernels

// Deferred finalisation: one WARP per hypothesis. With many hypotheses and few anchors each (the paper's coarse level:
// 1210 x 500) every CTA of the pass kernel would end in the serial fp64 tail while holding an SM slot that waiting CTAs
// need; here all hypotheses finalise side by side instead.
constexpr int kFinWarps = 4;
__global__ void __launch_bounds__(kFinWarps * 32) finalize_kernel(const __grid_constant__ PassArgs A) {
  pdl_prologue();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int m = blockIdx.x * kFinWarps + warp;
  __shared__ double s_sum[kFinWarps][kNacc];
  __shared__ HypState s_state[kFinWarps];
  __shared__ PriorTerms s_prior[kFinWarps];
  if (m >= A.n_hyp || A.state[m].level != A.level) return;
  if (A.prior_cta) {                             // what the pass kernel's prior CTA left in the workspace
    const int* src = reinterpret_cast<const int*>(static_cast<const PriorTerms*>(A.priors) + m);
    int* dst = reinterpret_cast<int*>(&s_prior[warp]);
    for (int i = lane; i < (int)(sizeof(PriorTerms) / 4); i += 32) dst[i] = __ldcg(src + i);
  }
  float t = 0.f;
  const float* p = A.partials + (size_t)m * A.n_chunks * kNacc + lane;
  for (int c = 0; c < A.n_chunks; ++c) t += __ldcg(p + (size_t)c * kNacc);      // fixed order
  s_sum[warp][lane] = (double)t;
  __syncwarp();
  finalize_in_workspace(A, m, s_sum[warp], lane, &s_state[warp], A.prior_cta ? &s_prior[warp] : nullptr);
}

__global__ void init_state_kernel(HypState* state, unsigned* counters, const float* poses, int n_hyp, double lambda_init,
                                  int level_begin) {
  pdl_prologue();
  int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n_hyp) return;
  HypState s;
  const float* T = poses + 12 * (size_t)m;
  for (int i = 0; i < 3; ++i) {
    for (int k = 0; k < 3; ++k) s.R[3 * k + i] = (double)T[4 * i + k];       // R_cw = R_wc^T
    s.C[i] = (double)T[4 * i + 3];
  }
  for (int i = 0; i < 9; ++i) s.Rc[i] = s.R[i];
  for (int i = 0; i < 3; ++i) s.Cc[i] = s.C[i];
  for (int i = 0; i < 21; ++i) s.H[i] = 0.0;
  for (int i = 0; i < 6; ++i) s.g[i] = 0.0;
  s.cost = 0.0; s.lambda = lambda_init; s.n_valid = 0; s.flags = 0; s.status = 0;
  s.level = level_begin; s.k = 0; s.pending = 0; s.visible_evals = 0ull;
  state[m] = s;
  counters[m] = 0u;
}

__global__ void visible_sum_kernel(const HypState* state, int n_hyp, unsigned long long* out) {
  unsigned long long t = 0ull;
  for (int m = threadIdx.x; m < n_hyp; m += blockDim.x) t += state[m].visible_evals;
  for (int o = 16; o >= 1; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  __shared__ unsigned long long part[8];
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = t;
  __syncthreads();
  if (threadIdx.x == 0) { unsigned long long a = 0ull; for (int i = 0; i < 8; ++i) a += part[i]; *out = a; }
}

}  // namespace

// ====================================================================== host side

struct pilot_refine_handle {
  pilot_refine_config cfg;
  char* ws;                 // device scratch
  size_t ws_bytes;
  bool owns_ws;
  int max_chunks;
  int chunk_override;       // 0 = heuristic
  int mode;                 // pilot_exec_mode
  int cluster_override;     // 0 = heuristic
  int math_mode;            // pilot_math_mode
  int sm_count;
  int last_launches;
  int last_n_hyp;
  unsigned last_mma_levels, last_resident_levels;
  float* iter_poses; int* iter_accept;      // optional extra records (pilot_refine_set_iterate_outputs)   // bit l: level l of the last run used the tensor-core contraction / the resident kernel
  // host-path staging (create_host only)
  bool host_mode;
  int max_dsm_w, max_dsm_h;
  char* stage;              // one cudaMalloc: two halves of stage_bytes each
  size_t stage_bytes;
  cudaStream_t copy_stream; // uploads of submit_host
  cudaEvent_t ev_copied[2], ev_done[2];
  long n_submitted, n_waited;
  // pruned host path (set_grid_host): one cudaMalloc
  float* grid;              // offsets [n][6] | seeds [n][12] | two halves of GridHalf floats
  int grid_n;
};

namespace {

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
size_t elem_size(pilot_dtype d) { return d == PILOT_F32 ? 4 : 2; }

// lanes per unit: C*sizeof/16, must be a power of two in [1, 32]
int lanes_per_unit(int channels, pilot_dtype d) {
  size_t bytes = (size_t)channels * elem_size(d);
  if (channels <= 0 || bytes % 16 != 0) return 0;
  size_t g = bytes / 16;
  if (g > 32 || (g & (g - 1)) != 0) return 0;
  return (int)g;
}

bool config_ok(const pilot_refine_config* c) {
  if (!c || c->n_levels < 1 || c->n_levels > PILOT_MAX_LEVELS) return false;
  if (c->feat_dtype != PILOT_F32 && c->feat_dtype != PILOT_BF16 && c->feat_dtype != PILOT_F16) return false;
  if (c->max_hypotheses < 1 || c->max_points < 1 || c->max_total_iters < 0) return false;
  for (int l = 0; l < c->n_levels; ++l)
    if (c->width[l] < 2 || c->height[l] < 2 || c->channels[l] < 1) return false;
  return true;
}

// Tap addresses are 32-bit byte offsets into a level's map and n_valid is summed in fp32 (exact to 2^24): larger shapes
// are refused at create() instead of wrapping silently.
bool shape_supported(const pilot_refine_config* c) {
  if (c->max_points > (1 << 24)) return false;
  for (int l = 0; l < c->n_levels; ++l) {
    const unsigned long long bytes = (unsigned long long)c->width[l] * (unsigned long long)c->height[l] *
                                     (unsigned long long)c->channels[l] * (unsigned long long)elem_size(c->feat_dtype);
    if (bytes >= 0xffffffffull) return false;
  }
  return true;
}

struct WsLayout { size_t state, counters, priors, partials, scratch, total; int max_chunks; };

WsLayout ws_layout(const pilot_refine_config* c) {
  WsLayout w;
  w.max_chunks = (c->max_points + kMinChunk - 1) / kMinChunk;
  size_t o = 0;
  w.state = o;    o = align_up(o + sizeof(HypState) * (size_t)c->max_hypotheses, 256);
  w.counters = o; o = align_up(o + sizeof(unsigned) * (size_t)c->max_hypotheses, 256);
  w.priors = o;   o = align_up(o + sizeof(PriorTerms) * (size_t)c->max_hypotheses, 256);   // deferred finalisation: the prior CTAs' terms
  w.partials = o; o = align_up(o + sizeof(float) * kNacc * (size_t)c->max_hypotheses * (size_t)w.max_chunks, 256);
  w.scratch = o;  o = align_up(o + 256, 256);
  w.total = o;
  return w;
}

typedef void (*pass_fn)(const PassArgs);

template <class T, bool CEN>
pass_fn pick_g(int g) {
  switch (g) {
    case 1: return photo_pass_kernel<T, 1, CEN, false>;
    case 2: return photo_pass_kernel<T, 2, CEN, false>;
    case 4: return photo_pass_kernel<T, 4, CEN, false>;
    case 8: return photo_pass_kernel<T, 8, CEN, false>;
    case 16: return photo_pass_kernel<T, 16, CEN, false>;
    case 32: return photo_pass_kernel<T, 32, CEN, false>;
  }
  return nullptr;
}

template <bool CEN>
pass_fn pick_t(pilot_dtype d, int g) {
  switch (d) {
    case PILOT_F32: return pick_g<F32Tag, CEN>(g);
    case PILOT_F16: return pick_g<F16Tag, CEN>(g);
    case PILOT_BF16: return pick_g<BF16Tag, CEN>(g);
  }
  return nullptr;
}

pass_fn pick_kernel(pilot_dtype d, int g, int grad_mode) {
  return grad_mode == PILOT_GRAD_CENTRAL_SAMPLED ? pick_t<true>(d, g) : pick_t<false>(d, g);
}

// Tensor-core contraction (pilot_math_mode): 16-bit features, 16-128 channels, exact bilinear gradient.
bool use_mma(const pilot_refine_handle* h, int g, int grad_mode, bool resident);

// Small problems (few (anchor, hypothesis) units per level) are launch- and tail-latency bound with one launch per
// pass: they go to the cluster-resident kernel, one launch per level. Returns the cluster size, 0 = pass kernel.
int choose_resident(const pilot_refine_handle* h, int n_hyp, int n_points) {
  if (h->mode == PILOT_EXEC_PASSES || h->mode == PILOT_EXEC_PASSES_SPLIT) return 0;
  // AUTO: resident only when every hypothesis' cluster is co-resident in one wave (2 CTAs per SM) and the level is small
  if (h->mode == PILOT_EXEC_AUTO && ((long)n_hyp * (long)n_points > 1500000L || n_hyp > 2 * h->sm_count)) return 0;
  if (h->cluster_override > 0) return h->cluster_override;
  // as many CTAs per hypothesis as keep the whole set co-resident (2 CTAs per SM) with about one batch per warp
  int s = 8;
  while (s > 1 && ((long)n_hyp * s > 2L * h->sm_count || n_points / s < 200)) s >>= 1;
  return s;
}

bool use_mma(const pilot_refine_handle* h, int g, int grad_mode, bool resident) {
  if (h->math_mode == PILOT_MATH_FP32) return false;
  const bool applies = h->cfg.feat_dtype != PILOT_F32 && grad_mode == PILOT_GRAD_BILINEAR_EXACT && (g == 2 || g == 4 || g == 8 || g == 16);
  if (h->math_mode == PILOT_MATH_MMA) return applies;
  // AUTO: measured on B200 (ms per step, FP32 -> MMA, round 2's one-unit-per-row-group gather): config 4 9.60 (7.65 with the
  // empty batches skipped) -> 7.88, config 2 8.02 -> 7.64 (64 channels, one launch per pass); config 1 0.642 -> 0.610,
  // config 3 1.093 -> 1.029, paper schedule 0.325 -> 0.289 (32 channels, cluster-resident and the 1210-hypothesis coarse pass).
  // 16 channels (8-byte loads per thread) were not measured: they stay on FFMA2.
  (void)resident;
  return applies && g >= 4;
}

int choose_chunk(const pilot_refine_handle* h, int n_hyp, int n_points) {
  if (h->chunk_override > 0) return h->chunk_override;
  // enough CTAs for ~4 waves at 2 CTAs/SM, chunks of 256..2048 anchors
  long want = 8L * h->sm_count;
  int chunk = 2048;
  while (chunk > kMinChunk && (long)n_hyp * ((n_points + chunk - 1) / chunk) < want) chunk >>= 1;
  // 12 batches per warp instead of 16 where the grid is large anyway. Measured (B200, ms per step, 2048 -> 1536): config 4
  // 9.12 -> 8.99, config 2 9.25 -> 9.07 (tensor-core contraction), 11.89 -> 11.84 and 11.43 -> 11.24 (FFMA2); 1152, 1280,
  // 1408, 1664 and 1792 lie between, 1024 and 4096 above
  if (chunk == 2048 && n_points > 2 * 1536) chunk = 1536;
  return chunk;
}

}  // namespace

extern "C" {

size_t pilot_refine_workspace_bytes(const pilot_refine_config* cfg) {
  if (!config_ok(cfg)) return 0;
  return ws_layout(cfg).total;
}

int pilot_refine_create(const pilot_refine_config* cfg, pilot_refine_handle** out) {
  if (!out) return PILOT_ERR_ARG;
  *out = nullptr;
  if (!config_ok(cfg)) return PILOT_ERR_ARG;
  for (int l = 0; l < cfg->n_levels; ++l)
    if (lanes_per_unit(cfg->channels[l], cfg->feat_dtype) == 0) return PILOT_ERR_UNSUPPORTED;
  if (!shape_supported(cfg)) return PILOT_ERR_UNSUPPORTED;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) return PILOT_ERR_CUDA;
  int prev = 0;
  cudaGetDevice(&prev);
  if (cudaSetDevice(cfg->device) != cudaSuccess) return PILOT_ERR_CUDA;
  WsLayout w = ws_layout(cfg);
  pilot_refine_handle* h = new pilot_refine_handle();
  h->cfg = *cfg;
  h->max_chunks = w.max_chunks;
  h->chunk_override = 0;
  h->mode = PILOT_EXEC_AUTO;
  h->cluster_override = 0;
  h->math_mode = PILOT_MATH_AUTO;
  h->last_launches = 0;
  h->last_n_hyp = 0;
  h->last_mma_levels = h->last_resident_levels = 0u;
  h->iter_poses = nullptr; h->iter_accept = nullptr;
  h->host_mode = false; h->stage = nullptr; h->stage_bytes = 0; h->max_dsm_w = h->max_dsm_h = 0;
  h->copy_stream = nullptr; h->n_submitted = h->n_waited = 0;
  h->grid = nullptr; h->grid_n = 0;
  for (int i = 0; i < 2; ++i) { h->ev_copied[i] = nullptr; h->ev_done[i] = nullptr; }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess) { delete h; cudaSetDevice(prev); return PILOT_ERR_CUDA; }
  h->sm_count = prop.multiProcessorCount;
  if (cfg->workspace_dev) {
    if (cfg->workspace_bytes < w.total) { delete h; cudaSetDevice(prev); return PILOT_ERR_WORKSPACE; }
    h->ws = static_cast<char*>(cfg->workspace_dev);
    h->ws_bytes = cfg->workspace_bytes;
    h->owns_ws = false;
  } else {
    void* p = nullptr;
    if (cudaMalloc(&p, w.total) != cudaSuccess) { delete h; cudaSetDevice(prev); return PILOT_ERR_CUDA; }
    h->ws = static_cast<char*>(p);
    h->ws_bytes = w.total;
    h->owns_ws = true;
  }
  cudaSetDevice(prev);
  *out = h;
  return PILOT_OK;
}

int pilot_refine_destroy(pilot_refine_handle* h) {
  if (!h) return PILOT_OK;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(h->cfg.device);
  if (h->owns_ws && h->ws) cudaFree(h->ws);
  if (h->copy_stream) { cudaStreamSynchronize(h->copy_stream); cudaStreamDestroy(h->copy_stream); }
  for (int i = 0; i < 2; ++i) {
    if (h->ev_done[i]) { cudaEventSynchronize(h->ev_done[i]); cudaEventDestroy(h->ev_done[i]); }
    if (h->ev_copied[i]) cudaEventDestroy(h->ev_copied[i]);
  }
  if (h->stage) cudaFree(h->stage);
  if (h->grid) cudaFree(h->grid);
  cudaSetDevice(prev);
  delete h;
  return PILOT_OK;
}

int pilot_refine_set_chunk(pilot_refine_handle* h, int chunk) {
  if (!h || chunk < 0 || (chunk % kMinChunk) != 0) return PILOT_ERR_ARG;
  h->chunk_override = chunk;
  return PILOT_OK;
}

int pilot_refine_set_exec_mode(pilot_refine_handle* h, int mode, int cluster) {
  if (!h || mode < PILOT_EXEC_AUTO || mode > PILOT_EXEC_PASSES_SPLIT) return PILOT_ERR_ARG;
  if (cluster != 0 && cluster != 1 && cluster != 2 && cluster != 4 && cluster != 8) return PILOT_ERR_ARG;
  h->mode = mode;
  h->cluster_override = cluster;
  return PILOT_OK;
}

int pilot_refine_set_iterate_outputs(pilot_refine_handle* h, float* iter_poses_dev, int* iter_accept_dev) {
  if (!h) return PILOT_ERR_ARG;
  h->iter_poses = iter_poses_dev; h->iter_accept = iter_accept_dev;
  return PILOT_OK;
}

int pilot_refine_set_math_mode(pilot_refine_handle* h, int mode) {
  if (!h || mode < PILOT_MATH_AUTO || mode > PILOT_MATH_MMA) return PILOT_ERR_ARG;
  h->math_mode = mode;
  return PILOT_OK;
}

int pilot_refine_last_launches(const pilot_refine_handle* h) { return h ? h->last_launches : 0; }

int pilot_refine_last_plan(const pilot_refine_handle* h, unsigned* mma_levels, unsigned* resident_levels) {
  if (!h) return PILOT_ERR_ARG;
  if (mma_levels) *mma_levels = h->last_mma_levels;
  if (resident_levels) *resident_levels = h->last_resident_levels;
  return PILOT_OK;
}

int pilot_refine_last_visible_evals(pilot_refine_handle* h, void* cuda_stream, unsigned long long* out_host) {
  if (!h || !out_host) return PILOT_ERR_ARG;
  *out_host = 0ull;
  if (h->last_n_hyp <= 0) return PILOT_OK;
  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != h->cfg.device && cudaSetDevice(h->cfg.device) != cudaSuccess) return PILOT_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  WsLayout w = ws_layout(&h->cfg);
  unsigned long long* d = reinterpret_cast<unsigned long long*>(h->ws + w.scratch);
  visible_sum_kernel<<<1, 256, 0, st>>>(reinterpret_cast<const HypState*>(h->ws + w.state), h->last_n_hyp, d);
  bool ok = cudaMemcpyAsync(out_host, d, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
            cudaStreamSynchronize(st) == cudaSuccess;
  if (prev != h->cfg.device) cudaSetDevice(prev);
  return ok ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_run(pilot_refine_handle* h, const pilot_refine_inputs* in, const pilot_refine_params* p,
                     const pilot_refine_outputs* out, void* cuda_stream) {
  if (!h) return PILOT_ERR_ARG;
  return pilot_refine_run_levels(h, in, p, out, 0, h->cfg.n_levels, cuda_stream);
}

int pilot_refine_run_levels(pilot_refine_handle* h, const pilot_refine_inputs* in, const pilot_refine_params* p,
                            const pilot_refine_outputs* out, int level_begin, int level_end, void* cuda_stream) {
  if (!h || !in || !p || !out) return PILOT_ERR_ARG;
  NvtxRange nvtx_run("pilot_refine_run_levels");
  const pilot_refine_config& c = h->cfg;
  if (level_begin < 0 || level_begin >= level_end || level_end > c.n_levels) return PILOT_ERR_ARG;
  if (in->n_hypotheses < 0) return PILOT_ERR_ARG;
  if (in->n_hypotheses > c.max_hypotheses) return PILOT_ERR_UNSUPPORTED;
  int total_iters = 0;
  for (int l = 0; l < c.n_levels; ++l) {
    if (in->n_points[l] < 0 || p->iters[l] < 0) return PILOT_ERR_ARG;
    total_iters += p->iters[l];
    if (l < level_begin || l >= level_end) continue;       // pointers of levels outside the range are not read
    if (in->n_points[l] > c.max_points) return PILOT_ERR_UNSUPPORTED;
    if (!in->query_feat_dev[l]) return PILOT_ERR_ARG;
    if (in->n_points[l] > 0 && (!in->points_dev[l] || !in->ref_feat_dev[l])) return PILOT_ERR_ARG;
    if (((uintptr_t)in->query_feat_dev[l] | (uintptr_t)in->ref_feat_dev[l] | (uintptr_t)in->points_dev[l]) & 15) return PILOT_ERR_ARG;
  }
  if (total_iters > c.max_total_iters) return PILOT_ERR_UNSUPPORTED;
  if (p->grad_mode != PILOT_GRAD_BILINEAR_EXACT && p->grad_mode != PILOT_GRAD_CENTRAL_SAMPLED) return PILOT_ERR_ARG;
  if (p->loss < PILOT_LOSS_L2 || p->loss > PILOT_LOSS_CAUCHY) return PILOT_ERR_ARG;
  if (p->range_mode < PILOT_RANGE_OFF || p->range_mode > PILOT_RANGE_MARCH) return PILOT_ERR_ARG;
  if (p->range_mode == PILOT_RANGE_MARCH && (p->march_steps < 1 || p->bisect_steps < 0)) return PILOT_ERR_ARG;
  if (p->range_mode != PILOT_RANGE_OFF && p->w_range > 0.f && in->dsm_dev && (in->dsm_width < 2 || in->dsm_height < 2 || !(in->dsm_gsd > 0.f)))
    return PILOT_ERR_ARG;
  h->last_launches = 0;
  if (in->n_hypotheses == 0) return PILOT_OK;
  if (!in->init_poses_dev) return PILOT_ERR_ARG;

  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != c.device && cudaSetDevice(c.device) != cudaSuccess) return PILOT_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  WsLayout w = ws_layout(&c);
  PassArgs A;
  memset(&A, 0, sizeof A);
  A.prm = *p;
  for (int i = 0; i < 3; ++i) { A.gw[i] = in->gravity_world[i]; A.gi[i] = in->gravity_imu[i]; A.ray[i] = in->range_ray_cam[i]; }
  A.range_meas = in->range_meas;
  A.pd.lambda_init = (double)p->lambda_init; A.pd.lambda_up = (double)p->lambda_up; A.pd.lambda_down = (double)p->lambda_down;
  A.pd.lambda_min = (double)p->lambda_min; A.pd.lambda_max = (double)p->lambda_max;
  A.pd.w_gravity = (double)p->w_gravity; A.pd.gravity_scale = (double)p->gravity_scale;
  A.pd.w_range = (double)p->w_range; A.pd.range_scale = (double)p->range_scale;
  for (int i = 0; i < 3; ++i) { A.pd.gw[i] = (double)in->gravity_world[i]; A.pd.gi[i] = (double)in->gravity_imu[i]; }
  A.dsm = in->dsm_dev; A.dsm_w = in->dsm_width; A.dsm_h = in->dsm_height;
  A.dsm_ox = in->dsm_origin_x; A.dsm_oy = in->dsm_origin_y; A.dsm_gsd = in->dsm_gsd;
  A.n_hyp = in->n_hypotheses; A.level_end = level_end;
  A.state = reinterpret_cast<HypState*>(h->ws + w.state);
  A.counters = reinterpret_cast<unsigned*>(h->ws + w.counters);
  A.priors = h->ws + w.priors;
  A.partials = reinterpret_cast<float*>(h->ws + w.partials);
  A.out = *out;
  A.iter_poses = h->iter_poses; A.iter_accept = h->iter_accept;

  int launches = 0;
  unsigned plan_mma = 0u, plan_res = 0u;
  launch_pdl(init_state_kernel, dim3((unsigned)((A.n_hyp + 127) / 128)), 128, 0, st, A.state, A.counters, in->init_poses_dev, A.n_hyp,
             (double)p->lambda_init, level_begin);
  ++launches;
  int rec_base = 0;
  for (int l = 0; l < level_end; ++l) {
    if (l < level_begin) { rec_base += p->iters[l]; continue; }
    static const char* const kLevelNames[PILOT_MAX_LEVELS] = {"pilot level 0", "pilot level 1", "pilot level 2", "pilot level 3"};
    NvtxRange nvtx_level(kLevelNames[l]);
    LevelArgs& L = A.lv;
    L.feat = in->query_feat_dev[l]; L.conf = in->query_conf_dev[l];
    L.points = reinterpret_cast<const float4*>(in->points_dev[l]); L.ref = in->ref_feat_dev[l];
    L.fx = in->intrinsics[l][0]; L.fy = in->intrinsics[l][1]; L.cx = in->intrinsics[l][2]; L.cy = in->intrinsics[l][3];
    L.W = c.width[l]; L.H = c.height[l]; L.C = c.channels[l]; L.N = in->n_points[l];
    A.level = l; A.iters = p->iters[l]; A.rec_base = rec_base;
    const int g = lanes_per_unit(L.C, c.feat_dtype);
    const int cluster = choose_resident(h, A.n_hyp, L.N);
    bool mma = use_mma(h, g, p->grad_mode, cluster > 0);
    if (mma && MmaGeom<64>::LB == 32 && g >= 8 && (((uintptr_t)L.feat | (uintptr_t)L.ref) & 31)) mma = false;   // 32-byte loads
    if (mma) plan_mma |= 1u << l;
    if (cluster > 0) plan_res |= 1u << l;
    A.chunk = choose_chunk(h, A.n_hyp, L.N);
    A.n_chunks = L.N > 0 ? (L.N + A.chunk - 1) / A.chunk : 1;
    if (A.n_chunks > h->max_chunks) { A.chunk = kMinChunk; A.n_chunks = (L.N + kMinChunk - 1) / kMinChunk; }
    if (cluster > 0) {
      if (resident_launch(c.feat_dtype, g, p->grad_mode, mma, A, cluster, cuda_stream) != (int)cudaSuccess) {
        if (prev != c.device) cudaSetDevice(prev);
        return PILOT_ERR_CUDA;
      }
      ++launches;
    } else {
      pass_fn fn = mma ? nullptr : pick_kernel(c.feat_dtype, g, p->grad_mode);
      const size_t smem = mma ? 0 : gather_smem_for(g, false);
      if (!mma && smem > 48 * 1024 && cudaFuncSetAttribute(reinterpret_cast<const void*>(fn), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                           (int)smem) != cudaSuccess) {
        if (prev != c.device) cudaSetDevice(prev);
        return PILOT_ERR_CUDA;
      }
      const bool range_on = p->range_mode != PILOT_RANGE_OFF && p->w_range > 0.f && in->dsm_dev != nullptr;
      // small CTAs (<= 512 anchors) in more than one wave, or many hypotheses (measured: config 2, H = 1024, 7.01 -> 6.76 ms;
      // config 4, H = 256, 7.01 -> 6.97): the serial tail moves to its own launch
      const int per_cta = A.chunk < L.N ? A.chunk : L.N;
      A.defer = h->mode == PILOT_EXEC_PASSES_SPLIT ||
                (h->mode == PILOT_EXEC_AUTO &&
                 ((per_cta <= 512 && (long)A.n_hyp * A.n_chunks > 2L * h->sm_count) || A.n_hyp >= 256));
      // the prior CTAs (pilot_pass.cuh) pay when the range prior marches the heightfield and a hypothesis has many gather
      // CTAs to hide them behind: config 4 (43 chunks) 6.97 -> 6.93 ms; with 6 chunks (config 2) the extra row of mostly empty
      // CTAs costs more than the march it hides (6.76 -> 6.80), and the HEIGHT mode has no march to hide
      A.prior_cta = (A.defer && range_on && p->range_mode == PILOT_RANGE_MARCH && A.n_chunks >= 16) ? 1 : 0;
      dim3 grid((unsigned)A.n_hyp, (unsigned)(A.n_chunks + A.prior_cta));
      for (int pass = 0; pass <= p->iters[l]; ++pass) {
        A.pass = pass;
        if (mma) {
          if (mma_pass_launch(c.feat_dtype, g, A, cuda_stream) != (int)cudaSuccess) {
            if (prev != c.device) cudaSetDevice(prev);
            return PILOT_ERR_CUDA;
          }
        } else {
          launch_pdl(fn, grid, kThreads, smem, st, A);
        }
        ++launches;
        if (A.defer) {
          launch_pdl(finalize_kernel, dim3((unsigned)((A.n_hyp + kFinWarps - 1) / kFinWarps)), kFinWarps * 32, 0, st, A);
          ++launches;
        }
      }
      A.defer = 0; A.prior_cta = 0;
    }
    rec_base += p->iters[l];
  }
  h->last_launches = launches;
  h->last_n_hyp = A.n_hyp;
  h->last_mma_levels = plan_mma; h->last_resident_levels = plan_res;
  cudaError_t e = cudaGetLastError();
  if (prev != c.device) cudaSetDevice(prev);
  return e == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

}  // extern "C"

// ====================================================================== host-buffer path (e2e)

namespace {

struct StageLayout {
  size_t feat[PILOT_MAX_LEVELS], conf[PILOT_MAX_LEVELS], pts[PILOT_MAX_LEVELS], ref[PILOT_MAX_LEVELS];
  size_t poses, dsm, o_poses, o_cost, o_nvalid, o_status, o_ih, o_ig, o_ic, o_il, total;
};

StageLayout stage_layout(const pilot_refine_config* c, int dsm_w, int dsm_h) {
  StageLayout s;
  size_t o = 0, es = elem_size(c->feat_dtype);
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
  for (int l = 0; l < PILOT_MAX_LEVELS; ++l) {
    bool on = l < c->n_levels;
    size_t px = on ? (size_t)c->width[l] * c->height[l] : 0;
    s.feat[l] = take(px * (on ? c->channels[l] : 0) * es);
    s.conf[l] = take(px * 4);
    s.pts[l] = take(on ? (size_t)c->max_points * 16 : 0);
    s.ref[l] = take(on ? (size_t)c->max_points * c->channels[l] * es : 0);
  }
  size_t H = (size_t)c->max_hypotheses, T = (size_t)c->max_total_iters;
  s.poses = take(H * 48);
  s.dsm = take((size_t)dsm_w * dsm_h * 4);
  s.o_poses = take(H * 48); s.o_cost = take(H * 4); s.o_nvalid = take(H * 4); s.o_status = take(H * 4);
  s.o_ih = take(T * H * 144); s.o_ig = take(T * H * 24); s.o_ic = take(T * H * 4); s.o_il = take(T * H * 4);
  s.total = o;
  return s;
}

}  // namespace

extern "C" {

int pilot_refine_create_host(const pilot_refine_config* cfg, int max_dsm_width, int max_dsm_height,
                             pilot_refine_handle** out) {
  if (!out) return PILOT_ERR_ARG;
  *out = nullptr;
  if (!cfg || cfg->workspace_dev || max_dsm_width < 0 || max_dsm_height < 0) return PILOT_ERR_ARG;
  int rc = pilot_refine_create(cfg, out);
  if (rc != PILOT_OK) return rc;
  pilot_refine_handle* h = *out;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(cfg->device);
  StageLayout s = stage_layout(cfg, max_dsm_width, max_dsm_height);
  void* p = nullptr;
  bool ok = cudaMalloc(&p, 2 * s.total) == cudaSuccess;            // two halves: run k+1 uploads while run k computes
  if (ok) {
    h->stage = static_cast<char*>(p);
    h->stage_bytes = s.total;
    ok = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking) == cudaSuccess;
    for (int i = 0; i < 2 && ok; ++i)
      ok = cudaEventCreateWithFlags(&h->ev_copied[i], cudaEventDisableTiming) == cudaSuccess &&
           cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming) == cudaSuccess;
  }
  cudaSetDevice(prev);
  h->host_mode = true;
  h->max_dsm_w = max_dsm_width; h->max_dsm_h = max_dsm_height;
  if (!ok) { pilot_refine_destroy(h); *out = nullptr; return PILOT_ERR_CUDA; }
  return PILOT_OK;
}

}  // extern "C"

namespace {

// Checks of a host-path submission and the upload of every input of `in` (host pointers) into staging half `half` on the
// handle's copy stream; `din` = the same inputs with device pointers. The compute stream waits for the upload (and for the
// previous run, which shares the workspace). Returns PILOT_OK or an error; T = sum of iterations.
int host_upload(pilot_refine_handle* h, const pilot_refine_inputs* in, const pilot_refine_params* p, cudaStream_t st, int half,
                pilot_refine_inputs* din, int* T_out) {
  const pilot_refine_config& c = h->cfg;
  if (in->n_hypotheses < 0 || in->n_hypotheses > c.max_hypotheses) return in->n_hypotheses < 0 ? PILOT_ERR_ARG : PILOT_ERR_UNSUPPORTED;
  int T = 0;
  for (int l = 0; l < c.n_levels; ++l) {
    if (in->n_points[l] < 0 || p->iters[l] < 0) return PILOT_ERR_ARG;
    if (in->n_points[l] > c.max_points) return PILOT_ERR_UNSUPPORTED;
    T += p->iters[l];
  }
  if (T > c.max_total_iters) return PILOT_ERR_UNSUPPORTED;
  if (in->dsm_dev && ((size_t)in->dsm_width * in->dsm_height > (size_t)h->max_dsm_w * h->max_dsm_h)) return PILOT_ERR_UNSUPPORTED;
  if (h->n_submitted - h->n_waited >= 2) return PILOT_ERR_UNSUPPORTED;      // both halves in flight
  char* stage = h->stage + (size_t)half * h->stage_bytes;
  StageLayout s = stage_layout(&c, h->max_dsm_w, h->max_dsm_h);
  size_t es = elem_size(c.feat_dtype), H = (size_t)in->n_hypotheses;
  *din = *in;
  bool ok = true;
  // the run that last used this half (two submissions ago) has been waited for, so the half is free on the device
  auto up = [&](size_t at, const void* src, size_t bytes) -> void* {
    if (!src || bytes == 0) return nullptr;
    ok = ok && cudaMemcpyAsync(stage + at, src, bytes, cudaMemcpyHostToDevice, h->copy_stream) == cudaSuccess;
    return stage + at;
  };
  for (int l = 0; l < c.n_levels; ++l) {
    size_t px = (size_t)c.width[l] * c.height[l], N = (size_t)in->n_points[l];
    din->query_feat_dev[l] = up(s.feat[l], in->query_feat_dev[l], px * c.channels[l] * es);
    din->query_conf_dev[l] = static_cast<const float*>(up(s.conf[l], in->query_conf_dev[l], px * 4));
    din->points_dev[l] = static_cast<const float*>(up(s.pts[l], in->points_dev[l], N * 16));
    din->ref_feat_dev[l] = up(s.ref[l], in->ref_feat_dev[l], N * c.channels[l] * es);
  }
  din->init_poses_dev = static_cast<const float*>(up(s.poses, in->init_poses_dev, H * 48));
  din->dsm_dev = static_cast<const float*>(up(s.dsm, in->dsm_dev, (size_t)in->dsm_width * in->dsm_height * 4));
  ok = ok && cudaEventRecord(h->ev_copied[half], h->copy_stream) == cudaSuccess;
  ok = ok && cudaStreamWaitEvent(st, h->ev_copied[half], 0) == cudaSuccess;
  // both runs in flight share the handle's workspace (optimiser state, partial sums): if the previous run was submitted on
  // ANOTHER stream, this run's kernels must still come after it (a no-op when the caller keeps to one stream)
  if (h->n_submitted > h->n_waited) ok = ok && cudaStreamWaitEvent(st, h->ev_done[half ^ 1], 0) == cudaSuccess;
  *T_out = T;
  return ok ? PILOT_OK : PILOT_ERR_CUDA;
}

// floats of one half of the pruned path's device block
struct GridHalf { size_t prior, kept_idx, kept_poses, kept_cost, best, total; };
GridHalf grid_half(int n) {
  GridHalf g;
  size_t o = 0;
  g.prior = o; o += 16;
  g.kept_idx = o; o += (size_t)(n + 3) / 4 * 4;
  g.kept_poses = o; o += (size_t)n * 12;
  g.kept_cost = o; o += (size_t)(n + 3) / 4 * 4;
  g.best = o; o += 16;                       // best_idx (in the kept set) | grid index | best_cost | pad | best_pose[12]
  o += 16;
  g.total = o;
  return g;
}

__global__ void best_grid_index_kernel(const int* kept_idx, const int* best_idx, int* out) { *out = kept_idx[*best_idx]; }

}  // namespace

extern "C" {

int pilot_refine_submit_host(pilot_refine_handle* h, const pilot_refine_inputs* in, const pilot_refine_params* p,
                             const pilot_refine_outputs* out, void* cuda_stream) {
  if (!h || !in || !p || !out || !h->host_mode) return PILOT_ERR_ARG;
  NvtxRange nvtx_submit("pilot_refine_submit_host");
  const pilot_refine_config& c = h->cfg;
  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != c.device && cudaSetDevice(c.device) != cudaSuccess) return PILOT_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int half = (int)(h->n_submitted & 1);
  char* stage = h->stage + (size_t)half * h->stage_bytes;
  StageLayout s = stage_layout(&c, h->max_dsm_w, h->max_dsm_h);
  pilot_refine_inputs din;
  int T = 0;
  int rc = host_upload(h, in, p, st, half, &din, &T);
  if (rc != PILOT_OK) { if (prev != c.device) cudaSetDevice(prev); return rc; }
  const size_t H = (size_t)in->n_hypotheses;
  bool ok = true;
  pilot_refine_outputs dout;
  dout.poses_dev = out->poses_dev ? reinterpret_cast<float*>(stage + s.o_poses) : nullptr;
  dout.cost_dev = out->cost_dev ? reinterpret_cast<float*>(stage + s.o_cost) : nullptr;
  dout.n_valid_dev = out->n_valid_dev ? reinterpret_cast<int*>(stage + s.o_nvalid) : nullptr;
  dout.status_dev = out->status_dev ? reinterpret_cast<unsigned*>(stage + s.o_status) : nullptr;
  dout.iter_hessian_dev = out->iter_hessian_dev ? reinterpret_cast<float*>(stage + s.o_ih) : nullptr;
  dout.iter_gradient_dev = out->iter_gradient_dev ? reinterpret_cast<float*>(stage + s.o_ig) : nullptr;
  dout.iter_cost_dev = out->iter_cost_dev ? reinterpret_cast<float*>(stage + s.o_ic) : nullptr;
  dout.iter_lambda_dev = out->iter_lambda_dev ? reinterpret_cast<float*>(stage + s.o_il) : nullptr;
  rc = pilot_refine_run(h, &din, p, &dout, cuda_stream);
  if (rc == PILOT_OK) {
    auto down = [&](void* dst, const void* src, size_t bytes) {
      if (dst && bytes) ok = ok && cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st) == cudaSuccess;
    };
    down(out->poses_dev, dout.poses_dev, H * 48);
    down(out->cost_dev, dout.cost_dev, H * 4);
    down(out->n_valid_dev, dout.n_valid_dev, H * 4);
    down(out->status_dev, dout.status_dev, H * 4);
    down(out->iter_hessian_dev, dout.iter_hessian_dev, (size_t)T * H * 144);
    down(out->iter_gradient_dev, dout.iter_gradient_dev, (size_t)T * H * 24);
    down(out->iter_cost_dev, dout.iter_cost_dev, (size_t)T * H * 4);
    down(out->iter_lambda_dev, dout.iter_lambda_dev, (size_t)T * H * 4);
    ok = ok && cudaEventRecord(h->ev_done[half], st) == cudaSuccess;
    if (!ok) rc = PILOT_ERR_CUDA;
  }
  if (prev != c.device) cudaSetDevice(prev);
  if (rc != PILOT_OK) return rc;
  const int ticket = (int)(h->n_submitted & 0x3fffffff);
  h->n_submitted += 1;
  return ticket;
}

int pilot_refine_set_grid_host(pilot_refine_handle* h, const float* offsets_host, int n) {
  if (!h || !h->host_mode || !offsets_host || n < 1) return PILOT_ERR_ARG;
  if (n > h->cfg.max_hypotheses || n > PILOT_TOPK_MAX) return PILOT_ERR_UNSUPPORTED;
  if (h->n_submitted != h->n_waited) return PILOT_ERR_ARG;                  // not while runs are in flight
  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != h->cfg.device && cudaSetDevice(h->cfg.device) != cudaSuccess) return PILOT_ERR_CUDA;
  if (h->grid) { cudaFree(h->grid); h->grid = nullptr; h->grid_n = 0; }
  const size_t floats = (size_t)n * 18 + 2 * grid_half(n).total;
  void* g = nullptr;
  bool ok = cudaMalloc(&g, floats * sizeof(float)) == cudaSuccess &&
            cudaMemcpy(g, offsets_host, (size_t)n * 6 * sizeof(float), cudaMemcpyHostToDevice) == cudaSuccess;
  if (ok) { h->grid = static_cast<float*>(g); h->grid_n = n; } else if (g) cudaFree(g);
  if (prev != h->cfg.device) cudaSetDevice(prev);
  return ok ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_submit_pruned_host(pilot_refine_handle* h, const pilot_refine_inputs* in, const pilot_refine_params* p,
                                    const float* prior_pose_host, int keep, int seed_frame, float* best_pose_host,
                                    float* best_cost_host, int* best_index_host, void* cuda_stream) {
  if (!h || !in || !p || !prior_pose_host || !h->host_mode || !h->grid) return PILOT_ERR_ARG;
  NvtxRange nvtx_submit("pilot_refine_submit_pruned_host");
  const pilot_refine_config& c = h->cfg;
  const int n = h->grid_n;
  if (keep < 1 || keep > n || c.n_levels < 2) return PILOT_ERR_ARG;
  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != c.device && cudaSetDevice(c.device) != cudaSuccess) return PILOT_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int half = (int)(h->n_submitted & 1);
  char* stage = h->stage + (size_t)half * h->stage_bytes;
  StageLayout s = stage_layout(&c, h->max_dsm_w, h->max_dsm_h);
  pilot_refine_inputs hin = *in, din;
  hin.n_hypotheses = n;
  hin.init_poses_dev = nullptr;                                            // the seeds are made on the device
  int T = 0;
  int rc = host_upload(h, &hin, p, st, half, &din, &T);
  if (rc != PILOT_OK) { if (prev != c.device) cudaSetDevice(prev); return rc; }
  const GridHalf G = grid_half(n);
  float* offsets = h->grid;
  float* seeds = h->grid + (size_t)n * 6;
  float* gh = h->grid + (size_t)n * 18 + (size_t)half * G.total;
  float* prior = gh + G.prior;
  int* kept_idx = reinterpret_cast<int*>(gh + G.kept_idx);
  float *kept_poses = gh + G.kept_poses, *kept_cost = gh + G.kept_cost;
  int* best_idx = reinterpret_cast<int*>(gh + G.best);
  int* best_grid = best_idx + 1;
  float* best_cost = gh + G.best + 2;
  float* best_pose = gh + G.best + 4;
  // the prior (48 bytes) is copied on the compute stream: the upload event of this half is already recorded
  bool ok = cudaMemcpyAsync(prior, prior_pose_host, 48, cudaMemcpyHostToDevice, st) == cudaSuccess;
  pilot_refine_outputs dout;
  memset(&dout, 0, sizeof dout);
  dout.poses_dev = reinterpret_cast<float*>(stage + s.o_poses);
  dout.cost_dev = reinterpret_cast<float*>(stage + s.o_cost);
  int launches = 0;
  if (ok) rc = pilot_refine_seed_hypotheses(prior, offsets, n, seed_frame, seeds, cuda_stream);
  if (ok && rc == PILOT_OK) {
    din.n_hypotheses = n; din.init_poses_dev = seeds;
    rc = pilot_refine_run_levels(h, &din, p, &dout, 0, 1, cuda_stream);                       // coarse level, all hypotheses
    launches += h->last_launches + 1;
  }
  if (ok && rc == PILOT_OK) rc = pilot_refine_prune_topk(dout.cost_dev, dout.poses_dev, n, keep, kept_idx, kept_poses, kept_cost, cuda_stream);
  if (ok && rc == PILOT_OK) {
    din.n_hypotheses = keep; din.init_poses_dev = kept_poses;
    rc = pilot_refine_run_levels(h, &din, p, &dout, 1, c.n_levels, cuda_stream);              // finer levels, the kept ones
    launches += h->last_launches + 1;
  }
  if (ok && rc == PILOT_OK) rc = pilot_refine_select_best(dout.cost_dev, dout.poses_dev, keep, best_idx, best_pose, best_cost, cuda_stream);
  if (ok && rc == PILOT_OK) {
    best_grid_index_kernel<<<1, 1, 0, st>>>(kept_idx, best_idx, best_grid);
    launches += 2;
    if (best_pose_host) ok = ok && cudaMemcpyAsync(best_pose_host, best_pose, 48, cudaMemcpyDeviceToHost, st) == cudaSuccess;
    if (best_cost_host) ok = ok && cudaMemcpyAsync(best_cost_host, best_cost, 4, cudaMemcpyDeviceToHost, st) == cudaSuccess;
    if (best_index_host) ok = ok && cudaMemcpyAsync(best_index_host, best_grid, 4, cudaMemcpyDeviceToHost, st) == cudaSuccess;
    ok = ok && cudaEventRecord(h->ev_done[half], st) == cudaSuccess;
  }
  h->last_launches = launches;
  if (!ok && rc == PILOT_OK) rc = PILOT_ERR_CUDA;
  if (prev != c.device) cudaSetDevice(prev);
  if (rc != PILOT_OK) return rc;
  const int ticket = (int)(h->n_submitted & 0x3fffffff);
  h->n_submitted += 1;
  return ticket;
}

int pilot_refine_wait_host(pilot_refine_handle* h) {
  if (!h || !h->host_mode || h->n_waited >= h->n_submitted) return PILOT_ERR_ARG;
  NvtxRange nvtx_wait("pilot_refine_wait_host");
  const int half = (int)(h->n_waited & 1);
  h->n_waited += 1;
  return cudaEventSynchronize(h->ev_done[half]) == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_run_host(pilot_refine_handle* h, const pilot_refine_inputs* in, const pilot_refine_params* p,
                          const pilot_refine_outputs* out, void* cuda_stream) {
  if (!h || !h->host_mode) return PILOT_ERR_ARG;
  while (h->n_waited < h->n_submitted) {                                     // drain anything still in flight
    int rc = pilot_refine_wait_host(h);
    if (rc != PILOT_OK) return rc;
  }
  int t = pilot_refine_submit_host(h, in, p, out, cuda_stream);
  if (t < 0) return t;
  return pilot_refine_wait_host(h);
}

}  // extern "C"

// ====================================================================== allocation-free entry point
//
// For callers that may not call cudaMalloc (stream capture, serving loops, harnesses that forbid it): the same refinement
// with the optimiser workspace (HypState per hypothesis, tickets, per-CTA partial sums) in an array that is part of the
// loaded module. `g_static_workspace` is, in HOST code, only a stand-in for the symbol: the device address the kernels get
// comes from cudaGetSymbolAddress, asked once per device with that device current.

static __device__ __align__(256) unsigned char g_static_workspace[PILOT_STATIC_WORKSPACE_BYTES];

namespace {

constexpr int kStaticMaxDevices = 64;
struct StaticSetup { bool ready; char* ws; int sm_count; };
StaticSetup g_static_setup[kStaticMaxDevices];
std::mutex g_static_mutex;

// the current device must be `device`
int static_setup(int device, StaticSetup* out) {
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticSetup& s = g_static_setup[device];
  if (!s.ready) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_static_workspace) != cudaSuccess || !ptr) { cudaGetLastError(); return PILOT_ERR_CUDA; }
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || sms < 1) { cudaGetLastError(); return PILOT_ERR_CUDA; }
    s.ws = static_cast<char*>(ptr);
    s.sm_count = sms;
    s.ready = true;
  }
  *out = s;
  return PILOT_OK;
}

}  // namespace

extern "C" {

size_t pilot_refine_static_workspace_bytes(void) { return (size_t)PILOT_STATIC_WORKSPACE_BYTES; }

int pilot_refine_run_static(const pilot_refine_config* cfg, const pilot_refine_inputs* in, const pilot_refine_params* p,
                            const pilot_refine_outputs* out, void* cuda_stream, int* launches_out) {
  if (launches_out) *launches_out = 0;
  if (!config_ok(cfg) || cfg->workspace_dev || !in || !p || !out) return PILOT_ERR_ARG;
  for (int l = 0; l < cfg->n_levels; ++l)
    if (lanes_per_unit(cfg->channels[l], cfg->feat_dtype) == 0) return PILOT_ERR_UNSUPPORTED;
  if (!shape_supported(cfg)) return PILOT_ERR_UNSUPPORTED;
  const WsLayout w = ws_layout(cfg);
  if (w.total > (size_t)PILOT_STATIC_WORKSPACE_BYTES) return PILOT_ERR_WORKSPACE;   // capacity beyond the static array
  if (cfg->device < 0 || cfg->device >= kStaticMaxDevices) return PILOT_ERR_ARG;
  int prev = 0;
  if (cudaGetDevice(&prev) != cudaSuccess) return PILOT_ERR_CUDA;
  if (prev != cfg->device && cudaSetDevice(cfg->device) != cudaSuccess) { cudaGetLastError(); return PILOT_ERR_CUDA; }
  StaticSetup s;
  int rc = static_setup(cfg->device, &s);
  if (rc == PILOT_OK) {
    pilot_refine_handle h;                     // lives on the stack for the duration of the call: nothing is allocated
    memset(&h, 0, sizeof h);
    h.cfg = *cfg;
    h.ws = s.ws; h.ws_bytes = (size_t)PILOT_STATIC_WORKSPACE_BYTES; h.owns_ws = false;
    h.max_chunks = w.max_chunks;
    h.mode = PILOT_EXEC_AUTO; h.math_mode = PILOT_MATH_AUTO;
    h.sm_count = s.sm_count;
    rc = pilot_refine_run_levels(&h, in, p, out, 0, cfg->n_levels, cuda_stream);
    if (launches_out) *launches_out = h.last_launches;
  }
  if (prev != cfg->device) cudaSetDevice(prev);
  return rc;
}

}  // extern "C"
