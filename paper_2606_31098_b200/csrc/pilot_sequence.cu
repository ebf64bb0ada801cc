// pilot_sequence.cu — streaming sequence runner (include/pilot_refine.h, "Streaming sequence").
//
// PAPER.md:110 (the previous frame's estimate is the next frame's prior) and supp IV PAPER.md:457-461 (the
// next frame's reference is prepared asynchronously). Two CUDA streams instead of the paper's two host
// threads: the library's copy stream fills one half of a double buffer with frame i+1 while the caller's
// compute stream refines frame i out of the other half; events order the reuse of each half. Nothing in
// step() synchronises with the host: seeding, refinement, arg-min and logging are all stream-ordered.
//
// Built only on the public entry points of pilot_refine.cu / pilot_hypotheses.cu. Shares no code with oracle/.
#include "../../include/pilot_refine.h"

#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace {

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
size_t elem_size(pilot_dtype d) { return d == PILOT_F32 ? 4 : 2; }

struct Slot {
  char* base;                                       // device
  char* pinned;                                     // host staging (page-locked), same layout
  bool ready_recorded;
  size_t feat[PILOT_MAX_LEVELS], conf[PILOT_MAX_LEVELS], pts[PILOT_MAX_LEVELS], ref[PILOT_MAX_LEVELS];
  pilot_refine_frame host;                          // scalars + which optional arrays are present
  cudaEvent_t ready, free_;                         // copy finished / refinement that read it finished
  bool free_recorded;
};

__global__ void log_row_kernel(const int* best_idx, const float* best_pose, const float* best_cost,
                               const int* n_valid, const unsigned* status, float* row) {
  const int t = threadIdx.x;
  const int b = best_idx[0];
  if (t < 12) row[t] = best_pose[t];
  else if (t == 12) row[12] = best_cost[0];
  else if (t == 13) row[13] = (float)b;
  else if (t == 14) row[14] = (float)n_valid[b];
  else if (t == 15) row[15] = (float)status[b];
}

}  // namespace

struct pilot_refine_sequence {
  pilot_refine_config cfg;
  pilot_refine_sequence_config sc;
  pilot_refine_handle* h;
  cudaStream_t copy_stream;
  Slot slot[2];
  size_t slot_bytes;
  char* mem;                // one cudaMalloc: slots, dsm, offsets, seeds, outputs, best, log
  char* pinned;             // one cudaHostAlloc: host staging of the two slots
  float *dsm, *offsets, *seeds, *poses, *cost, *prior, *best_cost, *log;
  int *n_valid, *best_idx;
  unsigned* status;
  long n_uploaded, n_stepped;
  int last_launches;
};

extern "C" {

int pilot_refine_sequence_create(const pilot_refine_config* cfg, const pilot_refine_sequence_config* sc,
                                 pilot_refine_sequence** out) {
  if (!out) return PILOT_ERR_ARG;
  *out = nullptr;
  if (!cfg || !sc || cfg->workspace_dev) return PILOT_ERR_ARG;
  if (sc->n_hypotheses < 1 || sc->n_hypotheses > cfg->max_hypotheses || !sc->offsets || sc->max_frames < 1)
    return PILOT_ERR_ARG;
  if (sc->seed_frame != PILOT_SEED_CAMERA && sc->seed_frame != PILOT_SEED_WORLD) return PILOT_ERR_ARG;
  if (sc->dsm && (sc->dsm_width < 2 || sc->dsm_height < 2 || !(sc->dsm_gsd > 0.f))) return PILOT_ERR_ARG;
  pilot_refine_handle* h = nullptr;
  int rc = pilot_refine_create(cfg, &h);
  if (rc != PILOT_OK) return rc;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(cfg->device);

  pilot_refine_sequence* s = new pilot_refine_sequence();
  memset(s, 0, sizeof *s);
  s->cfg = *cfg; s->sc = *sc; s->h = h;
  const size_t es = elem_size(cfg->feat_dtype), H = (size_t)sc->n_hypotheses;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
  for (int l = 0; l < cfg->n_levels; ++l) {
    size_t px = (size_t)cfg->width[l] * cfg->height[l];
    s->slot[0].feat[l] = take(px * cfg->channels[l] * es);
    s->slot[0].conf[l] = take(px * 4);
    s->slot[0].pts[l] = take((size_t)cfg->max_points * 16);
    s->slot[0].ref[l] = take((size_t)cfg->max_points * cfg->channels[l] * es);
  }
  s->slot_bytes = o;
  s->slot[1] = s->slot[0];
  const size_t dsm_bytes = sc->dsm ? (size_t)sc->dsm_width * sc->dsm_height * 4 : 0;
  o = 2 * s->slot_bytes;
  const size_t a_dsm = take(dsm_bytes), a_off = take(H * 24), a_seeds = take(H * 48), a_poses = take(H * 48),
               a_cost = take(H * 4), a_nv = take(H * 4), a_st = take(H * 4), a_prior = take(48), a_bc = take(4),
               a_bi = take(4), a_log = take((size_t)sc->max_frames * PILOT_SEQ_ROW * 4);
  void* p = nullptr;
  bool ok = cudaMalloc(&p, o) == cudaSuccess;
  if (ok) {
    s->mem = static_cast<char*>(p);
    s->slot[0].base = s->mem; s->slot[1].base = s->mem + s->slot_bytes;
    s->dsm = dsm_bytes ? reinterpret_cast<float*>(s->mem + a_dsm) : nullptr;
    s->offsets = reinterpret_cast<float*>(s->mem + a_off);
    s->seeds = reinterpret_cast<float*>(s->mem + a_seeds);
    s->poses = reinterpret_cast<float*>(s->mem + a_poses);
    s->cost = reinterpret_cast<float*>(s->mem + a_cost);
    s->n_valid = reinterpret_cast<int*>(s->mem + a_nv);
    s->status = reinterpret_cast<unsigned*>(s->mem + a_st);
    s->prior = reinterpret_cast<float*>(s->mem + a_prior);
    s->best_cost = reinterpret_cast<float*>(s->mem + a_bc);
    s->best_idx = reinterpret_cast<int*>(s->mem + a_bi);
    s->log = reinterpret_cast<float*>(s->mem + a_log);
    void* hp = nullptr;
    ok = ok && cudaHostAlloc(&hp, 2 * s->slot_bytes, cudaHostAllocDefault) == cudaSuccess;
    if (ok) {
      s->pinned = static_cast<char*>(hp);
      s->slot[0].pinned = s->pinned; s->slot[1].pinned = s->pinned + s->slot_bytes;
    }
    ok = ok && cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking) == cudaSuccess;
    for (int i = 0; i < 2 && ok; ++i) {
      ok = ok && cudaEventCreateWithFlags(&s->slot[i].ready, cudaEventDisableTiming) == cudaSuccess;
      ok = ok && cudaEventCreateWithFlags(&s->slot[i].free_, cudaEventDisableTiming) == cudaSuccess;
    }
    // static data: heightfield + offset table (synchronous, once)
    if (ok && dsm_bytes) ok = cudaMemcpy(s->dsm, sc->dsm, dsm_bytes, cudaMemcpyHostToDevice) == cudaSuccess;
    ok = ok && cudaMemcpy(s->offsets, sc->offsets, H * 24, cudaMemcpyHostToDevice) == cudaSuccess;
    ok = ok && cudaMemset(s->log, 0, (size_t)sc->max_frames * PILOT_SEQ_ROW * 4) == cudaSuccess;
    ok = ok && cudaMemset(s->prior, 0, 48) == cudaSuccess;
  }
  s->sc.offsets = nullptr; s->sc.dsm = nullptr;      // host pointers are not kept
  cudaSetDevice(prev);
  if (!ok) { pilot_refine_sequence_destroy(s); return PILOT_ERR_CUDA; }
  *out = s;
  return PILOT_OK;
}

int pilot_refine_sequence_destroy(pilot_refine_sequence* s) {
  if (!s) return PILOT_OK;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(s->cfg.device);
  if (s->copy_stream) cudaStreamSynchronize(s->copy_stream);
  for (int i = 0; i < 2; ++i) {
    if (s->slot[i].free_) { cudaEventSynchronize(s->slot[i].free_); cudaEventDestroy(s->slot[i].free_); }
    if (s->slot[i].ready) cudaEventDestroy(s->slot[i].ready);
  }
  if (s->copy_stream) cudaStreamDestroy(s->copy_stream);
  if (s->mem) cudaFree(s->mem);
  if (s->pinned) cudaFreeHost(s->pinned);
  cudaSetDevice(prev);
  pilot_refine_destroy(s->h);
  delete s;
  return PILOT_OK;
}

int pilot_refine_sequence_set_prior(pilot_refine_sequence* s, const float* pose_host, void* cuda_stream) {
  if (!s || !pose_host) return PILOT_ERR_ARG;
  // 48 bytes from pageable memory: staged by the runtime before the call returns
  cudaError_t e = cudaMemcpyAsync(s->prior, pose_host, 48, cudaMemcpyHostToDevice, static_cast<cudaStream_t>(cuda_stream));
  return e == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_sequence_upload(pilot_refine_sequence* s, const pilot_refine_frame* f) {
  if (!s || !f) return PILOT_ERR_ARG;
  if (s->n_uploaded - s->n_stepped >= 2) return PILOT_ERR_UNSUPPORTED;
  const pilot_refine_config& c = s->cfg;
  for (int l = 0; l < c.n_levels; ++l) {
    if (f->n_points[l] < 0 || !f->query_feat[l]) return PILOT_ERR_ARG;
    if (f->n_points[l] > c.max_points) return PILOT_ERR_UNSUPPORTED;
    if (f->n_points[l] > 0 && (!f->points[l] || !f->ref_feat[l])) return PILOT_ERR_ARG;
  }
  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != c.device && cudaSetDevice(c.device) != cudaSuccess) return PILOT_ERR_CUDA;
  Slot& S = s->slot[s->n_uploaded & 1];
  bool ok = true;
  // the refinement that last read this half must be over before it is overwritten
  if (S.free_recorded) ok = ok && cudaStreamWaitEvent(s->copy_stream, S.free_, 0) == cudaSuccess;
  const size_t es = elem_size(c.feat_dtype);
  // the caller's arrays are copied into page-locked staging first (so they may be pageable and reused at once);
  // the previous copy OUT of this staging half (two uploads ago) must have finished before it is overwritten
  if (S.ready_recorded && !f->arrays_pinned) ok = ok && cudaEventSynchronize(S.ready) == cudaSuccess;
  auto up = [&](size_t at, const void* src, size_t bytes) {
    if (!src || !bytes || !ok) return;
    if (f->arrays_pinned) {                     // the caller's page-locked arrays are the DMA source
      ok = cudaMemcpyAsync(S.base + at, src, bytes, cudaMemcpyHostToDevice, s->copy_stream) == cudaSuccess;
    } else {
      memcpy(S.pinned + at, src, bytes);
      ok = cudaMemcpyAsync(S.base + at, S.pinned + at, bytes, cudaMemcpyHostToDevice, s->copy_stream) == cudaSuccess;
    }
  };
  for (int l = 0; l < c.n_levels; ++l) {
    size_t px = (size_t)c.width[l] * c.height[l], N = (size_t)f->n_points[l];
    up(S.feat[l], f->query_feat[l], px * c.channels[l] * es);
    up(S.conf[l], f->query_conf[l], px * 4);
    up(S.pts[l], f->points[l], N * 16);
    up(S.ref[l], f->ref_feat[l], N * c.channels[l] * es);
  }
  ok = ok && cudaEventRecord(S.ready, s->copy_stream) == cudaSuccess;
  S.ready_recorded = true;
  S.host = *f;
  if (prev != c.device) cudaSetDevice(prev);
  if (!ok) return PILOT_ERR_CUDA;
  s->n_uploaded += 1;
  return PILOT_OK;
}

int pilot_refine_sequence_step(pilot_refine_sequence* s, const pilot_refine_params* p, void* cuda_stream) {
  if (!s || !p) return PILOT_ERR_ARG;
  if (s->n_stepped >= s->n_uploaded || s->n_stepped >= s->sc.max_frames) return PILOT_ERR_ARG;
  const pilot_refine_config& c = s->cfg;
  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != c.device && cudaSetDevice(c.device) != cudaSuccess) return PILOT_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  Slot& S = s->slot[s->n_stepped & 1];
  const int H = s->sc.n_hypotheses;
  bool ok = cudaStreamWaitEvent(st, S.ready, 0) == cudaSuccess;

  int rc = ok ? pilot_refine_seed_hypotheses(s->prior, s->offsets, H, s->sc.seed_frame, s->seeds, cuda_stream) : PILOT_ERR_CUDA;
  pilot_refine_inputs in;
  memset(&in, 0, sizeof in);
  in.n_hypotheses = H;
  for (int l = 0; l < c.n_levels; ++l) {
    in.n_points[l] = S.host.n_points[l];
    in.query_feat_dev[l] = S.base + S.feat[l];
    in.query_conf_dev[l] = S.host.query_conf[l] ? reinterpret_cast<const float*>(S.base + S.conf[l]) : nullptr;
    in.points_dev[l] = reinterpret_cast<const float*>(S.base + S.pts[l]);
    in.ref_feat_dev[l] = S.base + S.ref[l];
    for (int k = 0; k < 4; ++k) in.intrinsics[l][k] = S.host.intrinsics[l][k];
  }
  in.init_poses_dev = s->seeds;
  for (int k = 0; k < 3; ++k) {
    in.gravity_world[k] = s->sc.gravity_world[k];
    in.gravity_imu[k] = S.host.gravity_imu[k];
    in.range_ray_cam[k] = S.host.range_ray_cam[k];
  }
  in.range_meas = S.host.range_meas;
  in.dsm_dev = s->dsm; in.dsm_width = s->sc.dsm_width; in.dsm_height = s->sc.dsm_height;
  in.dsm_origin_x = s->sc.dsm_origin_x; in.dsm_origin_y = s->sc.dsm_origin_y; in.dsm_gsd = s->sc.dsm_gsd;
  pilot_refine_outputs out;
  memset(&out, 0, sizeof out);
  out.poses_dev = s->poses; out.cost_dev = s->cost; out.n_valid_dev = s->n_valid; out.status_dev = s->status;
  if (rc == PILOT_OK) rc = pilot_refine_run(s->h, &in, p, &out, cuda_stream);
  // lowest final objective -> output pose, which is also the next frame's prior
  if (rc == PILOT_OK) rc = pilot_refine_select_best(s->cost, s->poses, H, s->best_idx, s->prior, s->best_cost, cuda_stream);
  if (rc == PILOT_OK) {
    log_row_kernel<<<1, 16, 0, st>>>(s->best_idx, s->prior, s->best_cost, s->n_valid, s->status,
                                     s->log + (size_t)s->n_stepped * PILOT_SEQ_ROW);
    ok = cudaGetLastError() == cudaSuccess && cudaEventRecord(S.free_, st) == cudaSuccess;
    S.free_recorded = true;
    if (!ok) rc = PILOT_ERR_CUDA;
  }
  if (prev != c.device) cudaSetDevice(prev);
  if (rc != PILOT_OK) return rc;
  s->last_launches = pilot_refine_last_launches(s->h) + 3;
  s->n_stepped += 1;
  return PILOT_OK;
}

int pilot_refine_sequence_results(pilot_refine_sequence* s, int first, int count, float* results_host, void* cuda_stream) {
  if (!s || first < 0 || count < 0 || first + count > s->sc.max_frames || (count && !results_host)) return PILOT_ERR_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  bool ok = true;
  if (count)
    ok = cudaMemcpyAsync(results_host, s->log + (size_t)first * PILOT_SEQ_ROW, (size_t)count * PILOT_SEQ_ROW * 4,
                         cudaMemcpyDeviceToHost, st) == cudaSuccess;
  ok = ok && cudaStreamSynchronize(st) == cudaSuccess;
  return ok ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_sequence_last_frame(pilot_refine_sequence* s, float* seeds_host, float* poses_host, float* cost_host,
                                     void* cuda_stream) {
  if (!s) return PILOT_ERR_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const size_t H = (size_t)s->sc.n_hypotheses;
  bool ok = true;
  if (seeds_host) ok = ok && cudaMemcpyAsync(seeds_host, s->seeds, H * 48, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  if (poses_host) ok = ok && cudaMemcpyAsync(poses_host, s->poses, H * 48, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  if (cost_host) ok = ok && cudaMemcpyAsync(cost_host, s->cost, H * 4, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  ok = ok && cudaStreamSynchronize(st) == cudaSuccess;
  return ok ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_sequence_last_launches(const pilot_refine_sequence* s) { return s ? s->last_launches : 0; }

}  // extern "C"
