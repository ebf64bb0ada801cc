// pilot_unrolled.cu — backward pass through ALL the LM steps of an unrolled refinement (include/pilot_refine.h,
// pilot_refine_unrolled_backward; "the refinement is unrolled over nine coarse-to-fine steps" with a
// reprojection loss after every step, supp III-C Eq.7-8). The forward run records, per solve r, the
// accepted system (H_r, g_r, lambda_r), the pose it was built at and whether the step was accepted
// (pilot_refine_set_iterate_outputs). Reading the chain  T^{r+1} = exp(dxi_r^) T^r,  dxi_r = -(H_r + lambda_r D)^-1 g_r,
// (H_r, g_r) = photo(T^r, F_l, f^r_l)  backwards from the last pose, with q = dL/d eps at the current pose:
//   accepted step:  (dL/dH, dL/dg, q_pass) = lm_step_adjoint(H_r, g_r, lambda_r, q);   photo_backward at T^r adds
//                   dS/dF_l, dS/dref_l, dS/dconf_l for S = <dL/dH, H> + <dL/dg, g> and returns dS/d eps;
//                   q <- q_pass + dS/d eps
//   rejected step (or failed factorisation): the pose did not move, q stays
//   then            q <- q + w_r dL_r/d eps   (the supervision of the pose after r solves), r >= 1.
// Everything numerical runs in the kernels of pilot_supervision.cu and pilot_backward.cu; the two kernels here select by
// the accept flag and add 6-vectors. The host loop only sequences launches on one stream. Shares no code with oracle/.
#include "../../include/pilot_refine.h"

#include <cuda_runtime.h>
#include <stdint.h>

namespace {

// a rejected record contributes nothing: its dL/dH, dL/dg are zeroed before the transpose of the gather reads them
__global__ void mask_rejected_kernel(const int* __restrict__ accept, int n, float* GH, float* Gg) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n * 42) return;
  const int m = i / 42, c = i - m * 42;
  if (accept[m]) return;
  if (c < 36) GH[36 * m + c] = 0.f; else Gg[6 * m + (c - 36)] = 0.f;
}

// q <- (accepted ? q_pass + deps : q) + w lg;   loss += w ls     (qpass == nullptr: initialisation, q <- w lg, loss <- w ls)
__global__ void combine_kernel(const int* __restrict__ accept, const float* __restrict__ qpass, const float* __restrict__ deps,
                               const float* __restrict__ lg, const float* __restrict__ ls, float w, int n, float* q, float* loss) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n * 6) return;
  const int m = i / 6;
  float v = 0.f;
  if (qpass) v = accept[m] ? qpass[i] + deps[i] : q[i];
  if (lg) v += w * lg[i];
  q[i] = v;
  if (loss && i == 6 * m) loss[m] = (qpass ? loss[m] : 0.f) + (ls ? w * ls[m] : 0.f);
}

struct Scratch { float *lg, *ls, *q, *qpass, *deps, *dxi, *GH, *Gg; size_t total; };

Scratch carve(void* base, int H, int T) {
  Scratch s;
  size_t o = 0;
  auto take = [&](size_t floats) { float* p = base ? reinterpret_cast<float*>(static_cast<char*>(base) + o) : nullptr; o += (floats * 4 + 255) & ~(size_t)255; return p; };
  s.lg = take((size_t)T * H * 6);
  s.ls = take((size_t)T * H);
  s.q = take((size_t)H * 6);
  s.qpass = take((size_t)H * 6);
  s.deps = take((size_t)H * 6);
  s.dxi = take((size_t)H * 6);
  s.GH = take((size_t)H * 36);
  s.Gg = take((size_t)H * 6);
  s.total = o;
  return s;
}

}  // namespace

extern "C" size_t pilot_refine_unrolled_backward_scratch_bytes(int n_hypotheses, int total_iters) {
  if (n_hypotheses < 0 || total_iters < 0) return 0;
  return carve(nullptr, n_hypotheses, total_iters).total;
}

extern "C" int pilot_refine_unrolled_backward(const pilot_refine_config* cfg, const pilot_refine_inputs* in,
                                              const pilot_refine_params* p, const pilot_refine_unrolled_records* rec,
                                              const pilot_refine_supervision* sup, const pilot_refine_unrolled_grads* out,
                                              void* scratch_dev, size_t scratch_bytes, void* cuda_stream) {
  if (!cfg || !in || !p || !rec || !sup || !out) return PILOT_ERR_ARG;
  if (cfg->n_levels < 1 || cfg->n_levels > PILOT_MAX_LEVELS) return PILOT_ERR_ARG;
  const int H = in->n_hypotheses;
  if (H < 0) return PILOT_ERR_ARG;
  int T = 0;
  for (int l = 0; l < cfg->n_levels; ++l) { if (p->iters[l] < 0) return PILOT_ERR_ARG; T += p->iters[l]; }
  // the priors' terms depend on the pose but not on the features; their pose-dependence is not part of this chain
  if (p->w_gravity != 0.f || (p->range_mode != PILOT_RANGE_OFF && p->w_range != 0.f)) return PILOT_ERR_UNSUPPORTED;
  if (p->grad_mode != PILOT_GRAD_BILINEAR_EXACT) return PILOT_ERR_UNSUPPORTED;
  if (H == 0) return PILOT_OK;
  if (!rec->final_poses_dev || !sup->points_dev || !sup->step_weights) return PILOT_ERR_ARG;
  if (T > 0 && (!rec->iter_hessian_dev || !rec->iter_gradient_dev || !rec->iter_lambda_dev || !rec->iter_poses_dev || !rec->iter_accept_dev))
    return PILOT_ERR_ARG;
  const Scratch s = carve(scratch_dev, H, T);
  if (!scratch_dev || scratch_bytes < s.total || ((uintptr_t)scratch_dev & 255)) return PILOT_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int tb = 128;
  auto sup_grad = [&](const float* poses, int n, float* ls, float* lg) {
    return pilot_refine_reprojection_loss_grad(poses, n, sup->pose_star, sup->points_dev, sup->n_points, sup->intrinsics, sup->width,
                                               sup->height, p->z_near, sup->alpha, sup->scale, ls, nullptr, lg, cuda_stream);
  };
  // supervision value and gradient at the pose after r solves, r = 1 .. T (row r - 1): iterates 1 .. T-1, then the final pose
  int rc = PILOT_OK;
  if (T > 1) rc = sup_grad(rec->iter_poses_dev + (size_t)H * 12, (T - 1) * H, s.ls, s.lg);
  if (rc != PILOT_OK) return rc;
  if (T > 0) {
    rc = sup_grad(rec->final_poses_dev, H, s.ls + (size_t)(T - 1) * H, s.lg + (size_t)(T - 1) * H * 6);
    if (rc != PILOT_OK) return rc;
    combine_kernel<<<(H * 6 + tb - 1) / tb, tb, 0, st>>>(nullptr, nullptr, nullptr, s.lg + (size_t)(T - 1) * H * 6, s.ls + (size_t)(T - 1) * H,
                                                         sup->step_weights[T - 1], H, s.q, out->loss_dev);
  } else {
    combine_kernel<<<(H * 6 + tb - 1) / tb, tb, 0, st>>>(nullptr, nullptr, nullptr, nullptr, nullptr, 0.f, H, s.q, out->loss_dev);
  }
  int rec_end = T;
  for (int l = cfg->n_levels - 1; l >= 0; --l) {
    const int rec_begin = rec_end - p->iters[l];
    for (int r = rec_end - 1; r >= rec_begin; --r) {
      const size_t o = (size_t)r * H;
      rc = pilot_refine_lm_step_adjoint(rec->iter_hessian_dev + 36 * o, rec->iter_gradient_dev + 6 * o, rec->iter_lambda_dev + o, s.q, H,
                                        p->damp_mode, s.dxi, s.GH, s.Gg, s.qpass, nullptr, cuda_stream);
      if (rc != PILOT_OK) return rc;
      mask_rejected_kernel<<<(H * 42 + tb - 1) / tb, tb, 0, st>>>(rec->iter_accept_dev + o, H, s.GH, s.Gg);
      rc = pilot_refine_photo_backward(in->query_feat_dev[l], in->query_conf_dev[l], cfg->width[l], cfg->height[l], cfg->channels[l],
                                       cfg->feat_dtype, in->intrinsics[l], in->points_dev[l], in->ref_feat_dev[l], in->n_points[l],
                                       rec->iter_poses_dev + 12 * o, s.GH, s.Gg, H, p->loss, p->loss_scale, p->z_near,
                                       out->grad_feat_dev[l], out->grad_ref_dev[l], out->grad_conf_dev[l], s.deps, cuda_stream);
      if (rc != PILOT_OK) return rc;
      combine_kernel<<<(H * 6 + tb - 1) / tb, tb, 0, st>>>(rec->iter_accept_dev + o, s.qpass, s.deps, r >= 1 ? s.lg + (size_t)(r - 1) * H * 6 : nullptr,
                                                           r >= 1 ? s.ls + (size_t)(r - 1) * H : nullptr, r >= 1 ? sup->step_weights[r - 1] : 0.f,
                                                           H, s.q, out->loss_dev);
    }
    rec_end = rec_begin;
  }
  if (out->grad_init_pose_dev &&
      cudaMemcpyAsync(out->grad_init_pose_dev, s.q, (size_t)H * 6 * sizeof(float), cudaMemcpyDeviceToDevice, st) != cudaSuccess)
    return PILOT_ERR_CUDA;
  return cudaGetLastError() == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}
