// pilot_supervision.cu — forward value of the unrolled reprojection supervision (include/pilot_refine.h):
// L_k = 1/|V| sum_{j in V} rho_B(||p_j^k - p_j*||^2), supp Eq.(7)-(8), with Barron's general robust
// loss. One CTA per pose T^k; threads stride over the points (coalesced float4 loads), project under T* and T^k in
// double, and a fixed-order shared-memory tree ends the sum (deterministic, no atomics). HBM-bound by construction:
// 16 bytes per point per pose, served from L2 for every pose after the first. Shares no code with oracle/.
#include "../../include/pilot_refine.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

namespace {

constexpr int kSupThreads = 256;

struct SupArgs {
  double Rs[9], Cs[3];          // ground-truth pose T*: R_wc (row-major) and C
  double fx, fy, cx, cy, umax, vmax, z_near;
  double alpha, inv_c2;
  int mode;                     // 0 general, 1 alpha = 2, 2 alpha = 0, 3 alpha = -inf
};

__device__ __forceinline__ double barron(const SupArgs& a, double s) {
  const double z = s * a.inv_c2;
  switch (a.mode) {
    case 1: return 0.5 * z;
    case 2: return log1p(0.5 * z);
    case 3: return -expm1(-0.5 * z);
  }
  const double b = fabs(a.alpha - 2.0);
  return (b / a.alpha) * (pow(z / b + 1.0, 0.5 * a.alpha) - 1.0);
}

// p = pi(K, R_wc^T (P - C)); R_wc row-major
__device__ __forceinline__ void project(const double* R, const double* C, const SupArgs& a, const float4& P, double& u, double& v,
                                        double& Z) {
  const double dx = (double)P.x - C[0], dy = (double)P.y - C[1], dz = (double)P.z - C[2];
  const double X = R[0] * dx + R[3] * dy + R[6] * dz;
  const double Y = R[1] * dx + R[4] * dy + R[7] * dz;
  Z = R[2] * dx + R[5] * dy + R[8] * dz;
  u = a.fx * X / Z + a.cx;
  v = a.fy * Y / Z + a.cy;
}

__global__ void __launch_bounds__(kSupThreads) reprojection_loss_kernel(const float* __restrict__ poses, const float4* __restrict__ points,
                                                                         int n_points, const __grid_constant__ SupArgs a,
                                                                         float* __restrict__ loss, int* __restrict__ n_visible) {
  const int k = blockIdx.x;
  __shared__ double s_pose[12];
  __shared__ double s_sum[kSupThreads];
  __shared__ int s_cnt[kSupThreads];
  if (threadIdx.x < 12) s_pose[threadIdx.x] = (double)poses[12 * (size_t)k + threadIdx.x];
  __syncthreads();
  double R[9], C[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
#pragma unroll
    for (int j = 0; j < 3; ++j) R[3 * i + j] = s_pose[4 * i + j];
    C[i] = s_pose[4 * i + 3];
  }
  double sum = 0.0;
  int cnt = 0;
  for (int j = threadIdx.x; j < n_points; j += kSupThreads) {
    const float4 P = __ldg(points + j);
    double us, vs, zs, u, v, z;
    project(a.Rs, a.Cs, a, P, us, vs, zs);
    project(R, C, a, P, u, v, z);
    const bool vis = zs > a.z_near && us >= 0.0 && vs >= 0.0 && us <= a.umax && vs <= a.vmax && z > a.z_near;
    if (vis) {
      const double du = u - us, dv = v - vs;
      sum += barron(a, du * du + dv * dv);
      cnt += 1;
    }
  }
  s_sum[threadIdx.x] = sum;
  s_cnt[threadIdx.x] = cnt;
  __syncthreads();
  for (int h = kSupThreads / 2; h > 0; h >>= 1) {                // fixed order
    if (threadIdx.x < h) {
      s_sum[threadIdx.x] += s_sum[threadIdx.x + h];
      s_cnt[threadIdx.x] += s_cnt[threadIdx.x + h];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    loss[k] = s_cnt[0] > 0 ? (float)(s_sum[0] / (double)s_cnt[0]) : 0.f;
    if (n_visible) n_visible[k] = s_cnt[0];
  }
}

}  // namespace

extern "C" int pilot_refine_reprojection_loss(const float* poses_dev, int n_poses, const float pose_star[12],
                                              const float* points_dev, int n_points, const float intrinsics[4],
                                              int width, int height, float z_near, float alpha, float scale,
                                              float* loss_dev, int* n_visible_dev, void* cuda_stream) {
  if (n_poses < 0 || n_points < 0 || !pose_star || !intrinsics || width < 1 || height < 1 || !(scale > 0.f) ||
      !(intrinsics[0] > 0.f) || !(intrinsics[1] > 0.f) || isnan(alpha) || (isinf(alpha) && alpha > 0.f))
    return PILOT_ERR_ARG;
  if (n_poses == 0) return PILOT_OK;
  if (!poses_dev || !loss_dev || (n_points > 0 && (!points_dev || ((uintptr_t)points_dev & 15)))) return PILOT_ERR_ARG;
  SupArgs a;
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) a.Rs[3 * i + j] = (double)pose_star[4 * i + j];
    a.Cs[i] = (double)pose_star[4 * i + 3];
  }
  a.fx = intrinsics[0]; a.fy = intrinsics[1]; a.cx = intrinsics[2]; a.cy = intrinsics[3];
  a.umax = (double)(width - 1); a.vmax = (double)(height - 1); a.z_near = (double)z_near;
  a.alpha = (double)alpha; a.inv_c2 = 1.0 / ((double)scale * (double)scale);
  a.mode = alpha == 2.f ? 1 : (alpha == 0.f ? 2 : (isinf(alpha) ? 3 : 0));
  reprojection_loss_kernel<<<n_poses, kSupThreads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
      poses_dev, reinterpret_cast<const float4*>(points_dev), n_points, a, loss_dev, n_visible_dev);
  return cudaGetLastError() == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

// ====================================================================== backward pieces
//
// (1) dL_k / d eps for the left perturbation T_cw <- exp(eps^) T_cw of the optimised pose (the LM's own parametrisation):
//     1/|V| sum rho_B'(s_j) 2 (p_j - p_j*)^T J_uv(j); same CTA-per-pose layout as the forward kernel, seven sums.
// (2) one LM step dxi = -(H + lambda D)^-1 g, T' = exp(dxi^) T read backwards (Eq.8-9): one thread per
//     system, double: two Cholesky solves, the SE(3) left Jacobian by its series, Ad(exp(dxi^)).

namespace {

__device__ __forceinline__ double barron_d(const SupArgs& a, double s) {       // d rho / d s
  const double z = s * a.inv_c2;
  switch (a.mode) {
    case 1: return 0.5 * a.inv_c2;
    case 2: return 0.5 / (1.0 + 0.5 * z) * a.inv_c2;
    case 3: return 0.5 * exp(-0.5 * z) * a.inv_c2;
  }
  const double b = fabs(a.alpha - 2.0);
  return 0.5 * pow(z / b + 1.0, 0.5 * a.alpha - 1.0) * a.inv_c2;
}

__global__ void __launch_bounds__(kSupThreads) reprojection_grad_kernel(const float* __restrict__ poses, const float4* __restrict__ points,
                                                                         int n_points, const __grid_constant__ SupArgs a,
                                                                         float* __restrict__ loss, int* __restrict__ n_visible,
                                                                         float* __restrict__ grad) {
  const int k = blockIdx.x;
  __shared__ double s_pose[12];
  __shared__ double s_sum[7][kSupThreads];
  __shared__ int s_cnt[kSupThreads];
  if (threadIdx.x < 12) s_pose[threadIdx.x] = (double)poses[12 * (size_t)k + threadIdx.x];
  __syncthreads();
  double R[9], C[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
#pragma unroll
    for (int j = 0; j < 3; ++j) R[3 * i + j] = s_pose[4 * i + j];
    C[i] = s_pose[4 * i + 3];
  }
  double acc[7] = {0, 0, 0, 0, 0, 0, 0};
  int cnt = 0;
  for (int j = threadIdx.x; j < n_points; j += kSupThreads) {
    const float4 P = __ldg(points + j);
    double us, vs, zs, u, v, Z;
    project(a.Rs, a.Cs, a, P, us, vs, zs);
    const double dx = (double)P.x - C[0], dy = (double)P.y - C[1], dz = (double)P.z - C[2];
    const double X = R[0] * dx + R[3] * dy + R[6] * dz;
    const double Y = R[1] * dx + R[4] * dy + R[7] * dz;
    Z = R[2] * dx + R[5] * dy + R[8] * dz;
    u = a.fx * X / Z + a.cx;
    v = a.fy * Y / Z + a.cy;
    const bool vis = zs > a.z_near && us >= 0.0 && vs >= 0.0 && us <= a.umax && vs <= a.vmax && Z > a.z_near;
    if (vis) {
      const double du = u - us, dv = v - vs, s = du * du + dv * dv;
      acc[6] += barron(a, s);
      const double w = 2.0 * barron_d(a, s), wu = w * du, wv = w * dv;
      const double iz = 1.0 / Z, x = X * iz, y = Y * iz;
      acc[0] += wu * a.fx * iz;
      acc[1] += wv * a.fy * iz;
      acc[2] += -wu * a.fx * x * iz - wv * a.fy * y * iz;
      acc[3] += -wu * a.fx * x * y - wv * a.fy * (1.0 + y * y);
      acc[4] += wu * a.fx * (1.0 + x * x) + wv * a.fy * x * y;
      acc[5] += -wu * a.fx * y + wv * a.fy * x;
      cnt += 1;
    }
  }
#pragma unroll
  for (int i = 0; i < 7; ++i) s_sum[i][threadIdx.x] = acc[i];
  s_cnt[threadIdx.x] = cnt;
  __syncthreads();
  for (int h = kSupThreads / 2; h > 0; h >>= 1) {                // fixed order
    if (threadIdx.x < h) {
#pragma unroll
      for (int i = 0; i < 7; ++i) s_sum[i][threadIdx.x] += s_sum[i][threadIdx.x + h];
      s_cnt[threadIdx.x] += s_cnt[threadIdx.x + h];
    }
    __syncthreads();
  }
  if (threadIdx.x < 7) {
    const double inv = s_cnt[0] > 0 ? 1.0 / (double)s_cnt[0] : 0.0;
    if (threadIdx.x == 6) { if (loss) loss[k] = (float)(s_sum[6][0] * inv); if (n_visible) n_visible[k] = s_cnt[0]; }
    else grad[6 * (size_t)k + threadIdx.x] = (float)(s_sum[threadIdx.x][0] * inv);
  }
}

// A x = b for symmetric positive definite A (6x6, full storage), in place on b. false = not positive definite.
__device__ bool chol6_solve(const double (&A)[36], double (&b)[6]) {
  double L[36];
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j <= i; ++j) {
      double s = A[6 * i + j];
      for (int k = 0; k < j; ++k) s -= L[6 * i + k] * L[6 * j + k];
      if (i == j) { if (!(s > 0.0) || !isfinite(s)) return false; L[6 * i + i] = sqrt(s); }
      else L[6 * i + j] = s / L[6 * j + j];
    }
  for (int i = 0; i < 6; ++i) { double s = b[i]; for (int k = 0; k < i; ++k) s -= L[6 * i + k] * b[k]; b[i] = s / L[6 * i + i]; }
  for (int i = 5; i >= 0; --i) { double s = b[i]; for (int k = i + 1; k < 6; ++k) s -= L[6 * k + i] * b[k]; b[i] = s / L[6 * i + i]; }
  return true;
}

__device__ void hat3(const double* a, double (&K)[9]) { K[0] = 0; K[1] = -a[2]; K[2] = a[1]; K[3] = a[2]; K[4] = 0; K[5] = -a[0]; K[6] = -a[1]; K[7] = a[0]; K[8] = 0; }

__global__ void lm_step_adjoint_kernel(const float* __restrict__ Hs, const float* __restrict__ gs, const float* __restrict__ lams,
                                       const float* __restrict__ qs, int n, int damp_diag, float* __restrict__ dxi_out,
                                       float* __restrict__ GH_out, float* __restrict__ Gg_out, float* __restrict__ qprev_out,
                                       unsigned* __restrict__ status) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n) return;
  double A[36], Hd[6], g[6], q[6];
  const double lam = (double)lams[m];
  for (int i = 0; i < 36; ++i) A[i] = (double)Hs[36 * (size_t)m + i];
  for (int i = 0; i < 6; ++i)
    for (int j = i + 1; j < 6; ++j) A[6 * i + j] = A[6 * j + i] = 0.5 * (A[6 * i + j] + A[6 * j + i]);
  for (int i = 0; i < 6; ++i) {
    Hd[i] = A[7 * i];
    A[7 * i] += damp_diag ? lam * fmax(Hd[i], 1e-12) : lam;
    g[i] = (double)gs[6 * (size_t)m + i];
    q[i] = (double)qs[6 * (size_t)m + i];
  }
  double dxi[6];
  for (int i = 0; i < 6; ++i) dxi[i] = -g[i];
  bool ok = chol6_solve(A, dxi);                                   // dxi = -A^-1 g   (Eq.8)
  // ad(dxi) = [[phi^, rho^], [0, phi^]]
  double ad[36], Kp[9], Kr[9];
  hat3(dxi + 3, Kp); hat3(dxi, Kr);
  for (int i = 0; i < 36; ++i) ad[i] = 0.0;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) { ad[6 * i + j] = Kp[3 * i + j]; ad[6 * i + 3 + j] = Kr[3 * i + j]; ad[6 * (i + 3) + 3 + j] = Kp[3 * i + j]; }
  // v = J_l(dxi)^T q,  J_l = sum_n ad^n / (n + 1)!: accumulate t_n = (ad^T)^n q / (n + 1)!
  double v[6], t[6];
  for (int i = 0; i < 6; ++i) { v[i] = q[i]; t[i] = q[i]; }
  for (int nn = 1; nn < 24; ++nn) {
    double u[6];
    for (int i = 0; i < 6; ++i) { double s = 0.0; for (int k = 0; k < 6; ++k) s += ad[6 * k + i] * t[k]; u[i] = s / (double)(nn + 1); }
    for (int i = 0; i < 6; ++i) { t[i] = u[i]; v[i] += u[i]; }
  }
  double w[6];
  for (int i = 0; i < 6; ++i) w[i] = -v[i];
  ok = chol6_solve(A, w) && ok;                                    // w = -A^-1 v = dL/dg
  for (int i = 0; i < 6; ++i) {
    dxi_out[6 * (size_t)m + i] = (float)dxi[i];
    Gg_out[6 * (size_t)m + i] = (float)w[i];
    for (int j = 0; j < 6; ++j) {
      double gh = 0.5 * (w[i] * dxi[j] + dxi[i] * w[j]);
      if (i == j && damp_diag && Hd[i] > 1e-12) gh += lam * w[i] * dxi[i];
      GH_out[36 * (size_t)m + 6 * i + j] = (float)gh;
    }
  }
  if (qprev_out) {
    // Ad(exp(dxi^))^T q = exp(ad(dxi))^T q by the series sum_n (ad^T)^n q / n!
    double r[6], tt[6];
    for (int i = 0; i < 6; ++i) { r[i] = q[i]; tt[i] = q[i]; }
    for (int nn = 1; nn < 30; ++nn) {
      double u[6];
      for (int i = 0; i < 6; ++i) { double s = 0.0; for (int k = 0; k < 6; ++k) s += ad[6 * k + i] * tt[k]; u[i] = s / (double)nn; }
      for (int i = 0; i < 6; ++i) { tt[i] = u[i]; r[i] += u[i]; }
    }
    for (int i = 0; i < 6; ++i) qprev_out[6 * (size_t)m + i] = (float)r[i];
  }
  if (status) status[m] = ok ? 0u : PILOT_STATUS_CHOL_FAIL;
}

}  // namespace

extern "C" int pilot_refine_reprojection_loss_grad(const float* poses_dev, int n_poses, const float pose_star[12],
                                                   const float* points_dev, int n_points, const float intrinsics[4],
                                                   int width, int height, float z_near, float alpha, float scale,
                                                   float* loss_dev, int* n_visible_dev, float* grad_dev, void* cuda_stream) {
  if (n_poses < 0 || n_points < 0 || !pose_star || !intrinsics || width < 1 || height < 1 || !(scale > 0.f) ||
      !(intrinsics[0] > 0.f) || !(intrinsics[1] > 0.f) || isnan(alpha) || (isinf(alpha) && alpha > 0.f))
    return PILOT_ERR_ARG;
  if (n_poses == 0) return PILOT_OK;
  if (!poses_dev || !grad_dev || (n_points > 0 && (!points_dev || ((uintptr_t)points_dev & 15)))) return PILOT_ERR_ARG;
  SupArgs a;
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) a.Rs[3 * i + j] = (double)pose_star[4 * i + j];
    a.Cs[i] = (double)pose_star[4 * i + 3];
  }
  a.fx = intrinsics[0]; a.fy = intrinsics[1]; a.cx = intrinsics[2]; a.cy = intrinsics[3];
  a.umax = (double)(width - 1); a.vmax = (double)(height - 1); a.z_near = (double)z_near;
  a.alpha = (double)alpha; a.inv_c2 = 1.0 / ((double)scale * (double)scale);
  a.mode = alpha == 2.f ? 1 : (alpha == 0.f ? 2 : (isinf(alpha) ? 3 : 0));
  reprojection_grad_kernel<<<n_poses, kSupThreads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
      poses_dev, reinterpret_cast<const float4*>(points_dev), n_points, a, loss_dev, n_visible_dev, grad_dev);
  return cudaGetLastError() == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

extern "C" int pilot_refine_lm_step_adjoint(const float* hessian_dev, const float* gradient_dev, const float* lambda_dev,
                                            const float* q_dev, int n, int damp_mode, float* dxi_dev, float* grad_hessian_dev,
                                            float* grad_gradient_dev, float* q_prev_dev, unsigned* status_dev, void* cuda_stream) {
  if (n < 0 || (damp_mode != PILOT_DAMP_IDENTITY && damp_mode != PILOT_DAMP_DIAG)) return PILOT_ERR_ARG;
  if (n == 0) return PILOT_OK;
  if (!hessian_dev || !gradient_dev || !lambda_dev || !q_dev || !dxi_dev || !grad_hessian_dev || !grad_gradient_dev) return PILOT_ERR_ARG;
  lm_step_adjoint_kernel<<<(n + 63) / 64, 64, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
      hessian_dev, gradient_dev, lambda_dev, q_dev, n, damp_mode == PILOT_DAMP_DIAG, dxi_dev, grad_hessian_dev, grad_gradient_dev,
      q_prev_dev, status_dev);
  return cudaGetLastError() == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}
