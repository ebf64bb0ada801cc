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
