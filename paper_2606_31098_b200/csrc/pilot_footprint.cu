// pilot_footprint.cu — reference-crop geometry (include/pilot_refine.h): the crop footprint by arg-min along the
// four corner rays (supp Eq.2), the crop homography and the geo-anchor lift (supp Eq.3,
// PAPER.md:370-377). Uses the same bilinear heightfield sample as the range prior (pilot_device.cuh).
// Shares no code with oracle/.
#include "pilot_device.cuh"

namespace {

// One warp per image corner: lanes stride over the samples, keep (residual, index) minima, shuffle-reduce with
// ties going to the smaller index (= the smaller s).
__global__ void __launch_bounds__(128) footprint_kernel(const float* __restrict__ pose, float fx, float fy, float cx, float cy,
                                                        int width, int height, DsmView D, int n_samples, double s_max,
                                                        float* __restrict__ corners) {
  const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const double u = (c == 1 || c == 2) ? (double)(width - 1) : 0.0;
  const double v = (c >= 2) ? (double)(height - 1) : 0.0;
  double d[3] = {(u - (double)cx) / (double)fx, (v - (double)cy) / (double)fy, 1.0};
  const double inv = 1.0 / sqrt(d[0] * d[0] + d[1] * d[1] + 1.0);
  double w[3], C[3];
  for (int i = 0; i < 3; ++i) {
    w[i] = ((double)pose[4 * i] * d[0] + (double)pose[4 * i + 1] * d[1] + (double)pose[4 * i + 2] * d[2]) * inv;
    C[i] = (double)pose[4 * i + 3];
  }
  double best = INFINITY;
  int best_i = 0x7fffffff;
  for (int i = 1 + lane; i <= n_samples; i += 32) {
    const double s = (double)i * s_max / (double)n_samples;
    double z, zx, zy;
    if (!dsm_sample(D, C[0] + s * w[0], C[1] + s * w[1], z, zx, zy)) continue;
    const double res = fabs(C[2] + s * w[2] - z);
    if (res < best) { best = res; best_i = i; }       // ascending i within a lane: ties keep the smaller s
  }
  for (int o = 16; o; o >>= 1) {
    const double ob = __shfl_xor_sync(0xffffffffu, best, o);
    const int oi = __shfl_xor_sync(0xffffffffu, best_i, o);
    if (ob < best || (ob == best && oi < best_i)) { best = ob; best_i = oi; }
  }
  if (lane == 0) {
    float* o = corners + 4 * c;
    if (best_i == 0x7fffffff) {
      o[0] = o[1] = o[2] = o[3] = __int_as_float(0x7fc00000);
    } else {
      const double s = (double)best_i * s_max / (double)n_samples;
      o[0] = (float)(C[0] + s * w[0]); o[1] = (float)(C[1] + s * w[1]); o[2] = (float)(C[2] + s * w[2]);
      o[3] = (float)best;
    }
  }
}

// 8x8 linear solve (Gaussian elimination, partial pivoting) for the homography of 4 point pairs. false = singular.
__device__ bool solve_homography(const float* corners, double wc, double hc, double (&h)[9]) {
  const double src[4][2] = {{0.0, 0.0}, {wc, 0.0}, {wc, hc}, {0.0, hc}};
  double A[8][9];
  for (int k = 0; k < 4; ++k) {
    const double u = src[k][0], v = src[k][1], x = (double)corners[4 * k], y = (double)corners[4 * k + 1];
    if (!isfinite(x) || !isfinite(y)) return false;
    double r0[9] = {u, v, 1, 0, 0, 0, -u * x, -v * x, x};
    double r1[9] = {0, 0, 0, u, v, 1, -u * y, -v * y, y};
    for (int j = 0; j < 9; ++j) { A[2 * k][j] = r0[j]; A[2 * k + 1][j] = r1[j]; }
  }
  for (int col = 0; col < 8; ++col) {
    int piv = col;
    for (int r = col + 1; r < 8; ++r) if (fabs(A[r][col]) > fabs(A[piv][col])) piv = r;
    if (!(fabs(A[piv][col]) > 1e-300)) return false;
    if (piv != col) for (int j = 0; j < 9; ++j) { double t = A[col][j]; A[col][j] = A[piv][j]; A[piv][j] = t; }
    for (int r = col + 1; r < 8; ++r) {
      const double f = A[r][col] / A[col][col];
      for (int j = col; j < 9; ++j) A[r][j] -= f * A[col][j];
    }
  }
  for (int r = 7; r >= 0; --r) {
    double s = A[r][8];
    for (int j = r + 1; j < 8; ++j) s -= A[r][j] * h[j];
    h[r] = s / A[r][r];
  }
  h[8] = 1.0;
  bool ok = true;
  for (int i = 0; i < 8; ++i) ok = ok && isfinite(h[i]);
  return ok;
}

__global__ void __launch_bounds__(256) lift_kernel(const float* __restrict__ corners, int crop_w, int crop_h,
                                                   const float* __restrict__ pix, int n, DsmView D, float* __restrict__ pts) {
  __shared__ double s_h[9];
  __shared__ int s_ok;
  if (threadIdx.x == 0) {
    double h[9];
    s_ok = solve_homography(corners, (double)(crop_w - 1), (double)(crop_h - 1), h) ? 1 : 0;
    for (int i = 0; i < 9; ++i) s_h[i] = s_ok ? h[i] : 0.0;
  }
  __syncthreads();
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const double u = (double)pix[2 * k], v = (double)pix[2 * k + 1];
  const double q = s_h[6] * u + s_h[7] * v + s_h[8];
  const double x = (s_h[0] * u + s_h[1] * v + s_h[2]) / q, y = (s_h[3] * u + s_h[4] * v + s_h[5]) / q;
  double z = 0.0, zx, zy;
  const bool ok = s_ok && dsm_sample(D, x, y, z, zx, zy);
  float4 o = make_float4((float)x, (float)y, ok ? (float)z : 0.f, ok ? 1.f : 0.f);
  if (!s_ok) o = make_float4(0.f, 0.f, 0.f, 0.f);
  reinterpret_cast<float4*>(pts)[k] = o;
}

bool dsm_ok(const float* dsm, int w, int h, float gsd) { return dsm && w >= 2 && h >= 2 && gsd > 0.f; }

}  // namespace

extern "C" {

int pilot_refine_footprint(const float* pose_dev, const float intrinsics[4], int width, int height, const float* dsm_dev,
                           int dsm_width, int dsm_height, float dsm_origin_x, float dsm_origin_y, float dsm_gsd,
                           int n_samples, float s_max, float* corners_dev, void* cuda_stream) {
  if (!pose_dev || !intrinsics || !corners_dev || width < 2 || height < 2 || n_samples < 1 || !(s_max > 0.f) ||
      !(intrinsics[0] > 0.f) || !(intrinsics[1] > 0.f) || !dsm_ok(dsm_dev, dsm_width, dsm_height, dsm_gsd))
    return PILOT_ERR_ARG;
  const DsmView D = make_dsm_view(dsm_dev, dsm_width, dsm_height, dsm_origin_x, dsm_origin_y, dsm_gsd);
  footprint_kernel<<<1, 128, 0, static_cast<cudaStream_t>(cuda_stream)>>>(pose_dev, intrinsics[0], intrinsics[1], intrinsics[2],
                                                                          intrinsics[3], width, height, D, n_samples,
                                                                          (double)s_max, corners_dev);
  return cudaGetLastError() == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_lift_anchors(const float* corners_dev, int crop_width, int crop_height, const float* pix_dev, int n,
                              const float* dsm_dev, int dsm_width, int dsm_height, float dsm_origin_x, float dsm_origin_y,
                              float dsm_gsd, float* points_dev, void* cuda_stream) {
  if (n < 0 || crop_width < 2 || crop_height < 2 || !dsm_ok(dsm_dev, dsm_width, dsm_height, dsm_gsd)) return PILOT_ERR_ARG;
  if (n == 0) return PILOT_OK;
  if (!corners_dev || !pix_dev || !points_dev || ((uintptr_t)points_dev & 15)) return PILOT_ERR_ARG;
  const DsmView D = make_dsm_view(dsm_dev, dsm_width, dsm_height, dsm_origin_x, dsm_origin_y, dsm_gsd);
  lift_kernel<<<(n + 255) / 256, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(corners_dev, crop_width, crop_height,
                                                                                  pix_dev, n, D, points_dev);
  return cudaGetLastError() == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

}  // extern "C"
