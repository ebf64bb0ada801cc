// pilot_backward.cu — backward pass of the photo term (include/pilot_refine.h, pilot_refine_photo_backward): the transpose
// of the gather. Given dL/dH and dL/dg of the normal equations of one LM iteration (pilot_refine_lm_step_adjoint), it
// scatters dS/dF onto the query feature map, dS/dref onto the reference rows, dS/dconf onto the confidence map and sums
// dS/d eps per pose, S = <G_H, H> + <G_g, g> (Eq.1, Eq.2, Eq.8; "the refinement is unrolled",
// supp III-C PAPER.md:427-440). The formulas are derived in oracle/pilot_photo_backward.py's header; this
// file restates them for the GPU and shares no code with oracle/.
//
// One warp per (anchor, pose) unit at a time, lanes over the channels: pass 1 reduces nine channel dot products, the
// lane-uniform scalar algebra (projection, Jacobian, robust weight, alpha = J G_H J^T, beta = J G_g) runs in double, pass 2
// re-reads the taps (L1 hits) and adds the three C-vectors with fp32 atomics (the order of the additions, hence the last
// bits, varies from run to run: a training backward, not the parity-critical forward path).
#include "../../include/pilot_refine.h"

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

namespace {

constexpr int kBwdWarps = 8;

struct BwdArgs {
  const void* feat; const float* conf; const float4* points; const void* ref;
  const float* poses; const float* GH; const float* Gg;
  float* dfeat; float* dref; float* dconf; float* dpose;
  int W, H, C, N, n_poses, dtype, loss;
  double fx, fy, cx, cy, z_near, scale;
};

__device__ __forceinline__ float elem(const void* base, int dtype, size_t i) {
  if (dtype == PILOT_F32) return static_cast<const float*>(base)[i];
  if (dtype == PILOT_BF16) return __bfloat162float(static_cast<const __nv_bfloat16*>(base)[i]);
  return __half2float(static_cast<const __half*>(base)[i]);
}

__device__ __forceinline__ void loss_d2(int loss, double x, double scale, double& d1, double& d2) {
  d1 = 1.0; d2 = 0.0;
  if (!(scale > 0.0)) return;
  const double s2 = scale * scale;
  if (loss == PILOT_LOSS_HUBER) {
    if (x > s2) { const double sq = sqrt(x); d1 = scale / sq; d2 = -0.5 * scale / (x * sq); }
  } else if (loss == PILOT_LOSS_CAUCHY) {
    const double q = 1.0 + x / s2;
    d1 = 1.0 / q; d2 = -1.0 / (s2 * q * q);
  }
}

__device__ __forceinline__ double warp_sum(double v) {
  for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(kBwdWarps * 32) photo_backward_kernel(const __grid_constant__ BwdArgs a) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int m = blockIdx.x;
  __shared__ double s_R[9], s_C[3], s_GH[36], s_Gg[6];
  __shared__ double s_deps[kBwdWarps][6];
  if (threadIdx.x < 12) {
    const float* T = a.poses + 12 * (size_t)m;
    const int i = threadIdx.x / 4, k = threadIdx.x % 4;
    if (k < 3) s_R[3 * k + i] = (double)T[4 * i + k]; else s_C[i] = (double)T[4 * i + 3];      // R_cw = R_wc^T
  }
  if (threadIdx.x >= 32 && threadIdx.x < 68) {
    const int i = threadIdx.x - 32, r = i / 6, c = i % 6;
    s_GH[i] = 0.5 * ((double)a.GH[36 * (size_t)m + i] + (double)a.GH[36 * (size_t)m + 6 * c + r]);
  }
  if (threadIdx.x >= 96 && threadIdx.x < 102) s_Gg[threadIdx.x - 96] = (double)a.Gg[6 * (size_t)m + threadIdx.x - 96];
  __syncthreads();
  double deps[6] = {0, 0, 0, 0, 0, 0};
  const size_t C = (size_t)a.C;
  for (int j = blockIdx.y * kBwdWarps + warp; j < a.N; j += gridDim.y * kBwdWarps) {
    const float4 P = a.points[j];
    const double dx = (double)P.x - s_C[0], dy = (double)P.y - s_C[1], dz = (double)P.z - s_C[2];
    const double X = s_R[0] * dx + s_R[1] * dy + s_R[2] * dz;
    const double Y = s_R[3] * dx + s_R[4] * dy + s_R[5] * dz;
    const double Z = s_R[6] * dx + s_R[7] * dy + s_R[8] * dz;
    if (!(Z > a.z_near)) continue;
    const double u = a.fx * X / Z + a.cx, v = a.fy * Y / Z + a.cy;
    const double x0d = floor(u), y0d = floor(v);
    if (!(x0d >= 0.0) || !(y0d >= 0.0) || !(x0d + 1.0 <= (double)(a.W - 1)) || !(y0d + 1.0 <= (double)(a.H - 1))) continue;
    const int x0 = (int)x0d, y0 = (int)y0d;
    const float fa = (float)(u - x0d), fb = (float)(v - y0d);
    const size_t o00 = ((size_t)y0 * a.W + x0) * C, o10 = o00 + C, o01 = o00 + (size_t)a.W * C, o11 = o01 + C, oref = (size_t)j * C;
    // pass 1: nine dot products over the channels
    float d[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};            // gx.gx gx.gy gy.gy gx.r gy.r r.r gx.h gy.h r.h
    for (int c = lane; c < a.C; c += 32) {
      const float f00 = elem(a.feat, a.dtype, o00 + c), f10 = elem(a.feat, a.dtype, o10 + c);
      const float f01 = elem(a.feat, a.dtype, o01 + c), f11 = elem(a.feat, a.dtype, o11 + c);
      const float f = (1.f - fb) * ((1.f - fa) * f00 + fa * f10) + fb * ((1.f - fa) * f01 + fa * f11);
      const float gx = (1.f - fb) * (f10 - f00) + fb * (f11 - f01), gy = (1.f - fa) * (f01 - f00) + fa * (f11 - f10);
      const float r = f - elem(a.ref, a.dtype, oref + c), h = f11 - f01 - f10 + f00;
      d[0] += gx * gx; d[1] += gx * gy; d[2] += gy * gy; d[3] += gx * r; d[4] += gy * r; d[5] += r * r;
      d[6] += gx * h; d[7] += gy * h; d[8] += r * h;
    }
    double D[9];
#pragma unroll
    for (int i = 0; i < 9; ++i) D[i] = warp_sum((double)d[i]);
    // lane-uniform scalars
    double w = (double)P.w, wq_u = 0.0, wq_v = 0.0;
    const double A1 = (double)fa, B1 = (double)fb;
    if (a.conf) {
      const float* q = a.conf + (size_t)y0 * a.W + x0;
      const double q00 = q[0], q10 = q[1], q01 = q[a.W], q11 = q[a.W + 1];
      w *= (1 - B1) * ((1 - A1) * q00 + A1 * q10) + B1 * ((1 - A1) * q01 + A1 * q11);
      wq_u = (1 - B1) * (q10 - q00) + B1 * (q11 - q01);
      wq_v = (1 - A1) * (q01 - q00) + A1 * (q11 - q10);
    }
    const double xr = w * D[5];
    double d1, d2;
    loss_d2(a.loss, xr, a.scale, d1, d2);
    const double om = w * d1;
    const double iz = 1.0 / Z;
    const double J[2][6] = {{a.fx * iz, 0, -a.fx * X * iz * iz, -a.fx * X * Y * iz * iz, a.fx * (1 + X * X * iz * iz), -a.fx * Y * iz},
                            {0, a.fy * iz, -a.fy * Y * iz * iz, -a.fy * (1 + Y * Y * iz * iz), a.fy * X * Y * iz * iz, a.fy * X * iz}};
    double JG[2][6], al[2][2], be[2];
    for (int p = 0; p < 2; ++p) {
      be[p] = 0.0;
      for (int k = 0; k < 6; ++k) {
        double s = 0.0;
        for (int i = 0; i < 6; ++i) s += J[p][i] * s_GH[6 * i + k];
        JG[p][k] = s;
        be[p] += J[p][k] * s_Gg[k];
      }
    }
    for (int p = 0; p < 2; ++p)
      for (int q = 0; q < 2; ++q) { double s = 0.0; for (int k = 0; k < 6; ++k) s += JG[p][k] * J[q][k]; al[p][q] = s; }
    const double Q = al[0][0] * D[0] + 2 * al[0][1] * D[1] + al[1][1] * D[2] + be[0] * D[3] + be[1] * D[4];
    const double kr = Q * w * w * d2 * 2.0;                              // dS/dr = om (be0 gx + be1 gy) + kr r
    // pass 2: the three C-vectors, scattered
    {
      const float wf[4] = {(1.f - fa) * (1.f - fb), fa * (1.f - fb), (1.f - fa) * fb, fa * fb};
      const float wgx[4] = {-(1.f - fb), (1.f - fb), -fb, fb}, wgy[4] = {-(1.f - fa), -fa, (1.f - fa), fa};
      const float c_rx = (float)(om * be[0]), c_ry = (float)(om * be[1]), c_rr = (float)kr;
      const float c_xx = (float)(om * 2 * al[0][0]), c_xy = (float)(om * 2 * al[0][1]), c_yy = (float)(om * 2 * al[1][1]);
      for (int c = lane; c < a.C; c += 32) {
        const float f00 = elem(a.feat, a.dtype, o00 + c), f10 = elem(a.feat, a.dtype, o10 + c);
        const float f01 = elem(a.feat, a.dtype, o01 + c), f11 = elem(a.feat, a.dtype, o11 + c);
        const float f = (1.f - fb) * ((1.f - fa) * f00 + fa * f10) + fb * ((1.f - fa) * f01 + fa * f11);
        const float gx = (1.f - fb) * (f10 - f00) + fb * (f11 - f01), gy = (1.f - fa) * (f01 - f00) + fa * (f11 - f10);
        const float r = f - elem(a.ref, a.dtype, oref + c);
        const float Sr = c_rx * gx + c_ry * gy + c_rr * r;
        const float Sgx = c_xx * gx + c_xy * gy + c_rx * r, Sgy = c_xy * gx + c_yy * gy + c_ry * r;
        if (a.dfeat) {
          atomicAdd(a.dfeat + o00 + c, wf[0] * Sr + wgx[0] * Sgx + wgy[0] * Sgy);
          atomicAdd(a.dfeat + o10 + c, wf[1] * Sr + wgx[1] * Sgx + wgy[1] * Sgy);
          atomicAdd(a.dfeat + o01 + c, wf[2] * Sr + wgx[2] * Sgx + wgy[2] * Sgy);
          atomicAdd(a.dfeat + o11 + c, wf[3] * Sr + wgx[3] * Sgx + wgy[3] * Sgy);
        }
        if (a.dref) atomicAdd(a.dref + oref + c, -Sr);
      }
      if (a.conf && a.dconf && lane < 4) {
        const double Sw = Q * (d1 + xr * d2) * (double)P.w;
        atomicAdd(a.dconf + (size_t)(y0 + (lane >> 1)) * a.W + x0 + (lane & 1), (float)(Sw * (double)wf[lane]));
      }
    }
    if (lane == 0 && a.dpose) {
      // through (u, v): Sr.gx = om (be0 A11 + be1 A12) + kr b1, ...; Sgy.h = om (2 al01 gx.h + 2 al11 gy.h + be1 r.h)
      double Su = om * (be[0] * D[0] + be[1] * D[1]) + kr * D[3] + om * (2 * al[0][1] * D[6] + 2 * al[1][1] * D[7] + be[1] * D[8]);
      double Sv = om * (be[0] * D[1] + be[1] * D[2]) + kr * D[4] + om * (2 * al[0][0] * D[6] + 2 * al[0][1] * D[7] + be[0] * D[8]);
      if (a.conf) { const double Sw = Q * (d1 + xr * d2) * (double)P.w; Su += Sw * wq_u; Sv += Sw * wq_v; }
      for (int i = 0; i < 6; ++i) deps[i] += J[0][i] * Su + J[1][i] * Sv;
      // through J(X, Y, Z): M = om (2 A J G_H + b G_g^T)
      const double Am[2][2] = {{D[0], D[1]}, {D[1], D[2]}}, bm[2] = {D[3], D[4]};
      double M[2][6];
      for (int p = 0; p < 2; ++p)
        for (int k = 0; k < 6; ++k) M[p][k] = om * (2 * (Am[p][0] * JG[0][k] + Am[p][1] * JG[1][k]) + bm[p] * s_Gg[k]);
      const double iz2 = iz * iz, iz3 = iz2 * iz, fx = a.fx, fy = a.fy;
      const double SX = M[0][2] * (-fx * iz2) + M[0][3] * (-fx * Y * iz2) + M[0][4] * (2 * fx * X * iz2) + M[1][4] * (fy * Y * iz2) + M[1][5] * (fy * iz);
      const double SY = M[0][3] * (-fx * X * iz2) + M[0][5] * (-fx * iz) + M[1][2] * (-fy * iz2) + M[1][3] * (-2 * fy * Y * iz2) + M[1][4] * (fy * X * iz2);
      const double SZ = M[0][0] * (-fx * iz2) + M[0][2] * (2 * fx * X * iz3) + M[0][3] * (2 * fx * X * Y * iz3) + M[0][4] * (-2 * fx * X * X * iz3) + M[0][5] * (fx * Y * iz2) +
                        M[1][1] * (-fy * iz2) + M[1][2] * (2 * fy * Y * iz3) + M[1][3] * (2 * fy * Y * Y * iz3) + M[1][4] * (-2 * fy * X * Y * iz3) + M[1][5] * (-fy * X * iz2);
      // dp/d eps = [I | -p^]:  (-p^)^T Sp = p x Sp
      deps[0] += SX; deps[1] += SY; deps[2] += SZ;
      deps[3] += Y * SZ - Z * SY; deps[4] += Z * SX - X * SZ; deps[5] += X * SY - Y * SX;
    }
  }
  if (a.dpose) {
    if (lane == 0) for (int i = 0; i < 6; ++i) s_deps[warp][i] = deps[i];
    __syncthreads();
    if (threadIdx.x < 6) {
      double t = 0.0;
      for (int w2 = 0; w2 < kBwdWarps; ++w2) t += s_deps[w2][threadIdx.x];
      atomicAdd(a.dpose + 6 * (size_t)m + threadIdx.x, (float)t);
    }
  }
}

}  // namespace

extern "C" int pilot_refine_photo_backward(const void* query_feat_dev, const float* query_conf_dev, int width, int height, int channels,
                                           pilot_dtype feat_dtype, const float intrinsics[4], const float* points_dev,
                                           const void* ref_feat_dev, int n_points, const float* poses_dev,
                                           const float* grad_hessian_dev, const float* grad_gradient_dev, int n_poses,
                                           pilot_loss loss, float loss_scale, float z_near, float* grad_feat_dev, float* grad_ref_dev,
                                           float* grad_conf_dev, float* grad_pose_dev, void* cuda_stream) {
  if (width < 2 || height < 2 || channels < 1 || n_points < 0 || n_poses < 0 || !intrinsics) return PILOT_ERR_ARG;
  if (feat_dtype != PILOT_F32 && feat_dtype != PILOT_BF16 && feat_dtype != PILOT_F16) return PILOT_ERR_ARG;
  if (loss < PILOT_LOSS_L2 || loss > PILOT_LOSS_CAUCHY) return PILOT_ERR_ARG;
  if ((unsigned long long)width * height * channels >= 0xffffffffull) return PILOT_ERR_UNSUPPORTED;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (grad_pose_dev && n_poses > 0 && cudaMemsetAsync(grad_pose_dev, 0, sizeof(float) * 6 * (size_t)n_poses, st) != cudaSuccess) return PILOT_ERR_CUDA;
  if (n_poses == 0 || n_points == 0) return PILOT_OK;
  if (!query_feat_dev || !points_dev || !ref_feat_dev || !poses_dev || !grad_hessian_dev || !grad_gradient_dev) return PILOT_ERR_ARG;
  if ((uintptr_t)points_dev & 15) return PILOT_ERR_ARG;
  BwdArgs a;
  a.feat = query_feat_dev; a.conf = query_conf_dev; a.points = reinterpret_cast<const float4*>(points_dev); a.ref = ref_feat_dev;
  a.poses = poses_dev; a.GH = grad_hessian_dev; a.Gg = grad_gradient_dev;
  a.dfeat = grad_feat_dev; a.dref = grad_ref_dev; a.dconf = grad_conf_dev; a.dpose = grad_pose_dev;
  a.W = width; a.H = height; a.C = channels; a.N = n_points; a.n_poses = n_poses; a.dtype = (int)feat_dtype; a.loss = (int)loss;
  a.fx = intrinsics[0]; a.fy = intrinsics[1]; a.cx = intrinsics[2]; a.cy = intrinsics[3];
  a.z_near = (double)z_near; a.scale = (double)loss_scale;
  int gy = (n_points + kBwdWarps * 8 - 1) / (kBwdWarps * 8);
  if (gy < 1) gy = 1;
  if (gy > 512) gy = 512;
  photo_backward_kernel<<<dim3((unsigned)n_poses, (unsigned)gy), kBwdWarps * 32, 0, st>>>(a);
  return cudaGetLastError() == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}
