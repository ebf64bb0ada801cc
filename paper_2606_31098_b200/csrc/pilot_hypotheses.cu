// pilot_hypotheses.cu — the hypothesis set around the LM refinement (include/pilot_refine.h):
// sampling around a pose prior (supp II-C PAPER.md:381-386), top-k pruning by objective
// after the coarse level and the final arg-min. Everything stays on the
// device and on the caller's stream, so a frame never synchronises with the host between the seeding,
// the refinement of each level and the selection.
//
// Shares no code with oracle/.
#include "../../include/pilot_refine.h"

#include <cuda_runtime.h>
#include <math.h>

#include "pilot_pdl.cuh"
#include <stdint.h>

namespace {

// Order-preserving map float -> uint32 (NaN sorts last, like +inf but after it is canonicalised to +inf).
__device__ __forceinline__ unsigned orderable(float c) {
  if (isnan(c)) c = INFINITY;
  c += 0.0f;                                        // -0 -> +0: equal costs must compare equal
  unsigned b = __float_as_uint(c);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ unsigned long long make_key(float c, int idx) {
  return ((unsigned long long)orderable(c) << 32) | (unsigned)idx;   // ties -> lowest index
}

// exp([w]x) by Rodrigues in double (series near 0), row-major.
__device__ void rodrigues(const float* w, double (&E)[9]) {
  double x = w[0], y = w[1], z = w[2];
  double th2 = x * x + y * y + z * z, th = sqrt(th2), a, b;
  if (th < 1e-6) { a = 1.0 - th2 / 6.0; b = 0.5 - th2 / 24.0; }
  else { a = sin(th) / th; b = (1.0 - cos(th)) / th2; }
  double K[9] = {0, -z, y, z, 0, -x, -y, x, 0};
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      double k2 = K[3 * i] * K[j] + K[3 * i + 1] * K[3 + j] + K[3 * i + 2] * K[6 + j];
      E[3 * i + j] = (i == j ? 1.0 : 0.0) + a * K[3 * i + j] + b * k2;
    }
}

__global__ void seed_kernel(const float* __restrict__ base, const float* __restrict__ off, int n, int frame,
                            float* __restrict__ out) {
  pilot_internal::pdl_prologue();
  int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n) return;
  double R[9], C[3], E[9];
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) R[3 * i + j] = (double)base[4 * i + j];
    C[i] = (double)base[4 * i + 3];
  }
  rodrigues(off + 6 * (size_t)m, E);
  float* o = out + 12 * (size_t)m;
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) {
      double v = 0.0;
      for (int k = 0; k < 3; ++k)
        v += (frame == PILOT_SEED_CAMERA) ? R[3 * i + k] * E[3 * k + j] : E[3 * i + k] * R[3 * k + j];
      o[4 * i + j] = (float)v;
    }
    o[4 * i + 3] = (float)(C[i] + (double)off[6 * (size_t)m + 3 + i]);
  }
}

constexpr int kSelThreads = 1024;

__global__ void __launch_bounds__(kSelThreads) select_best_kernel(const float* __restrict__ cost,
                                                                  const float* __restrict__ poses, int n,
                                                                  int* best_idx, float* best_pose, float* best_cost) {
  pilot_internal::pdl_prologue();
  __shared__ unsigned long long s_key[kSelThreads / 32];
  unsigned long long k = ~0ull;
  for (int i = threadIdx.x; i < n; i += kSelThreads) {
    unsigned long long c = make_key(cost[i], i);
    k = c < k ? c : k;
  }
  for (int o = 16; o; o >>= 1) {
    unsigned long long t = __shfl_xor_sync(0xffffffffu, k, o);
    k = t < k ? t : k;
  }
  if ((threadIdx.x & 31) == 0) s_key[threadIdx.x >> 5] = k;
  __syncthreads();
  if (threadIdx.x < 32) {
    k = s_key[threadIdx.x];
    for (int o = 16; o; o >>= 1) {
      unsigned long long t = __shfl_xor_sync(0xffffffffu, k, o);
      k = t < k ? t : k;
    }
    const int b = (int)(unsigned)(k & 0xffffffffu);
    if (threadIdx.x == 0) {
      if (best_idx) best_idx[0] = b;
      if (best_cost) best_cost[0] = cost[b];
    }
    if (best_pose && poses && threadIdx.x < 12) best_pose[threadIdx.x] = poses[12 * (size_t)b + threadIdx.x];
  }
}

// One CTA: bitonic sort of n <= PILOT_TOPK_MAX 64-bit (cost, index) keys in shared memory.
__global__ void __launch_bounds__(kSelThreads) topk_kernel(const float* __restrict__ cost,
                                                           const float* __restrict__ poses, int n, int k, int n_pow2,
                                                           int* idx_out, float* poses_out, float* cost_out) {
  pilot_internal::pdl_prologue();
  extern __shared__ unsigned long long s[];
  for (int i = threadIdx.x; i < n_pow2; i += kSelThreads) s[i] = i < n ? make_key(cost[i], i) : ~0ull;
  __syncthreads();
  // A compare-exchange pass with stride <= 32 touches, per warp and per turn of the t loop, only that warp's own block of 64
  // keys (lo = 2t - (t & (stride-1)) over 32 consecutive t), so those passes - 51 of the 66 of a 2048-key sort - need only a
  // warp-level barrier; the CTA-wide one separates them from the passes with longer strides.
  for (int size = 2; size <= n_pow2; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int t = threadIdx.x; t < (n_pow2 >> 1); t += kSelThreads) {
        int lo = 2 * t - (t & (stride - 1));          // index with bit `stride` clear
        int hi = lo + stride;
        bool up = (lo & size) == 0;
        unsigned long long a = s[lo], b = s[hi];
        if ((a > b) == up) { s[lo] = b; s[hi] = a; }
      }
      if (stride > 32 || stride == 1) __syncthreads(); else __syncwarp();
    }
  }
  for (int i = threadIdx.x; i < k; i += kSelThreads) {
    int src = (int)(unsigned)(s[i] & 0xffffffffu);
    if (idx_out) idx_out[i] = src;
    if (cost_out) cost_out[i] = cost[src];
  }
  if (poses_out && poses)
    for (int i = threadIdx.x; i < 12 * k; i += kSelThreads) {
      int src = (int)(unsigned)(s[i / 12] & 0xffffffffu);
      poses_out[i] = poses[12 * (size_t)src + (i % 12)];
    }
}

}  // namespace

extern "C" {

int pilot_refine_grid_offsets(float xy_range, float xy_step, const float* yaw_deg, int n_yaw, const float up[3],
                              float* offsets_host, int capacity) {
  if (!(xy_range >= 0.f) || !(xy_step > 0.f) || n_yaw < 1 || !yaw_deg || !up) return PILOT_ERR_ARG;
  const int r = (int)floor((double)xy_range / (double)xy_step + 1e-6);
  const int side = 2 * r + 1;
  const long total = (long)side * side * n_yaw;
  if (total > 0x7fffffffL) return PILOT_ERR_ARG;
  if (!offsets_host || capacity < (int)total) return (int)total;
  const double deg = 3.14159265358979323846 / 180.0;
  size_t e = 0;
  for (int i = -r; i <= r; ++i)
    for (int j = -r; j <= r; ++j)
      for (int k = 0; k < n_yaw; ++k, ++e) {
        float* o = offsets_host + 6 * e;
        for (int a = 0; a < 3; ++a) o[a] = (float)((double)yaw_deg[k] * deg * (double)up[a]);
        o[3] = (float)((double)i * (double)xy_step);
        o[4] = (float)((double)j * (double)xy_step);
        o[5] = 0.f;
      }
  return (int)total;
}

int pilot_refine_seed_hypotheses(const float* base_pose_dev, const float* offsets_dev, int n, int frame,
                                 float* out_poses_dev, void* cuda_stream) {
  if (n < 0 || (frame != PILOT_SEED_CAMERA && frame != PILOT_SEED_WORLD)) return PILOT_ERR_ARG;
  if (n == 0) return PILOT_OK;
  if (!base_pose_dev || !offsets_dev || !out_poses_dev) return PILOT_ERR_ARG;
  return pilot_internal::launch_pdl(seed_kernel, dim3((unsigned)((n + 127) / 128)), 128, 0, static_cast<cudaStream_t>(cuda_stream),
                                    base_pose_dev, offsets_dev, n, frame, out_poses_dev) == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_select_best(const float* cost_dev, const float* poses_dev, int n, int* best_idx_dev,
                             float* best_pose_dev, float* best_cost_dev, void* cuda_stream) {
  if (n < 1 || !cost_dev || (best_pose_dev && !poses_dev)) return PILOT_ERR_ARG;
  return pilot_internal::launch_pdl(select_best_kernel, dim3(1), kSelThreads, 0, static_cast<cudaStream_t>(cuda_stream), cost_dev, poses_dev,
                                    n, best_idx_dev, best_pose_dev, best_cost_dev) == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

int pilot_refine_prune_topk(const float* cost_dev, const float* poses_dev, int n, int k, int* idx_out_dev,
                            float* poses_out_dev, float* cost_out_dev, void* cuda_stream) {
  if (!cost_dev || n < 1 || k < 1 || k > n || (poses_out_dev && !poses_dev)) return PILOT_ERR_ARG;
  if (n > PILOT_TOPK_MAX) return PILOT_ERR_UNSUPPORTED;
  int n_pow2 = 2;
  while (n_pow2 < n) n_pow2 <<= 1;
  const size_t smem = (size_t)n_pow2 * sizeof(unsigned long long);
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return PILOT_ERR_CUDA;
  return pilot_internal::launch_pdl(topk_kernel, dim3(1), kSelThreads, smem, static_cast<cudaStream_t>(cuda_stream), cost_dev, poses_dev, n, k,
                                    n_pow2, idx_out_dev, poses_out_dev, cost_out_dev) == cudaSuccess ? PILOT_OK : PILOT_ERR_CUDA;
}

}  // extern "C"
