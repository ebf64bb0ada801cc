// pilot_pass.cuh — the one-launch-per-pass photo kernel, shared by the two translation units
// that instantiate it with different CTA shapes: pilot_refine.cu (FFMA2 contraction: 4 warps, 128 registers) and
// pilot_pass_mma.cu (tensor-core contraction: 4 warps, 80 registers, 24 warps per SM). Shares no code with oracle/.
#pragma once
#include "pilot_device.cuh"

namespace {

template <class T, int G, bool CEN, bool MMA>
__global__ void __launch_bounds__(kThreads, PILOT_MIN_BLOCKS) photo_pass_kernel(const __grid_constant__ PassArgs A) {
  pdl_prologue();
  const int m = blockIdx.x;
  int chunk_idx = blockIdx.y;
  const HypState* st = A.state + m;
  if (st->level != A.level) return;             // finished this level early (failed factorisations)
  if (A.prior_cta) {
    // Row 0 of the grid: the priors' terms (heightfield ray-march of the range prior, algebra of both: supp Eq.5-6) depend only
    // on the candidate pose, so one warp per hypothesis evaluates them WHILE the other rows gather, and the deferred
    // finalisation adds 28 numbers instead of running the march's chain of dependent DSM samples on its own critical path.
    if (chunk_idx == 0) {
      if (threadIdx.x < 32) prior_terms_store(A, st->Rc, st->Cc, (int)threadIdx.x, static_cast<PriorTerms*>(A.priors) + m);
      return;
    }
    chunk_idx -= 1;
  }

  PILOT_DECLARE_ACC
  acc_zero<MMA>(acc, sacc);
  {
    const int begin = chunk_idx * A.chunk;
    const double* Rc = st->Rc;
    const double* Cc = st->Cc;
    if constexpr (MMA) {                          // the tensor-core gather re-reads the pose from shared memory
      __shared__ __align__(16) double s_pose[12 + 8];       // Rc[9] | Cc[3] | 16 floats: R, centre hi, centre lo (fp32 projection)
      if (threadIdx.x < 12) s_pose[threadIdx.x] = threadIdx.x < 9 ? st->Rc[threadIdx.x] : st->Cc[threadIdx.x - 9];
      else if (threadIdx.x < 32 + 16 && threadIdx.x >= 32) pose_to_float(st->Rc, st->Cc, (int)threadIdx.x - 32, reinterpret_cast<float*>(s_pose + 12));
      __syncthreads();
      Rc = s_pose; Cc = s_pose + 9;
    }
    photo_accumulate<T, G, CEN, MMA>(A, Rc, Cc, begin, min(begin + A.chunk, A.lv.N), (int)(threadIdx.x >> 5), kWarps, acc, sacc, red);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const float wtot = acc_warp_total<MMA>(acc, sacc, lane);
  __shared__ float s_part[kWarps][kNacc];
  __shared__ double s_sum[kNacc];                // the hypothesis' sums, converted by the lane that holds each
  __shared__ int s_last;
  __shared__ HypState s_state;                   // the last CTA's warp 0 finalises on a copy in shared memory
  s_part[warp][lane] = wtot;
  __syncthreads();
  if (warp == 0) {
    float t = 0.f;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) t += s_part[w][lane];                    // fixed order
    A.partials[((size_t)m * A.n_chunks + chunk_idx) * kNacc + lane] = t;
    if (A.defer) return;                         // finalize_kernel (next launch) ends the iteration
    __threadfence();
    __syncwarp();
    if (lane == 0) s_last = (atomicAdd(A.counters + m, 1u) == (unsigned)(A.n_chunks - 1));
  }
  if (A.defer) return;
  __syncthreads();
  if (!s_last || warp != 0) return;

  // last CTA of this hypothesis: fixed-order sum over chunks (deterministic), then the LM step
  __threadfence();
  float t = 0.f;
  const float* p = A.partials + (size_t)m * A.n_chunks * kNacc + lane;
  for (int c = 0; c < A.n_chunks; ++c) t += __ldcg(p + (size_t)c * kNacc);
  s_sum[lane] = (double)t;
  if (lane == 0) A.counters[m] = 0u;
  __syncwarp();
  finalize_in_workspace(A, m, s_sum, lane, &s_state);
}

}  // namespace
